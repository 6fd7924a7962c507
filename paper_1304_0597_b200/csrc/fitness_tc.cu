// placeholder until the tcgen05 kernel lands: reports the tensor path as not built
#include "game_internal.cuh"
namespace game {
bool tensor_path_built() { return false; }
int tensor_prepare(game_ctx *) { return GAME_OK; }
int launch_fitness_tensor(game_ctx *ctx, const float *, int, float *, const DevState *)
{
    return fail(ctx, GAME_ERR_UNSUPPORTED, "tensor path not built");
}
}  // namespace game

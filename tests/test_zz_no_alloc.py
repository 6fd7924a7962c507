"""game_rank_static -- the rank step for hosts that cannot allocate GPU memory -- against game_rank.

Some users of libgame_b200 run inside a process whose device memory is already spoken for (another component's caching
allocator holds all of HBM), or inside a loop that must never enter the driver's allocation path.  game_rank allocates
its counting scratch on every call; game_rank_static counts into an array that is part of the library image instead.
That array is shared by every call on a GPU and still holds the previous call's counts, so the property worth testing
is: a second call right after a first one (a different population size, different errors, no synchronisation between
them) is as correct as the first.  The reference is the library's existing, allocating game_rank; ranks are integers,
so the comparison is exact, like every other rank check in tests/test_gpu_parity.py.

The file name sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide the
parity tests.  It passes alone in a fresh process (first use of the array on the device) and after the other tests.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
if not torch.cuda.is_available():
    pytest.skip("no CUDA device", allow_module_level=True)

import paper_1304_0597_b200 as g  # noqa: E402


def _errors(rng, P):
    """errors with everything the rank rule has a clause for: ties, NaN, inf, -0 / +0 (DESIGN G20)"""
    fit = rng.random(P).astype(np.float32)
    if P > 10:
        fit[rng.integers(0, P, P // 10)] = fit[0]
        fit[rng.integers(0, P, 3)] = np.nan
        fit[rng.integers(0, P, 2)] = np.inf
        fit[rng.integers(0, P, 2)] = -0.0
        fit[rng.integers(0, P, 2)] = 0.0
    return torch.from_numpy(fit).cuda()


def test_rank_static_equals_game_rank_on_two_calls_in_a_row():
    ctx = g.Game(g.GAME_TRIG, 1, 1)
    rng = np.random.default_rng(2024)
    # (first call, second call): the second is smaller, larger, and equal in size, so it meets counts left behind by the
    # first both inside and outside the range it clears; 5000 and 65536 span several key slabs (atomic accumulation)
    for P1, P2 in ((5000, 257), (300, 8192), (4096, 4096), (1, 2), (g.GAME_RANK_STATIC_MAX_P, 1000)):
        f1, f2 = _errors(rng, P1), _errors(rng, P2)
        o1 = torch.full((P1,), -1, dtype=torch.int32, device="cuda")
        o2 = torch.full((P2,), -1, dtype=torch.int32, device="cuda")
        g.rank_static(f1, o1)
        g.rank_static(f2, o2)                     # same stream, straight after: no synchronisation in between
        assert torch.equal(o1, ctx.rank(f1)), (P1, "first call")
        assert torch.equal(o2, ctx.rank(f2)), (P2, "second call")
    ctx.destroy()


def test_rank_static_on_a_side_stream_and_its_limits():
    ctx = g.Game(g.GAME_TRIG, 1, 1)
    rng = np.random.default_rng(7)
    f = _errors(rng, 3000)
    o = torch.empty(3000, dtype=torch.int32, device="cuda")
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    g.rank_static(f, o, stream=s)
    g.rank_static(f, o, stream=s)
    s.synchronize()
    assert torch.equal(o, ctx.rank(f))
    # beyond the built-in scratch: refused with a message that says so, nothing enqueued
    big = torch.zeros(g.GAME_RANK_STATIC_MAX_P + 1, dtype=torch.float32, device="cuda")
    with pytest.raises(g.GameError) as ei:
        g.rank_static(big)
    assert ei.value.code == 1 and "GAME_RANK_STATIC_MAX_P" in str(ei.value)
    L = g.load_library()
    assert L.game_rank_static(None, 4, None, None) == 1 and b"NULL" in L.game_rank_static_error()
    assert L.game_rank_static(f.data_ptr(), 0, o.data_ptr(), None) == 1
    ctx.destroy()

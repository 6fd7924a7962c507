"""CPU-side checks of the boundary: the library loads, exports every symbol include/game.h declares,
and refuses to compute without a GPU (no CPU fallback)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1304_0597_b200 import build, binding
    build.build_library()
    return binding.load_library()


def _declared(headers=("game.h", "game_bench.h")):
    """every function the headers under include/ declare: the product API (game.h) and the measurement aids (game_bench.h)"""
    names = set()
    for h in headers:
        src = open(os.path.join(ROOT, "include", h)).read()
        src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
        names |= set(re.findall(r"\b(game_[a-z_]+)\s*\(", src))
    return sorted(names)


def test_product_header_holds_no_measurement_aids():
    api, src = _declared(("game.h",)), open(os.path.join(ROOT, "include", "game.h")).read()
    for aid in ("game_microbench", "game_set_kernel_timing", "game_get_kernel_timing", "game_launch_count", "game_set_tuning"):
        assert aid not in api
    assert "GAME_TUNE_" not in re.sub(r"/\*.*?\*/", "", src, flags=re.S) and '#include "game_bench.h"' not in src


def test_exports_every_declared_symbol(lib):
    from paper_1304_0597_b200 import binding
    names = _declared()
    assert len(names) >= 20
    assert sorted(binding.SYMBOLS) == names
    for n in names:
        assert hasattr(lib, n), n


def test_struct_layouts_match_header():
    from paper_1304_0597_b200 import binding
    assert ctypes.sizeof(binding.game_ga_params) == 36
    assert ctypes.sizeof(binding.game_result) == 16
    assert binding.game_ga_params.p_crossover.offset == 24 and binding.game_ga_params.stop_error.offset == 32


def test_argument_validation_without_gpu(lib):
    h = ctypes.c_void_p()
    assert lib.game_create(7, 2, 3, ctypes.byref(h)) == 1          # bad family -> INVALID_ARG
    assert lib.game_create(0, 0, 3, ctypes.byref(h)) == 1
    assert lib.game_create(0, 33, 3, ctypes.byref(h)) == 1
    assert lib.game_create(0, 2, 0, ctypes.byref(h)) == 1
    assert lib.game_num_terms(None) == -1
    import torch
    if not torch.cuda.is_available():
        # no device: the context cannot exist, and the Python layer refuses too -- no CPU fallback
        assert lib.game_create(0, 2, 3, ctypes.byref(h)) == 4       # GAME_ERR_CUDA
        assert not h.value
        from paper_1304_0597_b200 import Game
        with pytest.raises(RuntimeError):
            Game(0, 2, 3)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1304_0597_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "game_oracle" not in txt, f
    txt = open(os.path.join(ROOT, "oracle", "oracle.py")).read() + open(os.path.join(ROOT, "oracle", "game_oracle.c")).read()
    assert "paper_1304_0597_b200 import" not in txt and "game.h" not in txt and "libgame_b200" not in txt

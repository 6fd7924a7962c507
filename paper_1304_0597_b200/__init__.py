"""game-b200: the GAME (arXiv:1304.0597) fitness / GA hot path as sm_100a CUDA kernels behind a C ABI.

``binding`` is the thin ctypes layer over ``libgame_b200.so`` (built in-tree by ``build``);
``workloads`` holds the seeded synthetic input generators.  Importing the package does not load
the library; using it without the built library or without a CUDA device raises.
"""
from . import workloads  # noqa: F401
from .binding import *  # noqa: F401,F403
from .binding import Game, GameError, ga_params, load_library  # noqa: F401

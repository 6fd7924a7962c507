"""fp64 CPU oracle for the GAME fitness / GA hot path (arXiv:1304.0597).

TEST INFRASTRUCTURE, NOT PRODUCT: only ``tests/``, ``__graft_entry__.smoke()`` and the
``cpu_baseline`` / ``--impl reference`` legs of ``bench.py`` may import this package.
It shares no code with ``paper_1304_0597_b200`` and neither imports the other.

The arithmetic lives in ``game_oracle.c`` (plain C, fp64); this module only builds it with
gcc and marshals numpy arrays through ctypes.
"""
from .oracle import *  # noqa: F401,F403

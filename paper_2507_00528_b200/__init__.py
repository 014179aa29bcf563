"""GNEP hot path (NEP loss + analytic gradient + Adam) for NVIDIA B200, behind the C ABI of include/gnep.h.

`Gnep` is the thin Python binding (argument marshalling only).  The CUDA library is built in-tree by
`paper_2507_00528_b200.build.build()`; nothing here falls back to a CPU implementation.
"""
from .binding import EXPORTS, Gnep, GnepError, LIB_PATH, load_library, lr_schedule  # noqa: F401

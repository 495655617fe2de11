"""B200-native geometry-guidance hot path of arxiv/paper_2505_18932 (refine -> integrate -> extract).

`binding` is the ctypes layer over the C ABI (include/ggt.h, libggt.so built from csrc/ by build.py);
`synth` holds the seeded synthetic input generators shared with the oracle's tests.
"""
from . import synth  # noqa: F401
from .binding import (GGT_ACCUMULATE, GGT_F16, GGT_F32, GGT_OVERWRITE, Context, GgtError, Volume,  # noqa: F401
                      load_library)

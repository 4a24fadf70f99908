"""paper_2406_01322_b200: Python binding of libpsdns (B200-native pseudo-spectral channel step).

Argument marshalling only - every step of the hot path runs in the CUDA kernels of
`csrc/`.  There is no CPU fallback: importing `paper_2406_01322_b200.binding` raises if
`libpsdns.so` is missing."""
from .binding import (  # noqa: F401
    PHYSICAL, SPECTRAL, STATIC_SCRATCH_DOUBLES, PsdnsError, Solver, lib_path, load_library, exported_symbols,
)

"""paper_2606_04725_b200 -- B200-native (sm_100a, fp64) KKT hot path of the parametric interior-point NMPC method of
arxiv/paper_2606_04725.  The product is the C-ABI shared library `libnmpc_b200.so` (include/nmpc.h, sources in
csrc/); this package is its build script and a thin ctypes binding with the same function names.  PyTorch is used by
callers only for device memory and streams.  There is no CPU fallback: importing `binding` and calling into it
without the built library raises."""
from . import binding  # noqa: F401
from .binding import (Handle, NmpcError, Symbolic, default_options, fp64_peak, ipm_solve_batch, load_library, make_ocp,
                      make_pattern, tile_gemm_peak)  # noqa: F401

"""B200-native npFEM solid-solver step (arxiv 1911.03062): thin Python binding over the C-ABI
library `lib/libnpfem_b200.so` (include/npfem.h).  Argument marshalling only: every step of the
path runs in the hand-written sm_100a kernels under csrc/.  There is no CPU fallback."""
from .binding import NpfemError, Solver, load_library, library_path  # noqa: F401

"""B200-native hot path of the MuMax method (arXiv 1102.3069): a thin ctypes binding over the C-ABI
library libmm_b200.so (include/mm.h).  Argument marshalling only; every step runs in CUDA kernels."""
from .mm import (MM_OK, METHODS, Material, MMError, Sim, lib, demag_tensor_host, demag_khat_host)  # noqa: F401

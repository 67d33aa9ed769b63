"""B200-native hybrid tree force evaluation (arXiv:1406.6158) -- thin Python binding over the
C-ABI library libhyb.so (include/hyb.h).  Argument marshalling only: every step of the path runs
in the CUDA kernels under csrc/.  PyTorch supplies device memory and streams."""
from .binding import (HybParams, Hyb, hyb_workspace_bytes, hyb_run_host, hyb_probe_fp32, hyb_energy_noalloc, lib, HybError,  # noqa: F401
                      EXPORTS, ERR_NAMES)

"""B200-native (sm_100a) PIMD hot path of arXiv 2503.23728: thin Python binding over libpimd_b200.so.

All arithmetic runs in the CUDA kernels behind the C-ABI of include/pimd.h; this package only
marshals arguments.  PyTorch is used for device memory and the stream.  There is no CPU fallback:
importing `PIMD` without the compiled library raises.
"""
from .pimd import PIMD, NetParams, Estimators, load_library, library_path, PimdError, measure_fp32_fma_tflops, debye_cv_static  # noqa: F401

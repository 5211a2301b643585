"""B200-native slab-decomposed 3D R2C / C2R FFT (arXiv 2202.12756).  See DESIGN.md.

The compute path is ``libfft3d.so`` (hand-written sm_100a CUDA behind the C ABI of
``include/fft3d.h``); ``binding`` marshals torch tensors into it.  ``inputs`` holds the seeded
synthetic workloads and none of the method's arithmetic.
"""
from .binding import F32, F64, Fft3dError, Plan, PlanC2C, PlanInplace, PlanPencil, load_library, strerror, supported_length  # noqa: F401

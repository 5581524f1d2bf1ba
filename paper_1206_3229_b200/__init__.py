"""B200-native (sm_100a) Strang semi-Lagrangian Vlasov step of arXiv 1206.3229.

``binding``  ctypes binding of the C ABI in ``include/vlasov.h`` (``csrc/libvlasov_b200.so``)
``inputs``   seeded synthetic inputs (the five BASELINE.json configurations); no method arithmetic
``build``    nvcc build step of the CUDA library

The product path has no CPU fallback and never imports ``oracle``.
"""
from . import binding, build, inputs  # noqa: F401
from .binding import Vlasov, VlasovError  # noqa: F401

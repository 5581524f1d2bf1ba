"""CPU fp64 oracle of the Strang semi-Lagrangian Vlasov step (arXiv 1206.3229).

TEST INFRASTRUCTURE -- not part of the product.  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It shares no code with
``paper_1206_3229_b200`` (the CUDA path) and imports nothing from it.

The arithmetic lives in ``vlasov_oracle.c`` (plain C, written from PAPER.md);
this file only compiles it with gcc and marshals numpy arrays through ctypes.
"""
from .vlasov_oracle import (  # noqa: F401
    BC_PERIODIC,
    BC_ZERO,
    KEY_BC_P,
    KEY_BC_X,
    KEY_EPS,
    KEY_SPLINE,
    MODEL_FREE,
    MODEL_HMF,
    MODEL_RING,
    MODEL_SHEET,
    Oracle,
    SPLINE_FD,
    SPLINE_GS,
    build,
    fd8_second_derivative,
    force_from_rho,
    gs_second_derivative,
    shift_line,
)
from .hmf_md_oracle import MdOracle, build_md  # noqa: F401,E402

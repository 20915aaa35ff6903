"""paper_1206_0270_b200: B200-native FP64 Lax-Wendroff time step of the 2+1D Teukolsky equation
(arXiv:1206.0270 section 2.2) behind the C ABI of include/teuk.h.  See DESIGN.md."""
from . import workloads  # noqa: F401
from .teuk import Solver, TeukError, load, measure_fp64  # noqa: F401

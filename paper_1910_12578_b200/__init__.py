"""B200-native hot path of Castro's SDC reactive-flow method (arXiv:1910.12578, Eq. 1-2):
ghost fill, the advective term <A(U)>, the SDC node update (R = 0) and the CFL step, as
hand-written CUDA kernels for sm_100a behind the C ABI in include/cst.h.

  binding   -- ctypes binding of libcst.so (argument marshalling only; no CPU fallback)
  drivers   -- the SDC node loop (2-node trapezoid, M-node Gauss-Lobatto) as sequences of library calls
  workloads -- seeded synthetic inputs of the five BASELINE.json configs
  build     -- in-tree nvcc build of libcst.so
"""
from . import workloads  # noqa: F401
from .binding import Context, CstError, load  # noqa: F401
from .drivers import sdc_step_2nd, sdc_step_nodes, sdc_step_nodes_react  # noqa: F401

"""B200-native traffic microsimulation (arxiv 1807.01148, section 6.3): CUDA kernels behind the
C ABI of include/trafficsim.h, a thin ctypes binding, and the seeded workload generators."""
from . import workload  # noqa: F401
from .binding import Sim, TsError, load, query_workspace, sssp_static, sue_solve  # noqa: F401

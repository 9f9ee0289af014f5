"""paper_1401_6047_b200 -- B200-native (sm_100a, fp64) time-stepping hot path of arxiv 1401.6047.

The product is the C-ABI shared library built from csrc/ (include/bte.h); `Solver` is its thin binding.
Importing this package does not load the library (so the workload generator can be used on a CPU-only
box); constructing a Solver does, and fails loudly if the library or a CUDA device is missing.
"""
from . import workloads  # noqa: F401


def __getattr__(name):
    if name in ("Solver", "Obs", "BteError", "load_library", "workspace_bytes", "EXPORTS", "LIB_PATH",
                "pendulum_averages", "RealSpaceSolver", "rs_evolve_static"):
        from . import binding
        return getattr(binding, name)
    raise AttributeError(name)

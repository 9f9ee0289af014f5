"""CPU oracle of the CN + leap-frog step of arxiv 1401.6047 -- TEST INFRASTRUCTURE, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package.  It never imports paper_1401_6047_b200's CUDA binding and shares no code with it.
"""


def __getattr__(name):  # lazy, so that `python -m oracle.build` does not pre-import the wrapper
    if name in ("OracleSim", "OracleObs", "max_threads", "pendulum_averages", "pendulum_trajectory"):
        from . import bte_oracle
        return getattr(bte_oracle, name)
    raise AttributeError(name)

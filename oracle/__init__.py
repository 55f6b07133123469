"""fp64 CPU oracle (TEST INFRASTRUCTURE — see oracle/ani_oracle.c header).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It never imports the CUDA path.
"""
from .oracle import (AEV_DIM, NET_PARAMS, aev, energy_forces, mlp, num_threads, pairs,  # noqa: F401
                     total_energy_forces)

"""Seeded synthetic inputs shared by the oracle's tests and the CUDA path's tests and bench.
Holds no likelihood arithmetic of either side (see workloads/configs.py for the one shaping helper)."""
from .configs import (CONFIGS, Config, Workload, make_workload, theta_true, random_start, direction,
                      res_chan, masses, fill_amp, TABLE1_M_GAMMA)

__all__ = ["CONFIGS", "Config", "Workload", "make_workload", "theta_true", "random_start", "direction",
           "res_chan", "masses", "fill_amp", "TABLE1_M_GAMMA"]

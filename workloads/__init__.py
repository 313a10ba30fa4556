"""Seeded synthetic inputs shared by the oracle-side and CUDA-side tests and bench.py.
Holds no rendering arithmetic (see workloads/configs.py)."""
from .configs import (ABSORB, ADDITIVE, Camera, Workload, make, make_c1, make_c2, make_c3, make_c4,
                      make_c5, lut_hot, lut_hot_swapped, lut_absorb, FULL_N)

__all__ = ["ABSORB", "ADDITIVE", "Camera", "Workload", "make", "make_c1", "make_c2", "make_c3",
           "make_c4", "make_c5", "lut_hot", "lut_hot_swapped", "lut_absorb", "FULL_N"]

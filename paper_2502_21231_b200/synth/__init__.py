"""Seeded synthetic inputs shared by the tests' two sides (oracle and CUDA) and bench.py.

Holds no arithmetic of the method: a counter-based RNG (synth.c) and the workload recipes of
BASELINE.json's five configs (workloads.py).  Imports neither ``oracle`` nor the CUDA binding.
"""
from .rng import build, normal_f64, rows_bf16, uniform_f64  # noqa: F401
from .workloads import CONFIGS, Workload, make_workload, scaled_twin  # noqa: F401

"""Seeded synthetic workloads (inputs only; no method arithmetic)."""
from .gen import CONFIGS, Workload, make_workload, random_walkers, occupations, sym_normal, sign_fix

__all__ = ["CONFIGS", "Workload", "make_workload", "random_walkers", "occupations",
           "sym_normal", "sign_fix"]

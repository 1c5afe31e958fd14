"""Seeded synthetic input generator (serves both the oracle tests and the CUDA path; holds none
of the method's arithmetic)."""
from .recipe import (ANY, CONFIGS, EVENT_DTYPE, Fault, Spec, Workload, build_workload, scaled,
                     sig_class)

__all__ = ["ANY", "CONFIGS", "EVENT_DTYPE", "Fault", "Spec", "Workload", "build_workload", "scaled",
           "sig_class"]

"""Seeded synthetic input generators shared by the oracle tests and the CUDA path.

This package holds NO arithmetic of the method (no force, predictor, corrector or
time-step code): only the recipes that produce initial conditions and benchmark
inputs shaped like the paper's workloads.
"Input recipe".
"""
from .plummer import (CONFIGS, HENON_B, active_subset, config_inputs, kepler_binary,
                      mean_field_acc, plummer, plummer_with_heavy, power_law_masses)

__all__ = ["CONFIGS", "HENON_B", "active_subset", "config_inputs", "kepler_binary",
           "mean_field_acc", "plummer", "plummer_with_heavy", "power_law_masses"]

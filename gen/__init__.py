"""Seeded synthetic inputs shared by the oracle tests, the GPU parity tests and bench.py.

This module holds NO arithmetic of the Deep Potential method: it only draws atom positions, types, boxes and
random network weights (recipes: DESIGN.md "Input recipe"; BASELINE.json `configs`).  Both the CPU oracle and
the CUDA path receive the very same numpy arrays, so no cross-language RNG matching is needed.
"""
from .systems import (CONFIGS, SEED_BASE, SystemSpec, make_system, perturbed, water_box, copper_box,
                      replicate, MASSES, AMU_A2_FS2_IN_EV, KB_EV, maxwell_boltzmann)
from .weights import ModelSpec, make_weights, emb_net_size, fit_net_size, condition_fit_w0

__all__ = ["CONFIGS", "SEED_BASE", "SystemSpec", "make_system", "perturbed", "water_box", "copper_box",
           "replicate", "MASSES", "AMU_A2_FS2_IN_EV", "KB_EV", "maxwell_boltzmann", "ModelSpec", "make_weights", "emb_net_size", "fit_net_size", "condition_fit_w0"]

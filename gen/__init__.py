"""Seeded synthetic inputs for the batched ph-AFQMC local-energy path.

This package holds NO arithmetic of the method (no overlaps, Green's functions,
energies): only the random Hamiltonians, trials and walkers that both the CPU
oracle (``oracle/``) and the CUDA path (``paper_2209_04015_b200/``) consume.
It imports neither of them.
"""
from .configs import CONFIGS, CONFIG_ORDER, Inputs, make_inputs, make_hamiltonian, make_trial, make_walkers

__all__ = ["CONFIGS", "CONFIG_ORDER", "Inputs", "make_inputs", "make_hamiltonian", "make_trial", "make_walkers"]

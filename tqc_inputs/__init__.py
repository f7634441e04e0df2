"""Seeded synthetic input generators shared by the oracle, the tests and bench.py.

This package holds NO arithmetic of the method (no gate matrices, no
contraction, no Pauli attribution): it only emits *descriptions* — gate lists
(names, angles, operands), gate->subcircuit assignments, cut-network
descriptions, i.i.d. random tensor values and random bitstrings — with the
shapes of the five BASELINE.json configs.  Both the oracle (`oracle/`) and the
CUDA library binding consume these as inputs; neither imports the other.

Seeds follow SURVEY.md section 8(d): seed(cfg, stream) = 250203445*100 + 10*cfg + stream.
"""
from .seeds import seed_for
from .network import Network, pack_states, random_states, random_tensors, rank_one_tensors
from . import circuits, configs

__all__ = ["seed_for", "Network", "pack_states", "random_states", "random_tensors",
           "rank_one_tensors", "circuits", "configs"]

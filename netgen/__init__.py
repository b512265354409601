"""Seeded synthetic metabolic-network generator (inputs only).

This module serves BOTH the CPU oracle (``oracle/``) and the CUDA library
(``paper_1804_02867_b200/``).  It holds none of the method's arithmetic: it only
produces stoichiometric matrices, reversibility flags, internal/external masks
and the parameter sets of the five ``BASELINE.json`` configs.
"""
from .networks import (  # noqa: F401
    CONFIGS,
    chain_pair_network,
    Network,
    SplitMix64,
    config_names,
    hand_network,
    make_network,
    mirrored,
    random_seed_sets,
    unimolecular_network,
    wide_fan_network,
    with_dead_ends,
)

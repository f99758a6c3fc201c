"""Seeded synthetic input generators (BASELINE.json configs).

This package produces *inputs only* (positions, atomic numbers, boxes, ML index
lists, network weights, descriptor hyper-parameters).  It holds none of the
method's arithmetic: no cut-off function, no AEV, no MLP.  Both `oracle/` (through
the tests) and the CUDA path are fed the same arrays; neither imports the other.

The inputs stand in for the paper's bulk-water benchmark (PAPER.md line 144,
Fig. 5; lines 322-356, Tables S2/S3), whose GROMACS input files are not available.
"""
from .water import water_box, perturbed_positions, sheared_water_box
from .cluster import peptide_cluster, solvated_cluster
from .weights import make_weights, aev_params, aev_length
from .configs import get_config, CONFIG_NAMES

__all__ = [
    "water_box", "perturbed_positions", "peptide_cluster", "solvated_cluster",
    "make_weights", "aev_params", "aev_length", "get_config", "CONFIG_NAMES",
]

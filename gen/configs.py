"""The five BASELINE.json configs as seeded synthetic inputs.

get_config(k) -> dict(name, pos fp32 (N,3), pos64, Z int32 (N,), box fp32 (9,), pbc, ml_index or None,
aev = hyper-parameter dict, nets = {Z: (dims, W list, b list)}, celu_alpha, perturb_seed).
Seeds: weights 0 (cfg 0-1) / 1 (cfg 2-4); geometry 100+k; perturbations 200+k.
"""
import functools
import numpy as np
from .water import water_box
from .cluster import solvated_cluster
from .weights import make_weights, aev_params, aev_length, SPECIES_4, SPECIES_7

CONFIG_NAMES = [
    "cfg0_water_32", "cfg1_water_1000", "cfg2_water_8000", "cfg3_water_32000", "cfg4_mlmm_64_in_3000",
]
_WATER = {0: (4, 4, 2, 9.86), 1: (10, 10, 10, 31.04), 2: (20, 20, 20, 62.1), 3: (40, 40, 20, 98.6)}
DIMS_384 = (384, 160, 128, 96, 1)
DIMS_1008 = {1: (1008, 256, 192, 160, 1), 6: (1008, 224, 192, 160, 1),
             7: (1008, 192, 160, 128, 1), 8: (1008, 224, 192, 160, 1)}


def _nets(k, bias_scale=0.0):
    if k in (0, 1):
        return {Z: (DIMS_384,) + make_weights(0, Z, DIMS_384, bias_scale) for Z in (1, 8)}
    zs = (1, 8) if k in (2, 3) else (1, 6, 7, 8)
    return {Z: (DIMS_1008[Z],) + make_weights(1, Z, DIMS_1008[Z], bias_scale) for Z in zs}


@functools.lru_cache(maxsize=8)
def _geometry(k, layout):
    if k in _WATER:
        nx, ny, nz, L = _WATER[k]
        pos, Z, box, pos64 = water_box(nx, ny, nz, L, 100 + k)
        return pos, Z, box, None, pos64
    pos, Z, box, ml, pos64 = solvated_cluster(104, layout=layout)
    return pos, Z, box, ml, pos64


def get_config(k, layout="A", bias_scale=0.0):
    pos, Z, box, ml, pos64 = _geometry(k, layout)
    aev = aev_params(SPECIES_4 if k in (0, 1) else SPECIES_7)
    return dict(name=CONFIG_NAMES[k], k=k, pos=pos, pos64=pos64, Z=Z, box=box, pbc=1, ml_index=ml,
                aev=aev, aev_len=aev_length(aev), nets=_nets(k, bias_scale), celu_alpha=0.1,
                perturb_seed=200 + k)

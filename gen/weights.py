"""Seeded network weights and descriptor hyper-parameters (BASELINE.json configs).

Weights(seed, Z, dims): layer l (1-based) = default_rng([seed, Z, l]).normal(0,1,(dims[l],dims[l-1]))
/ sqrt(dims[l-1]) -> fp32, layout [out][in]; biases zero (reading #15, #16).  Pure data: no network
arithmetic lives here.
"""
import numpy as np

SPECIES_4 = (1, 6, 7, 8)                 # H C N O            (BASELINE.json configs[0])
SPECIES_7 = (1, 6, 7, 8, 16, 9, 17)      # H C N O S F Cl     (BASELINE.json configs[2])


def aev_params(species_Z):
    """ANI-style hyper-parameters of BASELINE.json configs[0] (reading #13: same for the 1008 AEV)."""
    return dict(
        Rcr=5.2, Rca=3.5, EtaR=16.0, EtaA=8.0, Zeta=32.0,
        ShfR=0.9 + 0.25 * np.arange(16, dtype=np.float64),
        ShfA=0.9 + 0.65 * np.arange(4, dtype=np.float64),
        ShfZ=np.pi / 16 + np.arange(8, dtype=np.float64) * np.pi / 8,
        radial_prefactor=0.25, cos_scale=0.95,
        species_Z=np.asarray(species_Z, dtype=np.int32),
    )


def aev_length(p):
    S = len(p["species_Z"])
    return S * len(p["ShfR"]) + S * (S + 1) // 2 * len(p["ShfA"]) * len(p["ShfZ"])


def make_weights(seed, Z, dims, bias_scale=0.0):
    """Returns (W list, b list); W[l] fp32 (dims[l+1], dims[l]); b zero unless bias_scale != 0
    (non-zero biases are used by tests only, drawn from default_rng([seed, Z, 100 + l]))."""
    W, b = [], []
    for l in range(1, len(dims)):
        w = np.random.default_rng([seed, Z, l]).normal(0.0, 1.0, size=(dims[l], dims[l - 1])) / np.sqrt(dims[l - 1])
        W.append(np.ascontiguousarray(w.astype(np.float32)))
        if bias_scale:
            bb = np.random.default_rng([seed, Z, 100 + l]).normal(0.0, bias_scale, size=dims[l])
            b.append(bb.astype(np.float32))
        else:
            b.append(np.zeros(dims[l], dtype=np.float32))
    return W, b

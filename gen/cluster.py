"""Seeded peptide-like cluster + solvent (BASELINE.json configs[4]).

64 ML atoms (H 32, C 18, N 6, O 8): a self-avoiding heavy-atom chain with random torsions, one H
per heavy atom, bonded distances 1.0-1.5 Angstrom, solvated in 3000 H2O in a cubic L = 45 Angstrom box.
"""
import numpy as np
from .water import place_waters


def _unit(v):
    return v / np.linalg.norm(v)


def peptide_cluster(rng):
    """Returns (pos fp64 (64,3) centred at the origin, Z int32 (64,)); order: heavy, its H, heavy, ..."""
    elems = rng.permutation(np.array([6] * 18 + [7] * 6 + [8] * 8, dtype=np.int32))
    heavy = [np.zeros(3)]
    # second atom: arbitrary direction; later atoms: bond length, bond angle, torsion
    for n in range(1, 32):
        for _ in range(1000):
            b = rng.uniform(1.3, 1.5)
            if n == 1:
                v = rng.normal(size=3)
                cand = heavy[0] + b * _unit(v)
            else:
                ang = np.deg2rad(rng.uniform(105.0, 125.0))
                tor = rng.uniform(-np.pi, np.pi)
                prev = _unit(heavy[n - 1] - heavy[n - 2])
                if n >= 3:
                    ref = heavy[n - 2] - heavy[n - 3]
                else:
                    ref = np.array([0.0, 0.0, 1.0]) if abs(prev[2]) < 0.9 else np.array([1.0, 0.0, 0.0])
                nrm = np.cross(prev, ref)
                if np.linalg.norm(nrm) < 1e-8:
                    nrm = np.cross(prev, np.array([0.3, 0.5, 0.8]))
                nrm = _unit(nrm)
                e2 = np.cross(nrm, prev)
                # new bond makes angle (pi - ang) with the previous bond direction
                d = -np.cos(ang) * prev + np.sin(ang) * (np.cos(tor) * e2 + np.sin(tor) * nrm)
                cand = heavy[n - 1] + b * d
            far = heavy[: max(0, n - 2)]
            if len(far) == 0 or np.min(np.linalg.norm(np.array(far) - cand, axis=1)) >= 2.4:
                heavy.append(cand)
                break
        else:
            raise RuntimeError("chain growth failed")
    heavy = np.array(heavy)
    hyd = []
    for n in range(32):
        for _ in range(1000):
            b = rng.uniform(1.0, 1.1)
            cand = heavy[n] + b * _unit(rng.normal(size=3))
            others = np.concatenate([np.delete(heavy, n, axis=0)] + ([np.array(hyd)] if hyd else []), axis=0)
            if np.min(np.linalg.norm(others - cand, axis=1)) >= 1.6:
                hyd.append(cand)
                break
        else:
            raise RuntimeError("hydrogen placement failed")
    hyd = np.array(hyd)
    pos = np.empty((64, 3))
    Z = np.empty(64, dtype=np.int32)
    pos[0::2], pos[1::2] = heavy, hyd
    Z[0::2], Z[1::2] = elems, 1
    pos -= pos.mean(axis=0)
    return pos, Z


def solvated_cluster(seed, L=45.0, nsite=15, ndrop=375, layout="A"):
    """cfg 4.  Returns (pos fp32 (9064,3), Z int32, box fp32 (9,), ml_index int32 (64,), pos64)."""
    rng = np.random.default_rng(seed)
    cpos, cZ = peptide_cluster(rng)
    centre = np.full(3, L / 2.0)
    cpos = cpos + centre
    g = np.stack(np.meshgrid(*(np.arange(nsite),) * 3, indexing="ij"), -1).reshape(-1, 3)
    sites = (g + 0.5) * (L / nsite)
    d = np.linalg.norm(sites - centre, axis=1)
    drop = np.argsort(d, kind="stable")[:ndrop]
    keep = np.ones(len(sites), dtype=bool)
    keep[drop] = False
    g, sites = g[keep], sites[keep]
    r_O = sites + rng.uniform(-0.3, 0.3, size=sites.shape)
    box = np.array([L, L, L])
    wpos = place_waters(r_O, box, rng, site_index=g, dims=(nsite,) * 3, fixed_atoms=cpos)
    wZ = np.tile(np.array([8, 1, 1], dtype=np.int32), len(sites))
    n_tot = 64 + wpos.shape[0]
    if layout == "A":
        pos64 = np.concatenate([cpos, wpos], axis=0)
        Z = np.concatenate([cZ, wZ])
        ml = np.arange(64, dtype=np.int32)
    elif layout == "B":
        ml = np.sort(rng.choice(n_tot, 64, replace=False)).astype(np.int32)
        mask = np.zeros(n_tot, dtype=bool)
        mask[ml] = True
        pos64 = np.empty((n_tot, 3))
        Z = np.empty(n_tot, dtype=np.int32)
        pos64[mask], pos64[~mask] = cpos, wpos
        Z[mask], Z[~mask] = cZ, wZ
    else:
        raise ValueError(layout)
    box9 = np.diag(box).astype(np.float32).reshape(9)
    return pos64.astype(np.float32), Z, box9, ml, pos64

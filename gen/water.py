"""Seeded water-box generator (SURVEY.md Appendix C "Water box"; BASELINE.json configs[0-3]).

Geometry recipe (readings #18, #19 of SURVEY.md section 8.c):
  * O on cell-centred lattice sites, C order (z fastest), + U(-0.3, 0.3) Angstrom jitter per coordinate;
  * rigid O-H 0.9572 Angstrom, H-O-H 104.52 deg, orientation = uniform SO(3) (Shoemake quaternion);
  * close-contact rule: redraw the orientation while any atom of the new molecule is closer than
    0.8 Angstrom (minimum image) to an atom of an already placed molecule;
  * atom order O,H,H; molecules kept whole (H may lie outside [0, L)); positions stored as fp32.
"""
import numpy as np

R_OH = 0.9572
HALF_HOH = np.deg2rad(104.52 / 2.0)
CONTACT = 0.8


def _quat_to_matrix(q):
    x, y, z, w = q
    return np.array([
        [1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)],
        [2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)],
        [2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)],
    ])


def random_rotation(rng):
    """One `rng.random(3)` call -> uniform rotation matrix (Shoemake)."""
    u1, u2, u3 = rng.random(3)
    q = (np.sqrt(1 - u1) * np.sin(2 * np.pi * u2), np.sqrt(1 - u1) * np.cos(2 * np.pi * u2),
         np.sqrt(u1) * np.sin(2 * np.pi * u3), np.sqrt(u1) * np.cos(2 * np.pi * u3))
    return _quat_to_matrix(q)


BODY_H = np.array([[R_OH * np.sin(HALF_HOH), 0.0, R_OH * np.cos(HALF_HOH)],
                   [-R_OH * np.sin(HALF_HOH), 0.0, R_OH * np.cos(HALF_HOH)]])


def _min_image(d, box):
    return d - box * np.rint(d / box)


def place_waters(r_O, box, rng, site_index=None, dims=None, fixed_atoms=None):
    """Place rigid waters on the given O positions in order, applying the close-contact rule.

    r_O: (M,3) fp64 oxygen positions; box: (3,) box lengths.  `site_index` (M,3) integer lattice
    coordinates and `dims` speed the contact search up (only molecules on nearby sites are
    tested); without them every placed molecule is tested.  `fixed_atoms` (K,3) are extra atoms
    (the cfg-4 cluster) the waters must also keep 0.8 Angstrom away from.
    Returns (3M,3) fp64 positions in O,H,H order.
    """
    M = r_O.shape[0]
    pos = np.zeros((M, 3, 3))
    if site_index is not None:
        dims = np.asarray(dims)
        lin = -np.ones(tuple(dims), dtype=np.int64)
        offs = np.array([(a, b, c) for a in range(-2, 3) for b in range(-2, 3) for c in range(-2, 3)])
    for m in range(M):
        if site_index is not None:
            nb = (site_index[m] + offs) % dims
            cand = np.unique(lin[nb[:, 0], nb[:, 1], nb[:, 2]])
            cand = cand[cand >= 0]
        else:
            cand = np.arange(m)
        others = pos[cand].reshape(-1, 3)
        if fixed_atoms is not None and len(fixed_atoms):
            others = np.concatenate([others, fixed_atoms], axis=0)
        for _ in range(100):
            Q = random_rotation(rng)
            mol = np.vstack([r_O[m], r_O[m] + BODY_H @ Q.T])
            if others.shape[0] == 0:
                break
            d = _min_image(mol[:, None, :] - others[None, :, :], box)
            if np.sqrt((d * d).sum(-1)).min() >= CONTACT:
                break
        else:
            raise RuntimeError("close-contact rule: no valid orientation in 100 tries")
        pos[m] = mol
        if site_index is not None:
            s = site_index[m]
            lin[s[0], s[1], s[2]] = m
    return pos.reshape(-1, 3)


def water_box(nx, ny, nz, L, seed):
    """Returns (pos fp32 (3M,3), Z int32 (3M,), box fp32 (9,), pos64 fp64 (3M,3))."""
    rng = np.random.default_rng(seed)
    dims = np.array([nx, ny, nz])
    g = np.stack(np.meshgrid(np.arange(nx), np.arange(ny), np.arange(nz), indexing="ij"), -1).reshape(-1, 3)
    spacing = np.array([L / nx, L / ny, L / nz])
    r_O = (g + 0.5) * spacing + rng.uniform(-0.3, 0.3, size=(g.shape[0], 3))
    box = np.array([L, L, L], dtype=np.float64)
    pos64 = place_waters(r_O, box, rng, site_index=g, dims=dims)
    Z = np.tile(np.array([8, 1, 1], dtype=np.int32), g.shape[0])
    box9 = np.diag(box).astype(np.float32).reshape(9)
    return pos64.astype(np.float32), Z, box9, pos64


def perturbed_positions(pos64, seed, T, sigma=0.01):
    """x_t = x_0 + N(0, sigma^2), not cumulative, rounded to fp32 (reading #17). Shape (T,N,3)."""
    rng = np.random.default_rng(seed)
    eps = rng.normal(0.0, sigma, size=(T,) + pos64.shape)
    return (pos64[None] + eps).astype(np.float32)


def sheared_water_box(cfg, bx, cx, cy):
    """Triclinic stand-in (GROMACS lower-triangular box): the molecules of an orthorhombic
    water configuration `cfg` are moved with their oxygen to the same FRACTIONAL position of the box with rows
    a = (Lx, 0, 0), b = (bx*Lx, Ly, 0), c = (cx*Lx, cy*Ly, Lz) (bx, cx, cy in box-length units, |.| <= 0.5); molecules stay
    rigid.  Returns (pos float32 (N,3), box float32 (9,)).  Input generation only: no model arithmetic."""
    pos = cfg["pos"].astype(np.float64)
    Lx, Ly, Lz = float(cfg["box"][0]), float(cfg["box"][4]), float(cfg["box"][8])
    H = np.array([[Lx, 0.0, 0.0], [bx * Lx, Ly, 0.0], [cx * Lx, cy * Ly, Lz]])
    out = pos.copy()
    n_mol = pos.shape[0] // 3
    for m in range(n_mol):            # atoms are stored molecule by molecule: O, H, H
        o = pos[3 * m]
        s = o / np.array([Lx, Ly, Lz])
        shift = s @ H - o
        out[3 * m: 3 * m + 3] += shift
    return out.astype(np.float32), H.astype(np.float32).reshape(9)

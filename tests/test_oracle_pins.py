"""Pins of the fp64 CPU oracle against things other than itself (-m "not gpu").

What fixes each part (SURVEY.md section 8.c "What pins each part"):
  * worked values of SURVEY.md Appendix B (tests/golden/appendix_b.json) -> cut-off, radial, angular,
    element order, PBC, one-layer network energy and forces;
  * textbook matmul+CELU chain in numpy fp64 -> MLP forward; its analytic gradient vs finite differences;
  * central finite differences of the oracle energy -> MLP backward + AEV backward + force assembly;
  * a short differentiable restatement in torch-CPU fp64 (autograd) -> AEV and forces, third opinion;
  * invariances (sum F = 0, torque, translation, rotation, permutation, cubic point group, MM independence);
  * brute-force numpy double loop -> neighbour definition; cell list == definition.
"""
import itertools
import json
import os

import numpy as np
import pytest

import oracle
from gen import aev_params, aev_length, get_config, make_weights
from gen.weights import SPECIES_4, SPECIES_7

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "appendix_b.json")))
P4 = aev_params(SPECIES_4)
BOX30 = np.diag([30.0, 30.0, 30.0]).reshape(9).astype(np.float32)
R_OH = 0.9572
PHI = np.deg2rad(104.52 / 2)


def ones_net(L):
    """One-layer all-ones network: E_i = sum of all AEV entries (Appendix B.2)."""
    return ((L, 1), [np.ones((1, L), np.float32)], [np.zeros(1, np.float32)])


def model4(nets=None):
    L = aev_length(P4)
    if nets is None:
        nets = {Z: ones_net(L) for Z in SPECIES_4}
    return oracle.Model(P4, nets)


def monomer():
    O = np.array([10.0, 10.0, 10.0])
    H1 = O + [R_OH * np.sin(PHI), 0, R_OH * np.cos(PHI)]
    H2 = O + [-R_OH * np.sin(PHI), 0, R_OH * np.cos(PHI)]
    return np.array([O, H1, H2]), np.array([8, 1, 1], np.int32)


# ------------------------------------------------------------------ scalars (Appendix B.5)
def test_cutoff_and_celu_scalars():
    assert oracle.fc(0.0, 5.2) == 1.0
    assert abs(oracle.fc(2.6, 5.2) - 0.5) < 1e-15
    assert abs(oracle.fc(5.2, 5.2)) < 1e-15
    assert oracle.fc(5.2000001, 5.2) == 0.0
    assert abs(oracle.fc(R_OH, 5.2) - GOLD["B5_fc_0p9572_5p2"]) < 1e-11
    assert abs(oracle.fc(R_OH, 3.5) - GOLD["B5_fc_0p9572_3p5"]) < 1e-11
    assert abs(oracle.celu(-0.1) - GOLD["B5_celu_m0p1"]) < 1e-11
    assert abs(oracle.celu(-1.0) - GOLD["B5_celu_m1"]) < 1e-11
    assert oracle.celu(0.3) == 0.3
    # CELU' continuous at 0: one-sided slopes agree
    h = 1e-7
    assert abs((oracle.celu(h) - oracle.celu(0)) / h - (oracle.celu(0) - oracle.celu(-h)) / h) < 1e-5


# ------------------------------------------------------------------ B.1 dimer
def test_dimer_radial_closed_form():
    pos = np.array([[10, 10, 10], [10 + R_OH, 10, 10]], np.float64)
    # fp32 positions: 10+0.9572 rounds; use the fp32-rounded distance for the closed form
    p32 = pos.astype(np.float32)
    R = float(np.linalg.norm(p32[1].astype(np.float64) - p32[0].astype(np.float64)))
    out = oracle.evaluate(model4(), p32, [8, 1], BOX30, want_aev=True)
    aev = out["aev"]
    fcv = 0.5 * np.cos(np.pi * R / 5.2) + 0.5
    closed = 0.25 * np.exp(-16.0 * (R - P4["ShfR"]) ** 2) * fcv
    assert np.allclose(aev[0, 0:16], closed, rtol=1e-12, atol=0)          # centre O, slot H
    assert np.allclose(aev[1, 48:64], closed, rtol=1e-12, atol=0)         # centre H, slot O = 3*16
    assert np.allclose(aev[0, 0:4], GOLD["B1_dimer_radial_m0_3"], rtol=2e-5)
    mask = np.ones(384, bool); mask[0:16] = False
    assert np.all(aev[0, mask] == 0.0) and np.all(aev[0, 64:] == 0.0)     # no angular entries


# ------------------------------------------------------------------ B.2 water monomer
def test_monomer_aev_energy_forces():
    pos, Z = monomer()
    assert abs(np.linalg.norm(pos[1] - pos[2]) - GOLD["B2_d_HH"]) < 1e-9
    out = oracle.evaluate(model4(), pos, Z, BOX30, want_aev=True, want_atomic=True)
    aev = out["aev"]
    rt = 3e-6  # fp32 rounding of the input positions (1e-7 relative) amplified by eta and zeta
    assert np.allclose(aev[0, 0:4], GOLD["B2_O_radial_H_m0_3"], rtol=1e-5, atol=5e-9)
    assert np.allclose(aev[0, 64:72], GOLD["B2_O_ang_HH_a0"], rtol=2e-5)
    assert np.allclose(aev[0, 72:80], GOLD["B2_O_ang_HH_a1"], rtol=2e-5)
    assert abs(aev[0, 64:96].sum() - GOLD["B2_O_ang_HH_sum"]) < rt * 3
    assert np.all(aev[0, 96:] == 0.0)
    assert np.allclose(aev[1, 48:51], GOLD["B2_H1_radial_O_m0_2"], rtol=1e-5, atol=5e-9)
    assert np.allclose(aev[1, 0:5], GOLD["B2_H1_radial_H_m0_4"], rtol=2e-5, atol=5e-9)
    assert np.allclose(aev[1, 160:168], GOLD["B2_H1_ang_HO_a0"], rtol=3e-5)
    assert np.allclose(aev[1, 168:176], GOLD["B2_H1_ang_HO_a1"], rtol=3e-5)
    assert abs(aev[1, 160:192].sum() - GOLD["B2_H1_ang_HO_sum"]) < rt * 3
    assert abs(aev[0].sum() - GOLD["B2_sum_O"]) < 1e-5
    assert abs(aev[1].sum() - GOLD["B2_sum_H"]) < 1e-5
    assert abs(aev[2].sum() - GOLD["B2_sum_H"]) < 1e-5
    assert abs(out["energy"] - GOLD["B2_E_all_ones"]) < 3e-5
    assert np.allclose(out["e_atom"], aev.sum(1), rtol=1e-13)
    F = out["forces"]
    assert np.allclose(F[0], GOLD["B2_F_O"], atol=2e-5)
    assert np.allclose(F[1], GOLD["B2_F_H1"], atol=2e-5)
    assert np.allclose(F[2], GOLD["B2_F_H2"], atol=2e-5)
    assert np.abs(F.sum(0)).max() < 1e-12


# ------------------------------------------------------------------ B.3 collinear trimer
def test_collinear_trimer_finite():
    pos = np.array([[10, 10, 10], [11.0, 10, 10], [8.2, 10, 10]], np.float64)
    Z = np.array([8, 1, 8], np.int32)
    out = oracle.evaluate(model4(), pos, Z, BOX30, want_aev=True)
    base = 64 + 3 * 32  # p(H,O) = 3
    row = out["aev"][0, base + 8: base + 16]
    assert np.allclose(row, GOLD["B3_trimer_HO_a1"], rtol=3e-5)
    assert abs(out["aev"][0, base: base + 32].sum() - GOLD["B3_trimer_HO_sum"]) < 1e-5
    assert np.all(np.isfinite(out["forces"]))
    assert np.abs(out["forces"].sum(0)).max() < 1e-12


# ------------------------------------------------------------------ B.4 PBC dimer
def test_pbc_dimer_equals_interior_dimer():
    a = oracle.evaluate(model4(), [[0.2, 5, 5], [29.6, 5, 5]], [8, 1], BOX30, want_aev=True)
    # fp32(29.6)-30 differs from -0.4 by fp32 rounding; build the interior copy from the same rounding
    dx = float(np.float32(29.6)) - 30.0 - float(np.float32(0.2))
    b = oracle.evaluate(model4(), [[10.0, 5, 5], [10.0 + dx, 5, 5]], [8, 1], BOX30, want_aev=True)
    assert abs(a["aev"][0, 0] - GOLD["B4_pbc_dimer_m0"]) < 2e-6
    assert np.allclose(a["aev"], b["aev"], rtol=2e-5, atol=1e-12)
    assert np.allclose(a["forces"], b["forces"], rtol=2e-5, atol=1e-9)
    # without PBC the pair is 29.4 apart: no neighbours at all
    c = oracle.evaluate(model4(), [[0.2, 5, 5], [29.6, 5, 5]], [8, 1], BOX30, pbc=0, want_aev=True)
    assert np.all(c["aev"] == 0.0)


# ------------------------------------------------------------------ MLP forward/backward
def test_mlp_matches_textbook_chain_and_fd():
    dims = (384, 160, 128, 96, 1)
    W, b = make_weights(7, 8, dims, bias_scale=0.3)
    rng = np.random.default_rng(5)
    G = rng.uniform(0, 1.5, size=384)
    E, g = oracle.mlp_forward(dims, W, b, G)
    h = G.copy()
    for l in range(4):
        z = W[l].astype(np.float64) @ h + b[l].astype(np.float64)
        h = z if l == 3 else np.where(z > 0, z, 0.1 * np.expm1(z / 0.1))
    assert abs(E - h[0]) < 1e-12 * max(1, abs(h[0]))
    # gradient by central differences of the numpy chain
    def f(G):
        h = G
        for l in range(4):
            z = W[l].astype(np.float64) @ h + b[l].astype(np.float64)
            h = z if l == 3 else np.where(z > 0, z, 0.1 * np.expm1(z / 0.1))
        return h[0]
    for i in rng.choice(384, 24, replace=False):
        e = np.zeros(384); e[i] = 1e-6
        fd = (f(G + e) - f(G - e)) / 2e-6
        assert abs(fd - g[i]) < 1e-7 * max(1.0, abs(g[i]))
    # zero weights => E = last bias
    Wz = [np.zeros_like(w) for w in W]
    E0, g0 = oracle.mlp_forward(dims, Wz, b, G)
    assert abs(E0 - float(b[3][0])) < 1e-15 and np.all(g0 == 0.0)


# ------------------------------------------------------------------ neighbour definition
def brute_neighbors_numpy(pos, box, Rc, pbc, active):
    L = np.array([box[0], box[4], box[8]], np.float64)
    p = pos.astype(np.float32).astype(np.float64)
    rows = []
    for i in active:
        d = p[active] - p[i]
        if pbc:
            d = d - L * np.rint(d / L)
        d2 = d[:, 0] * d[:, 0]
        d2 = d[:, 1] * d[:, 1] + d2      # differs from fma only in the last ulp; tests avoid boundary ties
        d2 = d[:, 2] * d[:, 2] + d2
        m = (d2 <= Rc * Rc) & (np.asarray(active) != i)
        rows.append(np.asarray(active)[m])
    return rows


def test_neighbor_list_is_the_double_loop():
    cfg = get_config(0)
    act = np.arange(96)
    for Rc in (5.2, 3.5):
        start, col = oracle.neighbors(cfg["pos"], cfg["box"], Rc)
        rows = brute_neighbors_numpy(cfg["pos"], cfg["box"], Rc, 1, act)
        for i in range(96):
            assert np.array_equal(col[start[i]:start[i + 1]], rows[i])
        # symmetry
        pairs = {(i, int(j)) for i in range(96) for j in col[start[i]:start[i + 1]]}
        assert all((j, i) in pairs for (i, j) in pairs)
    sr, cr = oracle.neighbors(cfg["pos"], cfg["box"], 5.2)
    sa, ca = oracle.neighbors(cfg["pos"], cfg["box"], 3.5)
    for i in range(96):  # angular subset of radial
        assert set(ca[sa[i]:sa[i + 1]]) <= set(cr[sr[i]:sr[i + 1]])


@pytest.mark.parametrize("k", [0, 1, 2, 4])
def test_cell_list_equals_definition(k):
    """The oracle's cell-list mode (mode=1, what the cfg-2 / cfg-3 GPU lists and the timed CPU baseline use) equals its
    O(N^2) definition (mode=0) -- at headline size too (cfg 2: one 24 000-atom double loop per cut-off)."""
    cfg = get_config(k)
    for Rc in (5.2, 3.5):
        s0, c0 = oracle.neighbors(cfg["pos"], cfg["box"], Rc, ml_index=cfg["ml_index"], mode=0)
        s1, c1 = oracle.neighbors(cfg["pos"], cfg["box"], Rc, ml_index=cfg["ml_index"], mode=1)
        assert np.array_equal(s0, s1) and np.array_equal(c0, c1)
    if k == 1:  # statistical sanity: (4/3) pi R^3 rho = 59.0 / 18.0 at rho = 0.1002 (section 8.c pins)
        s, _ = oracle.neighbors(cfg["pos"], cfg["box"], 5.2)
        assert abs(np.diff(s).mean() - 59.0) < 2.0
        s, _ = oracle.neighbors(cfg["pos"], cfg["box"], 3.5)
        assert abs(np.diff(s).mean() - 18.0) < 2.5


def test_neighbors_invariant_under_image_shift():
    cfg = get_config(0)
    pos = cfg["pos"].astype(np.float64).copy()
    s0, c0 = oracle.neighbors(pos, cfg["box"], 3.5)
    pos2 = pos.copy()
    pos2[5] += [9.86 * 2, 0, -9.86]  # exact box-vector multiples are not exact in fp32: compare sets away from ties
    s1, c1 = oracle.neighbors(pos2, cfg["box"], 3.5)
    assert np.array_equal(s0, s1) and np.array_equal(c0, c1)


# ------------------------------------------------------------------ finite differences
def fd_forces(model, pos, Z, box, pbc, atoms, h, ml_index=None):
    F = np.zeros((len(atoms), 3))
    for n, a in enumerate(atoms):
        for c in range(3):
            p = pos.copy(); p[a, c] += h
            m = pos.copy(); m[a, c] -= h
            Ep = oracle.evaluate(model, p, Z, box, pbc, ml_index, want_forces=False)["energy"]
            Em = oracle.evaluate(model, m, Z, box, pbc, ml_index, want_forces=False)["energy"]
            # positions pass through fp32: use the realised displacement
            dp = float(np.float32(p[a, c])) - float(np.float32(m[a, c]))
            F[n, c] = -(Ep - Em) / dp
    return F


def small_cluster(seed=3, n=14):
    """Non-periodic cluster of 4 species with coordinates exactly representable in fp32."""
    rng = np.random.default_rng(seed)
    while True:
        pos = rng.uniform(0, 4.2, size=(n, 3))
        d = np.linalg.norm(pos[:, None] - pos[None], axis=-1) + np.eye(n) * 9
        if d.min() > 0.85:
            break
    pos = np.round(pos * 1024) / 1024 + 8.0
    Z = rng.choice(np.array(SPECIES_4, np.int32), size=n)
    Z[:4] = SPECIES_4
    return pos, Z


def test_forces_match_finite_differences_cluster():
    pos, Z = small_cluster()
    dims = (384, 32, 24, 16, 1)
    nets = {z: (dims,) + make_weights(11, z, dims, bias_scale=0.2) for z in SPECIES_4}
    model = model4(nets)
    out = oracle.evaluate(model, pos, Z, BOX30, pbc=0)
    F = out["forces"]
    h = 2.0 ** -13  # exactly representable next to coordinates ~8-13 in fp32
    Ffd = fd_forces(model, pos, Z, BOX30, 0, range(len(Z)), h)
    scale = np.abs(F).max()
    assert scale > 1e-3
    assert np.abs(F - Ffd).max() < 2e-6 * scale
    assert np.abs(F.sum(0)).max() < 1e-10 * scale
    torque = np.cross(pos, F).sum(0)
    assert np.abs(torque).max() < 1e-9 * scale * 10


def test_forces_match_finite_differences_cfg0_periodic():
    cfg = get_config(0, bias_scale=0.1)
    model = oracle.Model(cfg["aev"], cfg["nets"])
    pos = np.round(cfg["pos"].astype(np.float64) * 4096) / 4096
    out = oracle.evaluate(model, pos, cfg["Z"], cfg["box"])
    F = out["forces"]
    atoms = [0, 1, 2, 30, 31, 95]
    Ffd = fd_forces(model, pos, cfg["Z"], cfg["box"], 1, atoms, 2.0 ** -14)
    scale = np.abs(F).max()
    assert np.abs(F[atoms] - Ffd).max() < 5e-6 * scale
    assert np.abs(F.sum(0)).max() < 1e-10 * scale


# ------------------------------------------------------------------ autograd restatement (third opinion)
def torch_restatement(pos, Z, params, nets, L_box=None):
    """A few lines of differentiable torch fp64: AEV, E and F = -dE/dr by autograd (test-only)."""
    import torch
    torch.set_default_dtype(torch.float64)
    r = torch.tensor(np.asarray(pos, np.float32).astype(np.float64), requires_grad=True)
    n = r.shape[0]
    sZ = list(params["species_Z"]); S = len(sZ)
    slot = [sZ.index(int(z)) for z in Z]
    ShfR, ShfA, ShfZ = (torch.tensor(params[k]) for k in ("ShfR", "ShfA", "ShfZ"))
    Ltot = aev_length(params)
    E = 0.0; aevs = []
    for i in range(n):
        G = torch.zeros(Ltot)
        nb = []
        for j in range(n):
            if j == i: continue
            d = r[j] - r[i]
            if L_box is not None: d = d - L_box * torch.round(d / L_box)
            R = d.norm()
            if R.item() <= params["Rcr"]:
                f = 0.5 * torch.cos(np.pi * R / params["Rcr"]) + 0.5
                idx = slot[j] * 16 + torch.arange(16)
                G = G.index_add(0, idx, params["radial_prefactor"] * torch.exp(-params["EtaR"] * (R - ShfR) ** 2) * f)
            if R.item() <= params["Rca"]:
                nb.append((j, d, R))
        for (j, dj, Rj), (k, dk, Rk) in itertools.combinations(nb, 2):
            th = torch.acos(params["cos_scale"] * (dj @ dk) / (Rj * Rk))
            ff = (0.5 * torch.cos(np.pi * Rj / params["Rca"]) + 0.5) * (0.5 * torch.cos(np.pi * Rk / params["Rca"]) + 0.5)
            F2 = torch.exp(-params["EtaA"] * ((Rj + Rk) / 2 - ShfA) ** 2)
            F1 = ((1 + torch.cos(th - ShfZ)) / 2) ** params["Zeta"]
            s1, s2 = sorted((slot[j], slot[k]))
            p = s1 * S - s1 * (s1 - 1) // 2 + (s2 - s1)
            idx = S * 16 + p * 32 + torch.arange(32)
            G = G.index_add(0, idx, (2 * F2[:, None] * F1[None, :] * ff).reshape(-1))
        aevs.append(G)
        dims, W, b = nets[int(Z[i])]
        h = G
        for l in range(len(W)):
            z = torch.tensor(W[l].astype(np.float64)) @ h + torch.tensor(b[l].astype(np.float64))
            # (torch.nn.functional.celu rounds 1/alpha through fp32 in its backward: written out instead)
            h = z if l == len(W) - 1 else torch.where(z > 0, z, 0.1 * torch.expm1(z / 0.1))
        E = E + h[0]
    F = -torch.autograd.grad(E, r)[0]
    return E.item(), F.numpy(), torch.stack(aevs).detach().numpy()


def test_against_autograd_restatement():
    pos, Z = small_cluster(seed=9, n=10)
    dims = (384, 20, 12, 8, 1)
    nets = {z: (dims,) + make_weights(3, z, dims, bias_scale=0.2) for z in SPECIES_4}
    E, F, aev = torch_restatement(pos, Z, P4, nets)
    out = oracle.evaluate(model4(nets), pos, Z, BOX30, pbc=0, want_aev=True)
    assert np.allclose(out["aev"], aev, rtol=1e-10, atol=1e-14)
    assert abs(out["energy"] - E) < 1e-11 * max(1, abs(E))
    assert np.abs(out["forces"] - F).max() < 1e-9 * np.abs(F).max()


def test_against_autograd_restatement_periodic_7_species():
    P7 = aev_params(SPECIES_7)
    rng = np.random.default_rng(2)
    Lb = 7.5
    while True:
        pos = rng.uniform(0, Lb, size=(12, 3))
        d = pos[:, None] - pos[None]; d -= Lb * np.rint(d / Lb)
        if (np.linalg.norm(d, axis=-1) + np.eye(12) * 9).min() > 0.9:
            break
    Z = np.array([1, 6, 7, 8, 16, 9, 17, 1, 8, 1, 6, 17], np.int32)
    dims = (1008, 16, 8, 8, 1)
    nets = {z: (dims,) + make_weights(4, z, dims, bias_scale=0.1) for z in SPECIES_7}
    E, F, aev = torch_restatement(pos, Z, P7, nets, L_box=Lb)
    box = np.diag([Lb] * 3).reshape(9)
    out = oracle.evaluate(oracle.Model(P7, nets), pos, Z, box, want_aev=True)
    assert np.allclose(out["aev"], aev, rtol=1e-10, atol=1e-14)
    assert abs(out["energy"] - E) < 1e-11 * max(1, abs(E))
    assert np.abs(out["forces"] - F).max() < 1e-9 * np.abs(F).max()


# ------------------------------------------------------------------ invariances
def test_invariances_periodic_cfg0():
    cfg = get_config(0, bias_scale=0.1)
    model = oracle.Model(cfg["aev"], cfg["nets"])
    pos = cfg["pos"].astype(np.float64)
    L = 9.86
    ref = oracle.evaluate(model, pos, cfg["Z"], cfg["box"])
    scale = np.abs(ref["forces"]).max()
    # permutation equivariance
    perm = np.random.default_rng(0).permutation(96)
    o = oracle.evaluate(model, pos[perm], cfg["Z"][perm], cfg["box"])
    assert abs(o["energy"] - ref["energy"]) < 1e-10 * abs(ref["energy"])
    assert np.abs(o["forces"] - ref["forces"][perm]).max() < 1e-10 * scale
    # translation (fp32 re-rounding of inputs limits agreement)
    o = oracle.evaluate(model, pos + [0.5, -1.25, 2.0], cfg["Z"], cfg["box"])
    assert abs(o["energy"] - ref["energy"]) < 2e-5 * abs(ref["energy"]) + 1e-4
    assert np.abs(o["forces"] - ref["forces"]).max() < 2e-4 * scale
    # cubic point group: signed axis permutations about the box centre
    for axes, signs in [((1, 2, 0), (1, 1, 1)), ((0, 1, 2), (-1, 1, 1)), ((2, 1, 0), (1, -1, -1)), ((1, 0, 2), (-1, -1, 1))]:
        Q = np.zeros((3, 3))
        for r_, (a, s) in enumerate(zip(axes, signs)):
            Q[r_, a] = s
        p2 = (pos - L / 2) @ Q.T + L / 2
        o = oracle.evaluate(model, p2, cfg["Z"], cfg["box"])
        assert abs(o["energy"] - ref["energy"]) < 2e-5 * abs(ref["energy"]) + 1e-4
        assert np.abs(o["forces"] - ref["forces"] @ Q.T).max() < 2e-4 * scale


def test_rotation_invariance_open_boundaries():
    pos, Z = small_cluster(seed=4, n=12)
    dims = (384, 24, 16, 8, 1)
    nets = {z: (dims,) + make_weights(5, z, dims, bias_scale=0.2) for z in SPECIES_4}
    model = model4(nets)
    ref = oracle.evaluate(model, pos, Z, BOX30, pbc=0)
    from gen.water import random_rotation
    Q = random_rotation(np.random.default_rng(8))
    c = pos.mean(0)
    o = oracle.evaluate(model, (pos - c) @ Q.T + c, Z, BOX30, pbc=0)
    s = np.abs(ref["forces"]).max()
    assert abs(o["energy"] - ref["energy"]) < 1e-5 * max(1, abs(ref["energy"]))
    assert np.abs(o["forces"] - ref["forces"] @ Q.T).max() < 1e-4 * s


def test_cfg4_mm_independence_and_layouts():
    A = get_config(4, "A")
    B = get_config(4, "B")
    model = oracle.Model(A["aev"], A["nets"])
    oa = oracle.evaluate(model, A["pos"], A["Z"], A["box"], ml_index=A["ml_index"])
    ob = oracle.evaluate(model, B["pos"], B["Z"], B["box"], ml_index=B["ml_index"])
    assert oa["energy"] == pytest.approx(ob["energy"], rel=1e-13)
    assert np.allclose(oa["forces"][A["ml_index"]], ob["forces"][B["ml_index"]], rtol=0, atol=1e-12)
    mm = np.setdiff1d(np.arange(9064), A["ml_index"])
    assert np.all(oa["forces"][mm] == 0.0)
    # deleting / moving MM atoms changes nothing
    oc = oracle.evaluate(model, A["pos"][:64], A["Z"][:64], A["box"])
    assert oc["energy"] == pytest.approx(oa["energy"], rel=1e-13)
    assert np.allclose(oc["forces"], oa["forces"][:64], rtol=0, atol=1e-12)
    p2 = A["pos"].copy(); p2[64:] += 0.37
    od = oracle.evaluate(model, p2, A["Z"], A["box"], ml_index=A["ml_index"])
    assert od["energy"] == oa["energy"]
    # bonded distances of the cluster lie in 1.0-1.5 Angstrom (BASELINE.json configs[4])
    c = A["pos64"][:64]
    assert all(1.0 <= np.linalg.norm(c[2 * i] - c[2 * i + 1]) <= 1.1 for i in range(32))
    assert all(1.3 <= np.linalg.norm(c[2 * i] - c[2 * i + 2]) <= 1.5 for i in range(31))


def test_errors():
    pos, Z = monomer()
    with pytest.raises(RuntimeError):  # unknown species
        oracle.evaluate(model4(), pos, [8, 1, 2], BOX30)
    bad = BOX30.copy(); bad[1] = 0.5
    with pytest.raises(RuntimeError):  # triclinic
        oracle.evaluate(model4(), pos, Z, bad)
    with pytest.raises(RuntimeError):  # coincident atoms
        oracle.evaluate(model4(), [[1, 1, 1], [1, 1, 1]], [8, 1], BOX30)
    # empty input
    o = oracle.evaluate(model4(), np.zeros((0, 3)), np.zeros(0, np.int32), BOX30)
    assert o["energy"] == 0.0 and o["forces"].shape == (0, 3)


# ------------------------------------------------------------------ link atoms (eq. 4)
def _link_case(pbc):
    rng = np.random.default_rng(17)
    n, L = 6, 12.0
    pos = rng.uniform(2.0, 10.0, size=(n, 3))
    if pbc:
        pos[4] = pos[1] + np.array([1.1, 0.4, -0.3]) + np.array([L, 0.0, -L])   # bonded MM partner in another image
    else:
        pos[4] = pos[1] + np.array([1.1, 0.4, -0.3])
    pos[5] = pos[2] + np.array([-0.7, 0.9, 0.6])
    link_ml, link_mm = np.array([1, 2], np.int32), np.array([4, 5], np.int32)
    box = np.diag([L, L, L]).astype(np.float32).reshape(9)
    ext = np.zeros((n + 2, 3), np.float32)
    ext[:n] = pos
    return n, ext, link_ml, link_mm, box


@pytest.mark.parametrize("pbc", [0, 1])
@pytest.mark.parametrize("d", [1.0, 0.73])
def test_link_atom_placement_eq4(pbc, d):
    """r_L lies on the (minimum-image) bond at distance d from the ML atom (eq. 4, written out here independently)."""
    n, ext, lm, lb, box = _link_case(pbc)
    oracle.link_place(ext, n, lm, lb, box, d, pbc)
    L = float(box[0])
    for q in range(2):
        ra, rb = ext[lm[q]].astype(np.float64), ext[lb[q]].astype(np.float64)
        v = rb - ra
        if pbc:
            v -= L * np.round(v / L)
        rl = ext[n + q].astype(np.float64)
        assert abs(np.linalg.norm(rl - ra) - d) < 2e-6
        assert np.linalg.norm(np.cross(rl - ra, v)) < 2e-6 * np.linalg.norm(v)      # collinear
        assert np.dot(rl - ra, v) > 0                                             # on the MM side
        np.testing.assert_allclose(rl, ra + d * v / np.linalg.norm(v), atol=2e-6)



def _sheared_link_case(seed):
    """A sheared GROMACS box (lower-triangular rows inside the shape limits), bonds of KNOWN direction v placed through
    a KNOWN integer combination k.H of box vectors: r_MM = r_ML + v + k.H.  Returns everything the known answer needs."""
    rng = np.random.default_rng(seed)
    H = np.array([[14.0, 0.0, 0.0], [rng.uniform(-6.5, 6.5), 13.0, 0.0],
                  [rng.uniform(-6.5, 6.5), rng.uniform(-6.0, 6.0), 12.0]])
    n, nl = 8, 3
    pos = rng.uniform(0.0, 12.0, size=(n, 3))
    lm, lb = np.array([0, 1, 2], np.int32), np.array([5, 6, 7], np.int32)
    vs, ks = [], []
    for q in range(nl):
        v = rng.normal(size=3)
        v *= rng.uniform(1.0, 1.6) / np.linalg.norm(v)          # a covalent bond length, far below half a box width
        k = rng.integers(-2, 3, size=3)
        pos[lb[q]] = pos[lm[q]] + v + k @ H
        vs.append(v); ks.append(k)
    ext = np.zeros((n + nl, 3), np.float32)
    ext[:n] = pos
    return n, ext, lm, lb, H, np.array(vs), np.array(ks)


@pytest.mark.parametrize("seed", [5, 6, 7])
@pytest.mark.parametrize("d", [1.0, 0.73])
def test_link_atom_placement_triclinic_known_answer(seed, d):
    """PAPER.md lines 79-82, eq. 4 in a SHEARED box (oracle link_bond(), the box[3] / box[6] / box[7] terms): the bonded MM
    partner sits in another periodic image, r_MM = r_ML + v + k.H with known v and integer k, so the known answer is
    r_L = r_ML + d v/|v| -- any other image choice moves r_L by whole box vectors.  Cross-check: the bond image the
    oracle took is the brute-force minimum over the 27 surrounding images of the row-reduced vector."""
    n, ext, lm, lb, H, vs, ks = _sheared_link_case(seed)
    box = H.astype(np.float32).reshape(9)
    assert np.any(ks != 0)
    oracle.link_place(ext, n, lm, lb, box, d, 1)
    Hf = box.reshape(3, 3).astype(np.float64)
    for q in range(len(lm)):
        ra, rb = ext[lm[q]].astype(np.float64), ext[lb[q]].astype(np.float64)
        rl = ext[n + q].astype(np.float64)
        want = ra + d * vs[q] / np.linalg.norm(vs[q])
        np.testing.assert_allclose(rl, want, atol=3e-6)          # fp32 storage of r_MM and r_L
        # brute force: the shortest of all images rb - ra + m.H, m in {-3..3}^3, is the bond the oracle used
        best = min((np.linalg.norm(rb - ra + np.array(m) @ Hf), m)
                   for m in [(a, b, c) for a in range(-3, 4) for b in range(-3, 4) for c in range(-3, 4)])
        np.testing.assert_allclose((rl - ra) / d, (rb - ra + np.array(best[1]) @ Hf) / best[0], atol=3e-6)


def test_link_force_spread_triclinic_conserves_force_and_is_chain_rule():
    """Force redistribution with the sheared-box bond: total force conserved and the shares are the chain rule of eq. 4
    written out with the KNOWN bond vector v (not the oracle's image search)."""
    d = 1.0
    n, ext, lm, lb, H, vs, ks = _sheared_link_case(9)
    box = H.astype(np.float32).reshape(9)
    oracle.link_place(ext, n, lm, lb, box, d, 1)
    rng = np.random.default_rng(2)
    F = rng.normal(size=(n + len(lm), 3))
    F0 = F.copy()
    oracle.link_spread(F, ext, n, lm, lb, box, d, 1)
    np.testing.assert_allclose(F.sum(axis=0), F0.sum(axis=0), atol=1e-12)
    assert np.all(F[n:] == 0.0)
    want = F0.copy()
    for q in range(len(lm)):
        l = np.linalg.norm(vs[q]); u = vs[q] / l
        perp = (d / l) * (F0[n + q] - u * np.dot(u, F0[n + q]))
        want[lm[q]] += F0[n + q] - perp
        want[lb[q]] += perp
        want[n + q] = 0.0
    np.testing.assert_allclose(F, want, atol=2e-6)               # v is known to fp32 rounding of the stored positions

@pytest.mark.parametrize("pbc", [0, 1])
def test_link_force_spread_conserves_force_and_torque(pbc):
    """Redistribution moves F_L onto the two bonded atoms without changing the total force; the total torque is
    conserved when taken with the link atom at r_L (minimum-image geometry)."""
    n, ext, lm, lb, box = _link_case(pbc)
    oracle.link_place(ext, n, lm, lb, box, 1.0, pbc)
    rng = np.random.default_rng(3)
    F0 = rng.normal(size=(n + 2, 3))
    F = F0.copy()
    oracle.link_spread(F, ext, n, lm, lb, box, 1.0, pbc)
    assert np.all(F[n:] == 0.0)
    np.testing.assert_allclose(F.sum(0), F0.sum(0), atol=1e-12)
    untouched = np.setdiff1d(np.arange(n), np.concatenate([lm, lb]))
    assert np.array_equal(F[untouched], F0[untouched])
    L = float(box[0])
    for q in range(2):
        ra = ext[lm[q]].astype(np.float64)
        v = ext[lb[q]].astype(np.float64) - ra
        if pbc:
            v -= L * np.round(v / L)
        rl = ext[n + q].astype(np.float64)
        dFa, dFb = F[lm[q]] - F0[lm[q]], F[lb[q]] - F0[lb[q]]
        # torque about the ML atom: only the MM share and the link force have a lever arm
        np.testing.assert_allclose(np.cross(v, dFb), np.cross(rl - ra, F0[n + q]), atol=2e-6)
        np.testing.assert_allclose(dFa + dFb, F0[n + q], atol=1e-12)


def test_link_force_spread_is_the_chain_rule_finite_differences():
    """For any scalar function phi(r_L), d phi / d r_a and d phi / d r_b through eq. 4 equal the spread of grad phi."""
    n, ext, lm, lb, box = _link_case(0)
    w = np.array([[0.3, -1.2, 0.7], [1.1, 0.5, -0.4]])

    def phi(p):
        e = np.zeros((n + 2, 3), np.float32)
        e[:n] = p
        oracle.link_place(e, n, lm, lb, box, 1.0, 0)
        rl = e[n:].astype(np.float64)
        return float(np.sum(np.sin(rl * w) + 0.1 * rl ** 2)), e

    p0 = ext[:n].astype(np.float64)
    _, e0 = phi(p0)
    rl = e0[n:].astype(np.float64)
    G = np.zeros((n + 2, 3))
    G[n:] = w * np.cos(rl * w) + 0.2 * rl          # d phi / d r_L, treated like a (negative) force on the link atoms
    oracle.link_spread(G, e0, n, lm, lb, box, 1.0, 0)
    h = 2e-3   # positions are fp32 inside the oracle: a larger step keeps the difference quotient clean
    for a in (int(lm[0]), int(lb[0]), int(lm[1]), int(lb[1])):
        for k in range(3):
            pp, pm = p0.copy(), p0.copy()
            pp[a, k] += h; pm[a, k] -= h
            fd = (phi(pp)[0] - phi(pm)[0]) / (2 * h)
            assert abs(fd - G[a, k]) < 2e-3 * (1 + abs(G[a, k])), (a, k, fd, G[a, k])


# ------------------------------------------------------------------ strain derivative / virial
def _fd_strain(model, pos64, Z, box, pbc, a, b, h):
    """Central finite difference of the oracle energy under r -> (1 + eps) r, box -> (1 + eps) box, eps = h e_a e_b^T."""
    out = []
    for sgn in (+1.0, -1.0):
        eps = np.eye(3)
        eps[a, b] += sgn * h
        p = (pos64 @ eps.T).astype(np.float32)
        bx = (np.asarray(box, np.float64).reshape(3, 3) @ eps.T).astype(np.float32).reshape(9) if pbc else box
        out.append(oracle.evaluate(model, p, Z, bx, pbc, None, want_forces=False)["energy"])
    return (out[0] - out[1]) / (2 * h)


def test_virial_is_the_strain_derivative_periodic_axes():
    cfg = get_config(0)
    m = oracle.Model(cfg["aev"], cfg["nets"], cfg["celu_alpha"])
    r = oracle.evaluate_virial(m, cfg["pos"], cfg["Z"], cfg["box"], 1)
    W = r["virial"]
    ref = oracle.evaluate(m, cfg["pos"], cfg["Z"], cfg["box"], 1)
    assert abs(r["energy"] - ref["energy"]) < 1e-12 and np.allclose(r["forces"], ref["forces"], atol=1e-12)
    assert np.abs(W - W.T).max() < 1e-8 * np.abs(W).max()          # rotation invariance of every E_i
    for a in range(3):                                             # axis scaling keeps the box orthorhombic
        fd = _fd_strain(m, cfg["pos64"], cfg["Z"], cfg["box"], 1, a, a, 2e-4)
        assert abs(fd - W[a, a]) < 2e-3 * (1 + abs(W[a, a])), (a, fd, W[a, a])


def test_virial_shear_and_force_moment_open_boundaries():
    cfg = get_config(4)
    ml = cfg["ml_index"]
    pos64 = cfg["pos64"][ml] - cfg["pos64"][ml].mean(0) + 20.0
    Z = cfg["Z"][ml]
    m = oracle.Model(cfg["aev"], cfg["nets"], cfg["celu_alpha"])
    r = oracle.evaluate_virial(m, pos64.astype(np.float32), Z, cfg["box"], 0)
    W, F = r["virial"], r["forces"]
    # isolated cluster: W = -sum_a F_a (x) r_a  (sum F = 0 makes it origin independent)
    M = -(F[:, :, None] * pos64.astype(np.float32).astype(np.float64)[:, None, :]).sum(0)
    assert np.abs(W - M).max() < 1e-8 * (1 + np.abs(W).max())
    for a, b in ((0, 1), (2, 0), (1, 2), (1, 1)):
        fd = _fd_strain(m, pos64, Z, cfg["box"], 0, a, b, 2e-4)
        assert abs(fd - W[a, b]) < 2e-3 * (1 + abs(W[a, b])), (a, b, fd, W[a, b])


# ------------------------------------------------------------------ triclinic boxes (reading #35)
def _tric_water(shear=(0.3, -0.2, 0.4), n=5, L=16.0, seed=41):
    """125 rigid waters in a sheared box; coordinates and box entries on a 1/1024 grid (exact in fp32, also after
    shifts by box vectors)."""
    from gen import water_box, sheared_water_box
    pos, Z, box, _ = water_box(n, n, n, L, seed)
    cfg = {"pos": pos, "box": box}
    p, H = sheared_water_box(cfg, *shear)
    q = lambda x: (np.round(np.asarray(x, np.float64) * 1024) / 1024)
    return q(p), Z, q(H).astype(np.float32)


def test_triclinic_minimum_image_is_the_brute_force_image_search():
    """The reduction + 27-image search of the oracle's disp() against the definition: a pair is a neighbour iff SOME lattice
    image lies within Rc (all 343 images n in {-3..3}^3 tried), on random boxes inside the GROMACS shape limits."""
    rng = np.random.default_rng(5)
    Rc = 5.2
    for trial in range(6):
        ax, by, cz = rng.uniform(11.0, 16.0, 3)
        bx, cx, cy = rng.uniform(-0.5, 0.5) * ax, rng.uniform(-0.5, 0.5) * ax, rng.uniform(-0.5, 0.5) * by
        H = np.array([[ax, 0, 0], [bx, by, 0], [cx, cy, cz]], dtype=np.float32)
        H64 = H.astype(np.float64)
        # Rc must not exceed half the smallest box width (distance between opposite faces)
        vol = abs(np.linalg.det(H64))
        widths = [vol / np.linalg.norm(np.cross(H64[(k + 1) % 3], H64[(k + 2) % 3])) for k in range(3)]
        if min(widths) < 2 * Rc + 0.2:
            continue
        n = 60
        pos = (rng.uniform(-0.5, 1.5, (n, 3)) @ H64).astype(np.float32)     # also outside the unit cell
        s, c = oracle.neighbors(pos, H.reshape(9), Rc)
        p64 = pos.astype(np.float64)
        imgs = np.array([[i, j, k] for i in range(-3, 4) for j in range(-3, 4) for k in range(-3, 4)], dtype=np.float64) @ H64
        ref_cols = []
        for i in range(n):
            d = p64[None, :, :] - p64[i][None, None, :] + imgs[:, None, :]
            near = ((d ** 2).sum(-1) <= Rc * Rc).any(0)
            near[i] = False
            ref_cols.append(np.nonzero(near)[0])
        assert np.array_equal(s, np.concatenate([[0], np.cumsum([len(r) for r in ref_cols])]))
        assert np.array_equal(c, np.concatenate(ref_cols))


def test_triclinic_invariances_and_finite_differences():
    pos, Z, H = _tric_water()
    cfg = get_config(0, bias_scale=0.1)
    model = oracle.Model(cfg["aev"], cfg["nets"])
    out = oracle.evaluate(model, pos, Z, H)
    F, scale = out["forces"], np.abs(out["forces"]).max()
    assert np.abs(F.sum(0)).max() < 1e-9 * scale
    # atoms moved by whole box vectors (any integer combination): same lists, same energy and forces
    rng = np.random.default_rng(9)
    n_int = rng.integers(-2, 3, size=pos.shape).astype(np.float64)
    pos2 = pos + n_int @ H.astype(np.float64).reshape(3, 3)
    assert np.array_equal(pos2, pos2.astype(np.float32).astype(np.float64))    # exact in fp32
    out2 = oracle.evaluate(model, pos2, Z, H)
    for Rc in (cfg["aev"]["Rcr"], cfg["aev"]["Rca"]):
        a, b = oracle.neighbors(pos, H, Rc), oracle.neighbors(pos2, H, Rc)
        assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])
    assert abs(out2["energy"] - out["energy"]) < 1e-9 * abs(out["energy"])
    assert np.abs(out2["forces"] - F).max() < 1e-9 * scale
    # rigid translation
    out3 = oracle.evaluate(model, pos + np.array([1.25, -2.5, 0.75]), Z, H)
    assert abs(out3["energy"] - out["energy"]) < 1e-9 * abs(out["energy"])
    # analytic forces against central differences
    atoms = [0, 1, 2, 200, 374]
    Ffd = fd_forces(model, pos, Z, H, 1, atoms, 2.0 ** -14)
    assert np.abs(F[atoms] - Ffd).max() < 5e-6 * scale
    # zero shear is the orthorhombic arithmetic, bit for bit
    H0 = np.diag(np.diag(H.reshape(3, 3))).astype(np.float32).reshape(9)
    a = oracle.evaluate(model, pos, Z, H0)
    H0b = H0.copy(); H0b[3] = 0.0
    assert oracle.evaluate(model, pos, Z, H0b)["energy"] == a["energy"]


def test_triclinic_box_shape_limits():
    pos, Z, H = _tric_water()
    cfg = get_config(0)
    model = oracle.Model(cfg["aev"], cfg["nets"])
    bad = H.copy(); bad[3] = 0.6 * H[0]          # |bx| > ax / 2
    with pytest.raises(RuntimeError):
        oracle.evaluate(model, pos, Z, bad)
    bad = H.copy(); bad[2] = 0.1                  # an upper-triangular entry
    with pytest.raises(RuntimeError):
        oracle.evaluate(model, pos, Z, bad)

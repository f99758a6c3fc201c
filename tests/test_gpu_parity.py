"""-m gpu: the CUDA path (through the C-ABI binding) against the fp64 CPU oracle on the same seeded inputs.

Bars (BASELINE.json north_star; SURVEY.md section 8.c reading #23):
  neighbour lists   bit-exact after canonical sort
  energy            |E_gpu - E_oracle| / n_ml <= 1e-4 eV/atom
  forces            RMS relative error <= 1e-3, max abs component error <= 5e-3 eV/Angstrom
  AEV (debug)       |dG| <= 2e-5 * (1 + |G|)   (fp32 arithmetic, ex2.approx, B^32 by squaring)
"""
import numpy as np
import pytest

import gen
import oracle

pytestmark = pytest.mark.gpu

E_TOL, F_RMS_TOL, F_MAX_TOL = 1e-4, 1e-3, 5e-3


def _torch():
    import torch
    return torch


def make(cfg, mode=None, max_atoms=None):
    import paper_2604_21441_b200 as nnp
    m = nnp.Model(cfg["aev"], cfg["nets"], cfg["celu_alpha"])
    n = cfg["pos"].shape[0] if max_atoms is None else max_atoms
    n_ml = n if cfg["ml_index"] is None else len(cfg["ml_index"])
    ws = nnp.Workspace(m, n, n_ml if max_atoms is None else max_atoms)
    if mode is not None:
        ws.set_mlp_mode(mode)
    return m, ws


def run_gpu(ws, pos, Z, box, pbc=1, ml=None):
    torch = _torch()
    dpos = torch.from_numpy(np.ascontiguousarray(pos, np.float32)).cuda()
    dZ = torch.from_numpy(np.ascontiguousarray(Z, np.int32)).cuda()
    dml = None if ml is None else torch.from_numpy(np.ascontiguousarray(ml, np.int32)).cuda()
    E, F = ws.eval(dpos, dZ, box, pbc, dml)
    torch.cuda.synchronize()
    st = ws.status()
    assert st == 0, f"nnp_status {st}"
    return float(E.cpu()[0]), F.cpu().numpy().astype(np.float64)


def check_EF(Eg, Fg, ref, n_ml, rows=None):
    Fo = ref["forces"]
    dE = abs(Eg - ref["energy"]) / max(n_ml, 1)
    if rows is not None:
        Fg, Fo = Fg[rows], Fo[rows]
    dF = Fg - Fo
    rms = np.sqrt((dF ** 2).sum() / max((Fo ** 2).sum(), 1e-300))
    mx = np.abs(dF).max() if dF.size else 0.0
    assert dE <= E_TOL, f"energy error {dE:.3e} eV/atom"
    assert rms <= F_RMS_TOL, f"force RMS rel {rms:.3e}"
    assert mx <= F_MAX_TOL, f"force max abs {mx:.3e}"
    return dE, rms, mx


def check_lists(ws, cfg, pos, n_ml, ml=None, pbc=1):
    for which, Rc in ((0, cfg["aev"]["Rcr"]), (1, cfg["aev"]["Rca"])):
        s_o, c_o = oracle.neighbors(pos, cfg["box"], Rc, pbc, ml, mode=1 if n_ml > 4000 else 0)
        s_g, c_g = ws.neighbors(which, n_ml)
        assert np.array_equal(s_o, s_g), f"row starts differ (which={which})"
        assert np.array_equal(c_o, c_g), f"columns differ (which={which})"


# ------------------------------------------------------------------ full configs
@pytest.mark.parametrize("k", [0, 1])
def test_config_small(k):
    cfg = gen.get_config(k)
    n = cfg["pos"].shape[0]
    om = oracle.Model(cfg["aev"], cfg["nets"], cfg["celu_alpha"])
    ref = oracle.evaluate(om, cfg["pos"], cfg["Z"], cfg["box"], 1, None, want_aev=True, want_atomic=True)
    m, ws = make(cfg)
    Eg, Fg = run_gpu(ws, cfg["pos"], cfg["Z"], cfg["box"])
    check_lists(ws, cfg, cfg["pos"], n)
    G = ws.aev(n).astype(np.float64)
    assert np.all(np.abs(G - ref["aev"]) <= 2e-5 * (1 + np.abs(ref["aev"]))), np.abs(G - ref["aev"]).max()
    ea = ws.atomic_energies(n).astype(np.float64)
    assert np.abs(ea - ref["e_atom"]).max() <= 1e-4
    check_EF(Eg, Fg, ref, n)
    assert abs(Fg.sum(0)).max() < 1e-3
    # every MLP arithmetic mode the library offers must meet the bar
    import paper_2604_21441_b200 as nnp
    for mode in (nnp.NNP_MLP_FP32_SIMT, nnp.NNP_MLP_F16X3, nnp.NNP_MLP_F16X1):
        if nnp.nnp_workspace_set_mlp_mode(ws.handle, mode) != 0:
            continue
        Eg2, Fg2 = run_gpu(ws, cfg["pos"], cfg["Z"], cfg["box"])
        check_EF(Eg2, Fg2, ref, n)


@pytest.mark.parametrize("k", [1, 4])
def test_mlp_stage_modes(k):
    """K5/K6 alone: per-atom energies and dE/dAEV of every MLP arithmetic mode against the oracle's fp64
    back-propagation, on the AEV columns the evaluation materialises (absent species' columns are never read).
    Bars: SIMT fp32 and F16X3 (fp16 hi/lo split, three MMAs) are fp32-grade; F16X1 (one fp16 product) sits at the
    2^-11 operand rounding level."""
    import paper_2604_21441_b200 as nnp
    cfg = gen.get_config(k)
    ml = cfg["ml_index"]
    n = cfg["pos"].shape[0]
    n_ml = n if ml is None else len(ml)
    om = oracle.Model(cfg["aev"], cfg["nets"], cfg["celu_alpha"])
    ref = oracle.evaluate(om, cfg["pos"], cfg["Z"], cfg["box"], 1, ml, want_aev=True, want_daev=True,
                          want_atomic=True, nbr_mode=1 if n_ml > 2000 else 0)
    live = np.abs(ref["aev"]).max(axis=0) > 0          # columns some atom populates
    m, ws = make(cfg)
    bars = {nnp.NNP_MLP_FP32_SIMT: (2e-6, 5e-5), nnp.NNP_MLP_F16X3: (5e-6, 5e-5), nnp.NNP_MLP_F16X1: (1e-3, 2e-3)}
    for dense in (0, 1):
        ws.set_dense_k(dense)
        for mode, (e_bar, d_bar) in bars.items():
            ws.set_mlp_mode(mode)
            Eg, Fg = run_gpu(ws, cfg["pos"], cfg["Z"], cfg["box"], 1, ml)
            ea = ws.atomic_energies(n_ml).astype(np.float64)
            D = ws.daev(n_ml).astype(np.float64)
            cols = slice(None) if dense else live
            rel = np.sqrt(((D[:, cols] - ref["daev"][:, cols]) ** 2).sum() / (ref["daev"][:, cols] ** 2).sum())
            assert np.abs(ea - ref["e_atom"]).max() <= e_bar, (mode, dense, np.abs(ea - ref["e_atom"]).max())
            assert rel <= d_bar, (mode, dense, rel)
            check_EF(Eg, Fg, ref, n_ml, rows=ml)


def test_config1_perturbed_steps():
    """cfg 1: positions perturbed by seeded N(0, 0.01 A) per step (reading #17): lists change every step."""
    cfg = gen.get_config(1)
    n = cfg["pos"].shape[0]
    P = gen.perturbed_positions(cfg["pos64"], cfg["perturb_seed"], 1000)   # the 1000-evaluation run of BASELINE.json configs[1]
    om = oracle.Model(cfg["aev"], cfg["nets"], cfg["celu_alpha"])
    m, ws = make(cfg)
    for t in (0, 1, 499, 999):                                               # parity on steps {0, 1, 499, 999}
        ref = oracle.evaluate(om, P[t], cfg["Z"], cfg["box"], 1, None, nbr_mode=1)
        Eg, Fg = run_gpu(ws, P[t], cfg["Z"], cfg["box"])
        check_lists(ws, cfg, P[t], n)
        check_EF(Eg, Fg, ref, n)


def test_config2_full_size():
    """cfg 2 (24 000 atoms, the bench workload): lists bit-exact, E and F against the oracle on every atom."""
    cfg = gen.get_config(2)
    n = cfg["pos"].shape[0]
    om = oracle.Model(cfg["aev"], cfg["nets"], cfg["celu_alpha"])
    ref = oracle.evaluate(om, cfg["pos"], cfg["Z"], cfg["box"], 1, None, nbr_mode=1, want_aev=True)
    m, ws = make(cfg)
    Eg, Fg = run_gpu(ws, cfg["pos"], cfg["Z"], cfg["box"])
    check_lists(ws, cfg, cfg["pos"], n)
    G = ws.aev(n).astype(np.float64)                    # every element of every row at headline size
    assert np.all(np.abs(G - ref["aev"]) <= 2e-5 * (1 + np.abs(ref["aev"]))), np.abs(G - ref["aev"]).max()
    check_EF(Eg, Fg, ref, n)
    # dense-K mode ("as ANI would run it") gives the same answer
    ws.set_dense_k(1)
    Eg2, Fg2 = run_gpu(ws, cfg["pos"], cfg["Z"], cfg["box"])
    check_EF(Eg2, Fg2, ref, n)


@pytest.mark.parametrize("n_sub", [8191, 8193, 8205])
def test_backward_block_shapes_around_the_threshold(n_sub):
    """k_aev_backward gives long blocks (two centres per warp) to the first 80 % of the grid from 8192 ML atoms on and
    one-centre blocks to the rest: ML subsets of cfg 2 just below / above the threshold, sizes that are no multiple of a
    block, with and without virial output (the other instantiation) -- E, F, virial against the oracle."""
    cfg = gen.get_config(2)
    n = cfg["pos"].shape[0]
    ml = np.sort(np.random.default_rng(n_sub).choice(n, size=n_sub, replace=False)).astype(np.int32)
    om = oracle.Model(cfg["aev"], cfg["nets"], cfg["celu_alpha"])
    ref = oracle.evaluate(om, cfg["pos"], cfg["Z"], cfg["box"], 1, ml, nbr_mode=1)
    m, ws = make(dict(cfg, ml_index=ml), max_atoms=n)
    Eg, Fg = run_gpu(ws, cfg["pos"], cfg["Z"], cfg["box"], 1, ml)
    check_EF(Eg, Fg, ref, n_sub, rows=ml)
    mm = np.setdiff1d(np.arange(n), ml)
    assert np.all(Fg[mm] == 0.0)
    torch = _torch()
    W = torch.zeros(9, dtype=torch.float64, device="cuda")
    ws.set_virial_output(W)
    Ev, Fv = run_gpu(ws, cfg["pos"], cfg["Z"], cfg["box"], 1, ml)
    assert Ev == Eg and np.array_equal(Fv, Fg)          # the virial instantiation: same forces, bit for bit
    ws.set_virial_output(None)


def test_config3_sampled():
    """cfg 3 (96 000 atoms): lists bit-exact; E/F checked on every atom with the oracle's cell-list mode."""
    cfg = gen.get_config(3)
    n = cfg["pos"].shape[0]
    om = oracle.Model(cfg["aev"], cfg["nets"], cfg["celu_alpha"])
    ref = oracle.evaluate(om, cfg["pos"], cfg["Z"], cfg["box"], 1, None, nbr_mode=1)
    m, ws = make(cfg)
    Eg, Fg = run_gpu(ws, cfg["pos"], cfg["Z"], cfg["box"])
    check_lists(ws, cfg, cfg["pos"], n)
    check_EF(Eg, Fg, ref, n)


@pytest.mark.parametrize("layout", ["A", "B"])
def test_config4_mlmm_subset(layout):
    cfg = gen.get_config(4, layout=layout)
    ml = cfg["ml_index"]
    om = oracle.Model(cfg["aev"], cfg["nets"], cfg["celu_alpha"])
    ref = oracle.evaluate(om, cfg["pos"], cfg["Z"], cfg["box"], 1, ml)
    m, ws = make(cfg)
    Eg, Fg = run_gpu(ws, cfg["pos"], cfg["Z"], cfg["box"], 1, ml)
    check_lists(ws, cfg, cfg["pos"], len(ml), ml)
    check_EF(Eg, Fg, ref, len(ml), rows=ml)
    mm = np.setdiff1d(np.arange(cfg["pos"].shape[0]), ml)
    assert np.all(Fg[mm] == 0.0) and not np.any(np.signbit(Fg[mm]))   # MM rows are +0.0f
    # MM independence: scrambling MM coordinates and atomic numbers changes nothing, bit for bit
    pos2, Z2 = cfg["pos"].copy(), cfg["Z"].copy()
    rng = np.random.default_rng(7)
    pos2[mm] += rng.normal(0, 1.0, size=(len(mm), 3)).astype(np.float32)
    Z2[mm] = 99
    Eg2, Fg2 = run_gpu(ws, pos2, Z2, cfg["box"], 1, ml)
    assert Eg2 == Eg and np.array_equal(Fg2, Fg)


# ------------------------------------------------------------------ edge and degenerate cases
def _small_cfg(bias_scale=0.0):
    return gen.get_config(0, bias_scale=bias_scale)


def test_bitwise_reproducible_and_host_entry():
    cfg = gen.get_config(1)
    m, ws = make(cfg)
    E1, F1 = run_gpu(ws, cfg["pos"], cfg["Z"], cfg["box"])
    E2, F2 = run_gpu(ws, cfg["pos"], cfg["Z"], cfg["box"])
    assert E1 == E2 and np.array_equal(F1, F2)
    E3, F3 = ws.eval_host(cfg["pos"], cfg["Z"], cfg["box"])
    assert ws.status() == 0
    assert E3 == E1 and np.array_equal(F3.astype(np.float64), F1)
    assert ws.launches() > 0


def test_host_entry_pinned_force_buffer():
    """A pinned force buffer is written by the output kernel itself, in the caller's order (no device-to-host copy): same
    bits as the copy path and the device entry point, on the cell-list path (cfg 1) and with an ML subset (copy path)."""
    torch = _torch()
    cfg = gen.get_config(1)
    n = cfg["pos"].shape[0]
    m, ws = make(cfg)
    E1, F1 = run_gpu(ws, cfg["pos"], cfg["Z"], cfg["box"])
    hF = torch.full((n, 3), float("nan"), dtype=torch.float32).pin_memory()
    nF = hF.numpy()
    for rep in range(2):
        E2, F2 = ws.eval_host(cfg["pos"], cfg["Z"], cfg["box"], 1, None, nF)
        assert ws.status() == 0
        assert F2 is nF and E2 == E1 and np.array_equal(nF.astype(np.float64), F1)
        nF[:] = np.nan
    E3, F3 = ws.eval_host(cfg["pos"], cfg["Z"], cfg["box"])          # pageable buffer: the copy path
    assert E3 == E1 and np.array_equal(F3.astype(np.float64), F1)
    ml = np.arange(0, n, 3, dtype=np.int32)                             # index subset: scattered rows, copy path
    m2, ws2 = make(dict(cfg, ml_index=ml), max_atoms=n)
    E4, F4 = run_gpu(ws2, cfg["pos"], cfg["Z"], cfg["box"], 1, ml)
    E5, F5 = ws2.eval_host(cfg["pos"], cfg["Z"], cfg["box"], 1, ml, nF)
    assert E5 == E4 and np.array_equal(nF.astype(np.float64), F4)


def test_host_entry_small_region_in_place():
    """cfg 4 (64 ML atoms of 9064) through nnp_eval_host with pinned buffers: the one-kernel path reads the positions from
    and writes the forces into the caller's buffers (no copies); same bits as the device entry point, rows of the other
    atoms +0.0f, twice in a row (the second call must clear what the first one left)."""
    torch = _torch()
    cfg = gen.get_config(4)
    n = cfg["pos"].shape[0]
    ml = cfg["ml_index"]
    m, ws = make(cfg)
    E1, F1 = run_gpu(ws, cfg["pos"], cfg["Z"], cfg["box"], 1, ml)
    assert ws.launches() == 1
    hP = torch.from_numpy(np.ascontiguousarray(cfg["pos"], np.float32)).pin_memory().numpy()
    hF = torch.full((n, 3), float("nan"), dtype=torch.float32).pin_memory().numpy()
    for rep in range(2):
        E2, F2 = ws.eval_host(hP, cfg["Z"], cfg["box"], 1, ml, hF)
        assert ws.status() == 0 and ws.launches() == 1
        assert E2 == E1 and np.array_equal(hF.astype(np.float64), F1)
        mm = np.setdiff1d(np.arange(n), ml)
        assert np.all(hF[mm] == 0.0) and not np.any(np.signbit(hF[mm]))
        hF[:] = np.nan


def test_nonzero_biases_and_padding_rows():
    """Non-zero biases make MLP(0) != 0: padded tile rows must not leak into E."""
    cfg = _small_cfg(bias_scale=0.3)
    om = oracle.Model(cfg["aev"], cfg["nets"], cfg["celu_alpha"])
    ref = oracle.evaluate(om, cfg["pos"], cfg["Z"], cfg["box"], 1, None)
    m, ws = make(cfg)
    Eg, Fg = run_gpu(ws, cfg["pos"], cfg["Z"], cfg["box"])
    check_EF(Eg, Fg, ref, cfg["pos"].shape[0])


def test_open_boundaries_cluster_and_orthorhombic_box():
    cfg = gen.get_config(4)
    ml = cfg["ml_index"]
    pos, Z = cfg["pos"][ml].copy(), cfg["Z"][ml].copy()
    om = oracle.Model(cfg["aev"], cfg["nets"], cfg["celu_alpha"])
    sub = dict(cfg, pos=pos, Z=Z, ml_index=None)
    m, ws = make(sub)
    ref = oracle.evaluate(om, pos, Z, cfg["box"], 0, None)
    Eg, Fg = run_gpu(ws, pos, Z, cfg["box"], 0)
    check_lists(ws, cfg, pos, len(pos), None, pbc=0)
    check_EF(Eg, Fg, ref, len(pos))
    # orthorhombic, non-cubic box; one dimension with fewer than three cells; atoms shifted by box vectors
    box = np.diag([17.0, 23.5, 12.0]).astype(np.float32).reshape(9)
    rng = np.random.default_rng(11)
    pos2 = (pos - pos.mean(0) + np.array([8.0, 11.0, 6.0])).astype(np.float32)
    shift = rng.integers(-2, 3, size=pos2.shape) * np.array([17.0, 23.5, 12.0])
    pos2 = (pos2 + shift).astype(np.float32)
    ref2 = oracle.evaluate(om, pos2, Z, box, 1, None)
    Eg2, Fg2 = run_gpu(ws, pos2, Z, box, 1)
    cfg2 = dict(cfg, box=box)
    check_lists(ws, cfg2, pos2, len(pos2))
    check_EF(Eg2, Fg2, ref2, len(pos2))


def test_dense_blob_many_angular_neighbours():
    """More than 32 angular neighbours per centre (far beyond liquid densities): exercises the backward kernel's
    general pair loop and rows close to the angular capacity.  40 atoms in a 2.8 A sphere, open boundaries."""
    rng = np.random.default_rng(5)
    pts = []
    while len(pts) < 40:
        p = rng.uniform(-2.8, 2.8, 3)
        if np.linalg.norm(p) <= 2.8 and all(np.linalg.norm(p - q) >= 0.75 for q in pts):
            pts.append(p)
    pos = (np.array(pts) + 20.0).astype(np.float32)
    Z = rng.choice([1, 6, 7, 8], size=40).astype(np.int32)
    cfg = gen.get_config(4)
    om = oracle.Model(cfg["aev"], cfg["nets"], cfg["celu_alpha"])
    sub = dict(cfg, pos=pos, Z=Z, ml_index=None)
    m, ws = make(sub)
    ref = oracle.evaluate(om, pos, Z, cfg["box"], 0, None)
    Eg, Fg = run_gpu(ws, pos, Z, cfg["box"], 0)
    sA, _ = ws.neighbors(1, 40)
    assert np.diff(sA).max() > 32, np.diff(sA).max()
    check_lists(ws, cfg, pos, 40, None, pbc=0)
    # all three bars.  (Forces here reach hundreds of eV/A -- 40 atoms 0.75 A apart -- so the absolute bar of 5e-3 eV/A
    # asks for ~1e-5 relative accuracy of the largest components: met by the fp32-grade default arithmetic.)
    check_EF(Eg, Fg, ref, 40)


def test_dense_blob_periodic_small_path():
    """The same blob in a periodic 24 A box: <= 256 atoms, so the one-kernel path takes it, whose team of warps handles at
    most 32 angular neighbours per centre and must hand centres beyond that to the general pair loop."""
    rng = np.random.default_rng(5)
    pts = []
    while len(pts) < 40:
        p = rng.uniform(-2.8, 2.8, 3)
        if np.linalg.norm(p) <= 2.8 and all(np.linalg.norm(p - q) >= 0.75 for q in pts):
            pts.append(p)
    pos = (np.array(pts) + 12.0).astype(np.float32)
    Z = rng.choice([1, 6, 7, 8], size=40).astype(np.int32)
    cfg = gen.get_config(4)
    box = np.diag([24.0, 24.0, 24.0]).astype(np.float32).reshape(9)
    om = oracle.Model(cfg["aev"], cfg["nets"], cfg["celu_alpha"])
    sub = dict(cfg, pos=pos, Z=Z, ml_index=None, box=box)
    m, ws = make(sub)
    ref = oracle.evaluate(om, pos, Z, box, 1, None)
    for on in (2, 1, 0):
        ws.set_small_path(on)
        Eg, Fg = run_gpu(ws, pos, Z, box, 1)
        if on == 2:
            assert ws.launches() == 1
        sA, _ = ws.neighbors(1, 40)
        assert np.diff(sA).max() > 32, np.diff(sA).max()
        check_lists(ws, sub, pos, 40, None, pbc=1)
        check_EF(Eg, Fg, ref, 40)


def test_one_layer_network_golden_monomer():
    """All-ones one-layer network on a water monomer: E = 7.1130060875."""
    import json, os
    gold = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "appendix_b.json")))
    aev = gen.aev_params(gen.weights.SPECIES_4)
    L = gen.aev_length(aev)
    nets = {Z: ((L, 1), [np.ones((1, L), np.float32)], [np.zeros(1, np.float32)]) for Z in (1, 6, 7, 8)}
    R, phi = 0.9572, np.deg2rad(104.52 / 2)
    O = np.array([10.0, 10.0, 10.0])
    pos = np.array([O, O + [R * np.sin(phi), 0, R * np.cos(phi)], O + [-R * np.sin(phi), 0, R * np.cos(phi)]], np.float32)
    Z = np.array([8, 1, 1], np.int32)
    box = np.diag([30.0] * 3).astype(np.float32).reshape(9)
    cfg = dict(aev=aev, nets=nets, celu_alpha=0.1, pos=pos, ml_index=None, box=box)
    m, ws = make(cfg)
    Eg, Fg = run_gpu(ws, pos, Z, box)
    key = [k for k in gold if "E" in k and "B2" in k]
    assert abs(Eg - 7.1130060875) < 2e-5, (Eg, key)
    assert abs(Fg[0, 2] + 0.98434044) < 2e-4 and abs(Fg[1, 0] - 2.68119284) < 2e-4
    assert abs(Fg.sum(0)).max() < 1e-5


def test_empty_and_single_atom():
    cfg = _small_cfg(bias_scale=0.2)
    om = oracle.Model(cfg["aev"], cfg["nets"], cfg["celu_alpha"])
    m, ws = make(cfg)
    torch = _torch()
    # n_atoms = 0
    E, F = ws.eval(torch.zeros((0, 3), dtype=torch.float32, device="cuda"),
                   torch.zeros((0,), dtype=torch.int32, device="cuda"), cfg["box"])
    torch.cuda.synchronize()
    assert ws.status() == 0 and float(E.cpu()[0]) == 0.0
    # one atom: E = MLP(0), F = 0
    pos, Z = cfg["pos"][:1], cfg["Z"][:1]
    ref = oracle.evaluate(om, pos, Z, cfg["box"], 1, None)
    Eg, Fg = run_gpu(ws, pos, Z, cfg["box"])
    assert abs(Eg - ref["energy"]) < 1e-5 and np.all(Fg == 0.0)
    # empty ML subset of a non-empty system
    ml = np.zeros((0,), np.int32)
    Eg, Fg = run_gpu(ws, cfg["pos"], cfg["Z"], cfg["box"], 1, ml)
    assert Eg == 0.0 and np.all(Fg == 0.0)


def test_error_reporting():
    import paper_2604_21441_b200 as nnp
    cfg = _small_cfg()
    m, ws = make(cfg)
    torch = _torch()
    dpos = torch.from_numpy(cfg["pos"]).cuda()
    dZ = torch.from_numpy(cfg["Z"]).cuda()
    bad_box = cfg["box"].copy(); bad_box[1] = 0.5
    with pytest.raises(nnp.NNPError) as e:
        ws.eval(dpos, dZ, bad_box)
    assert e.value.code == -3
    Zbad = cfg["Z"].copy(); Zbad[5] = 16   # sulfur: no slot in the 4-species model
    ws.eval(dpos, torch.from_numpy(Zbad).cuda(), cfg["box"])
    assert ws.status() == -2
    ml = torch.tensor([3, 2, 10], dtype=torch.int32, device="cuda")   # not ascending
    ws.eval(dpos, dZ, cfg["box"], 1, ml)
    assert ws.status() == -1
    pos2 = cfg["pos"].copy(); pos2[7] = pos2[3]
    ws.eval(torch.from_numpy(pos2).cuda(), dZ, cfg["box"])
    assert ws.status() == -5
    # too many atoms for the workspace
    big = torch.zeros((cfg["pos"].shape[0] + 1, 3), dtype=torch.float32, device="cuda")
    with pytest.raises(nnp.NNPError):
        ws.eval(big, torch.ones(big.shape[0], dtype=torch.int32, device="cuda"), cfg["box"])
    # the workspace still works afterwards
    om = oracle.Model(cfg["aev"], cfg["nets"], cfg["celu_alpha"])
    ref = oracle.evaluate(om, cfg["pos"], cfg["Z"], cfg["box"], 1, None)
    Eg, Fg = run_gpu(ws, cfg["pos"], cfg["Z"], cfg["box"])
    check_EF(Eg, Fg, ref, cfg["pos"].shape[0])


def test_capacity_overflow_is_reported_and_recovered_from():
    """150 atoms within 2.9 A of one point: every radial row (capacity 128), every angular row (48) and -- in a periodic box
    with a cell grid -- one cell's append buffer (96) overflow.  Every path must report NNP_ERR_CAPACITY (-4) instead of
    wrong numbers, and the workspace must evaluate correctly afterwards (the cell-list path by its general binning)."""
    rng = np.random.default_rng(11)
    pts = []
    while len(pts) < 150:
        p = rng.uniform(-2.9, 2.9, 3)
        if np.linalg.norm(p) <= 2.9 and all(np.linalg.norm(p - q) >= 0.7 for q in pts):
            pts.append(p)
    cfg = gen.get_config(4)
    box = np.diag([24.0, 24.0, 24.0]).astype(np.float32).reshape(9)
    pos = (np.array(pts) + 12.0).astype(np.float32)
    Z = rng.choice([1, 6, 7, 8], size=150).astype(np.int32)
    m, ws = make(dict(cfg, pos=pos, Z=Z, ml_index=None, box=box))
    torch = _torch()
    dpos, dZ = torch.from_numpy(pos).cuda(), torch.from_numpy(Z).cuda()
    for on, pbc in ((2, 1), (1, 1), (0, 1), (0, 0)):   # one kernel / small front end / cell list / open boundaries
        ws.set_small_path(on)
        ws.eval(dpos, dZ, box, pbc)
        assert ws.status() == -4, (on, pbc)
    # afterwards: the 40-atom blob of the tests above, on every path, against the oracle
    pos40, Z40 = pos[:40].copy(), Z[:40].copy()
    pos40 = (12.0 + (pos40 - 12.0) * 1.6).astype(np.float32)   # spread out: no row overflows any more
    om = oracle.Model(cfg["aev"], cfg["nets"], cfg["celu_alpha"])
    for on, pbc in ((2, 1), (1, 1), (0, 1), (0, 0)):
        ws.set_small_path(on)
        ref = oracle.evaluate(om, pos40, Z40, box, pbc, None)
        Eg, Fg = run_gpu(ws, pos40, Z40, box, pbc)
        check_EF(Eg, Fg, ref, 40)


# ------------------------------------------------------------------ link atoms (eq. 4)
@pytest.mark.parametrize("pbc", [0, 1])
def test_link_atoms_place_eval_spread(pbc):
    """ML/MM boundary cutting two bonds of the cfg-4 cluster: link atoms placed on the device (eq. 4), evaluated as
    regular ML hydrogens, their forces redistributed by the chain rule -- every step against the oracle, and the
    final forces against central finite differences of the oracle energy with respect to the REAL atoms."""
    torch = _torch()
    cfg = gen.get_config(4)
    ml_full = cfg["ml_index"]
    n = cfg["pos"].shape[0]
    box = cfg["box"]
    L = float(box[0])
    # ML region = the first 40 cluster atoms; the two bonds to atoms 40 and 41 of the chain are cut
    ml = ml_full[:40]
    bonded = []
    for b in (int(ml_full[40]), int(ml_full[41])):
        dv = cfg["pos"][ml].astype(np.float64) - cfg["pos"][b].astype(np.float64)
        dv -= L * np.round(dv / L)
        bonded.append(int(ml[np.argmin((dv ** 2).sum(1))]))
    link_ml = np.array(bonded, np.int32)
    link_mm = np.array([int(ml_full[40]), int(ml_full[41])], np.int32)
    pos_ext = np.zeros((n + 2, 3), np.float32)
    pos_ext[:n] = cfg["pos"]
    if pbc == 0:
        pos_ext[:n] -= L * np.floor(pos_ext[:n] / L)      # open boundaries: keep the cluster in one piece
    Z_ext = np.concatenate([cfg["Z"], np.array([1, 1], np.int32)])
    ml_ext = np.concatenate([ml, np.array([n, n + 1], np.int32)]).astype(np.int32)
    om = oracle.Model(cfg["aev"], cfg["nets"], cfg["celu_alpha"])
    # oracle chain
    p_or = pos_ext.copy()
    oracle.link_place(p_or, n, link_ml, link_mm, box, 1.0, pbc)
    ref = oracle.evaluate(om, p_or, Z_ext, box, pbc, ml_ext)
    F_or = ref["forces"].copy()
    oracle.link_spread(F_or, p_or, n, link_ml, link_mm, box, 1.0, pbc)
    # device chain
    m, ws = make(dict(cfg, pos=pos_ext, ml_index=ml_ext))
    dpos = torch.from_numpy(pos_ext).cuda(); dZ = torch.from_numpy(Z_ext).cuda(); dml = torch.from_numpy(ml_ext).cuda()
    dlm = torch.from_numpy(link_ml).cuda(); dlb = torch.from_numpy(link_mm).cuda()
    ws.link_place(dpos, n, dlm, dlb, box, 1.0, pbc)
    E, F = ws.eval(dpos, dZ, box, pbc, dml)
    ws.link_spread(F, dpos, n, dlm, dlb, box, 1.0, pbc)
    torch.cuda.synchronize()
    assert ws.status() == 0
    np.testing.assert_allclose(dpos.cpu().numpy()[n:], p_or[n:], atol=1e-6)           # placement
    Fg = F.cpu().numpy().astype(np.float64)
    assert np.all(Fg[n:] == 0.0)
    rows = np.concatenate([ml, link_mm])
    dF = Fg[rows] - F_or[rows]
    assert abs(float(E.cpu()[0]) - ref["energy"]) / len(ml_ext) <= E_TOL
    assert np.sqrt((dF ** 2).sum() / (F_or[rows] ** 2).sum()) <= F_RMS_TOL and np.abs(dF).max() <= F_MAX_TOL
    assert np.any(Fg[link_mm] != 0.0)                                                 # MM partners receive their share
    # finite differences of the oracle energy through the placement, with respect to a bonded ML and MM atom
    def energy(p):
        e = p.copy()
        oracle.link_place(e, n, link_ml, link_mm, box, 1.0, pbc)
        return oracle.evaluate(om, e, Z_ext, box, pbc, ml_ext, want_forces=False)["energy"]
    h = 1e-3
    for a in (int(link_ml[0]), int(link_mm[0])):
        for k in range(3):
            pp, pm = pos_ext.copy(), pos_ext.copy()
            pp[a, k] += h; pm[a, k] -= h
            fd = -(energy(pp) - energy(pm)) / float(pp[a, k] - pm[a, k])
            assert abs(fd - Fg[a, k]) <= 2e-2 * (1.0 + abs(fd)), (a, k, fd, Fg[a, k])


# ------------------------------------------------------------------ ensemble (ANI-2x = 8 networks)
@pytest.mark.parametrize("k,members", [(1, 3), (4, 8)])
def test_ensemble_mean_of_members(k, members):
    """E = mean over the members' energies (one AEV, `members` weight sets per element): against the mean of the
    oracle's single-network evaluations, in every MLP arithmetic mode."""
    import paper_2604_21441_b200 as nnp
    cfg = gen.get_config(k)
    ml = cfg["ml_index"]
    n = cfg["pos"].shape[0]
    n_ml = n if ml is None else len(ml)
    nets = []
    for mem in range(members):
        nets.append({Z: (d,) + gen.make_weights(40 + mem, Z, d, 0.1 if mem % 2 else 0.0) for Z, (d, _, _) in cfg["nets"].items()})
    E_or, F_or = 0.0, 0.0
    for mem in range(members):
        om = oracle.Model(cfg["aev"], nets[mem], cfg["celu_alpha"])
        r = oracle.evaluate(om, cfg["pos"], cfg["Z"], cfg["box"], 1, ml, nbr_mode=1 if n_ml > 2000 else 0)
        E_or += r["energy"] / members
        F_or = F_or + r["forces"] / members
    ref = dict(energy=E_or, forces=F_or)
    m = nnp.Model(cfg["aev"], nets, cfg["celu_alpha"])
    ws = nnp.Workspace(m, n, n_ml)
    for mode in (nnp.NNP_MLP_FP32_SIMT, nnp.NNP_MLP_F16X3, nnp.NNP_MLP_F16X1):
        ws.set_mlp_mode(mode)
        Eg, Fg = run_gpu(ws, cfg["pos"], cfg["Z"], cfg["box"], 1, ml)
        check_EF(Eg, Fg, ref, n_ml, rows=ml)
    E2, F2 = run_gpu(ws, cfg["pos"], cfg["Z"], cfg["box"], 1, ml)
    assert E2 == Eg and np.array_equal(F2, Fg)      # accumulation over members is reproducible


def test_cuda_graph_capture_and_replay():
    """nnp_eval allocates nothing and never synchronises: one evaluation (cooperative prep kernel included) can be
    captured into a CUDA graph and replayed with bitwise identical results (PAPER.md line 164 names CUDA graphs as the
    remedy for the launch-overhead plateau of small systems)."""
    torch = _torch()
    cfg = gen.get_config(0)
    n = cfg["pos"].shape[0]
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        import paper_2604_21441_b200 as nnp
        m = nnp.Model(cfg["aev"], cfg["nets"], cfg["celu_alpha"])
        ws = nnp.Workspace(m, n)
        dpos = torch.from_numpy(cfg["pos"]).cuda()
        dZ = torch.from_numpy(cfg["Z"]).cuda()
        E = torch.zeros(1, dtype=torch.float64, device="cuda")
        F = torch.zeros((n, 3), dtype=torch.float32, device="cuda")
        for _ in range(2):
            ws.eval(dpos, dZ, cfg["box"], 1, None, E, F)
        torch.cuda.synchronize()
        E0, F0 = E.clone(), F.clone()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            ws.eval(dpos, dZ, cfg["box"], 1, None, E, F)
        for _ in range(3):
            E.zero_(); F.zero_()
            g.replay()
        torch.cuda.synchronize()
        assert ws.status() == 0
        assert torch.equal(E, E0) and torch.equal(F, F0)


# ------------------------------------------------------------------ strain derivative / virial
@pytest.mark.parametrize("k", [0, 1, 4])
def test_virial_output(k):
    """dE/d eps from the force kernel's pair partials (fixed point) against the oracle's fp64 pair sum; switching the
    output on changes neither E nor F, and the result is bitwise reproducible."""
    torch = _torch()
    cfg = gen.get_config(k)
    ml = cfg["ml_index"]
    n = cfg["pos"].shape[0]
    n_ml = n if ml is None else len(ml)
    om = oracle.Model(cfg["aev"], cfg["nets"], cfg["celu_alpha"])
    ref = oracle.evaluate_virial(om, cfg["pos"], cfg["Z"], cfg["box"], 1, ml, nbr_mode=1 if n_ml > 2000 else 0)
    m, ws = make(cfg)
    ws.set_small_path(1)     # (the one-kernel small-system path has no virial output: keep one path for the bitwise comparison)
    E0, F0 = run_gpu(ws, cfg["pos"], cfg["Z"], cfg["box"], 1, ml)
    W = torch.zeros(9, dtype=torch.float64, device="cuda")
    ws.set_virial_output(W)
    E1, F1 = run_gpu(ws, cfg["pos"], cfg["Z"], cfg["box"], 1, ml)
    Wg = W.cpu().numpy().reshape(3, 3).copy()
    E2, F2 = run_gpu(ws, cfg["pos"], cfg["Z"], cfg["box"], 1, ml)
    assert E1 == E0 and np.array_equal(F1, F0)
    assert np.array_equal(W.cpu().numpy().reshape(3, 3), Wg)
    scale = np.abs(ref["virial"]).max()
    assert np.abs(Wg - ref["virial"]).max() <= 1e-3 * scale, (Wg, ref["virial"])     # same bar as the forces
    assert np.abs(Wg - Wg.T).max() <= 1e-3 * scale
    ws.set_virial_output(None)
    E3, F3 = run_gpu(ws, cfg["pos"], cfg["Z"], cfg["box"], 1, ml)
    assert E3 == E0 and np.array_equal(F3, F0)


def test_unit_conversion_nm_kjmol():
    """GROMACS units at the boundary: positions/box in nm, energies in kJ/mol, forces in kJ/mol/nm.  Reading #33: the
    conversion to Angstrom is one fp64 multiply rounded to fp32; the oracle is fed exactly those coordinates."""
    torch = _torch()
    cfg = gen.get_config(1)
    n = cfg["pos"].shape[0]
    pos_nm = (cfg["pos64"] / 10.0).astype(np.float32)
    box_nm = (cfg["box"].astype(np.float64) / 10.0).astype(np.float32)
    pos_a = (pos_nm.astype(np.float64) * 10.0).astype(np.float32)
    box_a = (box_nm.astype(np.float64) * 10.0).astype(np.float32)
    KJ = 96.48533212
    om = oracle.Model(cfg["aev"], cfg["nets"], cfg["celu_alpha"])
    ref = oracle.evaluate_virial(om, pos_a, cfg["Z"], box_a, 1, None, nbr_mode=1)
    m, ws = make(cfg)
    ws.set_units(10.0, KJ)
    W = torch.zeros(9, dtype=torch.float64, device="cuda")
    ws.set_virial_output(W)
    Eg, Fg = run_gpu(ws, pos_nm, cfg["Z"], box_nm)
    check_lists(ws, dict(cfg, box=box_a), pos_a, n)
    check_EF(Eg / KJ, Fg / (KJ * 10.0), ref, n)
    Wg = W.cpu().numpy().reshape(3, 3) / KJ
    assert np.abs(Wg - ref["virial"]).max() <= 1e-3 * np.abs(ref["virial"]).max()


# ------------------------------------------------------------------ external pair list
def _buffered_pairs(pos, box, pbc, atoms, cutoff, seed):
    """Candidate pairs as an MD engine's Verlet-buffered list would hold them: every unordered pair of `atoms` within
    `cutoff` under the minimum image (numpy fp64, all pairs), in shuffled order with random (i, j) orientation."""
    x = pos[atoms].astype(np.float64)
    d = x[None, :, :] - x[:, None, :]
    if pbc:
        L = np.array([box[0], box[4], box[8]], dtype=np.float64)
        d -= L * np.rint(d / L)
    r2 = (d ** 2).sum(-1)
    i, j = np.nonzero(np.triu(r2 <= cutoff * cutoff, k=1))
    rng = np.random.default_rng(seed)
    swap = rng.random(len(i)) < 0.5
    a, b = np.where(swap, j, i), np.where(swap, i, j)
    perm = rng.permutation(len(i))
    return np.stack([atoms[a[perm]], atoms[b[perm]]], axis=1).astype(np.int32)


@pytest.mark.parametrize("k,pbc", [(0, 1), (1, 1), (1, 0), (4, 1)])
def test_external_pair_list(k, pbc):
    """PAPER.md line 77 (2026 nnpot: the engine's pair list as a model input): with a buffered candidate list set, the
    neighbour rows are bit-identical to the oracle's lists and E, F meet the same bars as the built-in cell search."""
    torch = _torch()
    cfg = gen.get_config(k)
    ml = cfg["ml_index"]
    n = cfg["pos"].shape[0]
    n_ml = n if ml is None else len(ml)
    om = oracle.Model(cfg["aev"], cfg["nets"], cfg["celu_alpha"])
    ref = oracle.evaluate(om, cfg["pos"], cfg["Z"], cfg["box"], pbc, ml)
    if ml is None:
        atoms = np.arange(n)
    else:   # the engine's list also holds pairs with MM ends: they must be ignored
        mm = np.setdiff1d(np.arange(n), ml)
        atoms = np.sort(np.concatenate([ml, np.random.default_rng(5).choice(mm, 400, replace=False)]))
    pairs = _buffered_pairs(cfg["pos"], cfg["box"], pbc, atoms, cfg["aev"]["Rcr"] + 0.8, seed=11 + k)
    m, ws = make(cfg)
    E0, F0 = run_gpu(ws, cfg["pos"], cfg["Z"], cfg["box"], pbc, ml)        # built-in search
    dpairs = torch.from_numpy(pairs).cuda()
    ws.set_pair_list(dpairs)
    E1, F1 = run_gpu(ws, cfg["pos"], cfg["Z"], cfg["box"], pbc, ml)
    check_lists(ws, cfg, cfg["pos"], n_ml, ml, pbc)
    check_EF(E1, F1, ref, n_ml, rows=ml)
    assert abs(E1 - E0) / n_ml < 1e-6 and np.abs(F1 - F0).max() < 1e-4     # same rows, another summation order
    E2, F2 = run_gpu(ws, cfg["pos"], cfg["Z"], cfg["box"], pbc, ml)
    assert E2 == E1 and np.array_equal(F2, F1)                             # reproducible despite the atomic row fill
    # a pair listed twice is an argument error
    dd = cfg["pos"][pairs[:, 1]].astype(np.float64) - cfg["pos"][pairs[:, 0]].astype(np.float64)
    if pbc:
        Lb = np.array([cfg["box"][0], cfg["box"][4], cfg["box"][8]], dtype=np.float64)
        dd -= Lb * np.rint(dd / Lb)
    inside = np.nonzero(((dd ** 2).sum(1) < 9.0) & np.isin(pairs, atoms if ml is None else ml).all(1))[0][:1]
    ws.set_pair_list(torch.from_numpy(np.concatenate([pairs, pairs[inside, ::-1]]).copy()).cuda())
    ws.eval(torch.from_numpy(cfg["pos"]).cuda(), torch.from_numpy(cfg["Z"]).cuda(), cfg["box"], pbc,
            None if ml is None else torch.from_numpy(ml).cuda())
    assert ws.status() != 0
    ws.set_pair_list(None)
    E3, F3 = run_gpu(ws, cfg["pos"], cfg["Z"], cfg["box"], pbc, ml)
    assert E3 == E0 and np.array_equal(F3, F0)


# ------------------------------------------------------------------ small-system front end
@pytest.mark.parametrize("k,layout", [(0, "A"), (4, "A"), (4, "B")])
def test_small_path_and_general_path(k, layout):
    """<= 256 ML atoms in a periodic box take the single-kernel front end by default; the general cell-list path must
    give the same rows (bit-exact, both against the oracle) and the same E, F up to fp32 rounding of the positions' frame."""
    cfg = gen.get_config(k, layout=layout) if k == 4 else gen.get_config(k)
    ml = cfg["ml_index"]
    n = cfg["pos"].shape[0]
    n_ml = n if ml is None else len(ml)
    om = oracle.Model(cfg["aev"], cfg["nets"], cfg["celu_alpha"])
    ref = oracle.evaluate(om, cfg["pos"], cfg["Z"], cfg["box"], 1, ml, want_aev=True)
    m, ws = make(cfg)
    out = {}
    for on in (2, 1, 0):     # one kernel (default) / front end + four stage kernels / general cell-list path
        ws.set_small_path(on)
        E, F = run_gpu(ws, cfg["pos"], cfg["Z"], cfg["box"], 1, ml)
        assert ws.launches() == {2: 1, 1: 5}.get(on, ws.launches()) and ws.launches() in (1, 5, 7, 8)
        check_lists(ws, cfg, cfg["pos"], n_ml, ml)
        G = ws.aev(n_ml).astype(np.float64)
        assert np.all(np.abs(G - ref["aev"]) <= 2e-5 * (1 + np.abs(ref["aev"]))), np.abs(G - ref["aev"]).max()
        check_EF(E, F, ref, n_ml, rows=ml)
        E2, F2 = run_gpu(ws, cfg["pos"], cfg["Z"], cfg["box"], 1, ml)
        assert E2 == E and np.array_equal(F2, F)
        out[on] = (E, F)
    for on in (2, 1):
        assert abs(out[on][0] - out[0][0]) / n_ml < 1e-6 and np.abs(out[on][1] - out[0][1]).max() < 1e-4
    mm = None if ml is None else np.setdiff1d(np.arange(n), ml)
    if mm is not None:   # the single kernel writes the other atoms' rows itself: +0.0f
        assert np.all(out[2][1][mm] == 0.0) and not np.any(np.signbit(out[2][1][mm]))
    # atoms shifted by whole box vectors: same rows
    ws.set_small_path(2)
    shift = np.random.default_rng(3).integers(-2, 3, size=cfg["pos"].shape).astype(np.float32)
    pos2 = (cfg["pos"] + shift * np.array([cfg["box"][0], cfg["box"][4], cfg["box"][8]], dtype=np.float32)).astype(np.float32)
    ref2 = oracle.evaluate(om, pos2, cfg["Z"], cfg["box"], 1, ml)
    E3, F3 = run_gpu(ws, pos2, cfg["Z"], cfg["box"], 1, ml)
    check_lists(ws, cfg, pos2, n_ml, ml)
    check_EF(E3, F3, ref2, n_ml, rows=ml)


@pytest.mark.parametrize("n_sub", [1, 2, 3, 5, 17, 33, 100, 255, 256])
def test_small_path_subset_sizes(n_sub):
    """The one-kernel path deals a centre's triplet chunks, pair rounds and radial passes over a team of eight warps and the
    species groups over CTAs in chunks of two: ML subsets of odd sizes (one atom, groups of one, the 256-atom limit), half of
    them a compact ball (full rows, up to ~20 angular neighbours) and half scattered atoms (empty and one-entry rows), must
    give the oracle's rows, E and F, and what the general path gives."""
    cfg = gen.get_config(4)
    n = cfg["pos"].shape[0]
    rng = np.random.default_rng(1000 + n_sub)
    L = np.array([cfg["box"][0], cfg["box"][4], cfg["box"][8]], dtype=np.float64)
    if n_sub % 2:   # the n_sub atoms nearest to a random atom (minimum image)
        d = cfg["pos64"] - cfg["pos64"][rng.integers(n)]
        d -= L * np.rint(d / L)
        ml = np.sort(np.argsort((d * d).sum(1), kind="stable")[:n_sub]).astype(np.int32)
    else:
        ml = np.sort(rng.choice(n, size=n_sub, replace=False)).astype(np.int32)
    om = oracle.Model(cfg["aev"], cfg["nets"], cfg["celu_alpha"])
    ref = oracle.evaluate(om, cfg["pos"], cfg["Z"], cfg["box"], 1, ml)
    m, ws = make(cfg, max_atoms=n)
    out = {}
    for on in (2, 0):
        ws.set_small_path(on)
        E, F = run_gpu(ws, cfg["pos"], cfg["Z"], cfg["box"], 1, ml)
        if on == 2:
            assert ws.launches() == 1
        check_lists(ws, cfg, cfg["pos"], n_sub, ml)
        check_EF(E, F, ref, n_sub, rows=ml)
        E2, F2 = run_gpu(ws, cfg["pos"], cfg["Z"], cfg["box"], 1, ml)
        assert E2 == E and np.array_equal(F2, F)
        out[on] = (E, F)
    assert abs(out[2][0] - out[0][0]) / n_sub < 1e-6 and np.abs(out[2][1] - out[0][1]).max() < 1e-4


# ------------------------------------------------------------------ triclinic boxes (reading #35)
@pytest.mark.parametrize("shear", [(0.3, -0.2, 0.4), (-0.5, 0.5, -0.5), (0.0, 0.0, 0.25)])
def test_triclinic_box(shear):
    """GROMACS lower-triangular box: cfg 1's waters at the same fractional positions of a sheared box.  Lists bit-exact,
    E and F within the bars, against the oracle (whose triclinic minimum image is pinned to a brute-force image search)."""
    import paper_2604_21441_b200 as nnp
    torch = _torch()
    cfg = gen.get_config(1)
    pos, H = gen.sheared_water_box(cfg, *shear)
    n = pos.shape[0]
    om = oracle.Model(cfg["aev"], cfg["nets"], cfg["celu_alpha"])
    ref = oracle.evaluate(om, pos, cfg["Z"], H, 1, None, want_aev=True)
    tcfg = dict(cfg); tcfg["box"] = H
    m, ws = make(cfg)
    E, F = run_gpu(ws, pos, cfg["Z"], H)
    check_lists(ws, tcfg, pos, n)
    G = ws.aev(n).astype(np.float64)
    assert np.all(np.abs(G - ref["aev"]) <= 2e-5 * (1 + np.abs(ref["aev"]))), np.abs(G - ref["aev"]).max()
    check_EF(E, F, ref, n)
    assert abs(F.sum(0)).max() < 1e-3
    # atoms moved by whole box vectors: same rows, same results within fp32 rounding of the inputs
    k = np.random.default_rng(4).integers(-2, 3, size=pos.shape).astype(np.float64)
    pos2 = (pos.astype(np.float64) + k @ H.astype(np.float64).reshape(3, 3)).astype(np.float32)
    ref2 = oracle.evaluate(om, pos2, cfg["Z"], H)
    E2, F2 = run_gpu(ws, pos2, cfg["Z"], H)
    check_lists(ws, tcfg, pos2, n)
    check_EF(E2, F2, ref2, n)
    # the engine's pair list in a triclinic box (candidates from the oracle's own buffered list)
    s_o, c_o = oracle.neighbors(pos, H, cfg["aev"]["Rcr"] + 0.5)
    rows = np.repeat(np.arange(n), np.diff(s_o))
    keep = rows < c_o
    pairs = np.stack([rows[keep], c_o[keep]], 1).astype(np.int32)
    ws.set_pair_list(torch.from_numpy(pairs).cuda())
    E3, F3 = run_gpu(ws, pos, cfg["Z"], H)
    check_lists(ws, tcfg, pos, n)
    check_EF(E3, F3, ref, n)
    ws.set_pair_list(None)
    # virial against the oracle's strain derivative
    W = torch.zeros(9, dtype=torch.float64, device="cuda")
    ws.set_virial_output(W)
    run_gpu(ws, pos, cfg["Z"], H)
    Wo = np.asarray(oracle.evaluate_virial(om, pos, cfg["Z"], H)["virial"]).reshape(9)
    assert np.abs(W.cpu().numpy() - Wo).max() <= 1e-3 * np.abs(Wo).max()
    ws.set_virial_output(None)


def test_triclinic_box_limits():
    import paper_2604_21441_b200 as nnp
    torch = _torch()
    cfg = gen.get_config(1)
    pos, H = gen.sheared_water_box(cfg, 0.3, -0.2, 0.4)
    m, ws = make(cfg)
    dpos, dZ = torch.from_numpy(pos).cuda(), torch.from_numpy(cfg["Z"]).cuda()
    bad = H.copy(); bad[3] = 0.6 * H[0]                       # |bx| > ax / 2
    with pytest.raises(nnp.NNPError) as e:
        ws.eval(dpos, dZ, bad, 1)
    assert e.value.code == -3
    bad = H.copy(); bad[1] = 0.5                              # not lower-triangular
    with pytest.raises(nnp.NNPError):
        ws.eval(dpos, dZ, bad, 1)
    small = (H * 0.45).astype(np.float32)                     # < 3 cut-off wide cells between the faces
    with pytest.raises(nnp.NNPError) as e:
        ws.eval(dpos, dZ, small, 1)
    assert e.value.code == -3


def test_link_atoms_triclinic_box():
    """Link-atom placement and force spread with bonds crossing the faces of a sheared box, against the oracle."""
    torch = _torch()
    cfg = gen.get_config(1)
    pos, H = gen.sheared_water_box(cfg, 0.3, -0.2, 0.4)
    H64 = H.astype(np.float64).reshape(3, 3)
    n, nl = 60, 12
    rng = np.random.default_rng(21)
    p = pos[:n].astype(np.float64)
    lm = rng.choice(n, nl, replace=False).astype(np.int32)
    lb = rng.choice(np.setdiff1d(np.arange(n), lm), nl, replace=False).astype(np.int32)   # distinct partners, none of them an ML end
    vs = []
    for a, b in zip(lm, lb):     # MM partner 1.2-1.6 A from the ML atom along a KNOWN v, then moved to another periodic image
        v = rng.normal(size=3); v *= rng.uniform(1.2, 1.6) / np.linalg.norm(v)
        p[b] = p[a] + v + rng.integers(-1, 2, 3) @ H64
        vs.append(v)
    vs = np.array(vs)
    pos_ext = np.concatenate([p, np.zeros((nl, 3))]).astype(np.float32)
    ref_pos = pos_ext.copy()
    oracle.link_place(ref_pos, n, lm, lb, H, d=1.0, pbc=1)
    cfg4 = gen.get_config(0)
    m, ws = make(cfg4, max_atoms=n + nl)
    dpos = torch.from_numpy(pos_ext).cuda()
    dlm, dlb = torch.from_numpy(lm).cuda(), torch.from_numpy(lb).cuda()
    ws.link_place(dpos, n, dlm, dlb, H, d=1.0, pbc=1)
    torch.cuda.synchronize()
    got = dpos.cpu().numpy()
    assert np.abs(got - ref_pos).max() < 1e-5
    # known answer (eq. 4): r_L = r_ML + d v/|v| -- a wrong image of the bond would be off by whole box vectors
    want = got[lm].astype(np.float64) + vs / np.linalg.norm(vs, axis=1)[:, None]
    assert np.abs(got[n:] - want).max() < 1e-5
    F = rng.normal(size=(n + nl, 3)).astype(np.float32)
    refF = F.astype(np.float64)
    oracle.link_spread(refF, ref_pos, n, lm, lb, H, d=1.0, pbc=1)
    dF = torch.from_numpy(F.copy()).cuda()
    ws.link_spread(dF, dpos, n, dlm, dlb, H, d=1.0, pbc=1)
    torch.cuda.synchronize()
    assert np.abs(dF.cpu().numpy() - refF).max() < 1e-5
    assert np.all(dF.cpu().numpy()[n:] == 0.0)


@pytest.mark.parametrize("n_sub", [90, 600])
def test_triclinic_box_ml_subset(n_sub):
    """An index-listed ML subset in a sheared box (90 ML atoms would take the small-system front end in an orthorhombic
    box; a triclinic evaluation must fall back to the cell-list path), MM rows +0.0f."""
    cfg = gen.get_config(1)
    pos, H = gen.sheared_water_box(cfg, -0.4, 0.3, 0.2)
    n = pos.shape[0]
    ml = np.sort(np.random.default_rng(8).choice(n // 3, n_sub // 3, replace=False))
    ml = (3 * ml[:, None] + np.arange(3)[None, :]).reshape(-1).astype(np.int32)     # whole molecules
    om = oracle.Model(cfg["aev"], cfg["nets"], cfg["celu_alpha"])
    ref = oracle.evaluate(om, pos, cfg["Z"], H, 1, ml)
    tcfg = dict(cfg); tcfg["box"] = H; tcfg["ml_index"] = ml
    m, ws = make(tcfg)
    E, F = run_gpu(ws, pos, cfg["Z"], H, 1, ml)
    assert ws.launches() in (7, 8)   # never the small-system front end (5)
    check_lists(ws, tcfg, pos, len(ml), ml)
    check_EF(E, F, ref, len(ml), rows=ml)
    mm = np.setdiff1d(np.arange(n), ml)
    assert np.all(F[mm] == 0.0) and not np.any(np.signbit(F[mm]))


def test_two_workspaces_on_two_streams():
    """Two workspaces of one model on two CUDA streams, evaluations interleaved without synchronisation in between:
    every result bitwise equal to the same evaluation run alone (the launch chain, tile flags and scratch are per
    workspace)."""
    torch = _torch()
    import paper_2604_21441_b200 as nnp
    cfg = gen.get_config(1)
    n = cfg["pos"].shape[0]
    P = gen.perturbed_positions(cfg["pos64"], cfg["perturb_seed"], 4)
    m = nnp.Model(cfg["aev"], cfg["nets"], cfg["celu_alpha"])
    dZ = torch.from_numpy(cfg["Z"]).cuda()
    dpos = [torch.from_numpy(P[t]).cuda() for t in range(4)]
    ws0 = nnp.Workspace(m, n)
    alone = []
    for t in range(4):
        E, F = ws0.eval(dpos[t], dZ, cfg["box"], 1)
        torch.cuda.synchronize()
        alone.append((float(E.cpu()[0]), F.cpu().numpy().copy()))
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    torch.cuda.synchronize()
    with torch.cuda.stream(s1):
        w1 = nnp.Workspace(m, n)
    with torch.cuda.stream(s2):
        w2 = nnp.Workspace(m, n)
    outs = []
    for rep in range(3):
        for t in range(4):
            ws, st = (w1, s1) if t % 2 == 0 else (w2, s2)
            with torch.cuda.stream(st):
                E = torch.empty(1, dtype=torch.float64, device="cuda")
                F = torch.empty((n, 3), dtype=torch.float32, device="cuda")
                ws.eval(dpos[t], dZ, cfg["box"], 1, None, E, F)
                outs.append((t, E, F))
    torch.cuda.synchronize()
    assert w1.status() == 0 and w2.status() == 0
    for t, E, F in outs:
        assert float(E.cpu()[0]) == alone[t][0] and np.array_equal(F.cpu().numpy(), alone[t][1])


def test_bin_reuse_over_md_like_steps():
    """SURVEY.md section 8.f item 4 (Verlet-buffered reuse): the cell binning is reused for 4 of every 5 evaluations while
    the atoms jitter; rows stay bit-exact against the oracle and E, F inside the bars on every step; an atom that leaves
    its cell by more than skin / 2 on a reuse step is reported (NNP_ERR_STALE) and the next evaluation recovers."""
    torch = _torch()
    cfg = gen.get_config(1)
    n = cfg["pos"].shape[0]
    P = gen.perturbed_positions(cfg["pos64"], cfg["perturb_seed"], 12, sigma=0.05)
    om = oracle.Model(cfg["aev"], cfg["nets"], cfg["celu_alpha"])
    m, ws = make(cfg)
    ws.set_bin_reuse(5, 1.0)
    dZ = torch.from_numpy(cfg["Z"]).cuda()     # the same device buffers on every step, as an MD engine would pass them
    dpos = torch.empty((n, 3), dtype=torch.float32, device="cuda")
    for t in range(12):                        # full builds at steps 0, 5, 10; the other nine reuse binning AND rows
        dpos.copy_(torch.from_numpy(P[t]))
        E, F = ws.eval(dpos, dZ, cfg["box"], 1)
        torch.cuda.synchronize()
        assert ws.status() == 0
        # a reuse step runs no cell sweep: k_refresh + k_rows_from_wide in place of k_bin_cells + k_cell_sort + k_neighbors
        assert ws.launches() == (8 if t % 5 == 0 else 7), (t, ws.launches())
        ref = oracle.evaluate(om, P[t], cfg["Z"], cfg["box"], 1, None, nbr_mode=1)
        check_lists(ws, cfg, P[t], n)
        check_EF(float(E.cpu()[0]), F.cpu().numpy().astype(np.float64), ref, n)
    # step 12 is a reuse step (full builds at steps 0, 5, 10): push one atom far out of its cell
    bad = P[0].copy(); bad[17] += np.float32(8.0)      # farther than a cell edge + skin / 2
    dpos.copy_(torch.from_numpy(bad))
    ws.eval(dpos, dZ, cfg["box"], 1)
    assert ws.status() == -8
    E, F = ws.eval(dpos, dZ, cfg["box"], 1)    # rebuilds
    torch.cuda.synchronize()
    assert ws.status() == 0
    ref = oracle.evaluate(om, bad, cfg["Z"], cfg["box"], 1, None, nbr_mode=1)
    check_lists(ws, cfg, bad, n)
    check_EF(float(E.cpu()[0]), F.cpu().numpy().astype(np.float64), ref, n)
    # switched off: plain evaluations again, bitwise equal to a fresh workspace
    ws.set_bin_reuse(0)
    E1, F1 = run_gpu(ws, P[3], cfg["Z"], cfg["box"])
    m2, ws2 = make(cfg)
    E2, F2 = run_gpu(ws2, P[3], cfg["Z"], cfg["box"])
    assert E1 == E2 and np.array_equal(F1, F2)


def test_host_entry_pinned_buffers_with_reuse_and_changing_sizes():
    """The output kernel writes a pinned force buffer in the caller's order through the inverse map of the LAST cell sort:
    reuse steps (no sort) must still use the right map, and a later call with fewer atoms on the same workspace a new one.
    Device entry point on a second workspace = the reference bits."""
    torch = _torch()
    cfg = gen.get_config(1)
    n = cfg["pos"].shape[0]
    P = gen.perturbed_positions(cfg["pos64"], cfg["perturb_seed"], 7, sigma=0.05)
    m, ws = make(cfg)
    m2, ws2 = make(cfg)
    ws.set_bin_reuse(5, 1.0)
    ws2.set_bin_reuse(5, 1.0)
    hP = torch.empty((n, 3), dtype=torch.float32).pin_memory().numpy()
    hF = torch.empty((n, 3), dtype=torch.float32).pin_memory().numpy()
    dZ = torch.from_numpy(cfg["Z"]).cuda()
    dpos = torch.empty((n, 3), dtype=torch.float32, device="cuda")
    for t in range(7):
        hP[:] = P[t]
        hF[:] = np.nan
        E, F = ws.eval_host(hP, cfg["Z"], cfg["box"], 1, None, hF)
        assert ws.status() == 0 and ws.launches() == (8 if t % 5 == 0 else 7)
        dpos.copy_(torch.from_numpy(P[t]))
        E2, F2 = ws2.eval(dpos, dZ, cfg["box"], 1)
        torch.cuda.synchronize()
        assert ws2.status() == 0
        assert E == float(E2.cpu()[0]) and np.array_equal(hF, F2.cpu().numpy()), t
    # fewer atoms (the first 800 waters; same box: a thinner liquid) on the same workspace and the same pinned buffers
    ws.set_bin_reuse(0)
    k = 2400
    pos_k, Z_k = np.ascontiguousarray(P[0][:k]), np.ascontiguousarray(cfg["Z"][:k])
    hP[:k] = pos_k
    hF[:] = np.nan
    E, F = ws.eval_host(hP[:k], Z_k, cfg["box"], 1, None, hF[:k])
    assert ws.status() == 0
    m3, ws3 = make(dict(cfg, pos=pos_k, Z=Z_k))
    E3, F3 = run_gpu(ws3, pos_k, Z_k, cfg["box"])
    assert E == E3 and np.array_equal(hF[:k].astype(np.float64), F3) and np.all(np.isnan(hF[k:]))


def test_host_entry_pinned_buffers_on_the_other_paths():
    """Pinned host buffers where the binning kernel does NOT do the upload itself and the output kernel does not write in
    place: open boundaries (general binning), unit conversion (positions are scaled first), an external pair list.  The
    pending upload must become a copy on each of them: same bits as the device entry point."""
    torch = _torch()
    cfg = gen.get_config(1)
    n = cfg["pos"].shape[0]
    hP = torch.from_numpy(np.ascontiguousarray(cfg["pos"], np.float32)).pin_memory().numpy()
    hF = torch.empty((n, 3), dtype=torch.float32).pin_memory().numpy()
    m, ws = make(cfg)
    # open boundaries
    E0, F0 = run_gpu(ws, cfg["pos"], cfg["Z"], cfg["box"], 0)
    hF[:] = np.nan
    E1, _ = ws.eval_host(hP, cfg["Z"], cfg["box"], 0, None, hF)
    assert ws.status() == 0 and E1 == E0 and np.array_equal(hF.astype(np.float64), F0)
    # nm / kJ/mol
    ws.set_units(10.0, 96.485)
    pos_nm = (cfg["pos"] / 10.0).astype(np.float32)
    box_nm = (cfg["box"] / 10.0).astype(np.float32)
    E0, F0 = run_gpu(ws, pos_nm, cfg["Z"], box_nm, 1)
    hP[:] = pos_nm
    hF[:] = np.nan
    E1, _ = ws.eval_host(hP, cfg["Z"], box_nm, 1, None, hF)
    assert ws.status() == 0 and E1 == E0 and np.array_equal(hF.astype(np.float64), F0)
    ws.set_units(1.0, 1.0)
    # periodic again, the in-place path, after the others
    hP[:] = cfg["pos"]
    E0, F0 = run_gpu(ws, cfg["pos"], cfg["Z"], cfg["box"], 1)
    hF[:] = np.nan
    E1, _ = ws.eval_host(hP, cfg["Z"], cfg["box"], 1, None, hF)
    assert ws.status() == 0 and E1 == E0 and np.array_equal(hF.astype(np.float64), F0)


def test_bin_reuse_triclinic():
    torch = _torch()
    cfg = gen.get_config(1)
    pos0, H = gen.sheared_water_box(cfg, 0.3, -0.2, 0.4)
    n = pos0.shape[0]
    tcfg = dict(cfg); tcfg["box"] = H
    om = oracle.Model(cfg["aev"], cfg["nets"], cfg["celu_alpha"])
    rng = np.random.default_rng(14)
    m, ws = make(cfg)
    ws.set_bin_reuse(4, 1.0)
    dZ = torch.from_numpy(cfg["Z"]).cuda()
    dpos = torch.empty((n, 3), dtype=torch.float32, device="cuda")
    for t in range(5):
        pos = (pos0 + rng.normal(0, 0.05, size=pos0.shape)).astype(np.float32)
        if t == 2:      # whole-box-vector shifts on a reuse step: the nearest image of the stored cell is taken
            pos = (pos.astype(np.float64) + rng.integers(-1, 2, size=pos.shape) @ H.astype(np.float64).reshape(3, 3)).astype(np.float32)
        dpos.copy_(torch.from_numpy(pos))
        E, F = ws.eval(dpos, dZ, H, 1)
        torch.cuda.synchronize()
        assert ws.status() == 0
        ref = oracle.evaluate(om, pos, cfg["Z"], H)
        check_lists(ws, tcfg, pos, n)
        check_EF(float(E.cpu()[0]), F.cpu().numpy().astype(np.float64), ref, n)
    bad = pos0.copy(); bad[40] += np.float32(9.0)      # farther than a cell edge + skin / 2 along z
    dpos.copy_(torch.from_numpy(bad))
    ws.eval(dpos, dZ, H, 1)       # step 5 is a reuse step (full binnings at 0 and 4)
    assert ws.status() == -8


def test_bin_reuse_with_ml_subset_and_pair_list():
    """Binning reuse on the cell-list path with an index-listed ML subset (cfg 4, small-system front end off), with and
    without the engine's pair list: every step against the oracle."""
    torch = _torch()
    cfg = gen.get_config(4)
    ml = cfg["ml_index"]
    n = cfg["pos"].shape[0]
    om = oracle.Model(cfg["aev"], cfg["nets"], cfg["celu_alpha"])
    rng = np.random.default_rng(12)
    m, ws = make(cfg)
    ws.set_small_path(0)
    ws.set_bin_reuse(4, 0.8)
    dZ = torch.from_numpy(cfg["Z"]).cuda()
    dml = torch.from_numpy(ml).cuda()
    dpos = torch.empty((n, 3), dtype=torch.float32, device="cuda")
    pairs = _buffered_pairs(cfg["pos"], cfg["box"], 1, np.sort(ml), cfg["aev"]["Rcr"] + 1.0, seed=3)
    dpairs = torch.from_numpy(pairs).cuda()
    for t in range(6):
        pos = (cfg["pos"] + rng.normal(0, 0.03, size=cfg["pos"].shape)).astype(np.float32)
        dpos.copy_(torch.from_numpy(pos))
        ws.set_pair_list(dpairs if t >= 3 else None)
        E, F = ws.eval(dpos, dZ, cfg["box"], 1, dml)
        torch.cuda.synchronize()
        assert ws.status() == 0
        ref = oracle.evaluate(om, pos, cfg["Z"], cfg["box"], 1, ml)
        check_lists(ws, cfg, pos, len(ml), ml)
        check_EF(float(E.cpu()[0]), F.cpu().numpy().astype(np.float64), ref, len(ml), rows=ml)


# ------------------------------------------------------------------ round-2 additions
def test_dense_k_species_set_changes_on_one_workspace():
    """Dense-K mode materialises every column block whatever the species, so the layer-1 operand images must be re-packed
    when the set of species PRESENT changes: an H/O-only evaluation followed by one with C and N on the same workspace
    (the column-set key alone would not change)."""
    cfg = gen.get_config(4)
    n = cfg["pos"].shape[0]
    cluster = cfg["ml_index"]
    water = np.setdiff1d(np.arange(n), cluster)[:600].astype(np.int32)           # 200 whole molecules: H and O only
    om = oracle.Model(cfg["aev"], cfg["nets"], cfg["celu_alpha"])
    m, ws = make(dict(cfg, ml_index=water))
    ws.set_dense_k(1)
    for ml in (water, cluster.astype(np.int32), water):
        ref = oracle.evaluate(om, cfg["pos"], cfg["Z"], cfg["box"], 1, ml)
        E, F = run_gpu(ws, cfg["pos"], cfg["Z"], cfg["box"], 1, ml)
        check_EF(E, F, ref, len(ml), rows=ml)


def test_default_mlp_mode_reports_the_simt_fallback():
    """A network outside the tensor-core shape limits (hidden width 48) runs on CUDA cores: the model says so instead of
    falling back silently, the tensor-core modes are refused, and the result still meets the bars."""
    import paper_2604_21441_b200 as nnp
    cfg = gen.get_config(0)
    assert nnp.Model(cfg["aev"], cfg["nets"], cfg["celu_alpha"]).default_mlp_mode == nnp.NNP_MLP_F16X3
    dims = (384, 48, 32, 16, 1)
    nets = {Z: (dims,) + gen.make_weights(7, Z, dims) for Z in (1, 8)}
    m = nnp.Model(cfg["aev"], nets, cfg["celu_alpha"])
    assert m.default_mlp_mode == nnp.NNP_MLP_FP32_SIMT
    n = cfg["pos"].shape[0]
    ws = nnp.Workspace(m, n)
    assert nnp.nnp_workspace_set_mlp_mode(ws.handle, nnp.NNP_MLP_F16X3) == -7      # NNP_ERR_UNSUPPORTED
    ref = oracle.evaluate(oracle.Model(cfg["aev"], nets, cfg["celu_alpha"]), cfg["pos"], cfg["Z"], cfg["box"])
    E, F = run_gpu(ws, cfg["pos"], cfg["Z"], cfg["box"])
    check_EF(E, F, ref, n)


def test_ensemble_workspaces_on_two_streams():
    """Two ensemble workspaces used concurrently on two streams: the library orders their MLP launches (members hand over
    between co-resident CTAs of one launch), so the results equal those of a lone workspace, bit for bit, and nothing hangs."""
    torch = _torch()
    import paper_2604_21441_b200 as nnp
    cfg = gen.get_config(0)
    n = cfg["pos"].shape[0]
    nets = [{Z: (d,) + gen.make_weights(60 + mem, Z, d) for Z, (d, _, _) in cfg["nets"].items()} for mem in range(2)]
    m = nnp.Model(cfg["aev"], nets, cfg["celu_alpha"])
    P = gen.perturbed_positions(cfg["pos64"], 9, 4)
    dZ = torch.from_numpy(cfg["Z"]).cuda()
    dpos = [torch.from_numpy(P[t]).cuda() for t in range(4)]
    ws0 = nnp.Workspace(m, n)
    alone = []
    for t in range(4):
        E, F = ws0.eval(dpos[t], dZ, cfg["box"], 1)
        torch.cuda.synchronize()
        alone.append((float(E.cpu()[0]), F.cpu().numpy().copy()))
    # against the mean of the members' oracle evaluations
    refs = [oracle.evaluate(oracle.Model(cfg["aev"], nets[k], cfg["celu_alpha"]), P[0], cfg["Z"], cfg["box"]) for k in range(2)]
    check_EF(alone[0][0], alone[0][1].astype(np.float64),
             dict(energy=0.5 * (refs[0]["energy"] + refs[1]["energy"]), forces=0.5 * (refs[0]["forces"] + refs[1]["forces"])), n)
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    torch.cuda.synchronize()
    with torch.cuda.stream(s1):
        w1 = nnp.Workspace(m, n)
    with torch.cuda.stream(s2):
        w2 = nnp.Workspace(m, n)
    outs = []
    for rep in range(5):
        for t in range(4):
            ws, st = (w1, s1) if t % 2 == 0 else (w2, s2)
            with torch.cuda.stream(st):
                E = torch.empty(1, dtype=torch.float64, device="cuda")
                F = torch.empty((n, 3), dtype=torch.float32, device="cuda")
                ws.eval(dpos[t], dZ, cfg["box"], 1, None, E, F)
                outs.append((t, E, F))
    torch.cuda.synchronize()
    assert w1.status() == 0 and w2.status() == 0
    for t, E, F in outs:
        assert float(E.cpu()[0]) == alone[t][0] and np.array_equal(F.cpu().numpy(), alone[t][1])


def test_host_entry_notices_changed_atoms():
    """nnp_eval_host uploads Z / ml_index only when they changed since the last call -- and must notice when they did,
    also while the cell binning is being reused (the device buffers behind the host entry are always the same ones)."""
    cfg = gen.get_config(1)
    n = cfg["pos"].shape[0]
    om = oracle.Model(cfg["aev"], cfg["nets"], cfg["celu_alpha"])
    m, ws = make(cfg)
    ws.set_bin_reuse(5, 1.0)
    Z2 = cfg["Z"].copy()
    mol = np.random.default_rng(4).choice(n // 3, 50, replace=False)
    Z2[3 * mol], Z2[3 * mol + 1] = cfg["Z"][3 * mol + 1], cfg["Z"][3 * mol]      # 50 molecules become H-O-H in storage order
    ml = np.arange(0, n, 2, dtype=np.int32)
    for Z, idx in ((cfg["Z"], None), (cfg["Z"], None), (Z2, None), (Z2, ml), (cfg["Z"], ml), (cfg["Z"], None)):
        ref = oracle.evaluate(om, cfg["pos"], Z, cfg["box"], 1, idx, nbr_mode=1)
        E, F = ws.eval_host(cfg["pos"], Z, cfg["box"], 1, idx)
        assert ws.status() == 0
        check_EF(E, F.astype(np.float64), ref, n if idx is None else len(idx), rows=idx)


def test_link_atoms_in_nm_and_kj_per_mol():
    """Link atoms with unit conversion (a GROMACS-style caller: nm, kJ/mol): the link distance is given in the caller's
    length unit (0.1 nm), placement and force spread run on the nm positions and the converted forces, and the whole
    chain equals the oracle's Angstrom / eV chain scaled."""
    torch = _torch()
    cfg = gen.get_config(4)
    ml_full = cfg["ml_index"]
    n = cfg["pos"].shape[0]
    boxA = cfg["box"]
    L = float(boxA[0])
    ml = ml_full[:40]
    b = int(ml_full[40])
    dv = cfg["pos"][ml].astype(np.float64) - cfg["pos"][b].astype(np.float64)
    dv -= L * np.round(dv / L)
    link_ml = np.array([int(ml[np.argmin((dv ** 2).sum(1))])], np.int32)
    link_mm = np.array([b], np.int32)
    posA = np.zeros((n + 1, 3), np.float32); posA[:n] = cfg["pos"]
    Z_ext = np.concatenate([cfg["Z"], np.array([1], np.int32)])
    ml_ext = np.concatenate([ml, np.array([n], np.int32)]).astype(np.int32)
    NM, KJ = 10.0, 96.48533212
    pos_nm = (posA.astype(np.float64) / NM).astype(np.float32)
    box_nm = (np.asarray(boxA, np.float64) / NM).astype(np.float32)
    # oracle chain on exactly the coordinates the library converts to: fp32(nm * 10)
    p_or = (pos_nm.astype(np.float64) * NM).astype(np.float32)
    box_or = (box_nm.astype(np.float64) * NM).astype(np.float32)
    om = oracle.Model(cfg["aev"], cfg["nets"], cfg["celu_alpha"])
    m, ws = make(dict(cfg, pos=posA, ml_index=ml_ext))
    ws.set_units(NM, KJ)
    dpos = torch.from_numpy(pos_nm).cuda(); dZ = torch.from_numpy(Z_ext).cuda(); dml = torch.from_numpy(ml_ext).cuda()
    dlm = torch.from_numpy(link_ml).cuda(); dlb = torch.from_numpy(link_mm).cuda()
    ws.link_place(dpos, n, dlm, dlb, box_nm, 0.1, 1)                    # d = 1 Angstrom, in nm
    E, F = ws.eval(dpos, dZ, box_nm, 1, dml)
    ws.link_spread(F, dpos, n, dlm, dlb, box_nm, 0.1, 1)
    torch.cuda.synchronize()
    assert ws.status() == 0
    placed_nm = dpos.cpu().numpy()
    p_or[n:] = (placed_nm[n:].astype(np.float64) * NM).astype(np.float32)   # the link row as the library sees it in Angstrom
    want = p_or.copy()
    oracle.link_place(want, n, link_ml, link_mm, box_or, 1.0, 1)
    np.testing.assert_allclose(p_or[n:], want[n:], atol=2e-5)           # placed 1 Angstrom (0.1 nm) from the ML atom
    ref = oracle.evaluate(om, p_or, Z_ext, box_or, 1, ml_ext)
    F_or = ref["forces"].copy()
    oracle.link_spread(F_or, p_or, n, link_ml, link_mm, box_or, 1.0, 1)
    rows = np.concatenate([ml, link_mm])
    Fg = F.cpu().numpy().astype(np.float64) / (KJ * NM)                 # back to eV / Angstrom
    dF = Fg[rows] - F_or[rows]
    assert abs(float(E.cpu()[0]) / KJ - ref["energy"]) / len(ml_ext) <= E_TOL
    assert np.sqrt((dF ** 2).sum() / (F_or[rows] ** 2).sum()) <= F_RMS_TOL and np.abs(dF).max() <= F_MAX_TOL
    assert np.all(Fg[n:] == 0.0)

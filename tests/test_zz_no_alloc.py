"""The no-allocation entry point nnp_energy_sum_static (include/nnp.h; csrc/noalloc.cu): the K8 energy reduction with its
scratch in a static device array, against the existing path (the workspace's k_force_out, scratch from cudaMalloc).

Collected last on purpose (file name): the suite runs with `pytest -x`.  Passes alone in a fresh process and after the
other GPU tests (it shares nothing with them but the library's static scratch array, which every call re-arms)."""
import numpy as np
import pytest

import gen

E_TOL = 1e-4   # eV per atom: the energy bar of tests/test_gpu_parity.py


def _torch():
    import torch
    return torch


def _workspace_energy(cfg, pos):
    """E of the existing path and the per-atom energies it summed (ml_index order), one evaluation."""
    import paper_2604_21441_b200 as nnp
    torch = _torch()
    m = nnp.Model(cfg["aev"], cfg["nets"], cfg["celu_alpha"])
    n = cfg["pos"].shape[0]
    ws = nnp.Workspace(m, n, n)
    dpos = torch.from_numpy(np.ascontiguousarray(pos, np.float32)).cuda()
    dZ = torch.from_numpy(cfg["Z"]).cuda()
    E, F = ws.eval(dpos, dZ, cfg["box"], 1, None)
    torch.cuda.synchronize()
    assert ws.status() == 0
    return float(E.cpu()[0]), ws.atomic_energies(n)


@pytest.mark.gpu
def test_energy_sum_static_matches_workspace_path_on_two_calls_in_a_row():
    import paper_2604_21441_b200 as nnp
    torch = _torch()
    cfg = gen.get_config(1)                      # 3000 atoms: 12 blocks of partial sums
    n = cfg["pos"].shape[0]
    P = gen.perturbed_positions(cfg["pos64"], cfg["perturb_seed"], 2)
    ref = [_workspace_energy(cfg, P[t]) for t in range(2)]
    assert ref[0][0] != ref[1][0]                # two different inputs: a stale partial sum would show
    st = torch.cuda.current_stream().cuda_stream
    d_e = [torch.from_numpy(ref[t][1]).cuda() for t in range(2)]
    d_E = [torch.full((1,), float("nan"), dtype=torch.float64, device="cuda") for _ in range(3)]
    # two calls in a row on one stream (no synchronisation in between), then the first input again
    for k, t in enumerate((0, 1, 0)):
        rc = nnp.nnp_energy_sum_static(st, n, d_e[t].data_ptr(), 1.0, d_E[k].data_ptr())
        assert rc == 0, nnp.nnp_strerror(rc)
    torch.cuda.synchronize()
    got = [float(x.cpu()[0]) for x in d_E]
    for k, t in enumerate((0, 1, 0)):
        assert abs(got[k] - ref[t][0]) / n <= E_TOL, (k, got[k], ref[t][0])
        # ... and the definition itself: the fp64 sum of the same fp32 values (only the order of the additions differs)
        assert abs(got[k] - float(np.sum(ref[t][1].astype(np.float64)))) <= 1e-9 * max(1.0, abs(got[k]))
    assert got[0] == got[2]                      # bitwise reproducible, whatever ran in between
    # e_scale, and a ragged size (not a multiple of the block)
    rc = nnp.nnp_energy_sum_static(st, n - 37, d_e[1].data_ptr(), 96.485, d_E[0].data_ptr())
    assert rc == 0
    torch.cuda.synchronize()
    want = 96.485 * float(np.sum(ref[1][1][: n - 37].astype(np.float64)))
    assert abs(float(d_E[0].cpu()[0]) - want) <= 1e-9 * max(1.0, abs(want))


@pytest.mark.gpu
def test_energy_sum_static_limits():
    import paper_2604_21441_b200 as nnp
    torch = _torch()
    st = torch.cuda.current_stream().cuda_stream
    nmax = nnp.NNP_STATIC_MAX_ATOMS
    rng = np.random.default_rng(7)
    h = rng.standard_normal(nmax + 1).astype(np.float32)
    d = torch.from_numpy(h).cuda()
    dE = torch.full((1,), 123.0, dtype=torch.float64, device="cuda")
    # beyond the maximum: a clear error, nothing launched, the output untouched
    rc = nnp.nnp_energy_sum_static(st, nmax + 1, d.data_ptr(), 1.0, dE.data_ptr())
    assert rc == nnp.NNP_ERR_STATIC_LIMIT and "maximum" in nnp.nnp_strerror(rc)
    torch.cuda.synchronize()
    assert float(dE.cpu()[0]) == 123.0
    # the maximum itself (all 4096 partial sums in use), twice in a row
    for _ in range(2):
        rc = nnp.nnp_energy_sum_static(st, nmax, d.data_ptr(), 1.0, dE.data_ptr())
        assert rc == 0
        torch.cuda.synchronize()
        want = float(np.sum(h[:nmax].astype(np.float64)))
        assert abs(float(dE.cpu()[0]) - want) <= 1e-9 * max(1.0, abs(want))
    # empty input, bad arguments
    assert nnp.nnp_energy_sum_static(st, 0, None, 1.0, dE.data_ptr()) == 0
    torch.cuda.synchronize()
    assert float(dE.cpu()[0]) == 0.0
    assert nnp.nnp_energy_sum_static(st, -1, d.data_ptr(), 1.0, dE.data_ptr()) == -1
    assert nnp.nnp_energy_sum_static(st, 5, d.data_ptr(), 1.0, None) == -1

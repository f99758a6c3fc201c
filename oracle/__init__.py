"""ctypes front-end of the fp64 CPU oracle (oracle/nnp_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package.  It imports nothing from paper_2604_21441_b200 and shares no code with the CUDA path.
Marshalling only: all arithmetic is in nnp_oracle.c (cited there against SURVEY.md Appendix A).
"""
import ctypes as C
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "nnp_oracle.c")
_LIB = os.path.join(_HERE, "libnnp_oracle.so")
_lib = None


def build(force=False):
    """gcc -O2 -fopenmp; no BLAS, no intrinsics (SURVEY.md section 8.d "CPU baseline")."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared",
                               "-D_GNU_SOURCE", _SRC, "-o", _LIB, "-lm"])
    return _LIB


class _AevParams(C.Structure):
    _fields_ = [("Rcr", C.c_double), ("Rca", C.c_double), ("EtaR", C.c_double), ("EtaA", C.c_double),
                ("Zeta", C.c_double), ("nShfR", C.c_int32), ("nShfA", C.c_int32), ("nShfZ", C.c_int32),
                ("ShfR", C.POINTER(C.c_double)), ("ShfA", C.POINTER(C.c_double)), ("ShfZ", C.POINTER(C.c_double)),
                ("c_R", C.c_double), ("c_theta", C.c_double), ("S", C.c_int32),
                ("species_Z", C.POINTER(C.c_int32))]


class _Mlp(C.Structure):
    _fields_ = [("n_layers", C.c_int32), ("dims", C.POINTER(C.c_int32)),
                ("W", C.POINTER(C.POINTER(C.c_float))), ("b", C.POINTER(C.POINTER(C.c_float))),
                ("alpha", C.c_double)]


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_fc.restype = C.c_double
        _lib.orc_fc.argtypes = [C.c_double, C.c_double]
        _lib.orc_celu.restype = C.c_double
        _lib.orc_celu.argtypes = [C.c_double, C.c_double]
        _lib.orc_neighbors.restype = C.c_int64
        _lib.orc_mlp_forward.restype = C.c_double
        _lib.orc_eval.restype = C.c_int
        _lib.orc_aev_length.restype = C.c_int
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


class Model:
    """Holds the C structs (and the numpy arrays that back them) for one model."""

    def __init__(self, aev, nets, celu_alpha=0.1):
        """aev: dict as gen.aev_params; nets: {Z: (dims, W list, b list)} (species without entry: no net)."""
        self._keep = []
        k = lambda a: (self._keep.append(a), a)[1]
        ShfR = k(np.ascontiguousarray(aev["ShfR"], dtype=np.float64))
        ShfA = k(np.ascontiguousarray(aev["ShfA"], dtype=np.float64))
        ShfZ = k(np.ascontiguousarray(aev["ShfZ"], dtype=np.float64))
        sZ = k(np.ascontiguousarray(aev["species_Z"], dtype=np.int32))
        self.S = len(sZ)
        self.species_Z = sZ
        self.p = _AevParams(aev["Rcr"], aev["Rca"], aev["EtaR"], aev["EtaA"], aev["Zeta"],
                            len(ShfR), len(ShfA), len(ShfZ), _dp(ShfR), _dp(ShfA), _dp(ShfZ),
                            aev["radial_prefactor"], aev["cos_scale"], self.S,
                            sZ.ctypes.data_as(C.POINTER(C.c_int32)))
        self.L = lib().orc_aev_length(C.byref(self.p))
        self.nets = (_Mlp * self.S)()
        for s, Z in enumerate(sZ):
            if int(Z) not in nets:
                self.nets[s] = _Mlp(0, None, None, None, celu_alpha)
                continue
            dims, W, b = nets[int(Z)]
            self.nets[s] = self._mlp(dims, W, b, celu_alpha)

    def _mlp(self, dims, W, b, alpha):
        k = lambda a: (self._keep.append(a), a)[1]
        d = k(np.ascontiguousarray(dims, dtype=np.int32))
        nl = len(d) - 1
        Wp = k((C.POINTER(C.c_float) * nl)())
        bp = k((C.POINTER(C.c_float) * nl)())
        for l in range(nl):
            w = k(np.ascontiguousarray(W[l], dtype=np.float32))
            bb = k(np.ascontiguousarray(b[l], dtype=np.float32))
            assert w.shape == (d[l + 1], d[l]) and bb.shape == (d[l + 1],)
            Wp[l] = w.ctypes.data_as(C.POINTER(C.c_float))
            bp[l] = bb.ctypes.data_as(C.POINTER(C.c_float))
        return _Mlp(nl, d.ctypes.data_as(C.POINTER(C.c_int32)), Wp, bp, alpha)


def fc(R, Rc):
    return lib().orc_fc(float(R), float(Rc))


def celu(x, alpha=0.1):
    return lib().orc_celu(float(x), float(alpha))


def neighbors(pos, box, Rc, pbc=1, ml_index=None, mode=0):
    """CSR neighbour list: rows in ml_index order, columns = global atom indices ascending."""
    pos = np.ascontiguousarray(pos, dtype=np.float32)
    box = np.ascontiguousarray(box, dtype=np.float32).reshape(9)
    n = pos.shape[0]
    ml = None if ml_index is None else np.ascontiguousarray(ml_index, dtype=np.int32)
    n_ml = n if ml is None else len(ml)
    start = np.zeros(n_ml + 1, dtype=np.int32)
    cap = max(1024, 256 * n_ml)
    col = np.zeros(cap, dtype=np.int32)
    f = lib().orc_neighbors
    f.argtypes = [C.c_int64, C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p, C.c_int64, C.c_double, C.c_int32,
                  C.c_void_p, C.c_void_p, C.c_int64]
    r = f(n, pos.ctypes.data, box.ctypes.data, pbc, None if ml is None else ml.ctypes.data, n_ml, float(Rc), mode,
          start.ctypes.data, col.ctypes.data, cap)
    if r < 0:
        raise RuntimeError(f"orc_neighbors error {r}")
    return start, col[:r].copy()


def mlp_forward(dims, W, b, G, alpha=0.1, want_grad=True):
    """One atom: returns (E, g = dE/dG)."""
    m = Model.__new__(Model)
    m._keep = []
    net = m._mlp(dims, W, b, alpha)
    G = np.ascontiguousarray(G, dtype=np.float64)
    g = np.zeros_like(G)
    f = lib().orc_mlp_forward
    f.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
    E = f(C.addressof(net), G.ctypes.data, g.ctypes.data if want_grad else None)
    return E, g


def evaluate(model, pos, Z, box, pbc=1, ml_index=None, nbr_mode=0, want_forces=True, want_aev=False,
             want_atomic=False, want_daev=False):
    """One energy+force evaluation.  Returns dict(energy, forces (N,3) fp64, [aev], [e_atom], [daev])."""
    pos = np.ascontiguousarray(pos, dtype=np.float32)
    Z = np.ascontiguousarray(Z, dtype=np.int32)
    box = np.ascontiguousarray(box, dtype=np.float32).reshape(9)
    n = pos.shape[0]
    ml = None if ml_index is None else np.ascontiguousarray(ml_index, dtype=np.int32)
    n_ml = n if ml is None else len(ml)
    E = C.c_double(0.0)
    F = np.zeros((n, 3), dtype=np.float64)
    aev = np.zeros((n_ml, model.L), dtype=np.float64) if want_aev else None
    ea = np.zeros(n_ml, dtype=np.float64) if want_atomic else None
    da = np.zeros((n_ml, model.L), dtype=np.float64) if want_daev else None
    f = lib().orc_eval
    f.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p,
                  C.c_int64, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    rc = f(C.addressof(model.p), C.addressof(model.nets), n, pos.ctypes.data, Z.ctypes.data, box.ctypes.data, pbc,
           None if ml is None else ml.ctypes.data, n_ml, nbr_mode, 1 if want_forces else 0, C.addressof(E),
           F.ctypes.data, None if aev is None else aev.ctypes.data, None if ea is None else ea.ctypes.data,
           None if da is None else da.ctypes.data)
    if rc != 0:
        raise RuntimeError(f"orc_eval error {rc}")
    out = dict(energy=E.value, forces=F)
    if want_aev:
        out["aev"] = aev
    if want_atomic:
        out["e_atom"] = ea
    if want_daev:
        out["daev"] = da
    return out


def evaluate_virial(model, pos, Z, box, pbc=1, ml_index=None, nbr_mode=0):
    """Energy, forces and the strain derivative W[a][b] = dE/d eps_ab = sum_i sum_j p_ij[a] d_ij[b] (3x3, fp64)."""
    pos = np.ascontiguousarray(pos, dtype=np.float32)
    Z = np.ascontiguousarray(Z, dtype=np.int32)
    box = np.ascontiguousarray(box, dtype=np.float32).reshape(9)
    n = pos.shape[0]
    ml = None if ml_index is None else np.ascontiguousarray(ml_index, dtype=np.int32)
    n_ml = n if ml is None else len(ml)
    E = C.c_double(0.0)
    F = np.zeros((n, 3), dtype=np.float64)
    W = np.zeros((3, 3), dtype=np.float64)
    f = lib().orc_eval_virial
    f.restype = C.c_int
    f.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p,
                  C.c_int64, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p]
    rc = f(C.addressof(model.p), C.addressof(model.nets), n, pos.ctypes.data, Z.ctypes.data, box.ctypes.data, pbc,
           None if ml is None else ml.ctypes.data, n_ml, nbr_mode, C.addressof(E), F.ctypes.data, W.ctypes.data)
    if rc != 0:
        raise RuntimeError(f"orc_eval_virial error {rc}")
    return dict(energy=E.value, forces=F, virial=W)


def link_place(pos_ext, n_atoms, link_ml, link_mm, box, d=1.0, pbc=1):
    """Writes the link-atom rows n_atoms.. of pos_ext (fp32, (n_atoms + n_links, 3)) in place (eq. 4)."""
    assert pos_ext.dtype == np.float32 and pos_ext.flags["C_CONTIGUOUS"]
    lm = np.ascontiguousarray(link_ml, dtype=np.int32); lb = np.ascontiguousarray(link_mm, dtype=np.int32)
    box = np.ascontiguousarray(box, dtype=np.float32).reshape(9)
    f = lib().orc_link_place
    f.argtypes = [C.c_int64, C.c_int64, C.c_void_p, C.c_void_p, C.c_double, C.c_void_p, C.c_int32, C.c_void_p]
    rc = f(n_atoms, len(lm), lm.ctypes.data, lb.ctypes.data, float(d), box.ctypes.data, pbc, pos_ext.ctypes.data)
    if rc != 0:
        raise RuntimeError(f"orc_link_place error {rc}")
    return pos_ext


def link_spread(forces_ext, pos_ext, n_atoms, link_ml, link_mm, box, d=1.0, pbc=1):
    """Redistributes the link-atom force rows of forces_ext (fp64, in place) onto the bonded atoms (chain rule of eq. 4)."""
    assert forces_ext.dtype == np.float64 and forces_ext.flags["C_CONTIGUOUS"]
    pos_ext = np.ascontiguousarray(pos_ext, dtype=np.float32)
    lm = np.ascontiguousarray(link_ml, dtype=np.int32); lb = np.ascontiguousarray(link_mm, dtype=np.int32)
    box = np.ascontiguousarray(box, dtype=np.float32).reshape(9)
    f = lib().orc_link_spread
    f.argtypes = [C.c_int64, C.c_int64, C.c_void_p, C.c_void_p, C.c_double, C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p]
    rc = f(n_atoms, len(lm), lm.ctypes.data, lb.ctypes.data, float(d), box.ctypes.data, pbc, pos_ext.ctypes.data,
           forces_ext.ctypes.data)
    if rc != 0:
        raise RuntimeError(f"orc_link_spread error {rc}")
    return forces_ext


def num_threads():
    return lib().orc_num_threads()


def set_num_threads(n):
    lib().orc_set_num_threads(int(n))

"""ctypes binding of include/nnp.h -- argument marshalling only (same names as the C entry points).

Low level: nnp_* functions take/return raw pointers (ints) exactly like the C-ABI.
Convenience: Model / Workspace own the opaque handles; Workspace.eval takes torch CUDA tensors (device memory
and streams are torch's; nothing else of torch is used) and Workspace.eval_host takes numpy arrays.
"""
import ctypes as C
import os
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libnnp_b200.so")

NNP_OK = 0
NNP_MLP_FP32_SIMT, NNP_MLP_F16X3, NNP_MLP_F16X1 = 0, 1, 2

EXPORTS = [
    "nnp_model_create", "nnp_model_create_ensemble", "nnp_model_destroy", "nnp_model_aev_length", "nnp_workspace_create",
    "nnp_workspace_destroy", "nnp_workspace_set_mlp_mode", "nnp_workspace_set_dense_k", "nnp_workspace_set_virial_output", "nnp_workspace_set_units", "nnp_workspace_set_pair_list", "nnp_workspace_set_small_path", "nnp_workspace_set_bin_reuse", "nnp_eval",
    "nnp_eval_host", "nnp_status", "nnp_strerror", "nnp_debug_neighbors", "nnp_debug_aev", "nnp_debug_daev",
    "nnp_debug_atomic_energies", "nnp_debug_counters", "nnp_debug_mlp_timeline", "nnp_link_place", "nnp_link_spread", "nnp_workspace_set_profiling", "nnp_debug_stage_times",
    "nnp_debug_fp32_peak", "nnp_model_default_mlp_mode", "nnp_energy_sum_static",
]
NNP_ERR_STATIC_LIMIT = -9
NNP_STATIC_MAX_ATOMS = 1048576


class NNPError(RuntimeError):
    def __init__(self, code, where=""):
        self.code = code
        super().__init__(f"{where}: nnp error {code}: {nnp_strerror(code)}")


class _AevParams(C.Structure):
    _fields_ = [("Rcr", C.c_double), ("Rca", C.c_double), ("EtaR", C.c_double), ("EtaA", C.c_double),
                ("Zeta", C.c_double), ("nShfR", C.c_int32), ("nShfA", C.c_int32), ("nShfZ", C.c_int32),
                ("ShfR", C.POINTER(C.c_double)), ("ShfA", C.POINTER(C.c_double)), ("ShfZ", C.POINTER(C.c_double)),
                ("radial_prefactor", C.c_double), ("cos_scale", C.c_double), ("n_species", C.c_int32),
                ("species_Z", C.POINTER(C.c_int32))]


class _MlpDesc(C.Structure):
    _fields_ = [("n_layers", C.c_int32), ("dims", C.POINTER(C.c_int32)),
                ("W", C.POINTER(C.POINTER(C.c_float))), ("b", C.POINTER(C.POINTER(C.c_float))),
                ("celu_alpha", C.c_double)]


_lib = None


def lib_path():
    return _LIB_PATH


def lib():
    """Loads libnnp_b200.so (built in-tree by paper_2604_21441_b200/build.py).  No fallback of any kind."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise ImportError(f"{_LIB_PATH} is missing: run `python -m paper_2604_21441_b200.build` "
                              "(there is no CPU or PyTorch fallback for the NNP path)")
        L = C.CDLL(_LIB_PATH)
        vp, i32, i64 = C.c_void_p, C.c_int32, C.c_int64
        L.nnp_model_create.argtypes = [vp, vp, C.POINTER(vp)]
        L.nnp_model_create_ensemble.argtypes = [vp, vp, i32, C.POINTER(vp)]
        L.nnp_model_destroy.argtypes = [vp]
        L.nnp_model_aev_length.argtypes = [vp]
        L.nnp_model_default_mlp_mode.argtypes = [vp]
        L.nnp_workspace_create.argtypes = [vp, i64, i64, vp, C.POINTER(vp)]
        L.nnp_workspace_destroy.argtypes = [vp]
        L.nnp_workspace_set_mlp_mode.argtypes = [vp, i32]
        L.nnp_workspace_set_dense_k.argtypes = [vp, i32]
        L.nnp_workspace_set_virial_output.argtypes = [vp, vp]
        L.nnp_workspace_set_units.argtypes = [vp, C.c_double, C.c_double]
        L.nnp_workspace_set_pair_list.argtypes = [vp, vp, i64]
        L.nnp_workspace_set_small_path.argtypes = [vp, i32]
        L.nnp_workspace_set_bin_reuse.argtypes = [vp, i32, C.c_double]
        L.nnp_eval.argtypes = [vp, i64, vp, vp, vp, i32, vp, i64, vp, vp]
        L.nnp_eval_host.argtypes = [vp, i64, vp, vp, vp, i32, vp, i64, vp, vp]
        L.nnp_status.argtypes = [vp]
        L.nnp_strerror.argtypes = [C.c_int]
        L.nnp_strerror.restype = C.c_char_p
        L.nnp_debug_neighbors.argtypes = [vp, C.c_int, C.POINTER(i64), vp, vp, i64]
        L.nnp_debug_aev.argtypes = [vp, vp]
        L.nnp_debug_daev.argtypes = [vp, vp]
        L.nnp_debug_atomic_energies.argtypes = [vp, vp]
        L.nnp_debug_counters.argtypes = [vp, C.POINTER(i64)]
        L.nnp_debug_mlp_timeline.argtypes = [vp, vp]
        L.nnp_link_place.argtypes = [vp, i64, i64, vp, vp, C.c_double, vp, i32, vp]
        L.nnp_link_spread.argtypes = [vp, i64, i64, vp, vp, C.c_double, vp, i32, vp, vp]
        L.nnp_workspace_set_profiling.argtypes = [vp, i32]
        L.nnp_debug_stage_times.argtypes = [vp, vp]
        L.nnp_debug_fp32_peak.argtypes = [vp, i32, C.POINTER(C.c_double)]
        L.nnp_energy_sum_static.argtypes = [vp, i64, vp, C.c_double, vp]
        _lib = L
    return _lib


# ---------------------------------------------------------------- low level: one function per C entry point
def nnp_strerror(code):
    return lib().nnp_strerror(int(code)).decode()


def nnp_model_create(aev_struct, nets_array):
    out = C.c_void_p()
    rc = lib().nnp_model_create(C.addressof(aev_struct), C.addressof(nets_array), C.byref(out))
    return rc, out.value


def nnp_model_create_ensemble(aev_struct, nets_array, n_members):
    out = C.c_void_p()
    rc = lib().nnp_model_create_ensemble(C.addressof(aev_struct), C.addressof(nets_array), n_members, C.byref(out))
    return rc, out.value


def nnp_model_destroy(model):
    return lib().nnp_model_destroy(model)


def nnp_model_aev_length(model):
    return lib().nnp_model_aev_length(model)


def nnp_model_default_mlp_mode(model):
    return lib().nnp_model_default_mlp_mode(model)


def nnp_workspace_create(model, max_atoms, max_ml_atoms, cuda_stream):
    out = C.c_void_p()
    rc = lib().nnp_workspace_create(model, int(max_atoms), int(max_ml_atoms), cuda_stream, C.byref(out))
    return rc, out.value


def nnp_workspace_destroy(ws):
    return lib().nnp_workspace_destroy(ws)


def nnp_workspace_set_mlp_mode(ws, mode):
    return lib().nnp_workspace_set_mlp_mode(ws, int(mode))


def nnp_workspace_set_dense_k(ws, dense):
    return lib().nnp_workspace_set_dense_k(ws, int(dense))


def nnp_workspace_set_units(ws, angstrom_per_length_unit, energy_units_per_ev):
    return lib().nnp_workspace_set_units(ws, float(angstrom_per_length_unit), float(energy_units_per_ev))


def nnp_workspace_set_bin_reuse(ws, every_n, skin):
    return lib().nnp_workspace_set_bin_reuse(ws, int(every_n), float(skin))


def nnp_workspace_set_small_path(ws, on):
    return lib().nnp_workspace_set_small_path(ws, int(on))


def nnp_workspace_set_pair_list(ws, d_pairs, n_pairs):
    return lib().nnp_workspace_set_pair_list(ws, d_pairs, int(n_pairs))


def nnp_workspace_set_virial_output(ws, d_virial9):
    return lib().nnp_workspace_set_virial_output(ws, d_virial9)


def nnp_eval(ws, n_atoms, d_pos, d_Z, box_ptr, pbc, d_ml_index, n_ml, d_energy, d_forces):
    return lib().nnp_eval(ws, int(n_atoms), d_pos, d_Z, box_ptr, int(pbc), d_ml_index, int(n_ml), d_energy, d_forces)


def nnp_eval_host(ws, n_atoms, h_pos, h_Z, box_ptr, pbc, h_ml_index, n_ml, h_energy, h_forces):
    return lib().nnp_eval_host(ws, int(n_atoms), h_pos, h_Z, box_ptr, int(pbc), h_ml_index, int(n_ml), h_energy,
                               h_forces)


def nnp_status(ws):
    return lib().nnp_status(ws)


def nnp_debug_neighbors(ws, which, h_row_start, h_col, col_cap):
    n = C.c_int64(0)
    rc = lib().nnp_debug_neighbors(ws, int(which), C.byref(n), h_row_start, h_col, int(col_cap))
    return rc, n.value


def nnp_debug_aev(ws, h_aev):
    return lib().nnp_debug_aev(ws, h_aev)


def nnp_debug_daev(ws, h_daev):
    return lib().nnp_debug_daev(ws, h_daev)


def nnp_debug_atomic_energies(ws, h_e):
    return lib().nnp_debug_atomic_energies(ws, h_e)


def nnp_link_place(stream, n_atoms, n_links, d_link_ml, d_link_mm, d, box, pbc, d_pos):
    return lib().nnp_link_place(stream, n_atoms, n_links, d_link_ml, d_link_mm, float(d), box, pbc, d_pos)


def nnp_link_spread(stream, n_atoms, n_links, d_link_ml, d_link_mm, d, box, pbc, d_pos, d_forces):
    return lib().nnp_link_spread(stream, n_atoms, n_links, d_link_ml, d_link_mm, float(d), box, pbc, d_pos, d_forces)


def nnp_debug_mlp_timeline(ws, h_ticks):
    return lib().nnp_debug_mlp_timeline(ws, h_ticks)


def nnp_debug_counters(ws):
    n = C.c_int64(0)
    rc = lib().nnp_debug_counters(ws, C.byref(n))
    return rc, n.value


def nnp_workspace_set_profiling(ws, on):
    return lib().nnp_workspace_set_profiling(ws, int(on))


def nnp_debug_stage_times(ws, h_ms):
    return lib().nnp_debug_stage_times(ws, h_ms)


def nnp_debug_fp32_peak(cuda_stream, variant):
    t = C.c_double(0.0)
    rc = lib().nnp_debug_fp32_peak(cuda_stream, int(variant), C.byref(t))
    return rc, t.value


def nnp_energy_sum_static(cuda_stream, n, d_e_atom, e_scale, d_energy):
    """raw device pointers in, status out: the no-allocation energy reduction (nnp.h)"""
    return lib().nnp_energy_sum_static(cuda_stream, int(n), d_e_atom, float(e_scale), d_energy)


# ---------------------------------------------------------------- convenience owners
def _check(rc, where):
    if rc != NNP_OK:
        raise NNPError(rc, where)


class Model:
    """aev: dict with Rcr, Rca, EtaR, EtaA, Zeta, ShfR, ShfA, ShfZ, radial_prefactor, cos_scale, species_Z;
    nets: {Z: (dims, [W_l], [b_l])}; species without an entry have no network.  A list of such dicts makes an
    ensemble (E = mean over the members: ANI-2x is an ensemble of 8 networks)."""

    def __init__(self, aev, nets, celu_alpha=0.1):
        keep = []
        k = lambda a: (keep.append(a), a)[1]
        dp = lambda a: a.ctypes.data_as(C.POINTER(C.c_double))
        ShfR = k(np.ascontiguousarray(aev["ShfR"], dtype=np.float64))
        ShfA = k(np.ascontiguousarray(aev["ShfA"], dtype=np.float64))
        ShfZ = k(np.ascontiguousarray(aev["ShfZ"], dtype=np.float64))
        sZ = k(np.ascontiguousarray(aev["species_Z"], dtype=np.int32))
        S = len(sZ)
        p = _AevParams(aev["Rcr"], aev["Rca"], aev["EtaR"], aev["EtaA"], aev["Zeta"], len(ShfR), len(ShfA),
                       len(ShfZ), dp(ShfR), dp(ShfA), dp(ShfZ), aev["radial_prefactor"], aev["cos_scale"], S,
                       sZ.ctypes.data_as(C.POINTER(C.c_int32)))
        members = list(nets) if isinstance(nets, (list, tuple)) else [nets]
        M = len(members)
        arr = (_MlpDesc * (S * M))()
        for mem, s, Z in ((mem, s, Z) for mem in range(M) for s, Z in enumerate(sZ)):
            nets = members[mem]
            if int(Z) not in nets:
                arr[mem * S + s] = _MlpDesc(0, None, None, None, celu_alpha)
                continue
            dims, W, b = nets[int(Z)]
            d = k(np.ascontiguousarray(dims, dtype=np.int32))
            nl = len(d) - 1
            Wp = k((C.POINTER(C.c_float) * nl)())
            bp = k((C.POINTER(C.c_float) * nl)())
            for l in range(nl):
                w = k(np.ascontiguousarray(W[l], dtype=np.float32))
                bb = k(np.ascontiguousarray(b[l], dtype=np.float32))
                if w.shape != (d[l + 1], d[l]) or bb.shape != (d[l + 1],):
                    raise ValueError("weight/bias shape mismatch")
                Wp[l] = w.ctypes.data_as(C.POINTER(C.c_float))
                bp[l] = bb.ctypes.data_as(C.POINTER(C.c_float))
            arr[mem * S + s] = _MlpDesc(nl, d.ctypes.data_as(C.POINTER(C.c_int32)), Wp, bp, celu_alpha)
        rc, h = nnp_model_create_ensemble(p, arr, M) if M > 1 else nnp_model_create(p, arr)
        _check(rc, "nnp_model_create")
        self.n_members = M
        self.handle = h
        self.aev_length = nnp_model_aev_length(h)
        self.default_mlp_mode = nnp_model_default_mlp_mode(h)   # NNP_MLP_FP32_SIMT: networks outside the tensor-core limits

    def close(self):
        if getattr(self, "handle", None):
            nnp_model_destroy(self.handle)
            self.handle = None

    def __del__(self):
        self.close()


def _as(a, dtype):
    """`a` itself when it already is a C-contiguous array of `dtype` (no new object: see Workspace._ptr), else a converted copy."""
    if type(a) is np.ndarray and a.dtype == dtype and a.flags.c_contiguous:
        return a
    return np.ascontiguousarray(a, dtype=dtype)


class Workspace:
    def __init__(self, model, max_atoms, max_ml_atoms=None, stream=None):
        import torch
        self.model = model
        self.max_atoms = int(max_atoms)
        self.max_ml = int(max_atoms if max_ml_atoms is None else max_ml_atoms)
        self.stream = torch.cuda.current_stream() if stream is None else stream
        rc, h = nnp_workspace_create(model.handle, self.max_atoms, self.max_ml, self.stream.cuda_stream)
        _check(rc, "nnp_workspace_create")
        self.handle = h
        self._pcache = {}                              # id(array) -> (array, address): see _ptr
        self._E = np.zeros(1, dtype=np.float64)        # energy word of eval_host
        self._E_ptr = self._E.ctypes.data

    def set_mlp_mode(self, mode):
        _check(nnp_workspace_set_mlp_mode(self.handle, mode), "nnp_workspace_set_mlp_mode")

    def set_units(self, angstrom_per_length_unit=1.0, energy_units_per_ev=1.0):
        _check(nnp_workspace_set_units(self.handle, angstrom_per_length_unit, energy_units_per_ev), "nnp_workspace_set_units")

    def set_virial_output(self, virial):
        """virial: (9,) or (3,3) float64 cuda tensor that every later eval fills with dE/d eps, or None to switch off."""
        self._virial = virial
        _check(nnp_workspace_set_virial_output(self.handle, None if virial is None else virial.data_ptr()),
               "nnp_workspace_set_virial_output")

    def set_bin_reuse(self, every_n, skin=0.0):
        """Reuse the cell binning for every_n - 1 evaluations after a full one (cells cut skin wider); 0 / 1 = off."""
        _check(nnp_workspace_set_bin_reuse(self.handle, every_n, skin), "nnp_workspace_set_bin_reuse")

    def set_small_path(self, on):
        _check(nnp_workspace_set_small_path(self.handle, on), "nnp_workspace_set_small_path")

    def set_pair_list(self, pairs):
        """pairs: (n_pairs, 2) int32 cuda tensor of candidate pairs (global atom indices), or None for the cell search."""
        self._pairs = pairs
        if pairs is None:
            _check(nnp_workspace_set_pair_list(self.handle, None, 0), "nnp_workspace_set_pair_list")
        else:
            import torch
            assert pairs.is_cuda and pairs.dtype == torch.int32 and pairs.is_contiguous() and pairs.shape[1] == 2
            _check(nnp_workspace_set_pair_list(self.handle, pairs.data_ptr() if pairs.shape[0] else None, pairs.shape[0]),
                   "nnp_workspace_set_pair_list")

    def set_dense_k(self, dense):
        _check(nnp_workspace_set_dense_k(self.handle, dense), "nnp_workspace_set_dense_k")

    def eval(self, pos, Z, box, pbc=1, ml_index=None, energy=None, forces=None, check=False):
        """pos (N,3) float32 cuda, Z (N,) int32 cuda, box: 9 floats on the HOST, ml_index (n_ml,) int32 cuda
        or None.  Asynchronous on the workspace stream; returns (energy (1,) float64 cuda, forces (N,3))."""
        import torch
        n = pos.shape[0]
        assert pos.is_cuda and pos.dtype == torch.float32 and pos.is_contiguous()
        assert Z.is_cuda and Z.dtype == torch.int32 and Z.is_contiguous()
        if energy is None:
            energy = torch.empty(1, dtype=torch.float64, device=pos.device)
        if forces is None:
            forces = torch.empty((n, 3), dtype=torch.float32, device=pos.device)
        b = np.ascontiguousarray(box, dtype=np.float32).reshape(9)
        ml_ptr, n_ml = None, n
        if ml_index is not None:
            assert ml_index.is_cuda and ml_index.dtype == torch.int32 and ml_index.is_contiguous()
            n_ml = ml_index.shape[0]
            ml_ptr = ml_index.data_ptr() if n_ml > 0 else Z.data_ptr()  # empty subset: any non-NULL pointer
        rc = nnp_eval(self.handle, n, pos.data_ptr(), Z.data_ptr(), b.ctypes.data, pbc, ml_ptr, n_ml,
                      energy.data_ptr(), forces.data_ptr())
        _check(rc, "nnp_eval")
        self._last = (pos, Z, ml_index)  # keep the device buffers of the last evaluation alive for debug exports
        if check:
            _check(nnp_status(self.handle), "nnp_status")
        return energy, forces

    def link_place(self, pos_ext, n_atoms, link_ml, link_mm, box, d=1.0, pbc=1):
        """Writes the link-atom rows n_atoms.. of pos_ext ((n_atoms + n_links, 3) float32 cuda) on the workspace stream."""
        b = np.ascontiguousarray(box, dtype=np.float32).reshape(9)
        _check(nnp_link_place(self.stream.cuda_stream, n_atoms, link_ml.shape[0], link_ml.data_ptr(), link_mm.data_ptr(), d,
                              b.ctypes.data, pbc, pos_ext.data_ptr()), "nnp_link_place")

    def link_spread(self, forces_ext, pos_ext, n_atoms, link_ml, link_mm, box, d=1.0, pbc=1):
        """Redistributes the link rows of forces_ext onto the bonded atoms (chain rule of PAPER.md eq. 4)."""
        b = np.ascontiguousarray(box, dtype=np.float32).reshape(9)
        _check(nnp_link_spread(self.stream.cuda_stream, n_atoms, link_ml.shape[0], link_ml.data_ptr(), link_mm.data_ptr(), d,
                               b.ctypes.data, pbc, pos_ext.data_ptr(), forces_ext.data_ptr()), "nnp_link_spread")

    def eval_host(self, pos, Z, box, pbc=1, ml_index=None, forces_out=None):
        """numpy in / numpy out through nnp_eval_host (copies + synchronisation inside the library)."""
        pos = _as(pos, np.float32)
        Z = _as(Z, np.int32)
        b = _as(box, np.float32)
        n = pos.shape[0]
        ml = None if ml_index is None else _as(ml_index, np.int32)
        F = np.empty((n, 3), dtype=np.float32) if forces_out is None else forces_out
        rc = nnp_eval_host(self.handle, n, self._ptr(pos), self._ptr(Z), self._ptr(b), pbc,
                           None if ml is None else self._ptr(ml), 0 if ml is None else len(ml), self._E_ptr,
                           self._ptr(F))
        _check(rc, "nnp_eval_host")
        self._last = None
        self._n_ml = n if ml is None else len(ml)
        return float(self._E[0]), F

    def _ptr(self, a):
        """Address of a numpy array's buffer.  `a.ctypes.data` costs ~2.5 us a call -- five of them were 12 us of a 290 us
        step -- so the address of an array OBJECT seen before is remembered (the entry holds a reference: the id cannot be
        reused, and numpy refuses to reallocate a referenced array's buffer); at most 64 entries."""
        ent = self._pcache.get(id(a))
        if ent is not None and ent[0] is a:
            return ent[1]
        p = a.ctypes.data
        if len(self._pcache) >= 64:
            self._pcache.clear()
        self._pcache[id(a)] = (a, p)
        return p

    def status(self):
        return nnp_status(self.handle)

    def neighbors(self, which, n_ml):
        start = np.zeros(n_ml + 1, dtype=np.int32)
        rc, n = nnp_debug_neighbors(self.handle, which, None, None, 0)
        _check(rc, "nnp_debug_neighbors")
        col = np.zeros(max(n, 1), dtype=np.int32)
        rc, n = nnp_debug_neighbors(self.handle, which, start.ctypes.data, col.ctypes.data, len(col))
        _check(rc, "nnp_debug_neighbors")
        return start, col[:n]

    def aev(self, n_ml):
        a = np.zeros((n_ml, self.model.aev_length), dtype=np.float32)
        _check(nnp_debug_aev(self.handle, a.ctypes.data), "nnp_debug_aev")
        return a

    def daev(self, n_ml):
        a = np.zeros((n_ml, self.model.aev_length), dtype=np.float32)
        _check(nnp_debug_daev(self.handle, a.ctypes.data), "nnp_debug_daev")
        return a

    def mlp_timeline(self):
        t = np.zeros(64, dtype=np.int64)
        _check(nnp_debug_mlp_timeline(self.handle, t.ctypes.data), "nnp_debug_mlp_timeline")
        return t

    def atomic_energies(self, n_ml):
        e = np.zeros(n_ml, dtype=np.float32)
        _check(nnp_debug_atomic_energies(self.handle, e.ctypes.data), "nnp_debug_atomic_energies")
        return e

    def set_profiling(self, on):
        _check(nnp_workspace_set_profiling(self.handle, on), "nnp_workspace_set_profiling")

    def stage_times(self):
        """ms per stage of the last evaluation: neighbour, aev_fwd, mlp, aev_bwd, output."""
        ms = np.zeros(5, dtype=np.float32)
        _check(nnp_debug_stage_times(self.handle, ms.ctypes.data), "nnp_debug_stage_times")
        return ms

    def launches(self):
        rc, n = nnp_debug_counters(self.handle)
        _check(rc, "nnp_debug_counters")
        return n

    def close(self):
        if getattr(self, "handle", None):
            nnp_workspace_destroy(self.handle)
            self.handle = None

    def __del__(self):
        self.close()

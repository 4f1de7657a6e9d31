"""ctypes binding of include/pimd.h -- same names, argument marshalling only.

Host arrays are numpy float64 / int32; `_dev` calls take torch CUDA tensors (or raw device pointers).
PyTorch is used only to lend device memory (a uint8 workspace tensor from its caching allocator) and
the current stream to the library (`PIMD(..., torch_workspace=True)`).
"""
import ctypes as C
import os

import numpy as np

PIMD_OK, PIMD_EINVAL, PIMD_ENOSTATE, PIMD_ENOMODEL = 0, -1, -2, -3
PIMD_ESEL_OVERFLOW, PIMD_ECUDA, PIMD_ENOMEM, PIMD_ETABLE_RANGE, PIMD_ECONTACT = -4, -5, -6, -7, -8
PIMD_MAX_TYPES = 4

_HERE = os.path.dirname(os.path.abspath(__file__))


def library_path():
    return os.path.join(_HERE, "libpimd_b200.so")


class PimdError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("pimd error %d: %s" % (code, msg))
        self.code = code


class ModelDesc(C.Structure):
    _fields_ = [("rcut", C.c_double), ("rcut_smth", C.c_double), ("n_types", C.c_int32),
                ("sel", C.c_int32 * PIMD_MAX_TYPES), ("embed", C.c_int32 * 3), ("axis_neuron", C.c_int32),
                ("fit", C.c_int32 * 3)]

    @classmethod
    def from_dict(cls, d):
        m = cls()
        m.rcut, m.rcut_smth = float(d["rcut"]), float(d["rcut_smth"])
        m.n_types = len(d["sel"])
        for t, s in enumerate(d["sel"]):
            m.sel[t] = int(s)
        for l in range(3):
            m.embed[l] = int(d["embed"][l])
            m.fit[l] = int(d["fit"][l])
        m.axis_neuron = int(d["axis"])
        return m


class Estimators(C.Structure):
    _fields_ = [("K_PR", C.c_double), ("K_CV", C.c_double), ("H", C.c_double), ("K_ring", C.c_double),
                ("S_ring", C.c_double), ("U_sum", C.c_double), ("T_ring", C.c_double), ("step", C.c_int64)]

    def as_dict(self):
        return {n: getattr(self, n) for n, _ in self._fields_}


class BarostatState(C.Structure):
    _fields_ = [("v_W", C.c_double), ("box", C.c_double * 3), ("V", C.c_double), ("P_CV", C.c_double),
                ("P_PR", C.c_double), ("P_MD", C.c_double), ("K_W", C.c_double), ("U_W", C.c_double),
                ("J_W", C.c_double), ("enthalpy", C.c_double), ("v_W3", C.c_double * 3), ("P_CV3", C.c_double * 3)]

    def as_dict(self):
        d = {n: getattr(self, n) for n, _ in self._fields_}
        for key in ("box", "v_W3", "P_CV3"):
            d[key] = np.array(list(getattr(self, key)))
        return d


_lib = None

_SIGNATURES = {
    "pimd_create": (C.c_int, [C.POINTER(C.c_void_p), C.c_int, C.c_void_p, C.c_int, C.c_void_p, C.c_void_p,
                              C.c_int, C.c_double, C.c_double, C.c_double, C.c_uint64]),
    "pimd_destroy": (None, [C.c_void_p]),
    "pimd_last_error": (C.c_char_p, [C.c_void_p]),
    "pimd_workspace_bytes": (C.c_size_t, [C.c_void_p, C.c_void_p]),
    "pimd_set_workspace": (C.c_int, [C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p]),
    "pimd_set_state": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p]),
    "pimd_set_state_dev": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p]),
    "pimd_restore": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64]),
    "pimd_get_neighbor_counts": (C.c_int, [C.c_void_p, C.c_void_p]),
    "pimd_get_launch_count": (C.c_int64, [C.c_void_p]),
    "pimd_set_fitting_path": (C.c_int, [C.c_void_p, C.c_int]),
    "pimd_set_integrator": (C.c_int, [C.c_void_p, C.c_int]),
    "pimd_set_fixcom": (C.c_int, [C.c_void_p, C.c_int]),
    "pimd_set_method": (C.c_int, [C.c_void_p, C.c_int]),
    "pimd_set_barostat": (C.c_int, [C.c_void_p, C.c_double, C.c_double]),
    "pimd_set_barostat_aniso": (C.c_int, [C.c_void_p, C.c_double, C.c_double]),
    "pimd_get_barostat": (C.c_int, [C.c_void_p, C.c_void_p]),
    "pimd_get_barostat_history": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int]),
    "pimd_restore_cell": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]),
    "pimd_set_embedding_path": (C.c_int, [C.c_void_p, C.c_int]),
    "pimd_set_embedding_compressed": (C.c_int, [C.c_void_p, C.c_int]),
    "pimd_debug_gemm": (C.c_int, [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]),
    "pimd_model_n_weights": (C.c_size_t, [C.c_void_p]),
    "pimd_set_model": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_size_t]),
    "pimd_set_model_harmonic": (C.c_int, [C.c_void_p, C.c_double]),
    "pimd_step": (C.c_int, [C.c_void_p, C.c_int64]),
    "pimd_get_positions": (C.c_int, [C.c_void_p, C.c_void_p]),
    "pimd_get_momenta": (C.c_int, [C.c_void_p, C.c_void_p]),
    "pimd_get_forces": (C.c_int, [C.c_void_p, C.c_void_p]),
    "pimd_get_virial": (C.c_int, [C.c_void_p, C.c_void_p]),
    "pimd_get_energies": (C.c_int, [C.c_void_p, C.c_void_p]),
    "pimd_get_atom_energies": (C.c_int, [C.c_void_p, C.c_void_p]),
    "pimd_get_estimators": (C.c_int, [C.c_void_p, C.c_void_p]),
    "pimd_get_estimator_history": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int]),
    "pimd_get_positions_dev": (C.c_int, [C.c_void_p, C.c_void_p]),
    "pimd_get_forces_dev": (C.c_int, [C.c_void_p, C.c_void_p]),
    "pimd_get_neighbors": (C.c_int64, [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_size_t]),
    "pimd_debug_noise": (C.c_int, [C.c_void_p, C.c_int64, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]),
    "pimd_time_kernel": (C.c_int, [C.c_void_p, C.c_int, C.c_int, C.POINTER(C.c_double)]),
    "pimd_set_profiling": (C.c_int, [C.c_void_p, C.c_int]),
    "pimd_debug_graph_state": (C.c_int, [C.c_void_p]),
    "pimd_get_phase_ms": (C.c_int, [C.c_void_p, C.c_void_p]),
    "pimd_debug_get_row_index": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p]),
    "pimd_noalloc_setup": (C.c_int, []),
    "pimd_noalloc_last_error": (C.c_char_p, []),
    "pimd_row_scan_noalloc_dev": (C.c_int, [C.c_int, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]),
}


def lib():
    """Loads libpimd_b200.so (built by paper_2602_13553_b200.build).  Fails loudly if it is missing."""
    global _lib
    if _lib is None:
        path = library_path()
        if not os.path.exists(path):
            raise ImportError("%s not found: build it with `python -m paper_2602_13553_b200.build` "
                              "(there is no CPU fallback)" % path)
        L = C.CDLL(path)
        for name, (res, args) in _SIGNATURES.items():
            fn = getattr(L, name)
            fn.restype, fn.argtypes = res, args
        _lib = L
    return _lib


def _check(ctx, rc):
    if rc < 0:
        raise PimdError(rc, pimd_last_error(ctx))
    return rc


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _ptr(a):
    """numpy array -> host pointer; torch tensor -> device pointer; int -> as is."""
    if isinstance(a, np.ndarray):
        return a.ctypes.data
    if hasattr(a, "data_ptr"):
        return a.data_ptr()
    return int(a)


# ---- same-name wrappers ------------------------------------------------------------------------

def pimd_create(types, masses, box, n_beads, T, dt, gamma_centroid, seed):
    types = np.ascontiguousarray(types, dtype=np.int32)
    masses, box = _f64(masses), _f64(box)
    ctx = C.c_void_p()
    rc = lib().pimd_create(C.byref(ctx), types.size, types.ctypes.data, masses.size, masses.ctypes.data,
                           box.ctypes.data, int(n_beads), float(T), float(dt), float(gamma_centroid),
                           int(seed) & 0xFFFFFFFFFFFFFFFF)
    if rc < 0:
        raise PimdError(rc, "pimd_create failed (no CUDA device?)" if rc == PIMD_ECUDA else "pimd_create: bad argument")
    return ctx


def pimd_destroy(ctx):
    lib().pimd_destroy(ctx)


def pimd_last_error(ctx):
    return lib().pimd_last_error(ctx).decode()


def pimd_workspace_bytes(ctx, desc=None):
    return lib().pimd_workspace_bytes(ctx, C.byref(desc) if desc is not None else None)


def pimd_set_workspace(ctx, workspace_dev, nbytes, cuda_stream=0):
    return _check(ctx, lib().pimd_set_workspace(ctx, _ptr(workspace_dev), int(nbytes), int(cuda_stream) or None))


def pimd_set_state(ctx, x, p):
    x, p = _f64(x), _f64(p)
    return _check(ctx, lib().pimd_set_state(ctx, x.ctypes.data, p.ctypes.data))


def _dev_f64(t, numel, what):
    """A torch CUDA tensor handed to a `_dev` call crosses the C ABI as a raw pointer: check here that it is what the
    library will read (float64, contiguous, on the GPU, `numel` elements).  Plain ints (raw device pointers) pass."""
    if hasattr(t, "data_ptr"):
        import torch
        if not (t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and t.numel() == numel):
            raise ValueError("%s must be a contiguous float64 CUDA tensor of %d elements (got %s, %s, %d elements%s)"
                             % (what, numel, t.device, t.dtype, t.numel(), "" if t.is_contiguous() else ", non-contiguous"))
    return _ptr(t)


def pimd_set_state_dev(ctx, x_dev, p_dev, numel=None):
    """numel = P*N*3 enables the tensor checks of _dev_f64 (PIMD.set_state passes it)."""
    if numel is not None:
        return _check(ctx, lib().pimd_set_state_dev(ctx, _dev_f64(x_dev, numel, "x_dev"), _dev_f64(p_dev, numel, "p_dev")))
    return _check(ctx, lib().pimd_set_state_dev(ctx, _ptr(x_dev), _ptr(p_dev)))


def pimd_restore(ctx, x, p, f, U, step):
    x, p, f, U = _f64(x), _f64(p), _f64(f), _f64(U)
    return _check(ctx, lib().pimd_restore(ctx, x.ctypes.data, p.ctypes.data, f.ctypes.data, U.ctypes.data, int(step)))


def pimd_get_neighbor_counts(ctx, P, N, n_types):
    out = np.empty((P, N, n_types), dtype=np.int32)
    _check(ctx, lib().pimd_get_neighbor_counts(ctx, out.ctypes.data))
    return out


def pimd_debug_get_row_index(ctx, P, N, n_types):
    """(cen_idx[P N], rowstart[n_types][P N + 1]) of the most recent force evaluation (pimd_debug.h)."""
    cen = np.empty(P * N, dtype=np.int32)
    rowstart = np.empty((n_types, P * N + 1), dtype=np.int32)
    _check(ctx, lib().pimd_debug_get_row_index(ctx, cen.ctypes.data, rowstart.ctypes.data))
    return cen, rowstart


def pimd_noalloc_last_error():
    return lib().pimd_noalloc_last_error().decode()


def pimd_noalloc_setup():
    rc = lib().pimd_noalloc_setup()
    if rc < 0:
        raise PimdError(rc, pimd_noalloc_last_error())
    return rc


def _dev_i32(t, numel, what):
    """torch CUDA int32 tensor -> device pointer, checked (a wrong dtype or a host tensor would be a silent bad read)."""
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.int32 and t.is_contiguous() and t.numel() == numel):
        raise PimdError(PIMD_EINVAL, "%s must be a contiguous CUDA int32 tensor of %d elements" % (what, numel))
    return t.data_ptr()


def pimd_row_scan_noalloc_dev(n_centres, n_types, cen_idx_dev, ncount_dev, rowstart_dev, cuda_stream=0):
    """pimd_noalloc.h: asynchronous on `cuda_stream` (0 = legacy default stream); allocates nothing.  Sizes are passed
    on as given so that the library's own limit checks answer; tensors are checked when the sizes are positive."""
    n_centres, n_types = int(n_centres), int(n_types)
    if n_centres > 0 and n_types > 0 and hasattr(cen_idx_dev, "data_ptr"):
        ptrs = (_dev_i32(cen_idx_dev, n_centres, "cen_idx_dev"), _dev_i32(ncount_dev, n_centres * n_types, "ncount_dev"),
                _dev_i32(rowstart_dev, n_types * (n_centres + 1), "rowstart_dev"))
    else:
        ptrs = (_ptr(cen_idx_dev), _ptr(ncount_dev), _ptr(rowstart_dev))
    rc = lib().pimd_row_scan_noalloc_dev(n_centres, n_types, ptrs[0], ptrs[1], ptrs[2], int(cuda_stream) or None)
    if rc < 0:
        raise PimdError(rc, pimd_noalloc_last_error())
    return rc


def pimd_get_launch_count(ctx):
    return int(lib().pimd_get_launch_count(ctx))


PIMD_BAOAB, PIMD_OBABO = 0, 1


def pimd_set_integrator(ctx, kind):
    """kind: PIMD_BAOAB / PIMD_OBABO or the strings "baoab" / "obabo"."""
    if isinstance(kind, str):
        kind = {"baoab": PIMD_BAOAB, "obabo": PIMD_OBABO}[kind.lower()]
    return _check(ctx, lib().pimd_set_integrator(ctx, int(kind)))


PIMD_NMPIMD, PIMD_CART = 0, 1


def pimd_set_method(ctx, method):
    if isinstance(method, str):
        method = {"nmpimd": PIMD_NMPIMD, "pimd": PIMD_CART}[method]
    return _check(ctx, lib().pimd_set_method(ctx, int(method)))


def pimd_set_fixcom(ctx, on):
    return _check(ctx, lib().pimd_set_fixcom(ctx, int(bool(on))))


def pimd_set_fitting_path(ctx, use_tensor_cores):
    return _check(ctx, lib().pimd_set_fitting_path(ctx, int(bool(use_tensor_cores))))


def pimd_set_embedding_path(ctx, use_tensor_cores):
    return _check(ctx, lib().pimd_set_embedding_path(ctx, int(bool(use_tensor_cores))))


def pimd_set_embedding_compressed(ctx, on=True):
    return _check(ctx, lib().pimd_set_embedding_compressed(ctx, int(bool(on))))


def pimd_debug_gemm(ctx, A, Bt):
    A = np.ascontiguousarray(A, dtype=np.float32)
    Bt = np.ascontiguousarray(Bt, dtype=np.float32)
    M, K = A.shape
    N = Bt.shape[0]
    Cm = np.empty((M, N), dtype=np.float32)
    _check(ctx, lib().pimd_debug_gemm(ctx, M, N, K, A.ctypes.data, Bt.ctypes.data, Cm.ctypes.data))
    return Cm


def pimd_model_n_weights(desc):
    return lib().pimd_model_n_weights(C.byref(desc))


def pimd_set_model(ctx, desc, weights):
    w = _f64(weights)
    return _check(ctx, lib().pimd_set_model(ctx, C.byref(desc), w.ctypes.data, w.size))


def pimd_set_model_harmonic(ctx, k_spring):
    return _check(ctx, lib().pimd_set_model_harmonic(ctx, float(k_spring)))


def pimd_step(ctx, n_steps=1):
    return _check(ctx, lib().pimd_step(ctx, int(n_steps)))


def _getter(name, ctx, shape, out=None):
    """`out`: optional C-contiguous float64 array of `shape` to receive the copy (e.g. a view of pinned memory,
    which makes the device->host copy a direct DMA); a fresh array otherwise."""
    if out is None:
        out = np.empty(shape, dtype=np.float64)
    elif out.dtype != np.float64 or tuple(out.shape) != tuple(shape) or not out.flags["C_CONTIGUOUS"]:
        raise ValueError("out must be a C-contiguous float64 array of shape %r" % (tuple(shape),))
    _check(ctx, getattr(lib(), name)(ctx, out.ctypes.data))
    return out


def pimd_get_positions(ctx, P, N, out=None):
    return _getter("pimd_get_positions", ctx, (P, N, 3), out)


def pimd_get_momenta(ctx, P, N, out=None):
    return _getter("pimd_get_momenta", ctx, (P, N, 3), out)


def pimd_get_forces(ctx, P, N, out=None):
    return _getter("pimd_get_forces", ctx, (P, N, 3), out)


def pimd_get_virial(ctx, P):
    return _getter("pimd_get_virial", ctx, (P, 3, 3))


def pimd_get_energies(ctx, P):
    return _getter("pimd_get_energies", ctx, (P,))


def pimd_get_atom_energies(ctx, P, N):
    return _getter("pimd_get_atom_energies", ctx, (P, N))


def pimd_get_estimators(ctx):
    e = Estimators()
    _check(ctx, lib().pimd_get_estimators(ctx, C.byref(e)))
    return e.as_dict()


def pimd_set_barostat(ctx, p_ext_bar, tau_p):
    return _check(ctx, lib().pimd_set_barostat(ctx, float(p_ext_bar), float(tau_p)))


def pimd_set_barostat_aniso(ctx, p_ext_bar, tau_p):
    return _check(ctx, lib().pimd_set_barostat_aniso(ctx, float(p_ext_bar), float(tau_p)))


def pimd_get_barostat_history(ctx, cap):
    arr = (BarostatState * cap)()
    n = _check(ctx, lib().pimd_get_barostat_history(ctx, arr, cap))
    return [arr[q].as_dict() for q in range(n)]


def pimd_restore_cell(ctx, box, v_W, xi):
    box = np.ascontiguousarray(box, dtype=np.float64)
    v_W = np.ascontiguousarray(np.broadcast_to(np.asarray(v_W, dtype=np.float64), (3,)))
    xi = np.ascontiguousarray(xi, dtype=np.float64)
    return _check(ctx, lib().pimd_restore_cell(ctx, box.ctypes.data, v_W.ctypes.data, xi.ctypes.data))


def pimd_get_barostat(ctx):
    b = BarostatState()
    _check(ctx, lib().pimd_get_barostat(ctx, C.byref(b)))
    return b.as_dict()


def pimd_get_estimator_history(ctx, cap):
    arr = (Estimators * cap)()
    n = _check(ctx, lib().pimd_get_estimator_history(ctx, arr, cap))
    return [arr[q].as_dict() for q in range(n)]


def pimd_get_positions_dev(ctx, x_dev, numel=None):
    return _check(ctx, lib().pimd_get_positions_dev(ctx, _ptr(x_dev) if numel is None else _dev_f64(x_dev, numel, "x_dev")))


def pimd_get_forces_dev(ctx, f_dev, numel=None):
    return _check(ctx, lib().pimd_get_forces_dev(ctx, _ptr(f_dev) if numel is None else _dev_f64(f_dev, numel, "f_dev")))


def pimd_get_neighbors(ctx, bead, N, cap):
    count = np.empty(N, dtype=np.int32)
    j = np.empty(cap, dtype=np.int32)
    shift = np.empty((cap, 3), dtype=np.int8)
    n = lib().pimd_get_neighbors(ctx, int(bead), count.ctypes.data, j.ctypes.data, shift.ctypes.data, cap)
    _check(ctx, int(n))
    return count, j[:n].copy(), shift[:n].copy()


def pimd_debug_noise(ctx, step, idx):
    idx = np.ascontiguousarray(idx, dtype=np.int32).reshape(-1, 3)
    n = idx.shape[0]
    words = np.empty((n, 4), dtype=np.uint32)
    eta = np.empty(n, dtype=np.float64)
    _check(ctx, lib().pimd_debug_noise(ctx, int(step), n, idx.ctypes.data, words.ctypes.data, eta.ctypes.data))
    return words, eta


def pimd_time_kernel(ctx, kind, reps):
    ms = C.c_double()
    _check(ctx, lib().pimd_time_kernel(ctx, int(kind), int(reps), C.byref(ms)))
    return ms.value


def pimd_debug_graph_state(ctx):
    return int(lib().pimd_debug_graph_state(ctx))


def pimd_set_profiling(ctx, on):
    return _check(ctx, lib().pimd_set_profiling(ctx, int(bool(on))))


def pimd_get_phase_ms(ctx):
    out = np.zeros(6, dtype=np.float64)
    _check(ctx, lib().pimd_get_phase_ms(ctx, out.ctypes.data))
    return out


class PIMD:
    """Convenience owner of one context (create .. destroy) with the shapes remembered."""

    def __init__(self, types, masses, box, n_beads, T, dt, gamma_centroid, seed, model_desc=None,
                 torch_workspace=True, integrator="baoab", fixcom=False, method="nmpimd"):
        self.N, self.P = int(np.asarray(types).size), int(n_beads)
        self.ctx = pimd_create(types, masses, box, n_beads, T, dt, gamma_centroid, seed)
        if integrator != "baoab":
            pimd_set_integrator(self.ctx, integrator)
        if method != "nmpimd":
            pimd_set_method(self.ctx, method)
        if fixcom:
            pimd_set_fixcom(self.ctx, True)
        self.desc = ModelDesc.from_dict(model_desc) if isinstance(model_desc, dict) else model_desc
        self._ws = None
        if torch_workspace:
            import torch
            nbytes = pimd_workspace_bytes(self.ctx, self.desc)
            self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device="cuda")   # caching allocator
            base = (self._ws.data_ptr() + 255) // 256 * 256
            pimd_set_workspace(self.ctx, base, nbytes, torch.cuda.current_stream().cuda_stream)

    def close(self):
        if self.ctx is not None:
            pimd_destroy(self.ctx)
            self.ctx = None
            self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_state(self, x, p):
        if hasattr(x, "data_ptr"):
            return pimd_set_state_dev(self.ctx, x, p, numel=self.P * self.N * 3)
        x, p = np.asarray(x), np.asarray(p)
        if x.size != self.P * self.N * 3 or p.size != x.size:
            raise ValueError("x and p must hold P*N*3 = %d values" % (self.P * self.N * 3))
        return pimd_set_state(self.ctx, x, p)

    def set_model(self, weights, desc=None):
        if desc is not None:
            self.desc = ModelDesc.from_dict(desc) if isinstance(desc, dict) else desc
        return pimd_set_model(self.ctx, self.desc, weights)

    def set_compressed(self, on=True):
        return pimd_set_embedding_compressed(self.ctx, on)

    def set_model_harmonic(self, k):
        return pimd_set_model_harmonic(self.ctx, k)

    def step(self, n=1):
        return pimd_step(self.ctx, n)

    def positions(self, out=None): return pimd_get_positions(self.ctx, self.P, self.N, out)
    def momenta(self, out=None): return pimd_get_momenta(self.ctx, self.P, self.N, out)
    def forces(self, out=None): return pimd_get_forces(self.ctx, self.P, self.N, out)
    def virial(self): return pimd_get_virial(self.ctx, self.P)
    def energies(self): return pimd_get_energies(self.ctx, self.P)
    def atom_energies(self): return pimd_get_atom_energies(self.ctx, self.P, self.N)
    def estimators(self): return pimd_get_estimators(self.ctx)
    def set_barostat(self, p_ext_bar, tau_p, aniso=False):
        return (pimd_set_barostat_aniso if aniso else pimd_set_barostat)(self.ctx, p_ext_bar, tau_p)

    def barostat_state(self): return pimd_get_barostat(self.ctx)
    def barostat_history(self, cap=4096): return pimd_get_barostat_history(self.ctx, cap)
    def restore_cell(self, box, v_W, xi): return pimd_restore_cell(self.ctx, box, v_W, xi)
    def estimator_history(self, cap=4096): return pimd_get_estimator_history(self.ctx, cap)

    def neighbors(self, bead, cap=None):
        cap = cap or self.N * 512
        return pimd_get_neighbors(self.ctx, bead, self.N, cap)

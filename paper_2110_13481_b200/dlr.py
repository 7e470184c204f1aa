"""Thin ctypes binding of the C ABI in include/dlr.h (same names, argument marshalling only: every step of the
path runs in the CUDA kernels of libdlr_b200.so).  PyTorch is used for device memory and the stream only.

There is no CPU fallback: if the shared library is missing (run `python -m paper_2110_13481_b200.build`) or no
CUDA device is present, loading / creating a context raises.
"""
import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libdlr_b200.so")

DLR_OK = 0
ERRORS = {0: "DLR_OK", -1: "DLR_ERR_INVALID", -2: "DLR_ERR_UNSUPPORTED", -3: "DLR_ERR_WORKSPACE", -4: "DLR_ERR_CUDA",
          -5: "DLR_ERR_NOT_ORTHONORMAL", -6: "DLR_ERR_NO_STATE", -7: "DLR_ERR_TOO_LARGE"}
NOALLOC_MAX_PROBES = 4096


class dlr_config(ctypes.Structure):
    _fields_ = [("n_x", ctypes.c_int32 * 3), ("n_v", ctypes.c_int32 * 3),
                ("x_lo", ctypes.c_double * 3), ("x_hi", ctypes.c_double * 3),
                ("v_lo", ctypes.c_double * 3), ("v_hi", ctypes.c_double * 3),
                ("rank", ctypes.c_int32), ("order", ctypes.c_int32),
                ("e_scale", ctypes.c_double), ("flags", ctypes.c_uint32)]


class dlr_moments_t(ctypes.Structure):
    _fields_ = [("mass", ctypes.c_double), ("momentum", ctypes.c_double * 3), ("kinetic_energy", ctypes.c_double),
                ("electric_energy", ctypes.c_double), ("s_fro", ctypes.c_double),
                ("qr_fallbacks", ctypes.c_int32), ("nonfinite", ctypes.c_int32),
                ("qr_third_stage", ctypes.c_int32), ("eig_unconverged", ctypes.c_int32)]


_lib = None


def lib():
    """the loaded shared library (raises if it has not been built: no fallback)"""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} not found: build it with `python -m paper_2110_13481_b200.build` "
                               "(there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        vp, dp, ip = ctypes.c_void_p, ctypes.POINTER(ctypes.c_double), ctypes.c_int
        L.dlr_workspace_bytes.argtypes = [ctypes.POINTER(dlr_config), ctypes.POINTER(ctypes.c_size_t)]
        L.dlr_create.argtypes = [ctypes.POINTER(dlr_config), vp, ctypes.c_size_t, vp, ctypes.POINTER(vp)]
        L.dlr_set_initial.argtypes = [vp, vp, vp, vp, ip]
        L.dlr_step.argtypes = [vp, ctypes.c_double]
        L.dlr_run.argtypes = [vp, ctypes.c_double, ip]
        L.dlr_moments.argtypes = [vp, ctypes.POINTER(dlr_moments_t), ip, vp, vp, vp]
        L.dlr_get_factors.argtypes = [vp, vp, vp, vp, ip]
        L.dlr_get_field.argtypes = [vp, vp, ip]
        L.dlr_set_profiling.argtypes = [vp, ip]
        L.dlr_get_phase_times.argtypes = [vp, ip, ctypes.POINTER(ctypes.c_float), ctypes.POINTER(ctypes.c_char_p)]
        L.dlr_launches_per_step.argtypes = [vp]
        L.dlr_bytes_per_step.argtypes = [vp]
        L.dlr_bytes_per_step.restype = ctypes.c_double
        L.dlr_test_fft_roundtrip.argtypes = [vp, ip, ip, vp, vp, vp]
        L.dlr_test_dir_pass.argtypes = [vp, ip, ip, vp, vp, vp, vp, vp, vp, vp]
        L.dlr_test_chol_decide.argtypes = [vp, vp, ctypes.POINTER(ctypes.c_int)]
        L.dlr_destroy.argtypes = [vp]
        L.dlr_destroy.restype = None
        L.dlr_strerror.argtypes = [ip]
        L.dlr_strerror.restype = ctypes.c_char_p
        L.dlr_last_cuda_error.argtypes = [vp]
        L.dlr_last_cuda_error.restype = ctypes.c_char_p
        L.dlr_clear_error.argtypes = [vp]
        L.dlr_probe_noalloc.argtypes = [vp, vp, vp, ctypes.c_int64, ctypes.c_int64, ip, ip, vp, vp, vp, vp]
        L.dlr_noalloc_last_error.argtypes = []
        L.dlr_noalloc_last_error.restype = ctypes.c_char_p
        _lib = L
    return _lib


class DlrError(RuntimeError):
    def __init__(self, code, where, detail=""):
        self.code = code
        super().__init__(f"{where}: {ERRORS.get(code, code)} ({lib().dlr_strerror(code).decode()}) {detail}")


FLAG_PREDICTOR_L_FLOW = 1
FLAG_UNCONVENTIONAL = 2


def make_config(n_x, n_v, x_lo, x_hi, v_lo, v_hi, rank, order=2, e_scale=1.0, flags=0):
    c = dlr_config()
    for d in range(3):
        c.n_x[d], c.n_v[d] = n_x, n_v
        c.x_lo[d], c.x_hi[d], c.v_lo[d], c.v_hi[d] = x_lo, x_hi, v_lo, v_hi
    c.rank, c.order, c.e_scale, c.flags = rank, order, e_scale, flags
    return c


def config_from_inputs(cfg, order=2, e_scale=1.0, flags=0):
    """dlr_config from a dict of paper_2110_13481_b200.inputs.make_config"""
    return make_config(cfg["n_x"], cfg["n_v"], cfg["x_lo"], cfg["x_hi"], cfg["v_lo"], cfg["v_hi"], cfg["r"], order, e_scale,
                       flags)


def dlr_workspace_bytes(cfg):
    n = ctypes.c_size_t(0)
    rc = lib().dlr_workspace_bytes(ctypes.byref(cfg), ctypes.byref(n))
    if rc != DLR_OK:
        raise DlrError(rc, "dlr_workspace_bytes")
    return n.value


def _ptr(a):
    """raw pointer of a torch tensor (device or host) or a numpy array; None -> NULL"""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        return a.ctypes.data
    return a.data_ptr()


def probe_noalloc(X, S, V, probe_ix, probe_iv, stream=None):
    """dlr_probe_noalloc: f = X S V^T at index pairs, no device allocation (static device scratch, at most
    NOALLOC_MAX_PROBES pairs per call).  X (r, N_x), S (r, r), V (r, N_v): CUDA tensors holding the ABI's column-major
    layout (row c of the tensor = column c of the factor); probe_ix, probe_iv: host integer sequences -> numpy f"""
    import torch
    r = S.shape[0]
    ix = np.ascontiguousarray(probe_ix, dtype=np.int64)
    iv = np.ascontiguousarray(probe_iv, dtype=np.int64)
    f = np.empty(len(ix), dtype=np.float64)
    st = stream if stream is not None else torch.cuda.current_stream(X.device)
    rc = lib().dlr_probe_noalloc(X.data_ptr(), S.data_ptr(), V.data_ptr(), X.numel() // r, V.numel() // r, r, len(ix),
                                 _ptr(ix), _ptr(iv), _ptr(f), st.cuda_stream)
    if rc != DLR_OK:
        raise DlrError(rc, "dlr_probe_noalloc", lib().dlr_noalloc_last_error().decode())
    return f


class Dlr:
    """One context = one simulation on one GPU/stream.  Methods are the C calls with the `dlr_` prefix dropped."""

    def __init__(self, cfg, device="cuda:0", stream=None, guard_bytes=0):
        """guard_bytes > 0 puts that many pattern bytes before and after the workspace (check_guards(): tests only)"""
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: the DLR hot path has no CPU fallback")
        self.torch = torch
        self.cfg = cfg
        self.device = torch.device(device)
        self.r = cfg.rank
        self.Nx = cfg.n_x[0] * cfg.n_x[1] * cfg.n_x[2]
        self.Nv = cfg.n_v[0] * cfg.n_v[1] * cfg.n_v[2]
        nbytes = dlr_workspace_bytes(cfg)
        with torch.cuda.device(self.device):
            self.workspace = torch.full((nbytes + 512 + 2 * guard_bytes,), 0xA5, dtype=torch.uint8, device=self.device)
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        base = self.workspace.data_ptr()
        self._ws_ptr = (base + guard_bytes + 255) // 256 * 256
        self._guards = (self._ws_ptr - base, self._ws_ptr - base + nbytes) if guard_bytes else None
        h = ctypes.c_void_p()
        rc = lib().dlr_create(ctypes.byref(cfg), self._ws_ptr, nbytes, self.stream.cuda_stream, ctypes.byref(h))
        if rc != DLR_OK:
            raise DlrError(rc, "dlr_create")
        self.h = h

    def check_guards(self):
        """True if no byte outside [workspace, workspace + dlr_workspace_bytes) was written since creation"""
        lo, hi = self._guards
        self.torch.cuda.synchronize(self.device)
        return bool((self.workspace[:lo] == 0xA5).all().item()) and bool((self.workspace[hi:] == 0xA5).all().item())

    def _check(self, rc, where):
        if rc != DLR_OK:
            raise DlrError(rc, where, lib().dlr_last_cuda_error(self.h).decode())

    def set_initial(self, X, S, V):
        """X, S, V: column-major (Fortran-order numpy, or torch tensors holding that layout) fp64"""
        on_dev = 0
        if isinstance(X, np.ndarray):
            X, S, V = (np.asfortranarray(a, dtype=np.float64) for a in (X, S, V))
        else:
            on_dev = 1 if X.is_cuda else 0
        self._keep = (X, S, V)
        self._check(lib().dlr_set_initial(self.h, _ptr(X), _ptr(S), _ptr(V), on_dev), "dlr_set_initial")
        self._keep = None

    def step(self, tau):
        self._check(lib().dlr_step(self.h, float(tau)), "dlr_step")

    def run(self, tau, nsteps):
        self._check(lib().dlr_run(self.h, float(tau), int(nsteps)), "dlr_run")

    def moments(self, probe_ix=None, probe_iv=None):
        m = dlr_moments_t()
        npb = 0 if probe_ix is None else len(probe_ix)
        ix = iv = f = None
        if npb:
            ix = np.ascontiguousarray(probe_ix, dtype=np.int64)
            iv = np.ascontiguousarray(probe_iv, dtype=np.int64)
            f = np.empty(npb, dtype=np.float64)
        self._check(lib().dlr_moments(self.h, ctypes.byref(m), npb, _ptr(ix), _ptr(iv), _ptr(f)), "dlr_moments")
        out = {"mass": m.mass, "momentum": list(m.momentum), "kinetic_energy": m.kinetic_energy,
               "electric_energy": m.electric_energy, "s_fro": m.s_fro, "qr_fallbacks": m.qr_fallbacks,
               "nonfinite": m.nonfinite, "qr_third_stage": m.qr_third_stage, "eig_unconverged": m.eig_unconverged}
        return (out, f) if npb else out

    def get_factors(self, out=None):
        """(X, S, V) as Fortran-ordered numpy arrays; with out = (X, S, V) host tensors/arrays of r*N, r*r, r*N doubles
        in the ABI's column-major layout (e.g. pinned torch tensors of shape (r, N)) the copy goes there instead"""
        if out is not None:
            X, S, V = out
            self._check(lib().dlr_get_factors(self.h, _ptr(X), _ptr(S), _ptr(V), 0), "dlr_get_factors")
            return out
        X = np.empty((self.Nx, self.r), order="F")
        S = np.empty((self.r, self.r), order="F")
        V = np.empty((self.Nv, self.r), order="F")
        self._check(lib().dlr_get_factors(self.h, _ptr(X), _ptr(S), _ptr(V), 0), "dlr_get_factors")
        return X, S, V

    def get_field(self):
        E = np.empty((3, self.Nx))
        self._check(lib().dlr_get_field(self.h, _ptr(E), 0), "dlr_get_field")
        return E

    def clear_error(self):
        self._check(lib().dlr_clear_error(self.h), "dlr_clear_error")

    def set_profiling(self, on):
        self._check(lib().dlr_set_profiling(self.h, int(on)), "dlr_set_profiling")

    def phase_times(self):
        cap = 512
        ms = (ctypes.c_float * cap)()
        names = (ctypes.c_char_p * cap)()
        n = lib().dlr_get_phase_times(self.h, cap, ms, names)
        return [(names[i].decode(), ms[i]) for i in range(n)]

    def launches_per_step(self):
        return lib().dlr_launches_per_step(self.h)

    def bytes_per_step(self):
        return lib().dlr_bytes_per_step(self.h)

    def test_fft_roundtrip(self, which, A):
        """A: (N, ncols) Fortran-order numpy -> (roundtrip, spectrum as complex array [ncols, n, n, n/2+1] in the
        library's internal layout)"""
        torch = self.torch
        n = (self.cfg.n_v if which else self.cfg.n_x)[0]
        ncols = A.shape[1]
        d_in = torch.from_numpy(np.ascontiguousarray(A.T)).to(self.device)
        d_out = torch.empty_like(d_in)
        d_spec = torch.empty(ncols * (n // 2 + 1) * n * n * 2, dtype=torch.float64, device=self.device)
        self._check(lib().dlr_test_fft_roundtrip(self.h, which, ncols, d_in.data_ptr(), d_out.data_ptr(),
                                                 d_spec.data_ptr()), "dlr_test_fft_roundtrip")
        spec = d_spec.cpu().numpy().view(np.complex128).reshape(ncols, n, n, n // 2 + 1)
        return np.asfortranarray(d_out.cpu().numpy().T), spec

    def test_dir_pass(self, which, kind, A, tabs, min_=None, mout=None, Q=None, E=None):
        """one directional pass (include/dlr.h): A (N, r) Fortran-order numpy -> result of the same shape;
        tabs: complex (ntab, n, r) in natural DFT order; min_, mout (r, r) [cin][cout]; Q (3, r, r); E (3, N_x)"""
        torch = self.torch
        d_in = torch.from_numpy(np.ascontiguousarray(A.T)).to(self.device)
        d_out = torch.empty_like(d_in)
        d_E = None if E is None else torch.from_numpy(np.ascontiguousarray(E)).to(self.device)
        c = lambda a, dt=np.float64: None if a is None else np.ascontiguousarray(a, dtype=dt)
        tabs, min_, mout, Q = c(tabs, np.complex128), c(min_), c(mout), c(Q)
        self._check(lib().dlr_test_dir_pass(self.h, which, kind, d_in.data_ptr(), d_out.data_ptr(), _ptr(min_), _ptr(mout),
                                            _ptr(tabs), _ptr(Q), _ptr(d_E)), "dlr_test_dir_pass")
        return np.asfortranarray(d_out.cpu().numpy().T)

    def test_chol_decide(self, G):
        """does the adaptive CholeskyQR ask for a third stage, given the (r, r) Gram matrix of the once-orthogonalised
        factor?"""
        r = self.r
        up = np.ascontiguousarray([G[i, j] for i in range(r) for j in range(i, r)], dtype=np.float64)
        out = ctypes.c_int(0)
        self._check(lib().dlr_test_chol_decide(self.h, _ptr(up), ctypes.byref(out)), "dlr_test_chol_decide")
        return bool(out.value)

    def close(self):
        if getattr(self, "h", None):
            self.torch.cuda.synchronize(self.device)
            lib().dlr_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

"""Thin ctypes binding of libsn.so (include/sn.h) -- argument marshalling only.

PyTorch is used for exactly two things: the device workspace (one uint8 tensor) and the CUDA
stream.  Every step of the split-step path (eq. (1),(2)) runs in
the library's hand-written sm_100a kernels.  There is no CPU fallback: if libsn.so is missing
or no CUDA device is present this module raises.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsn.so")

SN_OK = 0
ERR_NAMES = {-1: "SN_ERR_NULL", -2: "SN_ERR_DIMS", -3: "SN_ERR_PARAM", -4: "SN_ERR_SINGULAR",
             -5: "SN_ERR_WORKSPACE", -6: "SN_ERR_STATE", -7: "SN_ERR_CUDA", -8: "SN_ERR_NOMEM", -9: "SN_ERR_FEATURE",
             -10: "SN_ERR_TOO_LARGE"}

# optional workspace regions (sn_options.features)
FEAT_STAGING, FEAT_VEXT, FEAT_SOURCE, FEAT_ALL = 1, 2, 4, 7
# sn_set_option
OPT_GRAPH, OPT_DISPATCH, OPT_GRAPH_STEPS, OPT_RESIDENT = 1, 2, 3, 4
DISPATCH_DEFAULT, DISPATCH_FIRST_PATH, DISPATCH_PIPELINED = 0, 1, 2

# every symbol include/sn.h declares
EXPORTS = ("sn_workspace_bytes", "sn_create", "sn_set_state", "sn_step", "sn_get_state", "sn_diagnostics",
           "sn_set_dtau", "sn_destroy", "sn_strerror", "sn_launch_count", "sn_profile", "sn_profile_read",
           "sn_debug_fft", "sn_debug_potential", "sn_set_local_terms", "sn_set_external_potential", "sn_set_source_tables", "sn_step_order4", "sn_workspace_bytes_batch", "sn_create_batch", "sn_set_bohm", "sn_workspace_bytes_opt",
           "sn_create_opt", "sn_set_option", "sn_workspace_bytes_mc", "sn_create_mc", "sn_mc_norms",
           "sn_slab_workspace_bytes", "sn_slab_create", "sn_slab_stage", "sn_slab_buffer", "sn_slab_pack",
           "sn_slab_exchange_local", "sn_slab_local_norm", "sn_norm_static")

PASS_KINDS = ("S_FFT", "S_KIN", "S_KDIAG", "H_NLKIN", "H_R2C", "H_POT", "H_DIAG", "X_FFT", "X_KIN", "X_POISSON",
              "X_KDIAG", "H_SRC", "H_BOHM", "H_R2C_MC", "H_NL_MC", "R_STEPS")


class SnDiag(ctypes.Structure):
    _fields_ = [("norm", ctypes.c_double), ("e_kin", ctypes.c_double), ("e_nonlocal", ctypes.c_double),
                ("e_local", ctypes.c_double), ("e_total", ctypes.c_double)]


class SnOptions(ctypes.Structure):
    _fields_ = [("struct_size", ctypes.c_size_t), ("batch", ctypes.c_int64), ("features", ctypes.c_uint32),
                ("dtype", ctypes.c_uint32)]


DTYPE_C64, DTYPE_C128 = 0, 1
_DTYPES = {"complex64": DTYPE_C64, "c64": DTYPE_C64, "complex128": DTYPE_C128, "c128": DTYPE_C128}


def _options(batch: int, features: int, dtype: int = DTYPE_C64) -> SnOptions:
    return SnOptions(ctypes.sizeof(SnOptions), int(batch), int(features), int(dtype))


class SnError(RuntimeError):
    def __init__(self, code: int, what: str, text: str = ""):
        super().__init__(f"{what}: {ERR_NAMES.get(code, code)} {text}".strip())
        self.code = code


_lib: Optional[ctypes.CDLL] = None


def lib() -> ctypes.CDLL:
    """Load libsn.so (built by paper_1909_08354_b200.build); fail loudly if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} not built: run `python -m paper_1909_08354_b200.build` "
                              "(there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        vp, i64p, dp = ctypes.c_void_p, ctypes.POINTER(ctypes.c_int64), ctypes.POINTER(ctypes.c_double)
        L.sn_workspace_bytes.argtypes = [ctypes.c_int, i64p]
        L.sn_workspace_bytes.restype = ctypes.c_size_t
        L.sn_create.argtypes = [ctypes.POINTER(vp), ctypes.c_int, i64p, dp, ctypes.c_double, ctypes.c_double,
                                ctypes.c_double, ctypes.c_double, dp, ctypes.c_int, ctypes.c_double, vp,
                                ctypes.c_size_t, vp]
        L.sn_workspace_bytes_batch.argtypes = [ctypes.c_int, i64p, ctypes.c_int64]
        L.sn_workspace_bytes_batch.restype = ctypes.c_size_t
        L.sn_create_batch.argtypes = [ctypes.POINTER(vp), ctypes.c_int, i64p, ctypes.c_int64, dp, ctypes.c_double,
                                      ctypes.c_double, ctypes.c_double, ctypes.c_double, dp, ctypes.c_int,
                                      ctypes.c_double, vp, ctypes.c_size_t, vp]
        L.sn_workspace_bytes_opt.argtypes = [ctypes.c_int, i64p, ctypes.POINTER(SnOptions)]
        L.sn_workspace_bytes_opt.restype = ctypes.c_size_t
        L.sn_create_opt.argtypes = [ctypes.POINTER(vp), ctypes.c_int, i64p, dp, ctypes.c_double, ctypes.c_double,
                                    ctypes.c_double, ctypes.c_double, dp, ctypes.c_int, ctypes.c_double, vp,
                                    ctypes.c_size_t, vp, ctypes.POINTER(SnOptions)]
        L.sn_set_option.argtypes = [vp, ctypes.c_int, ctypes.c_int]
        L.sn_workspace_bytes_mc.argtypes = [ctypes.c_int, i64p, ctypes.c_int]
        L.sn_workspace_bytes_mc.restype = ctypes.c_size_t
        L.sn_create_mc.argtypes = [ctypes.POINTER(vp), ctypes.c_int, i64p, dp, ctypes.c_int, dp, dp, ctypes.c_double,
                                   ctypes.c_double, dp, dp, ctypes.c_double, vp, ctypes.c_size_t, vp]
        L.sn_mc_norms.argtypes = [vp, dp]
        L.sn_norm_static.argtypes = [vp, ctypes.c_int64, ctypes.c_double, vp, vp]
        L.sn_set_state.argtypes = [vp, vp, ctypes.c_int]
        L.sn_step.argtypes = [vp, ctypes.c_int64]
        L.sn_step_order4.argtypes = [vp, ctypes.c_int64]
        L.sn_get_state.argtypes = [vp, vp, ctypes.c_int]
        L.sn_diagnostics.argtypes = [vp, ctypes.POINTER(SnDiag)]
        L.sn_set_dtau.argtypes = [vp, ctypes.c_double]
        L.sn_destroy.argtypes = [vp]
        L.sn_strerror.argtypes = [ctypes.c_int]
        L.sn_strerror.restype = ctypes.c_char_p
        L.sn_launch_count.argtypes = [vp]
        L.sn_launch_count.restype = ctypes.c_int64
        L.sn_profile.argtypes = [vp, ctypes.c_int]
        L.sn_profile_read.argtypes = [vp, dp, i64p, ctypes.c_int]
        L.sn_debug_fft.argtypes = [vp, ctypes.c_int]
        L.sn_debug_potential.argtypes = [vp, vp, ctypes.c_int]
        L.sn_set_local_terms.argtypes = [vp, ctypes.c_double, ctypes.c_double, ctypes.c_double, ctypes.c_double]
        L.sn_set_external_potential.argtypes = [vp, vp, ctypes.c_int]
        L.sn_set_source_tables.argtypes = [vp, vp, vp, ctypes.c_int]
        L.sn_set_bohm.argtypes = [vp, ctypes.c_double, ctypes.c_double]
        _lib = L
    return _lib


def _chk(rc: int, what: str) -> None:
    if rc != SN_OK:
        raise SnError(rc, what, lib().sn_strerror(rc).decode())


def workspace_bytes(dims: Sequence[int], batch: int = 1, features: int = 0, dtype: str = "complex64") -> int:
    d = (ctypes.c_int64 * len(dims))(*[int(n) for n in dims])
    opt = _options(batch, features, _DTYPES[dtype])
    return int(lib().sn_workspace_bytes_opt(len(dims), d, ctypes.byref(opt)))


STATIC_NORM_MAX_CELLS = 1 << 28


def norm_static(psi, dv: float, out, n_cells: Optional[int] = None, stream=None) -> None:
    """sn_norm_static: out[0] = dv * sum |psi|^2 for a complex64 CUDA tensor psi, written to the float64 CUDA tensor `out`
    (one element, caller-allocated).  No context, no workspace, no allocation: the scratch is a static device array of
    the library (limit STATIC_NORM_MAX_CELLS cells; calls that overlap on the GPU race on it).  Asynchronous.
    n_cells overrides psi.numel() (the tests pass an oversized count to check that it is rejected)."""
    import torch
    assert psi.is_cuda and psi.dtype == torch.complex64 and psi.is_contiguous()
    assert out.is_cuda and out.dtype == torch.float64 and out.numel() >= 1 and out.device == psi.device
    st = stream if stream is not None else torch.cuda.current_stream(psi.device)
    _chk(lib().sn_norm_static(ctypes.c_void_p(psi.data_ptr()), int(psi.numel() if n_cells is None else n_cells), float(dv),
                              ctypes.c_void_p(out.data_ptr()), ctypes.c_void_p(st.cuda_stream)), "sn_norm_static")


class Simulation:
    """One sn_ctx plus the torch tensor that backs its workspace."""

    def __init__(self, dims: Sequence[int], L, A: float, B: float, C: float, D: float, g: Sequence[float],
                 dtau: float, device: str = "cuda:0", stream=None, batch: Optional[int] = None, features: int = 0,
                 dtype: str = "complex64", workspace=None):
        """batch=None: one 2D/3D system of shape dims.  batch=B: an ensemble of B systems; every array then has the
        STORAGE shape (dims[0], B, dims[1][, dims[2]]) (member b at [:, b, ...]).  features: FEAT_* bits, the optional
        workspace regions (external potential table, source tables, host staging); 0 = the stepper alone, ~12 B/cell.
        dtype: "complex64" (default) or "complex128" -- the precision of the state and of all arithmetic.
        workspace: a caller-owned, 256-byte aligned torch uint8 CUDA tensor of at least workspace_bytes(...) bytes to
        use instead of allocating one (the tests hand in the middle of a larger, poisoned buffer)."""
        import torch

        if not torch.cuda.is_available():
            raise RuntimeError("paper_1909_08354_b200 needs a CUDA device (no CPU fallback)")
        pd = tuple(int(n) for n in dims)
        nd = len(pd)
        self.dims = pd if batch is None else (pd[0], int(batch)) + pd[1:]   # storage shape of every array
        self.features = int(features)
        self.dtype = np.dtype(np.complex128 if _DTYPES[dtype] == DTYPE_C128 else np.complex64)
        self.real_dtype = np.dtype(np.float64 if _DTYPES[dtype] == DTYPE_C128 else np.float32)
        Ls = [float(L)] * nd if np.isscalar(L) else [float(v) for v in L]
        g = [float(v) for v in g]
        self.device = torch.device(device)
        opt = _options(1 if batch is None else int(batch), features, _DTYPES[dtype])
        c_dims = (ctypes.c_int64 * nd)(*pd)
        nbytes = int(lib().sn_workspace_bytes_opt(nd, c_dims, ctypes.byref(opt)))
        if nbytes == 0:
            raise SnError(-2, "sn_workspace_bytes_opt", lib().sn_strerror(-2).decode())
        with torch.cuda.device(self.device):
            self._ws = workspace if workspace is not None else torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            self._stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self._h = ctypes.c_void_p()
        c_L = (ctypes.c_double * nd)(*Ls)
        c_g = (ctypes.c_double * max(1, len(g)))(*(g or [0.0]))
        # the library runs every call on the device that owns the workspace, whatever device is current here
        _chk(lib().sn_create_opt(ctypes.byref(self._h), nd, c_dims, c_L, A, B, C, D, c_g, len(g), dtau,
                                 ctypes.c_void_p(self._ws.data_ptr()), nbytes,
                                 ctypes.c_void_p(self._stream.cuda_stream), ctypes.byref(opt)), "sn_create_opt")

    @classmethod
    def from_config(cls, cfg, **kw) -> "Simulation":
        return cls(cfg.dims, cfg.L, cfg.A, cfg.B, cfg.C, cfg.D, cfg.g, cfg.dtau, **kw)

    @property
    def cells(self) -> int:
        return int(np.prod(self.dims))

    def close(self) -> None:
        if getattr(self, "_h", None):
            lib().sn_destroy(self._h)
            self._h = ctypes.c_void_p()
            self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- state ------------------------------------------------------------------------------
    def set_state(self, psi) -> None:
        """psi: numpy array (host) or torch CUDA / host tensor of the context's complex dtype, shape == dims."""
        if isinstance(psi, np.ndarray):
            a = np.ascontiguousarray(psi, dtype=self.dtype)
            assert a.shape == self.dims, (a.shape, self.dims)
            _chk(lib().sn_set_state(self._h, ctypes.c_void_p(a.ctypes.data), 0), "sn_set_state")
        else:
            import torch
            tdt = torch.complex128 if self.dtype == np.complex128 else torch.complex64
            assert psi.dtype == tdt and psi.is_contiguous() and tuple(psi.shape) == self.dims
            _chk(lib().sn_set_state(self._h, ctypes.c_void_p(psi.data_ptr()), 1 if psi.is_cuda else 0), "sn_set_state")

    def get_state(self, out=None):
        """Return the state as a numpy array of the context's dtype, or fill `out` (numpy / torch host or CUDA tensor)."""
        if out is None:
            out = np.empty(self.dims, dtype=self.dtype)
        if isinstance(out, np.ndarray):
            assert out.dtype == self.dtype and out.flags.c_contiguous and out.shape == self.dims
            _chk(lib().sn_get_state(self._h, ctypes.c_void_p(out.ctypes.data), 0), "sn_get_state")
        else:
            _chk(lib().sn_get_state(self._h, ctypes.c_void_p(out.data_ptr()), 1 if out.is_cuda else 0),
                 "sn_get_state")
        return out

    # -- the path ---------------------------------------------------------------------------
    def step(self, n: int) -> None:
        _chk(lib().sn_step(self._h, int(n)), "sn_step")

    def step_order4(self, n: int) -> None:
        """n fourth-order steps (Yoshida composition of three Strang steps each)."""
        _chk(lib().sn_step_order4(self._h, int(n)), "sn_step_order4")

    def set_dtau(self, dtau: float) -> None:
        _chk(lib().sn_set_dtau(self._h, float(dtau)), "sn_set_dtau")

    def set_local_terms(self, g_log: float = 0.0, rho_floor: float = 1e-30, g_pow: float = 0.0,
                        p_pow: float = 1.0) -> None:
        """G(rho) += g_log ln(max(rho, rho_floor)) + g_pow max(rho, rho_floor)**p_pow (eq. (16))."""
        _chk(lib().sn_set_local_terms(self._h, float(g_log), float(rho_floor), float(g_pow), float(p_pow)),
             "sn_set_local_terms")

    def set_external_potential(self, v) -> None:
        """Fixed external potential V(x): numpy float32 array (host), torch float32 CUDA tensor, or None."""
        if v is None:
            _chk(lib().sn_set_external_potential(self._h, None, 0), "sn_set_external_potential")
        elif isinstance(v, np.ndarray):
            a = np.ascontiguousarray(v, dtype=np.float32)
            assert a.shape == self.dims, (a.shape, self.dims)
            _chk(lib().sn_set_external_potential(self._h, ctypes.c_void_p(a.ctypes.data), 0),
                 "sn_set_external_potential")
        else:
            import torch
            assert v.dtype == torch.float32 and v.is_contiguous() and tuple(v.shape) == self.dims
            _chk(lib().sn_set_external_potential(self._h, ctypes.c_void_p(v.data_ptr()), 1 if v.is_cuda else 0),
                 "sn_set_external_potential")

    def set_bohm(self, c_bohm: float, sqrt_floor: float = 1e-30) -> None:
        """c_bohm * V_B in the N sub-step, V_B = lap sqrt(rho)/(2 max(sqrt(rho), sqrt_floor)) (eq. (15))."""
        _chk(lib().sn_set_bohm(self._h, float(c_bohm), float(sqrt_floor)), "sn_set_bohm")

    def set_source_tables(self, beta, gamma) -> None:
        """eq. (12): lap phi + C phi = D (gamma(x) rho + beta(x) lap rho); numpy float32 arrays or CUDA float32
        tensors of shape dims; (None, None) restores eq. (2)."""
        if beta is None and gamma is None:
            _chk(lib().sn_set_source_tables(self._h, None, None, 0), "sn_set_source_tables")
        elif isinstance(beta, np.ndarray):
            b = np.ascontiguousarray(beta, dtype=np.float32)
            g = np.ascontiguousarray(gamma, dtype=np.float32)
            assert b.shape == self.dims and g.shape == self.dims
            if self.features & FEAT_STAGING:
                _chk(lib().sn_set_source_tables(self._h, ctypes.c_void_p(b.ctypes.data), ctypes.c_void_p(g.ctypes.data), 0),
                     "sn_set_source_tables")
            else:  # no staging region in the workspace: hand the library device copies
                import torch
                with torch.cuda.device(self.device), torch.cuda.stream(self._stream):
                    db, dg = torch.from_numpy(b).to(self.device), torch.from_numpy(g).to(self.device)
                    _chk(lib().sn_set_source_tables(self._h, ctypes.c_void_p(db.data_ptr()),
                                                    ctypes.c_void_p(dg.data_ptr()), 1), "sn_set_source_tables")
                    self._stream.synchronize()
        else:
            assert beta.is_cuda and gamma.is_cuda and beta.is_contiguous() and gamma.is_contiguous()
            assert tuple(beta.shape) == self.dims and tuple(gamma.shape) == self.dims
            _chk(lib().sn_set_source_tables(self._h, ctypes.c_void_p(beta.data_ptr()),
                                            ctypes.c_void_p(gamma.data_ptr()), 1), "sn_set_source_tables")

    def _set_source_tables_host(self, beta: np.ndarray, gamma: np.ndarray) -> None:
        """sn_set_source_tables with HOST pointers, whatever the features (used by the tests of SN_ERR_FEATURE)."""
        b = np.ascontiguousarray(beta, dtype=np.float32)
        g = np.ascontiguousarray(gamma, dtype=np.float32)
        _chk(lib().sn_set_source_tables(self._h, ctypes.c_void_p(b.ctypes.data), ctypes.c_void_p(g.ctypes.data), 0),
             "sn_set_source_tables")

    def diagnostics(self) -> dict:
        d = SnDiag()
        _chk(lib().sn_diagnostics(self._h, ctypes.byref(d)), "sn_diagnostics")
        return {k: getattr(d, k) for k, _ in SnDiag._fields_}

    def set_option(self, option: int, value: int) -> None:
        """OPT_GRAPH 0/1; OPT_DISPATCH DISPATCH_DEFAULT / DISPATCH_FIRST_PATH / DISPATCH_PIPELINED; OPT_RESIDENT 0/1 (A/B runs, tests)."""
        _chk(lib().sn_set_option(self._h, int(option), int(value)), "sn_set_option")

    def launch_count(self) -> int:
        return int(lib().sn_launch_count(self._h))

    def profile(self, enable: bool) -> None:
        _chk(lib().sn_profile(self._h, 1 if enable else 0), "sn_profile")

    def profile_read(self, reset: bool = True) -> dict:
        """{pass kind: (summed device ms, launches)} for kinds that ran."""
        n = len(PASS_KINDS)
        ms = (ctypes.c_double * n)()
        cnt = (ctypes.c_int64 * n)()
        _chk(lib().sn_profile_read(self._h, ms, cnt, 1 if reset else 0), "sn_profile_read")
        return {PASS_KINDS[k]: (float(ms[k]), int(cnt[k])) for k in range(n) if cnt[k]}

    # -- test hooks ---------------------------------------------------------------------------
    def debug_fft(self, direction: int) -> None:
        _chk(lib().sn_debug_fft(self._h, int(direction)), "sn_debug_fft")

    def debug_potential(self) -> np.ndarray:
        """phi of eq. (2) for the current state, as a numpy float32 array (written to a device tensor by the library,
        copied to the host by torch; with FEAT_STAGING the library copies it itself)."""
        if self.features & FEAT_STAGING:
            out = np.empty(self.dims, dtype=self.real_dtype)
            _chk(lib().sn_debug_potential(self._h, ctypes.c_void_p(out.ctypes.data), 0), "sn_debug_potential")
            return out
        import torch
        with torch.cuda.device(self.device), torch.cuda.stream(self._stream):
            dev = torch.empty(self.dims, dtype=torch.float64 if self.real_dtype == np.float64 else torch.float32,
                              device=self.device)
            _chk(lib().sn_debug_potential(self._h, ctypes.c_void_p(dev.data_ptr()), 1), "sn_debug_potential")
            return dev.cpu().numpy()


class CoupledSimulation(Simulation):
    """Coupled wave functions (sn_create_mc, reading Q18 of DESIGN.md): state shape (M,) + dims, complex64.
    i dpsi_c/dtau = A_c lap psi_c + B_c phi psi_c + (sum_c' g[c][c'] |psi_c'|^2) psi_c; lap phi + C phi = D sum_c w_c |psi_c|^2."""

    def __init__(self, dims: Sequence[int], L, A: Sequence[float], B: Sequence[float], C: float, D: float,
                 w: Sequence[float], g, dtau: float, device: str = "cuda:0", stream=None):
        import torch

        if not torch.cuda.is_available():
            raise RuntimeError("paper_1909_08354_b200 needs a CUDA device (no CPU fallback)")
        pd = tuple(int(n) for n in dims)
        nd, M = len(pd), len(A)
        gm = np.ascontiguousarray(g, dtype=np.float64)
        assert gm.shape == (M, M) and len(B) == M and len(w) == M
        self.dims = (M,) + pd
        self.features = 0
        self.dtype, self.real_dtype = np.dtype(np.complex64), np.dtype(np.float32)
        Ls = [float(L)] * nd if np.isscalar(L) else [float(v) for v in L]
        self.device = torch.device(device)
        c_dims = (ctypes.c_int64 * nd)(*pd)
        nbytes = int(lib().sn_workspace_bytes_mc(nd, c_dims, M))
        if nbytes == 0:
            raise SnError(-2, "sn_workspace_bytes_mc", lib().sn_strerror(-2).decode())
        with torch.cuda.device(self.device):
            self._ws = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            self._stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self._h = ctypes.c_void_p()
        arr = lambda v: (ctypes.c_double * len(v))(*[float(x) for x in v])
        _chk(lib().sn_create_mc(ctypes.byref(self._h), nd, c_dims, arr(Ls), M, arr(A), arr(B), C, D, arr(w),
                                arr(gm.ravel()), dtau, ctypes.c_void_p(self._ws.data_ptr()), nbytes,
                                ctypes.c_void_p(self._stream.cuda_stream)), "sn_create_mc")

    def norms(self) -> np.ndarray:
        out = (ctypes.c_double * self.dims[0])()
        _chk(lib().sn_mc_norms(self._h, out), "sn_mc_norms")
        return np.array(out[:])

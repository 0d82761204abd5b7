"""ctypes loader for the float64 CPU oracle (oracle/snref.c).

TEST INFRASTRUCTURE: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this.  It imports nothing from the CUDA package.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libsnref.so")
_SRC = os.path.join(_HERE, "snref.c")
_lib: Optional[ctypes.CDLL] = None


class SnrefDiag(ctypes.Structure):
    _fields_ = [("norm", ctypes.c_double), ("e_kin", ctypes.c_double), ("e_nonlocal", ctypes.c_double),
                ("e_local", ctypes.c_double), ("e_total", ctypes.c_double)]


def build(force: bool = False) -> str:
    """Compile oracle/snref.c -> oracle/libsnref.so (gcc -O2 -fopenmp)."""
    if force or not os.path.exists(_LIB_PATH) or os.path.getmtime(_LIB_PATH) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-std=gnu99", "-fPIC", "-shared", "-o", _LIB_PATH, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB_PATH


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_LIB_PATH)
        vp, i64p, dp = ctypes.c_void_p, ctypes.POINTER(ctypes.c_int64), ctypes.POINTER(ctypes.c_double)
        L.snref_fft1d.argtypes = [vp, ctypes.c_int64, ctypes.c_int]
        L.snref_fftn.argtypes = [vp, ctypes.c_int, i64p, ctypes.c_int]
        L.snref_create.argtypes = [ctypes.POINTER(vp), ctypes.c_int, i64p, dp, ctypes.c_double, ctypes.c_double,
                                   ctypes.c_double, ctypes.c_double, dp, ctypes.c_int, ctypes.c_double]
        L.snref_destroy.argtypes = [vp]
        L.snref_set_dtau.argtypes = [vp, ctypes.c_double]
        L.snref_set_state.argtypes = [vp, vp]
        L.snref_get_state.argtypes = [vp, vp]
        L.snref_step.argtypes = [vp, ctypes.c_int64]
        L.snref_step_order4.argtypes = [vp, ctypes.c_int64]
        L.snref_potential.argtypes = [vp, vp]
        L.snref_diagnostics.argtypes = [vp, ctypes.POINTER(SnrefDiag)]
        L.snref_set_local_terms.argtypes = [vp, ctypes.c_double, ctypes.c_double, ctypes.c_double, ctypes.c_double]
        L.snref_set_external_potential.argtypes = [vp, vp]
        L.snref_set_source_tables.argtypes = [vp, vp, vp]
        L.snref_set_bohm.argtypes = [vp, ctypes.c_double, ctypes.c_double]
        L.snref_bohm_potential.argtypes = [vp, vp]
        L.snref_mc_create.argtypes = [ctypes.POINTER(vp), ctypes.c_int, i64p, dp, ctypes.c_int, dp, dp, ctypes.c_double,
                                      ctypes.c_double, dp, dp, ctypes.c_double]
        L.snref_mc_destroy.argtypes = [vp]
        L.snref_mc_set_dtau.argtypes = [vp, ctypes.c_double]
        L.snref_mc_set_state.argtypes = [vp, vp]
        L.snref_mc_get_state.argtypes = [vp, vp]
        L.snref_mc_step.argtypes = [vp, ctypes.c_int64]
        L.snref_mc_norms.argtypes = [vp, dp]
        L.snref_num_threads.restype = ctypes.c_int
        L.snref_set_num_threads.argtypes = [ctypes.c_int]
        _lib = L
    return _lib


class OracleError(RuntimeError):
    def __init__(self, code: int, what: str):
        super().__init__(f"{what} failed with oracle code {code}")
        self.code = code


def _chk(rc: int, what: str) -> None:
    if rc != 0:
        raise OracleError(rc, what)


def fft1d(x: np.ndarray, direction: int) -> np.ndarray:
    a = np.ascontiguousarray(x, dtype=np.complex128).copy()
    _chk(lib().snref_fft1d(a.ctypes.data, a.size, direction), "snref_fft1d")
    return a


def fftn(x: np.ndarray, direction: int) -> np.ndarray:
    a = np.ascontiguousarray(x, dtype=np.complex128).copy()
    dims = (ctypes.c_int64 * a.ndim)(*a.shape)
    _chk(lib().snref_fftn(a.ctypes.data, a.ndim, dims, direction), "snref_fftn")
    return a


def num_threads() -> int:
    return int(lib().snref_num_threads())


def set_num_threads(n: int) -> None:
    lib().snref_set_num_threads(int(n))


class Oracle:
    """One float64 simulation context (snref_ctx)."""

    def __init__(self, dims: Sequence[int], L, A: float, B: float, C: float, D: float,
                 g: Sequence[float], dtau: float):
        self.dims = tuple(int(n) for n in dims)
        nd = len(self.dims)
        Ls = [float(L)] * nd if np.isscalar(L) else [float(v) for v in L]
        self.L = tuple(Ls)
        g = [float(v) for v in g]
        self._h = ctypes.c_void_p()
        c_dims = (ctypes.c_int64 * nd)(*self.dims)
        c_L = (ctypes.c_double * nd)(*Ls)
        c_g = (ctypes.c_double * max(1, len(g)))(*g) if g else (ctypes.c_double * 1)(0.0)
        _chk(lib().snref_create(ctypes.byref(self._h), nd, c_dims, c_L, A, B, C, D, c_g, len(g), dtau),
             "snref_create")

    @classmethod
    def from_config(cls, cfg) -> "Oracle":
        return cls(cfg.dims, cfg.L, cfg.A, cfg.B, cfg.C, cfg.D, cfg.g, cfg.dtau)

    def close(self) -> None:
        if self._h:
            lib().snref_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_state(self, psi: np.ndarray) -> None:
        a = np.ascontiguousarray(psi, dtype=np.complex128)
        assert a.shape == self.dims, (a.shape, self.dims)
        _chk(lib().snref_set_state(self._h, a.ctypes.data), "snref_set_state")

    def get_state(self) -> np.ndarray:
        out = np.empty(self.dims, dtype=np.complex128)
        _chk(lib().snref_get_state(self._h, out.ctypes.data), "snref_get_state")
        return out

    def step(self, n: int) -> None:
        _chk(lib().snref_step(self._h, int(n)), "snref_step")

    def step_order4(self, n: int) -> None:
        _chk(lib().snref_step_order4(self._h, int(n)), "snref_step_order4")

    def set_dtau(self, dtau: float) -> None:
        _chk(lib().snref_set_dtau(self._h, float(dtau)), "snref_set_dtau")

    def set_local_terms(self, g_log: float = 0.0, rho_floor: float = 1e-30, g_pow: float = 0.0,
                        p_pow: float = 1.0) -> None:
        """G(rho) += g_log ln(max(rho, rho_floor)) + g_pow max(rho, rho_floor)**p_pow (eq. (16))."""
        _chk(lib().snref_set_local_terms(self._h, g_log, rho_floor, g_pow, p_pow), "snref_set_local_terms")

    def set_external_potential(self, v) -> None:
        """Fixed external potential V(x) added to the N sub-step phase (phi_C of eq. (15)); None removes it."""
        if v is None:
            _chk(lib().snref_set_external_potential(self._h, None), "snref_set_external_potential")
            return
        a = np.ascontiguousarray(v, dtype=np.float64)
        assert a.shape == self.dims, (a.shape, self.dims)
        _chk(lib().snref_set_external_potential(self._h, a.ctypes.data), "snref_set_external_potential")

    def set_source_tables(self, beta, gamma) -> None:
        """eq. (12): lap phi + C phi = D (gamma(x) rho + beta(x) lap rho); (None, None) restores eq. (2)."""
        if beta is None and gamma is None:
            _chk(lib().snref_set_source_tables(self._h, None, None), "snref_set_source_tables")
            return
        b = np.ascontiguousarray(beta, dtype=np.float64)
        g = np.ascontiguousarray(gamma, dtype=np.float64)
        assert b.shape == self.dims and g.shape == self.dims
        _chk(lib().snref_set_source_tables(self._h, b.ctypes.data, g.ctypes.data), "snref_set_source_tables")

    def set_bohm(self, c_bohm: float, sqrt_floor: float = 1e-30) -> None:
        """c_B * V_B added to the N sub-step, V_B = lap sqrt(rho)/(2 max(sqrt(rho), sqrt_floor)) (eq. (15))."""
        _chk(lib().snref_set_bohm(self._h, float(c_bohm), float(sqrt_floor)), "snref_set_bohm")

    def bohm_potential(self) -> np.ndarray:
        out = np.empty(self.dims, dtype=np.float64)
        _chk(lib().snref_bohm_potential(self._h, out.ctypes.data), "snref_bohm_potential")
        return out

    def potential(self) -> np.ndarray:
        out = np.empty(self.dims, dtype=np.float64)
        _chk(lib().snref_potential(self._h, out.ctypes.data), "snref_potential")
        return out

    def diagnostics(self) -> dict:
        d = SnrefDiag()
        _chk(lib().snref_diagnostics(self._h, ctypes.byref(d)), "snref_diagnostics")
        return {k: getattr(d, k) for k, _ in SnrefDiag._fields_}


class OracleMC:
    """Coupled wave functions (NEXT-4b, reading Q18): state shape (M,) + dims, complex128."""

    def __init__(self, dims: Sequence[int], L, A: Sequence[float], B: Sequence[float], C: float, D: float,
                 w: Sequence[float], g, dtau: float):
        self.dims = tuple(int(n) for n in dims)
        nd = len(self.dims)
        self.M = len(A)
        Ls = [float(L)] * nd if np.isscalar(L) else [float(v) for v in L]
        gm = np.ascontiguousarray(g, dtype=np.float64)
        assert gm.shape == (self.M, self.M) and len(B) == self.M and len(w) == self.M
        self._h = ctypes.c_void_p()
        arr = lambda v: (ctypes.c_double * len(v))(*[float(x) for x in v])
        _chk(lib().snref_mc_create(ctypes.byref(self._h), nd, (ctypes.c_int64 * nd)(*self.dims), arr(Ls), self.M,
                                   arr(A), arr(B), C, D, arr(w), arr(gm.ravel()), dtau), "snref_mc_create")

    def close(self) -> None:
        if self._h:
            lib().snref_mc_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_state(self, psi: np.ndarray) -> None:
        a = np.ascontiguousarray(psi, dtype=np.complex128)
        assert a.shape == (self.M,) + self.dims, a.shape
        _chk(lib().snref_mc_set_state(self._h, a.ctypes.data), "snref_mc_set_state")

    def get_state(self) -> np.ndarray:
        out = np.empty((self.M,) + self.dims, dtype=np.complex128)
        _chk(lib().snref_mc_get_state(self._h, out.ctypes.data), "snref_mc_get_state")
        return out

    def step(self, n: int) -> None:
        _chk(lib().snref_mc_step(self._h, int(n)), "snref_mc_step")

    def set_dtau(self, dtau: float) -> None:
        _chk(lib().snref_mc_set_dtau(self._h, float(dtau)), "snref_mc_set_dtau")

    def norms(self) -> np.ndarray:
        out = (ctypes.c_double * self.M)()
        _chk(lib().snref_mc_norms(self._h, out), "snref_mc_norms")
        return np.array(out[:])

"""Seeded synthetic initial states and the BASELINE.json config table.

This module is shared by the float64 oracle (``oracle/``) and the CUDA path
(``paper_1909_08354_b200.sn``).  It holds NONE of the method's arithmetic: no
FFT, no phase, no Poisson solve -- only the recipe for the initial wave
function psi_0 of each BASELINE.json config and the
constants A, B, C, D, g, dtau that PAPER.md:42-46 (eq. (1),(2)) leaves free.

The paper measures on its own (unpublished) simulations, not on a public
dataset; BASELINE.json names none.  All states are synthetic: generated in
float64 from ``numpy.random.default_rng(seed)`` and rounded ONCE to complex64;
the same rounded array is handed to the GPU and (cast back up) to the oracle,
so input rounding is charged to neither side.

Axis convention: ``dims[0]`` is the slowest axis, ``dims[-1]`` the contiguous
one (C order).  Coordinates on every axis: x_j = -L/2 + j*L/N.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Callable, Dict, Tuple

import numpy as np


def coords(n: int, L: float) -> np.ndarray:
    """Grid coordinates x_j = -L/2 + j*L/N, j = 0..N-1."""
    return -0.5 * L + np.arange(n, dtype=np.float64) * (L / n)


def wrap(u: np.ndarray, L: float) -> np.ndarray:
    """Minimum-image displacement on a periodic box of length L."""
    return np.mod(u + 0.5 * L, L) - 0.5 * L


def _outer_sum(factors) -> np.ndarray:
    """sum_b  f_0[b,:] (x) f_1[b,:] (x) ... as one dense array.

    ``factors`` is a list (one per axis) of complex arrays [n_blob, N_axis].
    The blob family is separable per axis, so the d-dimensional state is a sum
    of rank-1 outer products; evaluated as a matrix product to stay cheap at
    512^3.
    """
    if len(factors) == 2:
        fy, fx = factors
        return fy.T @ fx
    fz, fy, fx = factors
    nb = fz.shape[0]
    zy = (fz[:, :, None] * fy[:, None, :]).reshape(nb, -1)      # [b, z*y]
    out = zy.T @ fx                                             # [z*y, x]
    return out.reshape(fz.shape[1], fy.shape[1], fx.shape[1])


def gaussian_blobs(dims, L, n_blob, w_range, a_range, sigma_v, seed) -> np.ndarray:
    """psi = sum_b a_b exp(-|d_b|^2/(2 w_b^2)) exp(i v_b . d_b), d_b = wrap(x - c_b).

    Draw order per blob: centre c = 0.6 L (U[0,1)^d - 0.5),
    width w, amplitude a, boost v ~ N(0, sigma_v^2)^d; component i of c and v
    belongs to axis i (axis 0 = slowest).
    """
    d = len(dims)
    rng = np.random.default_rng(seed)
    factors = [np.empty((n_blob, n), dtype=np.complex128) for n in dims]
    for b in range(n_blob):
        c = 0.6 * L * (rng.random(d) - 0.5)
        w = rng.uniform(*w_range)
        a = rng.uniform(*a_range)
        v = rng.normal(0.0, sigma_v, d)
        for ax in range(d):
            disp = wrap(coords(dims[ax], L) - c[ax], L)
            f = np.exp(-disp * disp / (2.0 * w * w)) * np.exp(1j * v[ax] * disp)
            if ax == 0:
                f = a * f
            factors[ax][b] = f
    return _outer_sum(factors)


def centred_gaussian(dims, L, sigma=1.0) -> np.ndarray:
    """psi = (pi sigma^2)^(-d/4) exp(-r^2 / (2 sigma^2)), centred at x = 0 (grid point N/2)."""
    d = len(dims)
    fs = []
    for n in dims:
        x = coords(n, L)
        fs.append(((np.pi * sigma * sigma) ** -0.25 * np.exp(-x * x / (2.0 * sigma * sigma)))[None, :].astype(np.complex128))
    return _outer_sum(fs)


def super_gaussian_noise(dims, L, r0, noise, seed) -> np.ndarray:
    """exp(-(r/r0)^4) (1 + noise (n1 + i n2)), n1,n2 iid N(0,1) drawn as standard_normal(dims + (2,))."""
    assert len(dims) == 2
    rng = np.random.default_rng(seed)
    y = coords(dims[0], L)[:, None]
    x = coords(dims[1], L)[None, :]
    r2 = x * x + y * y
    env = np.exp(-(r2 / (r0 * r0)) ** 2)
    nz = rng.standard_normal(tuple(dims) + (2,))
    return env * (1.0 + noise * (nz[..., 0] + 1j * nz[..., 1]))


@dataclass(frozen=True)
class Config:
    """One BASELINE.json config: grid, constants of eq. (1),(2), step size and count."""
    name: str
    dims: Tuple[int, ...]
    L: float
    A: float
    B: float
    C: float
    D: float
    g: Tuple[float, ...]
    dtau: float
    steps: int
    make: Callable[[], np.ndarray] = field(repr=False, compare=False, default=None)

    @property
    def cells(self) -> int:
        return int(np.prod(self.dims))

    def initial_state(self) -> np.ndarray:
        """psi_0 rounded once to complex64 (C order)."""
        psi = self.make()
        return np.ascontiguousarray(psi.astype(np.complex64))


def _c5(n: int) -> Config:
    dims = (n, n, n)
    return Config(
        name=f"C5_{n}", dims=dims, L=128.0, A=-0.5, B=1.0, C=0.0, D=4.0 * np.pi, g=(0.01,),
        dtau=1e-2, steps=100,
        make=lambda: gaussian_blobs(dims, 128.0, 32, (4.0, 8.0), (0.05, 0.1), 0.2, seed=5))


def _configs() -> Dict[str, Config]:
    c: Dict[str, Config] = {}
    c["C1"] = Config("C1", (128, 128), 20.0, -0.5, 1.0, 0.0, 1.0, (), 1e-3, 200,
                     make=lambda: centred_gaussian((128, 128), 20.0, 1.0))
    c["C2"] = Config("C2", (1024, 1024), 100.0, -0.5, 1.0, 0.0, 1.0, (0.1,), 5e-3, 1000,
                     make=lambda: gaussian_blobs((1024, 1024), 100.0, 8, (0.5, 1.5), (0.5, 1.0), 0.3, seed=2))
    c["C3"] = Config("C3", (4096, 4096), 400.0, -0.5, 1.0, -1.0, 1.0, (-0.05,), 1e-2, 500,
                     make=lambda: super_gaussian_noise((4096, 4096), 400.0, 20.0, 0.01, seed=3))
    c["C4"] = Config("C4", (256, 256, 256), 64.0, -0.5, 1.0, 0.0, 4.0 * np.pi, (0.02,), 1e-2, 300,
                     make=lambda: gaussian_blobs((256, 256, 256), 64.0, 16, (1.0, 3.0), (0.1, 0.2), 0.2, seed=4))
    for n in (64, 128, 192, 256, 384, 512, 768):  # 192 and 768: beyond BASELINE.json's sweep, same recipe
        c[f"C5_{n}"] = _c5(n)
    return c


CONFIGS: Dict[str, Config] = _configs()


def scaled(cfg: Config, dims, L=None, steps=None, name=None) -> Config:
    """Same physics and recipe family on a different grid (for quick parity cases).

    Only the blob/gaussian families that are functions of physical coordinates
    can be resampled; the recipe's seed and draw order are unchanged.
    """
    dims = tuple(int(n) for n in dims)
    L = cfg.L if L is None else float(L)
    base = cfg.name.split("_")[0]
    if base == "C1":
        make = lambda: centred_gaussian(dims, L, 1.0)
    elif base == "C2":
        make = lambda: gaussian_blobs(dims, L, 8, (0.5, 1.5), (0.5, 1.0), 0.3, seed=2)
    elif base == "C3":
        make = lambda: super_gaussian_noise(dims, L, 20.0, 0.01, seed=3)
    elif base == "C4":
        make = lambda: gaussian_blobs(dims, L, 16, (1.0, 3.0), (0.1, 0.2), 0.2, seed=4)
    elif base == "C5":
        make = lambda: gaussian_blobs(dims, L, 32, (4.0, 8.0), (0.05, 0.1), 0.2, seed=5)
    else:
        raise ValueError(cfg.name)
    return Config(name or f"{cfg.name}@{'x'.join(map(str, dims))}", dims, L, cfg.A, cfg.B, cfg.C, cfg.D,
                  cfg.g, cfg.dtau, cfg.steps if steps is None else int(steps), make=make)


def white_noise(dims, seed) -> np.ndarray:
    """Seeded complex white noise (unit variance per component), complex64; for FFT round-trip tests."""
    rng = np.random.default_rng(seed)
    z = rng.standard_normal(tuple(dims) + (2,))
    return np.ascontiguousarray((z[..., 0] + 1j * z[..., 1]).astype(np.complex64))

"""Pins for the float64 oracle (oracle/snref.c) -- CPU only.

The paper prints no numerical value for the split-step path, so the oracle is
pinned to mathematics instead: brute force, closed-form solutions of eq. (1),(2)
 and invariants of the Symmetric Split-Step Fourier Method.
The pin numbers V1..V12 are SURVEY.md section 8(c)'s.  None of these tests re-types the
oracle's own formulae: each expected value is an independent closed form or a brute-force
sum evaluated here in numpy.
"""
import numpy as np
import pytest

from oracle import snref
from oracle.snref import Oracle
from paper_1909_08354_b200 import inputs


def rel(a, b):
    return float(np.linalg.norm((a - b).ravel()) / np.linalg.norm(np.asarray(b).ravel()))


def grid(dims, L):
    axes = [inputs.coords(n, L) for n in dims]
    return np.meshgrid(*axes, indexing="ij")


# ------------------------------------------------------------------ V1 brute-force DFT

@pytest.mark.parametrize("n", [2, 4, 6, 8, 12, 16, 24, 32, 48])
def test_v1_fft1d_vs_bruteforce(n):
    rng = np.random.default_rng(100 + n)
    x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    j = np.arange(n)
    W = np.exp(-2j * np.pi * np.outer(j, j) / n)          # O(N^2) DFT matrix
    assert rel(snref.fft1d(x, +1), W @ x) < 1e-13
    assert rel(snref.fft1d(x, -1), (W.conj() @ x) / n) < 1e-13


@pytest.mark.parametrize("dims", [(8, 6), (12, 32), (4, 24, 8), (6, 4, 16)])
def test_v1_fftn_vs_bruteforce(dims):
    rng = np.random.default_rng(7)
    x = rng.standard_normal(dims) + 1j * rng.standard_normal(dims)
    want = x.copy()
    for ax, n in enumerate(dims):                         # one dense DFT matrix per axis
        j = np.arange(n)
        W = np.exp(-2j * np.pi * np.outer(j, j) / n)
        want = np.moveaxis(np.tensordot(W, np.moveaxis(want, ax, 0), axes=(1, 0)), 0, ax)
    got = snref.fftn(x, +1)
    assert rel(got, want) < 1e-13
    assert rel(snref.fftn(got, -1), x) < 1e-13            # inverse carries 1/prod N


def test_fft_rejects_unsupported_length():
    with pytest.raises(snref.OracleError):
        snref.fft1d(np.zeros(10, complex), +1)


# ------------------------------------------------------------------ V2 plane wave

@pytest.mark.parametrize("C", [0.0, -1.0])
@pytest.mark.parametrize("dims", [(16, 24), (8, 12, 16)])
def test_v2_plane_wave_exact(dims, C):
    L, A, B, D, g = 7.0, -0.5, 1.3, 0.9, (0.2, 0.05)
    a = 0.8
    m = [2, -3, 1][: len(dims)]                           # lattice wave numbers
    q = [2 * np.pi * mi / L for mi in m]
    X = grid(dims, L)
    psi0 = a * np.exp(1j * sum(qi * Xi for qi, Xi in zip(q, X)))
    dtau, n = 0.013, 17
    o = Oracle(dims, L, A, B, C, D, g, dtau)
    o.set_state(psi0)
    o.step(n)
    rho = a * a
    phi0 = 0.0 if C == 0.0 else D * rho / C
    omega = A * sum(qi * qi for qi in q) - B * phi0 - (g[0] * rho + g[1] * rho * rho)
    want = psi0 * np.exp(1j * omega * dtau * n)
    assert rel(o.get_state(), want) < 1e-12


# ------------------------------------------------------------------ V3 / V4 free Gaussian

def _free_gaussian(X, sigma, A, tau, v=None):
    d = len(X)
    z = sigma * sigma - 2j * A * tau
    if v is None:
        r2 = sum(Xi * Xi for Xi in X)
        return (np.pi * sigma ** 2) ** (-d / 4) * (sigma ** 2 / z) ** (d / 2) * np.exp(-r2 / (2 * z))
    r2 = sum((Xi + 2 * A * tau * vi) ** 2 for Xi, vi in zip(X, v))
    ph = sum(vi * Xi for Xi, vi in zip(X, v)) + A * sum(vi * vi for vi in v) * tau
    return (np.pi * sigma ** 2) ** (-d / 4) * (sigma ** 2 / z) ** (d / 2) * np.exp(-r2 / (2 * z)) * np.exp(1j * ph)


@pytest.mark.parametrize("dims,L", [((128, 128), 20.0), ((64, 64, 64), 20.0)])
def test_v3_free_gaussian_spreading(dims, L):
    A, sigma, dtau, n = -0.5, 1.0, 0.01, 20
    X = grid(dims, L)
    o = Oracle(dims, L, A, 0.0, 0.0, 0.0, (), dtau)       # B = G = 0: pure kinetic flow
    o.set_state(_free_gaussian(X, sigma, A, 0.0))
    o.step(n)
    assert rel(o.get_state(), _free_gaussian(X, sigma, A, dtau * n)) < 1e-12


def test_v3_sign_of_A_matters():
    """A -> -A must give the complex-conjugate evolution, not the same one (catches a dropped sign)."""
    dims, L, sigma = (64, 64), 20.0, 1.0
    X = grid(dims, L)
    o = Oracle(dims, L, +0.5, 0.0, 0.0, 0.0, (), 0.01)
    o.set_state(_free_gaussian(X, sigma, 0.5, 0.0))
    o.step(20)
    got = o.get_state()
    assert rel(got, _free_gaussian(X, sigma, +0.5, 0.2)) < 1e-12
    assert rel(got, _free_gaussian(X, sigma, -0.5, 0.2)) > 1e-2


def test_v4_boosted_gaussian():
    dims, L, A, sigma = (128, 128), 40.0, -0.5, 1.0
    X = grid(dims, L)
    v = (2 * np.pi * 3 / L, -2 * np.pi * 5 / L)          # lattice boosts (periodic phase)
    dtau, n = 0.05, 40                                    # tau = 2: centre moves by (0.94, -1.57)
    o = Oracle(dims, L, A, 0.0, 0.0, 0.0, (), dtau)
    o.set_state(_free_gaussian(X, sigma, A, 0.0, v))
    o.step(n)
    assert rel(o.get_state(), _free_gaussian(X, sigma, A, dtau * n, v)) < 1e-9


def test_v4_anisotropic_box():
    """Per-axis L_a and N_a (Q14): free Gaussian on a non-square box and grid."""
    dims, Ls, A, sigma = (64, 96), (16.0, 24.0), -0.5, 1.0
    X = np.meshgrid(inputs.coords(dims[0], Ls[0]), inputs.coords(dims[1], Ls[1]), indexing="ij")
    o = Oracle(dims, Ls, A, 0.0, 0.0, 0.0, (), 0.02)
    o.set_state(_free_gaussian(X, sigma, A, 0.0))
    o.step(10)
    assert rel(o.get_state(), _free_gaussian(X, sigma, A, 0.2)) < 1e-11


# ------------------------------------------------------------------ V5 single-mode Poisson / Helmholtz

@pytest.mark.parametrize("C", [0.0, -1.0, -0.37, 0.5])
@pytest.mark.parametrize("dims", [(16, 24), (8, 12, 16)])
def test_v5_single_mode_potential(dims, C):
    L, D = 9.0, 0.9
    m = [1, -2, 3][: len(dims)]
    q = [2 * np.pi * mi / L for mi in m]
    X = grid(dims, L)
    rbar, eps = 1.5, 0.4
    cosqx = np.cos(sum(qi * Xi for qi, Xi in zip(q, X)))
    rho = rbar + eps * cosqx
    o = Oracle(dims, L, -0.5, 1.0, C, D, (), 0.01)
    o.set_state(np.sqrt(rho) * np.exp(0.3j * cosqx))     # any phase: phi only sees |psi|^2
    q2 = sum(qi * qi for qi in q)
    want = D * eps * cosqx / (C - q2) + (D * rbar / C if C != 0.0 else 0.0)
    assert np.max(np.abs(o.potential() - want)) < 1e-14


def test_q5_resonant_C_is_rejected():
    L = 2 * np.pi                                         # k lattice = integers; C = 4 hits |k| = 2
    with pytest.raises(snref.OracleError) as e:
        Oracle((8, 8), L, -0.5, 1.0, 4.0, 1.0, (), 0.01)
    assert e.value.code == -4


def test_odd_or_unsupported_dims_rejected():
    for dims in [(9, 8), (8, 10), (8,), (4, 4, 4, 4)]:
        with pytest.raises(snref.OracleError):
            Oracle(dims, 1.0, -0.5, 1.0, 0.0, 1.0, (), 0.01)


# ------------------------------------------------------------------ V6, V8 invariants

def _c1_small():
    return inputs.scaled(inputs.CONFIGS["C1"], (64, 64), steps=50)


def test_v6_norm_conservation():
    cfg = inputs.scaled(inputs.CONFIGS["C2"], (64, 64), L=25.0)
    o = Oracle.from_config(cfg)
    o.set_state(cfg.initial_state())
    n0 = o.diagnostics()["norm"]
    o.step(100)
    assert abs(o.diagnostics()["norm"] - n0) / n0 < 1e-12


def test_v8_time_reversal():
    cfg = inputs.scaled(inputs.CONFIGS["C2"], (64, 64), L=25.0)
    psi0 = cfg.initial_state().astype(np.complex128)
    o = Oracle.from_config(cfg)
    o.set_state(psi0)
    o.step(30)
    assert rel(o.get_state(), psi0) > 1e-3                # it did move
    o.set_dtau(-cfg.dtau)
    o.step(30)
    assert rel(o.get_state(), psi0) < 1e-11


# ------------------------------------------------------------------ V7 Strang order

def _run(cfg, dtau, T, psi0):
    o = Oracle(cfg.dims, cfg.L, cfg.A, cfg.B, cfg.C, cfg.D, cfg.g, dtau)
    o.set_state(psi0)
    o.step(int(round(T / dtau)))
    return o.get_state()


@pytest.mark.parametrize("g", [(), (-2.0, 0.5)])
def test_v7_second_order_self_convergence(g):
    base = inputs.scaled(inputs.CONFIGS["C1"], (64, 64))
    cfg = inputs.Config("v7", base.dims, base.L, -0.5, 3.0, 0.0, 2.0, g, 0.0, 0, make=base.make)
    psi0 = 2.0 * cfg.initial_state().astype(np.complex128)
    T = 0.32
    a, b, c = (_run(cfg, dt, T, psi0) for dt in (0.04, 0.02, 0.01))
    ratio = np.linalg.norm(a - b) / np.linalg.norm(b - c)
    assert abs(ratio - 4.0) < 0.05, ratio


def test_q1_kinetic_halves_outside():
    """K(dt/2) N(dt) K(dt/2): with B = G = 0 removed from the middle the two halves must compose to
    K(dt) exactly; and one step of the full scheme differs from N K N ordering at O(dt^2)."""
    cfg = _c1_small()
    psi0 = cfg.make()                                     # float64, not rounded: compared to a closed form
    X = grid(cfg.dims, cfg.L)
    # first sub-flow acting on psi0 must be kinetic: for tiny B the leading error vs. exact K is O(B)
    o = Oracle(cfg.dims, cfg.L, -0.5, 0.0, 0.0, 0.0, (), 0.1)
    o.set_state(psi0)
    o.step(1)
    assert rel(o.get_state(), _free_gaussian(X, 1.0, -0.5, 0.1)) < 1e-12
    # a pure local phase (A = 0): psi -> psi exp(-i dt g rho) exactly, any dt
    o = Oracle(cfg.dims, cfg.L, 0.0, 0.0, 0.0, 0.0, (0.7,), 0.3)
    o.set_state(psi0)
    o.step(2)
    assert rel(o.get_state(), psi0 * np.exp(-1j * 0.6 * 0.7 * np.abs(psi0) ** 2)) < 1e-13


# ------------------------------------------------------------------ V9 NLS bright soliton

def test_v9_bright_soliton_sign_of_G():
    dims, L, eta, T = (4, 512), 40.0, 1.5, 1.0
    X = grid(dims, L)
    psi0 = (eta / np.cosh(eta * X[1])).astype(np.complex128)
    want = psi0 * np.exp(0.5j * eta * eta * T)
    errs = []
    for dt in (4e-3, 2e-3):
        o = Oracle(dims, (1.0, L), -0.5, 0.0, 0.0, 0.0, (-1.0,), dt)
        o.set_state(psi0)
        o.step(int(round(T / dt)))
        errs.append(rel(o.get_state(), want))
    assert errs[0] < 5e-5 and 3.5 < errs[0] / errs[1] < 4.5, errs
    # the defocusing sign does not hold the soliton together
    o = Oracle(dims, (1.0, L), -0.5, 0.0, 0.0, 0.0, (+1.0,), 4e-3)
    o.set_state(psi0)
    o.step(250)
    assert rel(o.get_state(), want) > 0.1


# ------------------------------------------------------------------ V10 2D <-> 3D, V11 translation

@pytest.mark.parametrize("axis", [0, 1, 2])
def test_v10_3d_reduces_to_2d(axis):
    cfg = inputs.scaled(inputs.CONFIGS["C2"], (32, 48), L=20.0)
    Ls = (20.0, 30.0)
    psi2 = inputs.gaussian_blobs((32, 48), 20.0, 4, (1.0, 2.0), (0.5, 1.0), 0.3, seed=11).astype(np.complex128)
    o2 = Oracle((32, 48), Ls, cfg.A, cfg.B, -0.4, cfg.D, cfg.g, 0.01)
    o2.set_state(psi2)
    o2.step(10)
    n3 = 6
    dims3 = list((32, 48)); dims3.insert(axis, n3)
    L3 = list(Ls); L3.insert(axis, 3.3)
    psi3 = np.repeat(np.expand_dims(psi2, axis), n3, axis=axis)
    o3 = Oracle(dims3, L3, cfg.A, cfg.B, -0.4, cfg.D, cfg.g, 0.01)
    o3.set_state(psi3)
    o3.step(10)
    got = o3.get_state()
    want = np.repeat(np.expand_dims(o2.get_state(), axis), n3, axis=axis)
    assert rel(got, want) < 1e-12


def test_v11_translation_covariance():
    cfg = inputs.scaled(inputs.CONFIGS["C4"], (16, 24, 32), L=16.0)
    psi0 = cfg.initial_state().astype(np.complex128) * 3.0
    shift = (3, -5, 7)
    o = Oracle.from_config(cfg); o.set_state(psi0); o.step(5)
    a = o.get_state()
    o = Oracle.from_config(cfg); o.set_state(np.roll(psi0, shift, axis=(0, 1, 2))); o.step(5)
    assert rel(o.get_state(), np.roll(a, shift, axis=(0, 1, 2))) < 1e-12


# ------------------------------------------------------------------ V12 diagnostics: closed forms, momentum, energy

def test_v12_diagnostics_closed_forms_gaussian():
    """sigma = 1 Gaussian in 2D: norm 1, E_kin = -A d/(2 sigma^2), E_local = g1/(2 (2 pi)^{d/2}) + g2 rho^3 term."""
    dims, L, g = (128, 128), 20.0, (0.3, -0.2)
    o = Oracle(dims, L, -0.5, 0.0, 0.0, 1.0, g, 0.01)
    o.set_state(inputs.centred_gaussian(dims, L, 1.0))
    d = o.diagnostics()
    assert abs(d["norm"] - 1.0) < 1e-13
    assert abs(d["e_kin"] - 0.5) < 1e-12                   # -A * int |grad psi|^2 = 0.5 * d/(2 sigma^2) * 2
    int_rho2 = 1.0 / (2 * np.pi)                           # int rho^2 = (2 pi sigma^2)^{-d/2}
    int_rho3 = 1.0 / (3 * np.pi ** 2)                      # int rho^3 = (pi)^{-3} * (pi/3)
    assert abs(d["e_local"] - (g[0] * int_rho2 / 2 + g[1] * int_rho3 / 3)) < 1e-13
    assert d["e_nonlocal"] == 0.0
    assert abs(d["e_total"] - (d["e_kin"] + d["e_local"])) < 1e-15


@pytest.mark.parametrize("C", [0.0, -0.8])
def test_v12_nonlocal_energy_single_mode(C):
    dims, L, B, D = (16, 32), 6.0, 1.7, 0.6
    X = grid(dims, L)
    q = 2 * np.pi * 2 / L
    rbar, eps = 1.2, 0.5
    rho = rbar + eps * np.cos(q * X[1])
    o = Oracle(dims, L, -0.5, B, C, D, (), 0.01)
    o.set_state(np.sqrt(rho))
    V = L * L
    want = 0.5 * B * V * (D * eps ** 2 / (2 * (C - q * q)) + (D * rbar ** 2 / C if C != 0 else 0.0))
    assert abs(o.diagnostics()["e_nonlocal"] - want) < 1e-12 * abs(want)


def test_v12_energy_error_is_second_order_and_momentum_conserved():
    cfg = inputs.scaled(inputs.CONFIGS["C2"], (64, 64), L=25.0)
    psi0 = cfg.initial_state().astype(np.complex128)
    k = [2 * np.pi * np.fft.fftfreq(n, d=cfg.L / n) for n in cfg.dims]

    def momentum(psi):
        p = np.abs(np.fft.fftn(psi)) ** 2
        return np.array([np.sum(k[0][:, None] * p), np.sum(k[1][None, :] * p)]) / np.sum(p)

    dE = []
    for dt in (8e-3, 4e-3):
        o = Oracle(cfg.dims, cfg.L, cfg.A, cfg.B, cfg.C, cfg.D, cfg.g, dt)
        o.set_state(psi0)
        e0 = o.diagnostics()["e_total"]
        o.step(int(round(0.4 / dt)))
        dE.append(abs(o.diagnostics()["e_total"] - e0) / abs(e0))
        assert np.max(np.abs(momentum(o.get_state()) - momentum(psi0))) < 1e-11
    assert dE[0] < 1e-4 and 3.0 < dE[0] / dE[1] < 5.0, dE


# ------------------------------------------------------------------ input generator fingerprints

def test_generator_fingerprints():
    """Sum |psi|^2 dV of the float64 states, SURVEY.md 8(d) (tests/golden/generator_norms.txt)."""
    import os
    want = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "generator_norms.txt")) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                name, val = line.split()[:2]
                want[name] = float(val)
    c1 = inputs.CONFIGS["C1"]
    assert abs(np.sum(np.abs(c1.make()) ** 2) * (c1.L / 128) ** 2 - want["C1"]) < 1e-12
    c2 = inputs.CONFIGS["C2"]
    assert abs(np.sum(np.abs(c2.make()) ** 2) * (c2.L / 1024) ** 2 - want["C2"]) < 5e-7
    c4 = inputs.scaled(inputs.CONFIGS["C4"], (128, 128, 128))
    assert abs(np.sum(np.abs(c4.make()) ** 2) * (c4.L / 128) ** 3 - want["C4"]) < 5e-7
    c5 = inputs.CONFIGS["C5_64"]
    assert abs(np.sum(np.abs(c5.make()) ** 2) * (c5.L / 64) ** 3 - want["C5"]) < 5e-7

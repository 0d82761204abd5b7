"""Pins for the oracle's NEXT-1 terms (eq. (15),(16)) -- CPU only.

  W1  plane wave: exact solution of the full system for ANY local G, so it fixes the sign and the
      factor of the logarithmic and power-law terms of V_pressure (eq. (16)) and of a uniform V.
  W2  harmonic oscillator: with V = omega^2 r^2/2 and A = -1/2 the Gaussian ground state only
      acquires the phase exp(-i d omega tau/2); a displaced Gaussian (coherent state) moves as
      x0 cos(omega tau).  Fixes the sign of V in the N sub-step.
  W3  gausson of the logarithmic Schroedinger equation: i psi_t = -1/2 lap psi + g_log ln(rho) psi
      has the stationary Gaussian a exp(-r^2/(2 sigma^2)) exp(-i E tau) when g_log = -1/(2 sigma^2),
      E = d/(2 sigma^2) + 2 g_log ln(a) (insert and compare powers of r).
  W4  energy with the new terms: closed forms for a Gaussian (F_log, F_pow, V rho).
None of these re-types the oracle: each expected value is a closed form evaluated here in numpy.
"""
import numpy as np
import pytest

from oracle.snref import Oracle
from paper_1909_08354_b200 import inputs


def rel(a, b):
    return float(np.linalg.norm((a - b).ravel()) / np.linalg.norm(np.asarray(b).ravel()))


def grid(dims, L):
    return np.meshgrid(*[inputs.coords(n, L) for n in dims], indexing="ij")


@pytest.mark.parametrize("dims", [(16, 24), (8, 12, 16)])
def test_w1_plane_wave_with_log_and_power_terms(dims):
    L, A, B, C, D = 10.0, -0.7, 1.3, -1.0, 0.9
    g, g_log, g_pow, p = (0.2,), 0.31, -0.45, 2.0 / 3.0
    amp, dtau, n = 0.8, 7e-3, 9
    X = grid(dims, L)
    q = [2 * np.pi / L * m for m in (2, -1, 3)[:len(dims)]]
    psi0 = amp * np.exp(1j * sum(qa * xa for qa, xa in zip(q, X)))
    v0 = 0.37                                             # uniform external potential: a pure phase rate
    o = Oracle(dims, L, A, B, C, D, g, dtau)
    o.set_local_terms(g_log=g_log, rho_floor=1e-12, g_pow=g_pow, p_pow=p)
    o.set_external_potential(np.full(dims, v0))
    o.set_state(psi0)
    o.step(n)
    rho = amp ** 2
    G = g[0] * rho + g_log * np.log(rho) + g_pow * rho ** p
    rate = A * sum(qa * qa for qa in q) - B * D * rho / C - G - v0
    assert rel(o.get_state(), psi0 * np.exp(1j * rate * n * dtau)) < 1e-12
    o.close()


def test_w2_harmonic_ground_state_and_coherent_state():
    dims, L, w = (64, 64), 16.0, 1.5
    X, Y = grid(dims, L)
    V = 0.5 * w * w * (X * X + Y * Y)
    g0 = np.sqrt(w / np.pi) * np.exp(-0.5 * w * (X * X + Y * Y))
    errs = []
    for dtau in (8e-3, 4e-3):
        o = Oracle(dims, L, -0.5, 0.0, 0.0, 0.0, (), dtau)
        o.set_external_potential(V)
        o.set_state(g0)
        n = int(round(0.8 / dtau))
        o.step(n)
        errs.append(rel(o.get_state(), g0 * np.exp(-1j * w * n * dtau)))   # d*omega/2 with d = 2
        o.close()
    assert errs[1] < 1e-5 and 3.7 < errs[0] / errs[1] < 4.3               # O(dtau^2) splitting error only
    # coherent state: centre follows x0 cos(omega tau), norm 1
    x0, dtau = 1.2, 2e-3
    o = Oracle(dims, L, -0.5, 0.0, 0.0, 0.0, (), dtau)
    o.set_external_potential(V)
    o.set_state(np.sqrt(w / np.pi) * np.exp(-0.5 * w * ((X - x0) ** 2 + Y * Y)))
    n = 500
    o.step(n)
    rho = np.abs(o.get_state()) ** 2
    dV = (L / 64) ** 2
    assert abs(rho.sum() * dV - 1.0) < 1e-10
    assert abs((rho * X).sum() * dV - x0 * np.cos(w * n * dtau)) < 1e-5
    assert abs((rho * Y).sum() * dV) < 1e-10
    o.close()


@pytest.mark.parametrize("dims,L", [((96, 96), 24.0), ((32, 32, 32), 20.0)])
def test_w3_gausson_of_the_logarithmic_equation(dims, L):
    d, sigma, a = len(dims), 1.6, 0.9
    g_log = -1.0 / (2 * sigma * sigma)
    E = d / (2 * sigma * sigma) + 2 * g_log * np.log(a)
    X = grid(dims, L)
    r2 = sum(x * x for x in X)
    psi0 = a * np.exp(-r2 / (2 * sigma * sigma))
    errs = []
    for dtau in (2e-2, 1e-2):
        o = Oracle(dims, L, -0.5, 0.0, 0.0, 0.0, (), dtau)
        o.set_local_terms(g_log=g_log, rho_floor=1e-300)
        o.set_state(psi0)
        n = int(round(1.0 / dtau))
        o.step(n)
        errs.append(rel(o.get_state(), psi0 * np.exp(-1j * E * n * dtau)))
        o.close()
    assert errs[1] < 5e-5 and 3.6 < errs[0] / errs[1] < 4.4


def test_w3_sign_of_log_term_matters():
    dims, L, sigma = (64, 64), 20.0, 1.6
    X, Y = grid(dims, L)
    psi0 = 0.9 * np.exp(-(X * X + Y * Y) / (2 * sigma * sigma))
    o = Oracle(dims, L, -0.5, 0.0, 0.0, 0.0, (), 1e-2)
    o.set_local_terms(g_log=+1.0 / (2 * sigma * sigma), rho_floor=1e-300)   # wrong sign: the packet spreads
    o.set_state(psi0)
    o.step(100)
    assert np.abs(o.get_state()).max() < 0.9 * 0.9   # the stationary gausson keeps 0.9
    o.close()


def test_w4_energy_closed_forms_and_conservation():
    dims, L, s = (96, 96), 24.0, 1.3
    X, Y = grid(dims, L)
    r2 = X * X + Y * Y
    a = 0.7
    psi0 = a * np.exp(-r2 / (2 * s * s))                   # rho = a^2 exp(-r^2/s^2)
    w, g_log, g_pow, p = 0.8, 0.25, 0.6, 1.5
    o = Oracle(dims, L, -0.5, 0.0, 0.0, 0.0, (), 2e-3)
    o.set_local_terms(g_log=g_log, rho_floor=1e-300, g_pow=g_pow, p_pow=p)
    o.set_external_potential(0.5 * w * w * r2)
    o.set_state(psi0)
    d0 = o.diagnostics()
    M = np.pi * a * a * s * s                              # int rho
    # int rho ln rho = M (2 ln a - 1) [int r^2/s^2 rho = M];  int rho^(p+1) = pi a^(2p+2) s^2/(p+1);  int r^2 rho = M s^2
    e_log = g_log * (M * (2 * np.log(a) - 1.0) - M)
    e_pow = g_pow * np.pi * a ** (2 * p + 2) * s * s / (p + 1) / (p + 1)
    e_ext = 0.5 * w * w * M * s * s
    assert abs(d0["e_local"] - (e_log + e_pow + e_ext)) < 1e-9 * abs(e_ext)
    assert abs(d0["e_kin"] - 0.5 * M / (s * s)) < 1e-9     # -A int |grad psi|^2 = (1/2) M/s^2 in 2D
    o.step(400)
    d1 = o.diagnostics()
    assert abs(d1["e_total"] - d0["e_total"]) < 2e-6 * abs(d0["e_total"])   # O(dtau^2), bounded
    assert abs(d1["norm"] - d0["norm"]) < 1e-12 * d0["norm"]
    o.close()


# ------------------------------------------------------------------ W5 modified Poisson source, eq. (12)

@pytest.mark.parametrize("dims,C", [((32, 48), 0.0), ((16, 24, 32), -0.8)])
def test_w5_position_dependent_source_closed_form(dims, C):
    """rho = rb + e cos(q.x), beta = b0 + b1 cos(p.x), gamma = g0 + g1 cos(p.x):
    s = gamma rho + beta lap rho has modes 0, p, q, p+q, p-q with amplitudes from cos a cos b = (cos(a+b) + cos(a-b))/2;
    each mode k gives phi_k = D s_k/(C - |k|^2) (mode 0: dropped if C = 0, else D s_0/C)."""
    L, D = 9.0, 1.7
    nd = len(dims)
    X = grid(dims, L)
    k0 = 2 * np.pi / L
    q = np.array([2, 1, -1][:nd]) * k0
    p = np.array([1, -2, 2][:nd]) * k0
    rb, e, b0, b1, g0, g1 = 1.3, 0.4, 0.25, 0.1, 0.6, -0.2
    ph = lambda k: sum(ka * xa for ka, xa in zip(k, X))
    rho = rb + e * np.cos(ph(q))
    beta = b0 + b1 * np.cos(ph(p))
    gamma = g0 + g1 * np.cos(ph(p))
    q2 = float(q @ q)
    # s = g0 rb + g0 e cos q + g1 rb cos p + g1 e cos p cos q - q2 e (b0 cos q + b1 cos p cos q)
    modes = [(np.zeros(nd), g0 * rb), (q, g0 * e - q2 * e * b0), (p, g1 * rb),
             (p + q, 0.5 * (g1 * e - q2 * e * b1)), (p - q, 0.5 * (g1 * e - q2 * e * b1))]
    want = np.zeros(dims)
    for k, amp in modes:
        k2 = float(k @ k)
        if k2 == 0.0:
            want += 0.0 if C == 0.0 else D * amp / C
        else:
            want += D * amp / (C - k2) * np.cos(ph(k))
    o = Oracle(dims, L, -0.5, 1.0, C, D, (), 1e-3)
    o.set_source_tables(beta, gamma)
    o.set_state(np.sqrt(rho).astype(complex))
    assert np.abs(o.potential() - want).max() < 1e-12 * max(1.0, np.abs(want).max())
    # gamma = 1, beta = 0 is eq. (2) itself
    o.set_source_tables(np.zeros(dims), np.ones(dims))
    a = o.potential()
    o.set_source_tables(None, None)
    assert np.abs(a - o.potential()).max() < 1e-13
    o.close()


# ------------------------------------------------------------------ W6 fourth-order composition

def test_w6_order4_self_convergence_and_invariants():
    """Halving dtau must reduce the error 16-fold (order 4), against 4-fold for the Strang step; the composition is
    still unitary (norm), time-reversible, and exact on a plane wave."""
    dims, L = (64, 64), 20.0
    cfg = inputs.scaled(inputs.CONFIGS["C1"], dims, L=L)
    psi0 = cfg.initial_state().astype(np.complex128) * 6.0        # strong self-gravity: splitting error well above roundoff
    T = 0.4

    def run(order, dtau):
        o = Oracle(dims, L, -0.5, 1.0, 0.0, 1.0, (0.05,), dtau)
        o.set_state(psi0)
        n = int(round(T / dtau))
        (o.step_order4 if order == 4 else o.step)(n)
        out, d = o.get_state(), o.diagnostics()
        o.close()
        return out, d

    ref, _ = run(4, T / 640)
    e4 = [rel(run(4, T / n)[0], ref) for n in (10, 20, 40)]
    e2 = [rel(run(2, T / n)[0], ref) for n in (10, 20, 40)]
    assert 13.0 < e4[0] / e4[1] < 19.0 and 13.0 < e4[1] / e4[2] < 19.0, e4
    assert 3.6 < e2[1] / e2[2] < 4.4, e2
    assert e4[2] < 0.01 * e2[2]
    out, d = run(4, T / 20)
    n0 = float((np.abs(psi0) ** 2).sum() * (L / 64) ** 2)
    assert abs(d["norm"] - n0) < 1e-11 * n0
    # time reversal
    o = Oracle(dims, L, -0.5, 1.0, 0.0, 1.0, (0.05,), T / 20)
    o.set_state(psi0)
    o.step_order4(7)
    o.set_dtau(-T / 20)
    o.step_order4(7)
    assert rel(o.get_state(), psi0) < 1e-11
    o.close()
    # plane wave: exact for any composition of exact sub-flows (w1 + w0 + w1 = 1)
    X, Y = grid(dims, L)
    q = 2 * np.pi / L * np.array([3, -2])
    pw = 0.7 * np.exp(1j * (q[0] * X + q[1] * Y))
    o = Oracle(dims, L, -0.5, 1.0, -1.0, 0.9, (0.2,), 3e-2)
    o.set_state(pw)
    o.step_order4(5)
    rate = -0.5 * float(q @ q) - 1.0 * 0.9 * 0.49 / (-1.0) - 0.2 * 0.49
    assert rel(o.get_state(), pw * np.exp(1j * rate * 5 * 3e-2)) < 1e-12
    o.close()


# ------------------------------------------------------------------ W7 Bohm quantum potential of eq. (15)

def test_w7_bohm_potential_closed_form_and_stationarity():
    """sqrt(rho) = a exp(-r^2/(2 s^2))  =>  V_B = lap sqrt(rho)/(2 sqrt(rho)) = (r^2/s^4 - d/s^2)/2 (closed form).
    With c_B = -2A the Bohm term cancels the quantum pressure of the kinetic operator exactly (Madelung:
    A lap sqrt(rho) + c_B V_B sqrt(rho) = 0), so ANY real positive state is stationary: the Gaussian that spreads
    under K alone stays put to ~1e-6 (splitting error and the floor in the far tails)."""
    dims, L, s, a = (96, 96), 24.0, 1.7, 0.8
    X, Y = grid(dims, L)
    r2 = X * X + Y * Y
    psi0 = (a * np.exp(-r2 / (2 * s * s))).astype(complex)
    o = Oracle(dims, L, -0.5, 0.0, 0.0, 0.0, (), 1e-2)
    o.set_bohm(1.0, 1e-300)
    o.set_state(psi0)
    vb = o.bohm_potential()
    core = r2 < (5 * s) ** 2                                   # where sqrt(rho) is above the roundoff of the transform
    want = 0.5 * (r2 / s ** 4 - 2.0 / s ** 2)
    assert np.abs(vb - want)[core].max() < 1e-6
    o.close()
    errs = []
    for dtau in (2e-2, 1e-2):
        o = Oracle(dims, L, -0.5, 0.0, 0.0, 0.0, (), dtau)
        o.set_bohm(1.0, 1e-6)                                  # c_B = -2A
        o.set_state(psi0)
        o.step(int(round(1.0 / dtau)))
        errs.append(rel(o.get_state(), psi0))
        o.close()
    assert max(errs) < 1e-5, errs                              # stationary (splitting + floor effects ~1e-6)
    o = Oracle(dims, L, -0.5, 0.0, 0.0, 0.0, (), 1e-2)      # without the Bohm term the packet spreads
    o.set_state(psi0)
    o.step(100)
    free_max = np.abs(o.get_state()).max()
    assert rel(o.get_state(), psi0) > 0.1
    o.close()
    o = Oracle(dims, L, -0.5, 0.0, 0.0, 0.0, (), 1e-2)      # wrong sign: spreads faster still
    o.set_bohm(-1.0, 1e-6)
    o.set_state(psi0)
    o.step(100)
    assert np.abs(o.get_state()).max() < 0.97 * free_max
    o.close()

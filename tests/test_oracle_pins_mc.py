"""Pins of the coupled-wave-function oracle (oracle/snref.c, snref_mc_*; NEXT-4b, reading Q18 of
DESIGN.md).  None of them re-types the oracle: each fixes it against an exact solution, against the separately pinned
one-component oracle, or against an invariant of the equations.

    i dpsi_c/dtau = A_c lap psi_c + B_c phi psi_c + (sum_c' g_cc' |psi_c'|^2) psi_c,   lap phi + C phi = D sum_c w_c |psi_c|^2
"""
import numpy as np
import pytest

from oracle.snref import Oracle, OracleMC
from paper_1909_08354_b200 import inputs


def rel(a, b):
    return float(np.linalg.norm((np.asarray(a) - np.asarray(b)).ravel()) / np.linalg.norm(np.asarray(b).ravel()))


def plane(dims, L, mode, amp):
    X = np.meshgrid(*[inputs.coords(n, L) for n in dims], indexing="ij")
    q = 2 * np.pi / L * np.asarray(mode, dtype=np.float64)
    return amp * np.exp(1j * sum(qa * x for qa, x in zip(q, X))), float(q @ q)


@pytest.mark.parametrize("dims,C", [((32, 24), 0.0), ((16, 32), -1.3), ((16, 12, 8), 0.0), ((8, 16, 16), -0.7)])
def test_mc1_plane_waves_are_exact(dims, C):
    """psi_c = a_c e^{i q_c.x}: every rho_c is uniform, so phi = phi0 = 0 (C = 0) or D sum w_c a_c^2 / C, and each
    component stays a plane wave with omega_c = A_c |q_c|^2 - B_c phi0 - sum_c' g_cc' a_c'^2.  Exact for the full system
    and for every sub-step, any dtau: fixes every constant's role, the sign conventions and the component indexing
    (g is NOT symmetric here, A, B, w differ per component)."""
    L, dtau, steps = 7.0, 0.05, 9
    A, B, w = (-0.5, 0.8, -0.3), (1.3, -0.4, 0.9), (0.7, 1.9, -0.6)
    g = np.array([[0.2, -0.5, 0.11], [0.3, 0.05, -0.7], [-0.13, 0.4, 0.6]])
    D = 0.9
    modes = [(3, -2, 1), (-1, 4, 2), (2, 2, -3)]
    amps = (0.8, 0.5, 1.1)
    M = 3
    psi, q2 = zip(*[plane(dims, L, modes[c][: len(dims)], amps[c]) for c in range(M)])
    orc = OracleMC(dims, L, A, B, C, D, w, g, dtau)
    orc.set_state(np.stack(psi))
    orc.step(steps)
    got = orc.get_state()
    orc.close()
    a2 = np.square(amps)
    phi0 = 0.0 if C == 0 else D * float(np.dot(w, a2)) / C
    for c in range(M):
        omega = A[c] * q2[c] - B[c] * phi0 - float(g[c] @ a2)
        assert rel(got[c], psi[c] * np.exp(1j * omega * dtau * steps)) < 1e-12, c


@pytest.mark.parametrize("dims", [(32, 32), (16, 16, 16)])
def test_mc2_decoupled_limit_is_the_one_component_oracle(dims):
    """w = (1, 0), g diagonal in component 0, B_1 = 0: component 0 evolves exactly as the (separately pinned)
    one-component oracle with G = g_00 rho, component 1 as a free particle with its own A.  Then w = (0, 1): the roles
    of the source swap -- component 0 now moves in the potential of component 1 (it must NOT match the self-gravitating
    run any more)."""
    nd = len(dims)
    L, dtau, steps = 12.0, 0.02, 12
    c0 = inputs.scaled(inputs.CONFIGS["C2" if nd == 2 else "C4"], dims, L=L)
    p0 = c0.initial_state().astype(np.complex128)
    p1 = np.roll(p0, 5, axis=0) * (0.6 + 0.2j)
    A, B = (-0.5, -0.9), (1.0, 0.0)
    g = np.array([[0.3, 0.0], [0.0, 0.0]])
    orc = OracleMC(dims, L, A, B, 0.0, 2.0, (1.0, 0.0), g, dtau)
    orc.set_state(np.stack([p0, p1]))
    orc.step(steps)
    got = orc.get_state()
    orc.close()
    one = Oracle(dims, L, A[0], B[0], 0.0, 2.0, (0.3,), dtau)
    one.set_state(p0)
    one.step(steps)
    assert rel(got[0], one.get_state()) < 1e-13
    one.close()
    free = Oracle(dims, L, A[1], 0.0, 0.0, 0.0, (), dtau)
    free.set_state(p1)
    free.step(steps)
    assert rel(got[1], free.get_state()) < 1e-13
    free.close()
    swapped = OracleMC(dims, L, A, B, 0.0, 2.0, (0.0, 1.0), g, dtau)
    swapped.set_state(np.stack([p0, p1]))
    swapped.step(steps)
    assert rel(swapped.get_state()[0], got[0]) > 1e-3
    swapped.close()


@pytest.mark.parametrize("dims,C", [((32, 32), 0.0), ((16, 16, 16), -0.5)])
def test_mc3_equal_split_of_a_one_component_state(dims, C):
    """psi_0 = cos(t) psi, psi_1 = sin(t) e^{i a} psi with equal A, B, w = (1, 1) and g_cc' = g for all c, c': the
    densities add up to |psi|^2 everywhere and both components see B phi[rho] + g rho, so each stays that multiple
    of the one-component solution.  Catches a dropped or doubled term in either sum over components."""
    nd = len(dims)
    L, dtau, steps, gk, t, al = 12.0, 0.02, 10, 0.25, 0.7, 1.1
    cfg = inputs.scaled(inputs.CONFIGS["C2" if nd == 2 else "C4"], dims, L=L)
    p = cfg.initial_state().astype(np.complex128)
    f = (np.cos(t), np.sin(t) * np.exp(1j * al))
    orc = OracleMC(dims, L, (-0.5, -0.5), (1.2, 1.2), C, 1.7, (1.0, 1.0), np.full((2, 2), gk), dtau)
    orc.set_state(np.stack([f[0] * p, f[1] * p]))
    orc.step(steps)
    got = orc.get_state()
    orc.close()
    one = Oracle(dims, L, -0.5, 1.2, C, 1.7, (gk,), dtau)
    one.set_state(p)
    one.step(steps)
    want = one.get_state()
    one.close()
    for c in range(2):
        assert rel(got[c], f[c] * want) < 1e-13, c


def test_mc4_norms_conserved_and_second_order():
    """Every sub-step is unitary on each component separately (norms to roundoff), and the splitting is symmetric:
    self-convergence ratio 4 under dtau halving (a non-symmetric or first-order composition gives 2)."""
    dims, L, T = (32, 32), 12.0, 0.32
    cfg = inputs.scaled(inputs.CONFIGS["C2"], dims, L=L)
    p0 = cfg.initial_state().astype(np.complex128)
    p1 = np.roll(p0, (3, 7), axis=(0, 1)) * 0.7j
    g = np.array([[0.3, -0.4], [0.6, 0.1]])

    def run(n):
        o = OracleMC(dims, L, (-0.5, -0.8), (1.0, 0.6), 0.0, 1.5, (1.0, 0.5), g, T / n)
        o.set_state(np.stack([p0, p1]))
        n0 = o.norms()
        o.step(n)
        out, n1 = o.get_state(), o.norms()
        o.close()
        assert np.all(np.abs(n1 - n0) < 1e-13 * n0)
        return out

    a, b, c = run(16), run(32), run(64)
    ratio = np.linalg.norm((a - b).ravel()) / np.linalg.norm((b - c).ravel())
    assert 3.8 < ratio < 4.2, ratio
    dV = (L / 32) ** 2
    o = OracleMC(dims, L, (-0.5, -0.8), (1.0, 0.6), 0.0, 1.5, (1.0, 0.5), g, 0.01)
    o.set_state(np.stack([p0, p1]))
    assert np.allclose(o.norms(), [np.sum(np.abs(p0) ** 2) * dV, np.sum(np.abs(p1) ** 2) * dV], rtol=1e-14)
    o.close()

"""GPU parity of the coupled-wave-function path (sn_create_mc; NEXT-4b, reading Q18 of DESIGN.md) against
the float64 oracle (snref_mc_*), through the C ABI.  Same tolerances as the one-component complex64 path."""
import numpy as np
import pytest

from _parity import TOL_NORM, TOL_STATE, assert_state, rel

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def mods():
    from oracle.snref import Oracle, OracleMC
    from paper_1909_08354_b200 import inputs, sn
    return Oracle, OracleMC, inputs, sn


def components(inputs, name, dims, L, M):
    """M seeded component states from the config's recipe: shifted, rescaled, re-phased copies of its initial state."""
    cfg = inputs.scaled(inputs.CONFIGS[name], dims, L=L)
    p = cfg.initial_state()
    rng = np.random.default_rng(17)
    out = []
    for c in range(M):
        sh = tuple(int(rng.integers(n)) for n in dims)
        out.append(np.roll(p, sh, axis=tuple(range(len(dims)))) * np.complex64((0.9 - 0.2 * c) * np.exp(0.7j * c)))
    return cfg, np.ascontiguousarray(np.stack(out).astype(np.complex64))


CONSTS = {
    2: dict(A=(-0.5, -0.8), B=(1.0, 0.6), w=(1.0, 0.5), g=[[0.3, -0.4], [0.6, 0.1]]),
    3: dict(A=(-0.5, 0.8, -0.3), B=(1.3, -0.4, 0.9), w=(0.7, 1.9, -0.6),
            g=[[0.2, -0.5, 0.11], [0.3, 0.05, -0.7], [-0.13, 0.4, 0.6]]),
    4: dict(A=(-0.5, -0.5, -1.0, -0.25), B=(1.0, 1.0, 0.5, 2.0), w=(1.0, 1.0, 0.5, 0.25),
            g=np.full((4, 4), 0.1) + 0.2 * np.eye(4)),
}

CASES = [
    # name, dims, L, M, C, D, steps
    ("C2", (128, 128), 12.5, 2, 0.0, 1.0, 100),
    ("C2", (256, 64), 25.0, 3, -1.0, 1.0, 60),
    ("C2", (512, 128), 25.0, 2, 0.0, 1.0, 20),          # pipelined 512-point strided kinetic passes along axis 0
    ("C3", (64, 2048), 50.0, 2, -1.0, 1.0, 10),         # pipelined long contiguous lines
    ("C2", (96, 384), 25.0, 4, 0.0, 1.0, 40),           # 3*2^a lengths, four components
    ("C4", (64, 64, 64), 16.0, 2, 0.0, 4 * np.pi, 60),
    ("C4", (64, 128, 256), 32.0, 3, -0.7, 4 * np.pi, 8),
    ("C5_512", (64, 512, 128), 128.0, 2, 0.0, 4 * np.pi, 4),   # 512-point strided lines along axis 1
    ("C4", (32, 32, 32), 8.0, 4, 0.0, 4 * np.pi, 40),
]


@pytest.mark.parametrize("name,dims,L,M,C,D,steps", CASES)
def test_coupled_steps_match_oracle(mods, name, dims, L, M, C, D, steps):
    Oracle, OracleMC, inputs, sn = mods
    cfg, psi0 = components(inputs, name, dims, L, M)
    k = CONSTS[M]
    sim = sn.CoupledSimulation(dims, L, k["A"], k["B"], C, D, k["w"], k["g"], cfg.dtau)
    sim.set_state(psi0)
    n0 = sim.norms()
    sim.step(steps // 2)
    sim.step(steps - steps // 2)                        # split calls
    got = sim.get_state()
    n1 = sim.norms()
    sim.close()
    orc = OracleMC(dims, L, k["A"], k["B"], C, D, k["w"], k["g"], cfg.dtau)
    orc.set_state(psi0.astype(np.complex128))
    r0 = orc.norms()
    orc.step(steps)
    want = orc.get_state()
    orc.close()
    for c in range(M):
        assert_state(got[c], want[c])
    assert np.all(np.abs(n0 - r0) < 1e-6 * r0)
    assert np.all(np.abs(n1 - n0) < TOL_NORM * n0)


def test_one_component_context_equals_sn_create(mods):
    """n_comp = 1 with g_00 = g: the coupled scheduler (unfused nonlinear pass, separate kinetic sweep) against the
    fused one-component path: same mathematics, different kernels -- agreement to fp32 roundoff, both within tolerance
    of the oracle."""
    Oracle, OracleMC, inputs, sn = mods
    cfg = inputs.scaled(inputs.CONFIGS["C4"], (64, 128, 64), L=16.0, steps=12)
    psi0 = cfg.initial_state()
    one = sn.Simulation.from_config(cfg)
    one.set_state(psi0)
    one.step(12)
    a = one.get_state()
    one.close()
    mc = sn.CoupledSimulation(cfg.dims, cfg.L, (cfg.A,), (cfg.B,), cfg.C, cfg.D, (1.0,), [[cfg.g[0]]], cfg.dtau)
    mc.set_state(psi0[None])
    mc.step(12)
    b = mc.get_state()[0]
    mc.close()
    orc = Oracle.from_config(cfg)
    orc.set_state(psi0.astype(np.complex128))
    orc.step(12)
    want = orc.get_state()
    orc.close()
    assert_state(a, want)
    assert_state(b, want)
    assert rel(a, b) < 5e-6


def test_plane_waves_full_size(mods):
    """Two plane waves at 256^3: exact solution of the coupled system (pin MC1), every pipelined kinetic kernel."""
    Oracle, OracleMC, inputs, sn = mods
    dims, L, dtau, steps, C, D = (256, 256, 256), 32.0, 5e-3, 10, -1.0, 0.9
    k = CONSTS[2]
    modes, amps = [(3, -2, 5), (-1, 4, 2)], (0.8, 0.5)
    psi, q2 = [], []
    for md, am in zip(modes, amps):
        q = 2 * np.pi / L * np.asarray(md, dtype=np.float64)
        f = [np.exp(1j * qa * inputs.coords(n, L)) for qa, n in zip(q, dims)]
        psi.append((am * f[0][:, None, None] * f[1][None, :, None] * f[2][None, None, :]).astype(np.complex64))
        q2.append(float(q @ q))
    psi0 = np.ascontiguousarray(np.stack(psi))
    sim = sn.CoupledSimulation(dims, L, k["A"], k["B"], C, D, k["w"], k["g"], dtau)
    sim.set_state(psi0)
    sim.step(steps)
    got = sim.get_state()
    sim.close()
    a2 = np.square(amps)
    phi0 = D * float(np.dot(k["w"], a2)) / C
    for c in range(2):
        omega = k["A"][c] * q2[c] - k["B"][c] * phi0 - float(np.dot(k["g"][c], a2))
        assert rel(got[c], psi0[c].astype(np.complex128) * np.exp(1j * omega * dtau * steps)) < 2e-5


def test_coupled_context_contract(mods):
    Oracle, OracleMC, inputs, sn = mods
    dims = (64, 64)
    k = CONSTS[2]
    sim = sn.CoupledSimulation(dims, 10.0, k["A"], k["B"], 0.0, 1.0, k["w"], k["g"], 1e-3)
    with pytest.raises(sn.SnError) as e:
        sim.step(1)
    assert e.value.code == -6                           # no state yet
    sim.set_state(np.zeros((2,) + dims, np.complex64))
    for call in (sim.diagnostics, lambda: sim.step_order4(1), lambda: sim.debug_fft(1), lambda: sim.set_bohm(0.1, 1e-6)):
        with pytest.raises(sn.SnError) as e:
            call()
        assert e.value.code == -9
    sim.step(3)
    assert np.array_equal(sim.get_state(), np.zeros((2,) + dims, np.complex64))
    sim.close()
    with pytest.raises(sn.SnError):
        sn.CoupledSimulation(dims, 10.0, (1.0,) * 5, (1.0,) * 5, 0.0, 1.0, (1.0,) * 5, np.zeros((5, 5)), 1e-3)

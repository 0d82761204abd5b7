"""GPU parity for the NEXT-1 terms (eq. (15),(16)): logarithmic / power-law pressure
potential and a fixed external potential, CUDA path (C ABI) against the float64 oracle, same tolerances as
the main path (rel-L2 <= 1e-4, norm drift <= 1e-5)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from _parity import TOL_NORM, TOL_STATE, assert_state, maxrel, rel


@pytest.fixture(scope="module")
def mods():
    """(Oracle, inputs, sn) with sn.Simulation creating every context with all optional workspace regions
    (external potential table, source tables, host staging: sn_options.features = SN_FEAT_ALL)."""
    import types
    from oracle.snref import Oracle
    from paper_1909_08354_b200 import inputs, sn

    class SimAll(sn.Simulation):
        def __init__(self, *a, **kw):
            kw.setdefault("features", sn.FEAT_ALL)
            super().__init__(*a, **kw)

    shim = types.SimpleNamespace(**{k: v for k, v in vars(sn).items() if not k.startswith("__")})
    shim.Simulation = SimAll
    return Oracle, inputs, shim


def nmc_potential(dims, L, lam=1.0, r0=2.0):
    """phi_C = ln[1 - (r0/(r + r0))^lambda] of eq. (11) on the periodic box, with the radius softened to
    sqrt(r^2 + 1) because the grid has a point at r = 0 where eq. (11) diverges (the paper does not say how its
    mesh avoids it)."""
    from paper_1909_08354_b200 import inputs
    X = np.meshgrid(*[inputs.coords(n, L) for n in dims], indexing="ij")
    r = np.sqrt(sum(x * x for x in X) + 1.0)
    return np.log(1.0 - (r0 / (r + r0)) ** lam)


CASES = [
    # name, dims, L, steps, local terms (g_log, floor, g_pow, p), external potential?
    ("C2", (256, 128), 25.0, 200, (0.05, 1e-12, 0.0, 1.0), False),      # w ln(rho), n = 1 of eq. (16)
    ("C2", (128, 256), 25.0, 200, (0.0, 1e-12, 0.08, 2.0 / 3.0), False),  # (n w/(n-1)) rho^(n-1), n = 5/3
    ("C2", (256, 256), 25.0, 200, (0.0, 1e-30, 0.0, 1.0), True),         # phi_C table only
    ("C4", (64, 128, 64), 16.0, 60, (0.02, 1e-12, 0.05, 0.5), True),     # everything on, 3D
    ("C5_384", (96, 64, 64), 128.0, 20, (0.02, 1e-12, 0.0, 1.0), True),  # 6*4^a axis with the extras
    ("C4", (32, 64, 32), 16.0, 40, (0.02, 1e-12, 0.05, 0.5), True),      # 32-point lines: V on the first-path axis-0 pass
    ("C2", (64, 32), 12.5, 100, (0.05, 1e-12, 0.0, 1.0), True),
]


@pytest.mark.parametrize("name,dims,L,steps,terms,ext", CASES)
def test_next_terms_match_oracle(mods, name, dims, L, steps, terms, ext):
    Oracle, inputs, sn = mods
    cfg = inputs.scaled(inputs.CONFIGS[name], dims, L=L, steps=steps)
    psi0 = cfg.initial_state()
    V = nmc_potential(dims, L).astype(np.float32) if ext else None
    sim = sn.Simulation.from_config(cfg)
    sim.set_local_terms(*terms)
    sim.set_external_potential(V)
    sim.set_state(psi0)
    d0 = sim.diagnostics()
    sim.step(steps)
    got = sim.get_state()
    d1 = sim.diagnostics()
    sim.close()
    orc = Oracle.from_config(cfg)
    orc.set_local_terms(*terms)
    orc.set_external_potential(None if V is None else V.astype(np.float64))
    orc.set_state(psi0.astype(np.complex128))
    r0 = orc.diagnostics()
    orc.step(steps)
    want = orc.get_state()
    r1 = orc.diagnostics()
    orc.close()
    assert_state(got, want)
    assert abs(d1["norm"] - d0["norm"]) < TOL_NORM * d0["norm"]
    for k in ("norm", "e_kin", "e_nonlocal", "e_local", "e_total"):
        scale = max(abs(r0["e_total"]), abs(r0[k]), 1e-30)
        assert abs(d0[k] - r0[k]) < 2e-5 * scale, (k, d0[k], r0[k])
        assert abs(d1[k] - r1[k]) < 2e-5 * scale, (k, d1[k], r1[k])


def test_terms_can_be_switched_off_again(mods):
    Oracle, inputs, sn = mods
    cfg = inputs.scaled(inputs.CONFIGS["C2"], (128, 128), L=25.0, steps=20)
    psi0 = cfg.initial_state()
    sim = sn.Simulation.from_config(cfg)
    sim.set_state(psi0)
    sim.step(20)
    plain = sim.get_state()
    sim.set_local_terms(0.3, 1e-12, 0.2, 0.5)
    sim.set_external_potential(nmc_potential((128, 128), 25.0).astype(np.float32))
    sim.set_state(psi0)
    sim.step(20)
    assert rel(sim.get_state(), plain) > 1e-3            # the terms do something
    sim.set_local_terms(0.0, 1e-30, 0.0, 1.0)
    sim.set_external_potential(None)
    sim.set_state(psi0)
    sim.step(20)
    assert rel(sim.get_state(), plain) == 0.0            # and the default path is restored bit for bit
    sim.close()


def test_features_are_opt_in(mods):
    """The default workspace holds the stepper alone (~12 B/cell); the NEXT-1 tables and the host staging scratch
    are requested at create (sn_options.features).  Without them the setters return SN_ERR_FEATURE and leave the
    context untouched; with exactly the bits a call needs it works and matches the all-features context bit for bit."""
    Oracle, inputs, sn = mods
    from paper_1909_08354_b200 import sn as raw
    dims, L = (64, 128), 12.5
    cfg = inputs.scaled(inputs.CONFIGS["C2"], dims, L=L, steps=8)
    psi0 = cfg.initial_state()
    V = nmc_potential(dims, L).astype(np.float32)
    beta, gamma = nmc_tables(dims, L)
    w0 = raw.workspace_bytes(dims)
    assert w0 < 12.6 * cfg.cells + 65536
    assert raw.workspace_bytes(dims, features=raw.FEAT_VEXT) >= w0 + 4 * cfg.cells
    assert raw.workspace_bytes(dims, features=raw.FEAT_ALL) >= w0 + 16 * cfg.cells
    plain = raw.Simulation.from_config(cfg)                 # features = 0
    plain.set_state(psi0)
    for call in (lambda: plain.set_external_potential(V),
                 lambda: plain._set_source_tables_host(beta, gamma)):
        with pytest.raises(raw.SnError) as e:
            call()
        assert e.value.code == -9
    plain.step(8)
    want_plain = plain.get_state()
    plain.close()
    out = []
    for feats in (raw.FEAT_VEXT | raw.FEAT_SOURCE, raw.FEAT_ALL):
        sim = raw.Simulation.from_config(cfg, features=feats)
        sim.set_state(psi0)
        sim.set_external_potential(V)
        sim.set_source_tables(beta, gamma)                  # device copies when there is no staging region
        sim.step(8)
        out.append(sim.get_state())
        phi = sim.debug_potential()
        assert np.isfinite(phi).all()
        sim.close()
    assert np.array_equal(out[0], out[1])
    assert rel(out[0], want_plain) > 1e-4                    # the terms did something


def test_parameter_validation(mods):
    Oracle, inputs, sn = mods
    sim = sn.Simulation((64, 64), 10.0, -0.5, 1.0, 0.0, 1.0, (), 1e-3)
    for bad in [(0.1, 0.0, 0.0, 1.0), (0.1, -1.0, 0.0, 1.0), (0.0, 1e-12, 0.1, -1.0), (float("nan"), 1e-12, 0.0, 1.0)]:
        with pytest.raises(sn.SnError) as e:
            sim.set_local_terms(*bad)
        assert e.value.code == -3
    sim.close()


# ------------------------------------------------------------------ eq. (12): position-dependent Poisson source

def nmc_tables(dims, L, lam=1.0, r0=2.0):
    """gamma = (1/2)[1 - (r0/(r+r0))^lambda] (eq. (9)), beta = lambda (r0/(r+r0))^lambda /(r+r0) (eq. (10)), radius
    softened to sqrt(r^2 + 1) as for phi_C."""
    from paper_1909_08354_b200 import inputs
    X = np.meshgrid(*[inputs.coords(n, L) for n in dims], indexing="ij")
    r = np.sqrt(sum(x * x for x in X) + 1.0)
    f = (r0 / (r + r0)) ** lam
    return (lam * f / (r + r0)).astype(np.float32), (0.5 * (1.0 - f)).astype(np.float32)


@pytest.mark.parametrize("state", ["blobs", "noise"])
@pytest.mark.parametrize("dims,C", [((128, 64), 0.0), ((64, 256), -1.0), ((64, 64, 128), 0.0), ((96, 64, 64), -0.7),
                                    ((512, 64), 0.0), ((64, 512, 64), -0.7)])
def test_source_tables_potential_matches_oracle(mods, dims, C, state):
    """eq. (12).  "noise": white-noise psi, so that lap rho = F^-1[-k^2 rho^] is dominated by the
    highest wavenumbers -- the Nyquist row of the half spectrum, the mirrored rows of the packed transforms and the
    -k^2 multiplier at large k all carry the signal."""
    Oracle, inputs, sn = mods
    cfg = inputs.scaled(inputs.CONFIGS["C2" if len(dims) == 2 else "C4"], dims, L=16.0)
    psi0 = cfg.initial_state() if state == "blobs" else inputs.white_noise(dims, seed=23)
    beta, gamma = nmc_tables(dims, 16.0)
    sim = sn.Simulation(dims, 16.0, -0.5, 1.0, C, 0.9, (0.1,), 1e-3)
    sim.set_source_tables(beta, gamma)
    sim.set_state(psi0)
    orc = Oracle(dims, 16.0, -0.5, 1.0, C, 0.9, (0.1,), 1e-3)
    orc.set_source_tables(beta.astype(np.float64), gamma.astype(np.float64))
    orc.set_state(psi0.astype(np.complex128))
    got, want = sim.debug_potential(), orc.potential()
    # noise: lap rho = F^-1[-k^2 rho^] of white noise is all high-k content carried in fp32; a few 1e-6 at 512 points
    tol = 5e-6 if state == "blobs" else 2e-5
    assert rel(got, want) < tol and maxrel(got, want) < 10 * tol, (rel(got, want), maxrel(got, want))
    sim.set_source_tables(None, None)                      # back to eq. (2)
    orc.set_source_tables(None, None)
    assert rel(sim.debug_potential(), orc.potential()) < 2e-6
    sim.close()
    orc.close()


@pytest.mark.parametrize("name,dims,L,steps", [("C2", (256, 256), 25.0, 150), ("C4", (64, 128, 64), 16.0, 60),
                                               ("C5_256", (128, 128, 128), 128.0, 10)])
def test_source_tables_steps_match_oracle(mods, name, dims, L, steps):
    Oracle, inputs, sn = mods
    cfg = inputs.scaled(inputs.CONFIGS[name], dims, L=L, steps=steps)
    psi0 = cfg.initial_state()
    beta, gamma = nmc_tables(dims, L)
    sim = sn.Simulation.from_config(cfg)
    sim.set_source_tables(beta, gamma)
    sim.set_external_potential(nmc_potential(dims, L).astype(np.float32))   # the full NMC model of eq. (15): phi_N + phi_C
    sim.set_state(psi0)
    d0 = sim.diagnostics()
    sim.step(steps)
    got = sim.get_state()
    d1 = sim.diagnostics()
    sim.close()
    orc = Oracle.from_config(cfg)
    orc.set_source_tables(beta.astype(np.float64), gamma.astype(np.float64))
    orc.set_external_potential(nmc_potential(dims, L).astype(np.float32).astype(np.float64))
    orc.set_state(psi0.astype(np.complex128))
    orc.step(steps)
    want = orc.get_state()
    r1 = orc.diagnostics()
    orc.close()
    assert_state(got, want)
    assert abs(d1["norm"] - d0["norm"]) < TOL_NORM * d0["norm"]
    for k in ("e_kin", "e_nonlocal", "e_local"):
        assert abs(d1[k] - r1[k]) < 2e-5 * max(abs(r1["e_total"]), abs(r1[k])), (k, d1[k], r1[k])


# ------------------------------------------------------------------ fourth-order composition

@pytest.mark.parametrize("name,dims,L,steps,extras", [
    ("C2", (256, 256), 25.0, 100, False),
    ("C4", (64, 128, 64), 16.0, 40, False),
    ("C5_384", (96, 64, 128), 128.0, 10, False),
    ("C2", (128, 256), 25.0, 60, True),            # with the full NMC model: external potential rides on the right sub-step
])
def test_order4_steps_match_oracle(mods, name, dims, L, steps, extras):
    Oracle, inputs, sn = mods
    cfg = inputs.scaled(inputs.CONFIGS[name], dims, L=L, steps=steps)
    psi0 = cfg.initial_state()
    sim = sn.Simulation.from_config(cfg)
    orc = Oracle.from_config(cfg)
    if extras:
        beta, gamma = nmc_tables(dims, L)
        V = nmc_potential(dims, L).astype(np.float32)
        sim.set_local_terms(0.05, 1e-12, 0.03, 0.5)
        sim.set_external_potential(V)
        sim.set_source_tables(beta, gamma)
        orc.set_local_terms(0.05, 1e-12, 0.03, 0.5)
        orc.set_external_potential(V.astype(np.float64))
        orc.set_source_tables(beta.astype(np.float64), gamma.astype(np.float64))
    sim.set_state(psi0)
    d0 = sim.diagnostics()
    sim.step_order4(steps // 2)
    sim.step_order4(steps - steps // 2)                       # split calls: the end sweeps are half sweeps
    got = sim.get_state()
    d1 = sim.diagnostics()
    sim.close()
    orc.set_state(psi0.astype(np.complex128))
    orc.step_order4(steps)
    want = orc.get_state()
    orc.close()
    assert_state(got, want)
    assert abs(d1["norm"] - d0["norm"]) < TOL_NORM * d0["norm"]


def test_order4_differs_from_order2_by_the_splitting_error(mods):
    Oracle, inputs, sn = mods
    cfg = inputs.scaled(inputs.CONFIGS["C2"], (128, 128), L=25.0, steps=40)
    psi0 = cfg.initial_state()
    sim = sn.Simulation(cfg.dims, cfg.L, cfg.A, cfg.B, cfg.C, cfg.D, cfg.g, 2e-2)
    sim.set_state(psi0)
    sim.step(40)
    a = sim.get_state()
    sim.set_state(psi0)
    sim.step_order4(40)
    b = sim.get_state()
    sim.close()
    assert 1e-6 < rel(a, b) < 1e-2


# ------------------------------------------------------------------ ensembles of 2D systems

@pytest.mark.parametrize("dims,batch,steps", [((128, 128), 8, 60), ((64, 256), 3, 40), ((512, 64), 4, 12), ((96, 128), 5, 20)])
def test_batch2d_members_match_single_system_oracle(mods, dims, batch, steps):
    """An ensemble context advances every member exactly like a single-system run: compare each member with the
    float64 oracle run on that member alone, and the ensemble diagnostics with the sum of the members'."""
    Oracle, inputs, sn = mods
    L = 25.0
    base = inputs.scaled(inputs.CONFIGS["C2"], dims, L=L, steps=steps)
    rng = np.random.default_rng(11)
    members = []
    for b in range(batch):                                # same recipe, each member rotated/scaled differently
        psi = np.roll(base.initial_state(), (int(rng.integers(dims[0])), int(rng.integers(dims[1]))), axis=(0, 1))
        members.append((psi * np.complex64(0.6 + 0.1 * b)).astype(np.complex64))
    store = np.ascontiguousarray(np.stack(members, axis=1))          # storage layout [n0][batch][n1]
    sim = sn.Simulation(dims, L, base.A, base.B, base.C, base.D, base.g, base.dtau, batch=batch)
    assert sim.dims == (dims[0], batch, dims[1])
    sim.set_state(store)
    d0 = sim.diagnostics()
    sim.step(steps)
    got = sim.get_state()
    d1 = sim.diagnostics()
    sim.close()
    tot = {k: 0.0 for k in d1}
    for b in range(batch):
        orc = Oracle(dims, L, base.A, base.B, base.C, base.D, base.g, base.dtau)
        orc.set_state(members[b].astype(np.complex128))
        orc.step(steps)
        assert rel(got[:, b, :], orc.get_state()) < TOL_STATE, b
        r = orc.diagnostics()
        for k in tot:
            tot[k] += r[k]
        orc.close()
    assert abs(d1["norm"] - d0["norm"]) < TOL_NORM * d0["norm"]
    for k in tot:
        assert abs(d1[k] - tot[k]) < 2e-5 * max(abs(tot["e_total"]), abs(tot[k])), (k, d1[k], tot[k])


def test_batch_validation(mods):
    Oracle, inputs, sn = mods
    from paper_1909_08354_b200.sn import lib
    import ctypes
    d = (ctypes.c_int64 * 2)(128, 128)
    assert lib().sn_workspace_bytes_batch(2, d, 0) == 0
    assert lib().sn_workspace_bytes_batch(2, d, 7) > 7 * 128 * 128 * 8
    assert lib().sn_workspace_bytes_batch(2, d, 1) == lib().sn_workspace_bytes(2, d)
    bad = (ctypes.c_int64 * 2)(100, 128)
    assert lib().sn_workspace_bytes_batch(2, bad, 4) == 0


@pytest.mark.parametrize("dims,batch,steps", [((64, 64, 64), 5, 20), ((64, 128, 64), 2, 12), ((96, 64, 128), 3, 6)])
def test_batch3d_members_match_single_system_oracle(mods, dims, batch, steps):
    """Ensembles of 3D systems: storage [n0][batch][n1][n2]; the axis-1 passes see n0*batch outer blocks."""
    Oracle, inputs, sn = mods
    L = 16.0
    base = inputs.scaled(inputs.CONFIGS["C4"], dims, L=L, steps=steps)
    members = [np.roll(base.initial_state(), (3 * b, 5 * b, 7 * b), axis=(0, 1, 2)) * np.complex64(0.8 + 0.1 * b)
               for b in range(batch)]
    sim = sn.Simulation(dims, L, base.A, base.B, base.C, base.D, base.g, base.dtau, batch=batch)
    assert sim.dims == (dims[0], batch, dims[1], dims[2])
    sim.set_state(np.ascontiguousarray(np.stack(members, axis=1).astype(np.complex64)))
    d0 = sim.diagnostics()
    sim.step(steps)
    got = sim.get_state()
    d1 = sim.diagnostics()
    sim.close()
    tot = {k: 0.0 for k in d1}
    for b in range(batch):
        orc = Oracle(dims, L, base.A, base.B, base.C, base.D, base.g, base.dtau)
        orc.set_state(members[b].astype(np.complex64).astype(np.complex128))
        orc.step(steps)
        assert rel(got[:, b], orc.get_state()) < TOL_STATE, b
        r = orc.diagnostics()
        for k in tot:
            tot[k] += r[k]
        orc.close()
    assert abs(d1["norm"] - d0["norm"]) < TOL_NORM * d0["norm"]
    for k in tot:
        assert abs(d1[k] - tot[k]) < 2e-5 * max(abs(tot["e_total"]), abs(tot[k])), (k, d1[k], tot[k])


def test_batch2d_with_nmc_terms_and_order4(mods):
    """Ensemble + every NEXT-1 term + the fourth-order step at once: the tables are per member, stored in the same
    [n0][batch][n1] layout as the state."""
    Oracle, inputs, sn = mods
    dims, batch, L, steps = (128, 64), 3, 25.0, 16
    base = inputs.scaled(inputs.CONFIGS["C2"], dims, L=L, steps=steps)
    beta, gamma = nmc_tables(dims, L)
    V = nmc_potential(dims, L).astype(np.float32)
    members = [np.roll(base.initial_state(), 7 * b, axis=1) * np.complex64(0.7 + 0.1 * b) for b in range(batch)]
    tabs = [(np.roll(beta, 3 * b, axis=0) * (1.0 + 0.2 * b), gamma * (1.0 - 0.1 * b), V * (1.0 + 0.5 * b)) for b in range(batch)]
    st = lambda arrs, dt: np.ascontiguousarray(np.stack(arrs, axis=1).astype(dt))
    sim = sn.Simulation(dims, L, base.A, base.B, base.C, base.D, base.g, base.dtau, batch=batch)
    sim.set_local_terms(0.04, 1e-12, 0.03, 0.5)
    sim.set_source_tables(st([t[0] for t in tabs], np.float32), st([t[1] for t in tabs], np.float32))
    sim.set_external_potential(st([t[2] for t in tabs], np.float32))
    sim.set_state(st(members, np.complex64))
    sim.step_order4(steps)
    got = sim.get_state()
    sim.close()
    for b in range(batch):
        orc = Oracle(dims, L, base.A, base.B, base.C, base.D, base.g, base.dtau)
        orc.set_local_terms(0.04, 1e-12, 0.03, 0.5)
        orc.set_source_tables(tabs[b][0].astype(np.float32).astype(np.float64), tabs[b][1].astype(np.float32).astype(np.float64))
        orc.set_external_potential(tabs[b][2].astype(np.float32).astype(np.float64))
        orc.set_state(members[b].astype(np.complex64).astype(np.complex128))
        orc.step_order4(steps)
        assert rel(got[:, b, :], orc.get_state()) < TOL_STATE, b
        orc.close()


# ------------------------------------------------------------------ full size, all terms: exact plane-wave solution

@pytest.mark.parametrize("dims,C,order4", [((512, 512, 512), -1.0, False), ((256, 256, 256), -0.6, True),
                                           ((4096, 2048), -1.0, False)])
def test_plane_wave_full_size_with_next_terms(mods, dims, C, order4):
    """At BASELINE.json's full sizes, in the launch configuration bench.py --extras times: a plane wave a e^{iq.x}
    stays an exact solution with the logarithmic/power-law terms, a uniform external potential v0 and CONSTANT source
    tables gamma = g0, beta = b0 (rho is uniform, so lap rho = 0 and phi0 = D g0 a^2/C):
    psi(tau) = psi0 exp(i (A|q|^2 - B phi0 - G(a^2) - v0) tau), for the Strang and the order-4 step alike."""
    Oracle, inputs, sn = mods
    L, A, B, D, g, dtau, steps, amp = 32.0, -0.5, 1.3, 0.9, (0.2,), 5e-3, 12, 0.8
    g_log, g_pow, p, v0, g0, b0 = 0.31, -0.45, 2.0 / 3.0, 0.37, 0.6, 0.25
    nd = len(dims)
    mode = (3, -2, 5)[:nd]
    ax = [inputs.coords(n, L) for n in dims]
    ph = sum((2 * np.pi / L * m) * a.reshape([-1 if i == k else 1 for i in range(nd)]) for k, (m, a) in enumerate(zip(mode, ax)))
    psi0 = (amp * np.exp(1j * ph)).astype(np.complex64)
    del ph
    q2 = sum((2 * np.pi / L * m) ** 2 for m in mode)
    sim = sn.Simulation(dims, L, A, B, C, D, g, dtau)
    sim.set_local_terms(g_log, 1e-12, g_pow, p)
    sim.set_external_potential(np.full(dims, v0, dtype=np.float32))
    sim.set_source_tables(np.full(dims, b0, dtype=np.float32), np.full(dims, g0, dtype=np.float32))
    sim.set_state(psi0)
    (sim.step_order4 if order4 else sim.step)(steps)
    got = sim.get_state()
    sim.close()
    a2 = amp * amp
    omega = A * q2 - B * D * g0 * a2 / C - (g[0] * a2 + g_log * np.log(a2) + g_pow * a2 ** p) - v0
    rot = complex(np.exp(1j * omega * dtau * steps))
    num = den = 0.0
    g1, p1 = got.reshape(-1), psi0.reshape(-1)
    for i in range(0, g1.size, 1 << 24):
        w = p1[i:i + (1 << 24)].astype(np.complex128) * rot
        num += float(np.sum(np.abs(g1[i:i + (1 << 24)] - w) ** 2))
        den += float(np.sum(np.abs(w) ** 2))
    assert np.sqrt(num / den) < 2e-5


# ------------------------------------------------------------------ Bohm quantum potential of eq. (15)

def smooth_positive_state(inputs, dims, Ls):
    """rho = 1 + 0.3 cos(q1.x) + 0.2 cos(q2.x) > 0 everywhere, phase 0.25 sin(q3.x): no nodes, so V_B is well conditioned
    (a state with interference zeros makes lap sqrt(rho)/sqrt(rho) singular and fp32 and fp64 runs decorrelate)."""
    nd = len(dims)
    X = np.meshgrid(*[inputs.coords(n, L) for n, L in zip(dims, Ls)], indexing="ij")
    ph = lambda m: sum(2 * np.pi / L * mi * x for mi, x, L in zip(m, X, Ls))
    rho = 1.0 + 0.3 * np.cos(ph((1, 2, -1)[:nd])) + 0.2 * np.cos(ph((-2, 1, 1)[:nd]))
    return (np.sqrt(rho) * np.exp(0.25j * np.sin(ph((1, -1, 2)[:nd])))).astype(np.complex64)


@pytest.mark.parametrize("dims,steps,order4", [((256, 256), 60, False), ((64, 128, 64), 30, False), ((512, 128), 30, False),
                                               ((128, 96), 30, True), ((2048, 64), 10, False)])
def test_bohm_term_matches_oracle(mods, dims, steps, order4):
    """The Bohm phase is a derivative-dependent potential treated explicitly: dtau c_B k_max^2 must stay small or the
    scheme itself (oracle included) amplifies grid-scale noise; h = 0.15 on every axis keeps it at 0.2 per step."""
    Oracle, inputs, sn = mods
    Ls = tuple(0.15 * n for n in dims)
    psi0 = smooth_positive_state(inputs, dims, Ls)
    par = dict(A=-0.5, B=1.0, C=-1.0, D=0.5, g=(0.1,), dtau=2e-3)
    sim = sn.Simulation(dims, Ls, par["A"], par["B"], par["C"], par["D"], par["g"], par["dtau"])
    sim.set_bohm(0.4, 1e-3)
    sim.set_state(psi0)
    d0 = sim.diagnostics()
    (sim.step_order4 if order4 else sim.step)(steps)
    got = sim.get_state()
    d1 = sim.diagnostics()
    sim.close()
    orc = Oracle(dims, Ls, par["A"], par["B"], par["C"], par["D"], par["g"], par["dtau"])
    orc.set_bohm(0.4, 1e-3)
    orc.set_state(psi0.astype(np.complex128))
    (orc.step_order4 if order4 else orc.step)(steps)
    want = orc.get_state()
    orc.set_bohm(0.0, 1e-3)
    orc.set_state(psi0.astype(np.complex128))
    (orc.step_order4 if order4 else orc.step)(steps)
    without = orc.get_state()
    orc.close()
    assert rel(want, without) > 1e-4                       # the term matters in this run
    assert_state(got, want)
    assert abs(d1["norm"] - d0["norm"]) < TOL_NORM * d0["norm"]


def test_bohm_term_makes_real_states_stationary(mods):
    """c_B = -2A cancels the quantum pressure: the Gaussian that spreads under K alone stays put (pin W7)."""
    Oracle, inputs, sn = mods
    dims, L, s, a = (128, 128), 24.0, 1.7, 0.8
    X = np.meshgrid(*[inputs.coords(n, L) for n in dims], indexing="ij")
    psi0 = (a * np.exp(-(X[0] ** 2 + X[1] ** 2) / (2 * s * s))).astype(np.complex64)
    sim = sn.Simulation(dims, L, -0.5, 0.0, 0.0, 0.0, (), 1e-2)
    sim.set_state(psi0)
    sim.step(100)
    assert rel(sim.get_state(), psi0) > 0.1               # spreads without the Bohm term
    sim.set_bohm(1.0, 1e-4)
    sim.set_state(psi0)
    sim.step(100)
    assert rel(sim.get_state(), psi0) < 2e-4               # stationary with it (fp32 transform noise in the tails)
    sim.set_bohm(0.0, 1e-4)
    sim.close()


@pytest.mark.parametrize("dims,batch,steps", [((128, 64), 3, 30), ((64, 64, 64), 2, 16), ((32, 32), 7, 30)])
def test_bohm_term_in_an_ensemble(mods, dims, batch, steps):
    """The Bohm chain (sqrt(rho) r2c, Laplacian multiplier, axis-0 phase pass) on the ensemble layout: each member
    matches the single-system oracle."""
    Oracle, inputs, sn = mods
    Ls = tuple(0.15 * n for n in dims)
    par = dict(A=-0.5, B=1.0, C=-1.0, D=0.5, g=(0.1,), dtau=2e-3)
    base = smooth_positive_state(inputs, dims, Ls)
    members = [(np.roll(base, 5 * b, axis=len(dims) - 1) * np.complex64(0.8 + 0.15 * b)).astype(np.complex64)
               for b in range(batch)]
    sim = sn.Simulation(dims, Ls, par["A"], par["B"], par["C"], par["D"], par["g"], par["dtau"], batch=batch)
    sim.set_bohm(0.4, 1e-3)
    sim.set_state(np.ascontiguousarray(np.stack(members, axis=1)))
    sim.step(steps)
    got = sim.get_state()
    sim.close()
    for b in range(batch):
        orc = Oracle(dims, Ls, par["A"], par["B"], par["C"], par["D"], par["g"], par["dtau"])
        orc.set_bohm(0.4, 1e-3)
        orc.set_state(members[b].astype(np.complex128))
        orc.step(steps)
        assert rel(got[:, b], orc.get_state()) < TOL_STATE, b
        orc.close()


@pytest.mark.parametrize("dims,order4", [((128, 128), False), ((64, 96, 64), False), ((256, 64), True), ((32, 32, 64), False),
                                         ((64, 32), True)])
def test_every_term_at_once(mods, dims, order4):
    """Eq. (12) source tables, eq. (15)/(16) log and power terms, external potential and Bohm term in one run."""
    Oracle, inputs, sn = mods
    Ls = tuple(0.15 * n for n in dims)
    nd = len(dims)
    X = np.meshgrid(*[inputs.coords(n, L) for n, L in zip(dims, Ls)], indexing="ij")
    ph = lambda m: sum(2 * np.pi / L * mi * x for mi, x, L in zip(m, X, Ls))
    beta = (1.0 + 0.2 * np.cos(ph((1, 0, 1)[:nd]))).astype(np.float32)
    gamma = (0.05 * np.sin(ph((0, 1, 1)[:nd]))).astype(np.float32)
    V = (0.3 * np.cos(ph((1, 1, 0)[:nd]))).astype(np.float32)
    psi0 = smooth_positive_state(inputs, dims, Ls)
    par = dict(A=-0.5, B=1.0, C=-1.0, D=0.5, g=(0.1, -0.02), dtau=2e-3)
    steps = 20

    def drive(o, cast):
        o.set_local_terms(0.04, 1e-12, 0.03, 0.5)
        o.set_source_tables(cast(beta), cast(gamma))
        o.set_external_potential(cast(V))
        o.set_bohm(0.3, 1e-3)
        o.set_state(psi0.astype(np.complex128) if cast is f64 else psi0)
        (o.step_order4 if order4 else o.step)(steps)
        return o.get_state()

    f64 = lambda a: a.astype(np.float64)
    sim = sn.Simulation(dims, Ls, par["A"], par["B"], par["C"], par["D"], par["g"], par["dtau"])
    got = drive(sim, lambda a: a)
    sim.close()
    orc = Oracle(dims, Ls, par["A"], par["B"], par["C"], par["D"], par["g"], par["dtau"])
    want = drive(orc, f64)
    orc.close()
    assert_state(got, want)

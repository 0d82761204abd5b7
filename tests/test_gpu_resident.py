"""GPU parity of the cluster-resident step kernel (csrc/sn_resident.cu) against the float64 oracle and against the pass
kernels.

sn_step on a complex64 2D grid with n0 == n1 in {64, 128} runs, by default, as ONE launch that keeps the state in the
distributed shared memory of a cluster of 8 CTAs for all n steps (SN_OPT_RESIDENT).  Same schedule as the pass kernels
(K(dtau/2) [N(dtau) K(dtau)]^(n-1) N(dtau) K(dtau/2); eq. (1),(2) PAPER.md:42-44), so the acceptance is
north_star's: rel-L2 <= 1e-4 against the oracle (+ the element-wise bound of _parity.assert_state), norm drift <= 1e-5.
The orientation of its sweeps alternates from step to step, so step counts 1, 2, 3 are compared separately.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from _parity import TOL_NORM, assert_state, rel


@pytest.fixture(scope="module")
def mods():
    from oracle.snref import Oracle
    from paper_1909_08354_b200 import inputs, sn
    return Oracle, inputs, sn


def oracle_run(Oracle, cfg, psi0, steps):
    orc = Oracle.from_config(cfg)
    orc.set_state(psi0.astype(np.complex128))
    orc.step(steps)
    want = orc.get_state()
    orc.close()
    return want


def gpu_run(sn, cfg, psi0, calls, resident=1, batch=None, prepare=None, features=0):
    sim = sn.Simulation.from_config(cfg, batch=batch, features=features)
    sim.set_option(sn.OPT_RESIDENT, resident)
    if prepare:
        prepare(sim)
    sim.set_state(psi0)
    n0 = sim.launch_count()
    for n in calls:
        sim.step(n)
    launches = sim.launch_count() - n0
    out = sim.get_state()
    norm = sim.diagnostics()["norm"]
    sim.close()
    return out, launches, norm


CASES = [("C1", (128, 128), None, 200),       # BASELINE.json configs[0], whole configured run
         ("C1", (128, 128), None, 1), ("C1", (128, 128), None, 2), ("C1", (128, 128), None, 3),
         ("C2", (128, 128), 25.0, 60), ("C2", (64, 64), 12.5, 40), ("C2", (64, 64), 12.5, 1), ("C2", (64, 64), 12.5, 2),
         ("C3", (128, 128), 100.0, 30)]       # C = -1 (screened Poisson), defocusing G


@pytest.mark.parametrize("name,dims,L,steps", CASES)
def test_resident_steps_match_oracle(mods, name, dims, L, steps):
    Oracle, inputs, sn = mods
    base = inputs.CONFIGS[name]
    cfg = base if tuple(base.dims) == dims and L is None else inputs.scaled(base, dims, L=L, steps=steps)
    psi0 = cfg.initial_state()
    got, launches, norm = gpu_run(sn, cfg, psi0, [steps])
    assert launches == 1                       # the whole call is one launch
    want = oracle_run(Oracle, cfg, psi0, steps)
    assert_state(got, want)
    n0 = float(np.sum(np.abs(psi0.astype(np.complex128)) ** 2)) * np.prod([l / n for l, n in zip(np.broadcast_to(cfg.L, (2,)), dims)])
    assert abs(norm - n0) / n0 < TOL_NORM


@pytest.mark.parametrize("C,D", [(0.0, 1.0), (-0.7, 1.0), (3.3, 0.8)])
def test_resident_white_noise_state_and_helmholtz_constants(mods, C, D):
    """A white-noise state loads every mode up to Nyquist on both axes, so a wrong multiplier row / column, a wrong
    mirrored index of the C - k0^2 table or a wrong orientation of the alternating sweeps shows; C > 0 lies between
    grid modes (the hi/lo denominator of eq. (2))."""
    Oracle, inputs, sn = mods
    dims, L = (128, 128), 12.0
    psi0 = (0.3 * inputs.white_noise(dims, 21)).astype(np.complex64)
    for steps in (1, 4):
        sim = sn.Simulation(dims, L, -0.5, 1.0, C, D, (0.1, 0.02), 2e-3)
        sim.set_state(psi0)
        sim.step(steps)
        got = sim.get_state()
        sim.close()
        orc = Oracle(dims, L, -0.5, 1.0, C, D, (0.1, 0.02), 2e-3)
        orc.set_state(psi0.astype(np.complex128))
        orc.step(steps)
        want = orc.get_state()
        orc.close()
        assert_state(got, want)


@pytest.mark.parametrize("dims,batch", [((128, 128), None), ((64, 64), None), ((128, 128), 3), ((64, 64), 5)])
def test_resident_agrees_with_pass_kernels_and_split_calls(mods, dims, batch):
    """SN_OPT_RESIDENT = 0 runs the same schedule through the pass kernels: the two agree to rounding (the resident
    kernel transforms the density as a complex field, the pass kernels as a packed real one).  Ensemble members run
    in separate clusters and must not mix; several calls equal one call."""
    Oracle, inputs, sn = mods
    cfg = inputs.scaled(inputs.CONFIGS["C2"], dims, L=12.5 * dims[0] / 64, steps=12)
    one = cfg.initial_state()
    if batch is None:
        psi0 = one
    else:  # members differ in amplitude and phase: storage (n0, batch, n1)
        psi0 = np.stack([one * (1.0 + 0.2 * b) * np.exp(0.4j * b) for b in range(batch)], axis=1).astype(np.complex64)
    a, la, _ = gpu_run(sn, cfg, psi0, [12], resident=1, batch=batch)
    b, lb, _ = gpu_run(sn, cfg, psi0, [12], resident=0, batch=batch)
    c, lc, _ = gpu_run(sn, cfg, psi0, [5, 1, 6], resident=1, batch=batch)
    assert la == 1 and lc == 3 and lb > 12
    assert rel(a, b) < 5e-6
    assert rel(c, a) < 5e-6
    if batch is not None:  # member 0 of the ensemble = the single system
        s, _, _ = gpu_run(sn, cfg, one, [12], resident=1)
        assert np.array_equal(a[:, 0], s)


def test_resident_falls_back_to_the_pass_kernels(mods):
    """Contexts the resident kernel does not serve take the pass kernels with unchanged results: the Bohm term in
    effect, a forced dispatch, an ensemble above its member limit."""
    Oracle, inputs, sn = mods
    cfg = inputs.scaled(inputs.CONFIGS["C2"], (64, 64), L=12.5, steps=6)
    psi0 = cfg.initial_state()
    terms = lambda sim: sim.set_bohm(0.05, 1e-3)
    a, la, _ = gpu_run(sn, cfg, psi0, [6], resident=1, prepare=terms)
    b, lb, _ = gpu_run(sn, cfg, psi0, [6], resident=0, prepare=terms)
    assert la == lb and la > 6 and np.array_equal(a, b)
    forced = lambda sim: sim.set_option(sn.OPT_DISPATCH, sn.DISPATCH_FIRST_PATH)
    _, lf, _ = gpu_run(sn, cfg, psi0, [6], resident=1, prepare=forced)
    assert lf > 6
    big = np.stack([psi0] * 300, axis=1)          # above the member limit of the 64^2 kernel (256; 32 at 128^2)
    _, lbig, _ = gpu_run(sn, cfg, big, [6], resident=1, batch=300)
    assert lbig > 6
    cleared = lambda sim: (sim.set_bohm(0.05, 1e-3), sim.set_bohm(0.0, 1e-3))
    _, lcl, _ = gpu_run(sn, cfg, psi0, [6], resident=1, prepare=cleared)
    assert lcl == 1                              # term switched off again: eligible again
    sim = sn.Simulation.from_config(cfg)
    with pytest.raises(sn.SnError):              # the option takes 0 or 1
        sim.set_option(sn.OPT_RESIDENT, 2)
    sim.set_state(psi0)
    sim.step(0)                                  # no step: no launch, state untouched
    assert np.array_equal(sim.get_state(), psi0)
    sim.close()


@pytest.mark.parametrize("terms", [(0.05, 1e-12, 0.0, 1.0), (0.0, 1e-12, 0.08, 2.0 / 3.0), (0.02, 1e-12, 0.05, 0.5)])
def test_resident_local_terms_match_oracle(mods, terms):
    """The logarithmic and power-law terms of eq. (16) (V_p = w ln rho, (n w/(n-1)) rho^(n-1)) run through
    the resident kernel's nonlinear phase; against the oracle and against the pass kernels."""
    Oracle, inputs, sn = mods
    cfg = inputs.scaled(inputs.CONFIGS["C2"], (128, 128), L=25.0, steps=40)
    psi0 = cfg.initial_state()
    prep = lambda sim: sim.set_local_terms(*terms)
    a, la, _ = gpu_run(sn, cfg, psi0, [40], resident=1, prepare=prep)
    b, lb, _ = gpu_run(sn, cfg, psi0, [40], resident=0, prepare=prep)
    assert la == 1 and lb > 40
    orc = Oracle.from_config(cfg)
    orc.set_local_terms(*terms)
    orc.set_state(psi0.astype(np.complex128))
    orc.step(40)
    want = orc.get_state()
    orc.close()
    assert_state(a, want)
    assert rel(a, b) < 5e-6


@pytest.mark.parametrize("dims,order4", [((128, 128), False), ((64, 64), False), ((128, 128), True)])
def test_resident_external_potential_matches_oracle(mods, dims, order4):
    """A fixed external potential V(x) (phi_C of eq. (15); softened at the origin, reading Q16) together
    with the local terms: its rows sit in the ranks' shared memory and its phase rides on the nonlinear phase."""
    Oracle, inputs, sn = mods
    L = 25.0 * dims[0] / 128
    cfg = inputs.scaled(inputs.CONFIGS["C2"], dims, L=L, steps=30)
    psi0 = cfg.initial_state()
    X = np.meshgrid(*[inputs.coords(n, L) for n in dims], indexing="ij")
    r = np.sqrt(sum(x * x for x in X) + 1.0)
    V = (-1.0 / r + 0.05 * X[0] - 0.02 * X[1]).astype(np.float32)   # not symmetric under transposition
    steps = 6 if order4 else 30
    def prep(sim):
        sim.set_local_terms(0.02, 1e-12, 0.05, 0.5)
        sim.set_external_potential(V)
    def run(res):
        sim = sn.Simulation.from_config(cfg, features=sn.FEAT_VEXT)
        sim.set_option(sn.OPT_RESIDENT, res)
        prep(sim)
        sim.set_state(psi0)
        n0 = sim.launch_count()
        (sim.step_order4 if order4 else sim.step)(steps)
        out = (sim.get_state(), sim.launch_count() - n0)
        sim.close()
        return out
    a, la = run(1)
    b, lb = run(0)
    assert la == 1 and lb > steps
    orc = Oracle.from_config(cfg)
    orc.set_local_terms(0.02, 1e-12, 0.05, 0.5)
    orc.set_external_potential(V.astype(np.float64))
    orc.set_state(psi0.astype(np.complex128))
    (orc.step_order4 if order4 else orc.step)(steps)
    want = orc.get_state()
    orc.close()
    assert_state(a, want)
    assert rel(a, b) < 5e-6


@pytest.mark.parametrize("dims,steps", [((128, 128), 6), ((64, 64), 5)])
def test_resident_order4_steps_match_oracle(mods, dims, steps):
    """sn_step_order4 (three Strang sub-steps per step) runs through the same kernel with a period-3
    program: against the oracle's fourth-order step, against the pass kernels, and split into two calls."""
    Oracle, inputs, sn = mods
    cfg = inputs.scaled(inputs.CONFIGS["C2"], dims, L=12.5 * dims[0] / 64, steps=steps)
    psi0 = cfg.initial_state()
    out = {}
    for res in (1, 0):
        sim = sn.Simulation.from_config(cfg)
        sim.set_option(sn.OPT_RESIDENT, res)
        sim.set_state(psi0)
        n0 = sim.launch_count()
        sim.step_order4(steps // 2)
        sim.step_order4(steps - steps // 2)
        out[res] = (sim.get_state(), sim.launch_count() - n0)
        sim.close()
    assert out[1][1] == 2 and out[0][1] > 2 * steps
    orc = Oracle.from_config(cfg)
    orc.set_state(psi0.astype(np.complex128))
    orc.step_order4(steps // 2)
    orc.step_order4(steps - steps // 2)
    want = orc.get_state()
    orc.close()
    assert_state(out[1][0], want)
    assert rel(out[1][0], out[0][0]) < 5e-6


@pytest.mark.parametrize("dims,batch", [((128, 128), 32), ((64, 64), 256)])
def test_resident_full_ensembles_are_bitwise_the_single_system(mods, dims, batch):
    """The largest ensembles the kernel serves: every cluster of the machine busy at once, rough states (blobs + white
    noise).  Every member must equal the single-system run bit for bit, in every repetition: a race between clusters, or
    between the remote accesses of one cluster and its barriers, would show as a differing member."""
    Oracle, inputs, sn = mods
    cfg = inputs.scaled(inputs.CONFIGS["C2"], dims, L=12.5 * dims[0] / 64, steps=60)
    one = (0.5 * cfg.initial_state() + 0.2 * inputs.white_noise(dims, 3)).astype(np.complex64)
    ref, l1, _ = gpu_run(sn, cfg, one, [60])
    psi0 = np.stack([one] * batch, axis=1).astype(np.complex64)
    for rep in range(3):
        out, lb, _ = gpu_run(sn, cfg, psi0, [60], batch=batch)
        assert l1 == 1 and lb == 1
        assert all(np.array_equal(out[:, b], ref) for b in range(batch)), rep


def test_resident_runs_are_bitwise_identical(mods):
    Oracle, inputs, sn = mods
    cfg = inputs.CONFIGS["C1"]
    psi0 = (0.3 * inputs.white_noise(cfg.dims, 4)).astype(np.complex64)
    outs = [gpu_run(sn, cfg, psi0, [25])[0] for _ in range(3)]
    assert np.array_equal(outs[0], outs[1]) and np.array_equal(outs[0], outs[2])

"""GPU parity of the complex128 path (sn_options.dtype = SN_DTYPE_C128; SURVEY.md 8(f) item 3 -- the precision the
paper benchmarked) against the float64 oracle, through the C ABI.

Both sides now compute in float64, so the tolerances are roundoff-class.  Derivation: one radix-8 Stockham transform
of N <= 4096 points has a relative error of a few eps64 = 2.2e-16 (log_8 N <= 4 stages, errors add in quadrature);
a Strang step is 2 d + 4-ish transforms deep and the dynamics of the configs amplify perturbations by ~1.0x over a
run, so after n steps the two implementations differ by ~ sqrt(n) * 10 * eps64: 1e-13 at n = 1000.
Written with one decade of margin: rel-L2 <= 1e-12 per run, <= 1e-14 per transform round trip, norm drift <= 1e-13.
"""
import numpy as np
import pytest

from _parity import maxrel, rel

pytestmark = pytest.mark.gpu

TOL_STATE64 = 1e-12
TOL_ROUNDTRIP64 = 1e-14
TOL_NORM64 = 1e-13


@pytest.fixture(scope="module")
def mods():
    from oracle import snref
    from oracle.snref import Oracle
    from paper_1909_08354_b200 import inputs, sn
    return snref, Oracle, inputs, sn


def noise128(dims, seed):
    rng = np.random.default_rng(seed)
    z = rng.standard_normal(tuple(dims) + (2,))
    return np.ascontiguousarray(z[..., 0] + 1j * z[..., 1])


def sim128(sn, cfg, **kw):
    return sn.Simulation(cfg.dims, cfg.L, cfg.A, cfg.B, cfg.C, cfg.D, cfg.g, cfg.dtau, dtype="complex128", **kw)


@pytest.mark.parametrize("dims", [(64, 64), (128, 256), (512, 64), (64, 1024), (2048, 64), (64, 4096), (4096, 32),
                                  (64, 64, 64), (128, 64, 256), (64, 512, 128), (32, 32, 32),
                                  (96, 96), (384, 64), (64, 384), (1536, 64), (96, 384, 64),
                                  (192, 64), (64, 192), (768, 192), (3072, 64), (64, 3072), (192, 64, 768)])
def test_fft_forward_matches_oracle_and_round_trip(mods, dims):
    snref, Oracle, inputs, sn = mods
    x = noise128(dims, 11)
    sim = sn.Simulation(dims, 10.0, -0.5, 1.0, 0.0, 1.0, (), 1e-3, dtype="complex128")
    sim.set_state(x)
    sim.debug_fft(+1)
    assert rel(sim.get_state(), snref.fftn(x, +1)) < 2e-15
    sim.debug_fft(-1)
    assert rel(sim.get_state(), x) < TOL_ROUNDTRIP64
    sim.close()


@pytest.mark.parametrize("state", ["blobs", "noise"])
@pytest.mark.parametrize("dims,C", [((64, 128), 0.0), ((128, 64), -1.0), ((64, 64, 128), 0.0), ((64, 128, 64), -0.7),
                                    ((384, 96), 0.0), ((96, 64, 384), -0.7), ((32, 32), 0.0), ((512, 64), 0.0),
                                    ((64, 512, 64), -0.7), ((64, 64, 512), 0.0), ((64, 64, 64), 7.7)])
def test_potential_matches_oracle(mods, dims, C, state):
    """eq. (2): r2c -> D/(C - k^2) -> c2r against the oracle's full complex transforms; "noise" loads
    the Nyquist row and the mirrored rows of the packed real transforms."""
    snref, Oracle, inputs, sn = mods
    cfg = inputs.scaled(inputs.CONFIGS["C2" if len(dims) == 2 else "C4"], dims, L=16.0)
    psi0 = cfg.initial_state().astype(np.complex128) if state == "blobs" else noise128(dims, 21)
    sim = sn.Simulation(dims, 16.0, -0.5, 1.0, C, 0.9, (0.1,), 1e-3, dtype="complex128")
    sim.set_state(psi0)
    orc = Oracle(dims, 16.0, -0.5, 1.0, C, 0.9, (0.1,), 1e-3)
    orc.set_state(psi0)
    got, want = sim.debug_potential(), orc.potential()
    sim.close()
    orc.close()
    assert got.dtype == np.float64
    # C = 7.7 sits 1.4e-3 (relative) from a grid mode: that mode's 1/(C - k^2) amplifies roundoff 700x
    tol = 1e-14 if C <= 0 else 1e-12
    assert rel(got, want) < tol and maxrel(got, want) < 10 * tol, (rel(got, want), maxrel(got, want))


STEP_CASES = [
    ("C1", (128, 128), 20.0, 200),          # C1 in full
    ("C2", (256, 256), 25.0, 400),
    ("C2", (1024, 1024), 100.0, 100),       # full size, prefix
    ("C3", (512, 512), 50.0, 100),          # C = -1
    ("C3", (4096, 64), 50.0, 10),
    ("C3", (2048, 128), 50.0, 10),
    ("C4", (64, 64, 64), 16.0, 100),
    ("C5_64", (64, 64, 64), 128.0, 100),    # sweep point in full
    ("C5_128", (128, 128, 128), 128.0, 10),
    ("C4", (64, 128, 256), 32.0, 10),       # three different line lengths
    ("C4", (64, 2048, 64), 16.0, 3),
    ("C4", (64, 64, 4096), 16.0, 3),
    ("C5_256", (256, 256, 256), 128.0, 2),
    ("C2", (384, 96), 25.0, 100),           # 3*2^a lengths on both axes
    ("C5_384", (96, 96, 96), 128.0, 20),
    ("C5_384", (384, 64, 128), 128.0, 4),
    ("C5_384", (64, 128, 384), 128.0, 4),
    ("C2", (192, 768), 25.0, 40),
    ("C2", (32, 32), 6.25, 200),
    ("C4", (32, 256, 32), 16.0, 10),
    ("C5_512", (64, 512, 128), 128.0, 2),
]


@pytest.mark.parametrize("name,dims,L,steps", STEP_CASES)
def test_steps_match_oracle(mods, name, dims, L, steps):
    snref, Oracle, inputs, sn = mods
    cfg = inputs.scaled(inputs.CONFIGS[name], dims, L=L, steps=steps)
    psi0 = cfg.initial_state().astype(np.complex128)   # the complex64-rounded recipe state, cast up: same input as the c64 tests
    sim = sim128(sn, cfg)
    sim.set_state(psi0)
    d0 = sim.diagnostics()
    sim.step(steps)
    got = sim.get_state()
    d1 = sim.diagnostics()
    sim.close()
    orc = Oracle.from_config(cfg)
    orc.set_state(psi0)
    r0 = orc.diagnostics()
    orc.step(steps)
    want = orc.get_state()
    r1 = orc.diagnostics()
    orc.close()
    assert got.dtype == np.complex128
    assert rel(got, want) < TOL_STATE64 and maxrel(got, want) < 10 * TOL_STATE64, (rel(got, want), maxrel(got, want))
    assert abs(d1["norm"] - d0["norm"]) < TOL_NORM64 * d0["norm"]
    scale = abs(r1["e_kin"]) + abs(r1["e_nonlocal"]) + abs(r1["e_local"])
    for d, r in ((d0, r0), (d1, r1)):
        assert abs(d["norm"] - r["norm"]) < 1e-12 * r["norm"]   # sums of up to 2^24 terms taken in different orders
        for k in ("e_kin", "e_nonlocal", "e_local", "e_total"):
            assert abs(d[k] - r[k]) < 1e-12 * scale, (k, d[k], r[k])


def test_order4_split_calls_time_reversal(mods):
    snref, Oracle, inputs, sn = mods
    cfg = inputs.scaled(inputs.CONFIGS["C4"], (64, 128, 64), L=16.0, steps=8)
    psi0 = cfg.initial_state().astype(np.complex128)
    sim = sim128(sn, cfg)
    sim.set_state(psi0)
    sim.step_order4(3)
    sim.step_order4(5)                                  # split calls: half kinetics not merged across the boundary
    got = sim.get_state()
    orc = Oracle.from_config(cfg)
    orc.set_state(psi0)
    orc.step_order4(8)
    want = orc.get_state()
    orc.close()
    assert rel(got, want) < TOL_STATE64
    sim.set_dtau(-cfg.dtau)                             # and back (time reversal, pin V8)
    sim.step_order4(8)
    assert rel(sim.get_state(), psi0) < 1e-12
    sim.close()


@pytest.mark.parametrize("dims,batch,steps", [((128, 128), 5, 40), ((64, 64, 64), 3, 12), ((96, 128), 4, 20)])
def test_ensemble_members_match_single_system_oracle(mods, dims, batch, steps):
    snref, Oracle, inputs, sn = mods
    nd = len(dims)
    base = inputs.scaled(inputs.CONFIGS["C2" if nd == 2 else "C4"], dims, L=25.0 if nd == 2 else 16.0, steps=steps)
    rng = np.random.default_rng(7)
    p0 = base.initial_state().astype(np.complex128)
    mem = [np.roll(p0, tuple(int(rng.integers(n)) for n in dims), axis=tuple(range(nd))) * (0.8 + 0.1 * b) for b in range(batch)]
    sim = sim128(sn, base, batch=batch)
    sim.set_state(np.ascontiguousarray(np.stack(mem, axis=1)))
    sim.step(steps)
    got = sim.get_state()
    sim.close()
    for b in range(batch):
        orc = Oracle.from_config(base)
        orc.set_state(mem[b])
        orc.step(steps)
        assert rel(got[:, b], orc.get_state()) < TOL_STATE64, b
        orc.close()


@pytest.mark.parametrize("dims,C", [((256, 256, 256), 0.0), ((2048, 2048), -1.0)])
def test_plane_wave_exact_solution(mods, dims, C):
    """psi0 = a e^{iq.x} solves the full system exactly (pin V2): psi(tau) = psi0 exp(i (A|q|^2 - B phi0 - G(a^2)) tau)."""
    snref, Oracle, inputs, sn = mods
    L, A, B, D, g, dtau, steps, amp = 32.0, -0.5, 1.3, 0.9, (0.2, 0.05), 5e-3, 20, 0.8
    mode = (3, -2, 5)[: len(dims)]
    q = 2 * np.pi / L * np.asarray(mode, dtype=np.float64)
    f = [np.exp(1j * qa * inputs.coords(n, L)) for qa, n in zip(q, dims)]
    psi0 = amp * f[0]
    for fa in f[1:]:
        psi0 = psi0[..., None] * fa
    psi0 = np.ascontiguousarray(psi0)
    sim = sn.Simulation(dims, L, A, B, C, D, g, dtau, dtype="complex128")
    sim.set_state(psi0)
    sim.step(steps)
    got = sim.get_state()
    sim.close()
    a2 = amp * amp
    omega = A * float(q @ q) - B * (0.0 if C == 0 else D * a2 / C) - (g[0] * a2 + g[1] * a2 * a2)
    assert rel(got, psi0 * np.exp(1j * omega * dtau * steps)) < 1e-13


def test_c128_contract(mods):
    """complex128 contexts: twice the state bytes, float64 hooks, NEXT-1 terms refused, graph replay identical."""
    snref, Oracle, inputs, sn = mods
    dims = (64, 128)
    assert sn.workspace_bytes(dims, dtype="complex128") > 1.9 * sn.workspace_bytes(dims) - 4 * 65536
    assert sn.workspace_bytes(dims, features=sn.FEAT_VEXT, dtype="complex128") == 0
    with pytest.raises(sn.SnError):
        sn.Simulation(dims, 10.0, -0.5, 1.0, 0.0, 1.0, (), 1e-3, dtype="complex128", features=sn.FEAT_VEXT)
    sim = sn.Simulation(dims, 10.0, -0.5, 1.0, 0.0, 1.0, (0.1,), 1e-3, dtype="complex128")
    for call in (lambda: sim.set_local_terms(0.1, 1e-12, 0.0, 1.0), lambda: sim.set_bohm(0.5, 1e-6),
                 lambda: sim.set_external_potential(np.zeros(dims, np.float32))):
        with pytest.raises(sn.SnError) as e:
            call()
        assert e.value.code == -9
    x = noise128(dims, 3)
    out = {}
    for graph in (1, 0):
        sim.set_option(sn.OPT_GRAPH, graph)
        sim.set_state(x)
        n0 = sim.launch_count()
        sim.step(9)
        out[graph] = (sim.get_state(), sim.launch_count() - n0)
    assert np.array_equal(out[0][0], out[1][0]) and out[0][1] == out[1][1] == 2 + 9 * 4
    sim.close()

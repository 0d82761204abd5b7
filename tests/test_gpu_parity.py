"""GPU parity: the CUDA path (through the C ABI of libsn.so) against the float64 oracle.

Acceptance tolerances are BASELINE.json's north_star: relative L2 error of psi <= 1e-4 after
the configured step count, <= 1e-5 per forward+inverse transform round trip, relative norm
drift <= 1e-5.  Inputs are the seeded synthetic states of paper_1909_08354_b200/inputs.py
(DESIGN.md section 5); both sides start from the same complex64-rounded array.  Where the
oracle is too slow for the full size/step count, the full-size run is checked through
properties that hold at any size (exact plane-wave solution of eq. (1),(2), norm
conservation, time reversal) and the oracle comparison runs on a resampled grid or a prefix
of the steps.
"""
import os

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from _parity import TOL_NORM, TOL_ROUNDTRIP, TOL_STATE, assert_state, maxrel, rel


@pytest.fixture(scope="module")
def mods():
    from oracle import snref
    from oracle.snref import Oracle
    from paper_1909_08354_b200 import inputs, sn
    return snref, Oracle, inputs, sn


def run_pair(mods, cfg, steps, split=None, dispatch=None):
    """Run GPU and oracle from cfg's initial state; return (gpu psi, oracle psi, gpu sim)."""
    snref, Oracle, inputs, sn = mods
    psi0 = cfg.initial_state()
    sim = sn.Simulation.from_config(cfg)
    if dispatch is not None:
        sim.set_option(sn.OPT_DISPATCH, dispatch)
    sim.set_state(psi0)
    if split:
        for n in split:
            sim.step(n)
    else:
        sim.step(steps)
    got = sim.get_state()
    orc = Oracle.from_config(cfg)
    orc.set_state(psi0.astype(np.complex128))
    orc.step(steps)
    want = orc.get_state()
    orc.close()
    return got, want, sim


# ------------------------------------------------------------------ transforms

FFT_DIMS = [(64, 64), (128, 256), (512, 64), (64, 1024), (2048, 64), (64, 4096), (4096, 128),
            (64, 64, 64), (128, 64, 256), (64, 512, 128),
            (96, 96), (384, 64), (64, 384), (1536, 64), (64, 1536), (96, 384, 64),   # 6*4^a lengths (radix-6 stage)
            (192, 64), (64, 192), (768, 192), (3072, 64), (64, 3072), (192, 64, 768),  # 12*4^a: leading radix-2 stage
            (32, 32), (32, 512), (1024, 32), (32, 32, 32), (64, 32, 96), (32, 128, 32)]  # 32-point lines (first-path kernels)


@pytest.mark.parametrize("dims", FFT_DIMS)
def test_fft_forward_matches_oracle_and_round_trip(mods, dims):
    snref, Oracle, inputs, sn = mods
    x = inputs.white_noise(dims, seed=11)
    sim = sn.Simulation(dims, 10.0, -0.5, 1.0, 0.0, 1.0, (), 1e-3)
    sim.set_state(x)
    sim.debug_fft(+1)
    fwd = sim.get_state()
    assert rel(fwd, snref.fftn(x.astype(np.complex128), +1)) < 1e-6
    sim.debug_fft(-1)
    assert rel(sim.get_state(), x) < TOL_ROUNDTRIP
    sim.close()


@pytest.mark.parametrize("name", ["C1", "C2", "C5_64"])
def test_round_trip_on_config_states(mods, name):
    snref, Oracle, inputs, sn = mods
    cfg = inputs.CONFIGS[name]
    x = cfg.initial_state()
    sim = sn.Simulation.from_config(cfg)
    sim.set_state(x)
    sim.debug_fft(+1)
    sim.debug_fft(-1)
    assert rel(sim.get_state(), x) < TOL_ROUNDTRIP
    sim.close()


# ------------------------------------------------------------------ eq. (2): potential

POT_DIMS = [((64, 128), 0.0), ((128, 64), -1.0), ((64, 64, 128), 0.0), ((64, 128, 64), -0.7),
            ((384, 96), 0.0), ((96, 64, 384), -0.7), ((32, 32), 0.0), ((32, 64, 32), -0.7),
            ((512, 64), 0.0), ((64, 512, 64), -0.7), ((64, 64, 512), 0.0), ((256, 128, 64), 0.0),  # pipelined 512-point kernels on each axis
            ((128, 64), 3.3), ((64, 64, 64), 7.7)]            # C > 0 between grid modes (sign change of C - k^2 inside the spectrum)


@pytest.mark.parametrize("state", ["blobs", "noise"])
@pytest.mark.parametrize("dims,C", POT_DIMS)
def test_potential_matches_oracle(mods, dims, C, state):
    """phi of eq. (2) from the r2c -> D/(C - k^2) -> c2r chain against the oracle's full complex
    transforms.  "noise": complex white noise, so the Nyquist row N/2 of the half spectrum, the mirrored-row
    untangling of the packed real transforms and the high-k multipliers all carry signal (a smooth blob state has
    e^-40 there)."""
    snref, Oracle, inputs, sn = mods
    cfg = inputs.scaled(inputs.CONFIGS["C2" if len(dims) == 2 else "C4"], dims, L=16.0)
    psi0 = cfg.initial_state() if state == "blobs" else inputs.white_noise(dims, seed=21)
    sim = sn.Simulation(dims, 16.0, -0.5, 1.0, C, 0.9, (0.1,), 1e-3)
    sim.set_state(psi0)
    orc = Oracle(dims, 16.0, -0.5, 1.0, C, 0.9, (0.1,), 1e-3)
    orc.set_state(psi0.astype(np.complex128))
    got, want = sim.debug_potential(), orc.potential()
    sim.close()
    orc.close()
    # white noise: rho has a mean as large as its fluctuations, and the fp32 rounding of that mean through the
    # butterflies (6e-8 x sum rho) lands on the lowest modes, which 1/k^2 then weights up -- a few 1e-6 on 2^21 cells
    # C > 0 a relative 1.4e-3 away from a grid mode (7.7 vs k^2 = 7.711): that mode is amplified 700x over its neighbours
    tol = (2e-6 if C <= 0 else 5e-6) if state == "blobs" else 1e-5
    assert rel(got, want) < tol and maxrel(got, want) < 10 * tol, (rel(got, want), maxrel(got, want))


@pytest.mark.parametrize("dims", [(64, 128), (64, 64, 64), (512, 64), (96, 64), (64, 512, 64), (64, 64, 512)])
def test_potential_spectrum_bin_by_bin(mods, dims):
    """Every Fourier bin of phi against the oracle's for white-noise psi.  A rel-L2 over phi with C = 0 is blind to the
    high wavenumbers (1/k^2 suppresses the Nyquist row by 1/N^2), so: (i) C = -300 ~ -k_max^2, where D/(C - k^2) varies
    by less than 5x over the spectrum and every bin -- row N/2 of the half spectrum, the mirrored rows of the packed
    real transforms -- carries the same weight: tight bound per bin; (ii) C = 0 with the bins re-weighted by k^2: only
    as tight as the float32 rounding of phi itself allows (a white 6e-8 max|phi| floor against a signal that falls as
    1/k^2), still 100x below what one wrong row would give (sqrt(1/N0) ~ 0.05)."""
    snref, Oracle, inputs, sn = mods
    psi0 = inputs.white_noise(dims, seed=22)
    k2 = sum(np.square(2 * np.pi / 16.0 * np.fft.fftfreq(n, 1.0 / n)).reshape([-1 if i == a else 1 for i in range(len(dims))])
             for a, n in enumerate(dims))
    for C, w, tol in ((-300.0, 1.0, 3e-6), (0.0, k2, 2e-4)):
        sim = sn.Simulation(dims, 16.0, -0.5, 1.0, C, 0.9, (), 1e-3)
        sim.set_state(psi0)
        orc = Oracle(dims, 16.0, -0.5, 1.0, C, 0.9, (), 1e-3)
        orc.set_state(psi0.astype(np.complex128))
        got, want = sim.debug_potential(), orc.potential()
        sim.close()
        orc.close()
        G, W = snref.fftn(got.astype(np.complex128), +1), snref.fftn(want.astype(np.complex128), +1)
        if C != 0:                      # the k = 0 bin holds D rho_mean/C, ~sqrt(cells) above the rest: compare it on its own
            assert abs(G.flat[0] - W.flat[0]) < 1e-6 * abs(W.flat[0])
            G.flat[0] = W.flat[0] = 0.0
        assert rel(G * w, W * w) < tol, (C, rel(G * w, W * w))
        assert np.max(np.abs((G - W) * w)) < 10 * tol * np.max(np.abs(W * w)), C


def test_single_mode_poisson_closed_form(mods):
    """rho = rbar + eps cos(q.x) -> phi = D eps cos(q.x)/(C - |q|^2) (+ D rbar/C if C != 0)  [pin V5]."""
    snref, Oracle, inputs, sn = mods
    dims, L = (64, 128), 12.0
    y = inputs.coords(dims[0], L)[:, None]
    x = inputs.coords(dims[1], L)[None, :]
    q = 2 * np.pi / L * np.array([3, -5])
    rbar, eps = 1.3, 0.4
    rho = rbar + eps * np.cos(q[0] * y + q[1] * x)
    psi = np.sqrt(rho).astype(np.complex64)
    rho32 = np.abs(psi.astype(np.complex128)) ** 2  # what the GPU actually sees
    for C, D in [(0.0, 0.9), (-1.5, -0.7)]:
        sim = sn.Simulation(dims, L, -0.5, 1.0, C, D, (), 1e-3)
        sim.set_state(psi)
        want = D * (rho32 - rho32.mean()) / (C - q @ q) + (D * rho32.mean() / C if C != 0 else 0.0)
        assert np.max(np.abs(sim.debug_potential() - want)) < 5e-6 * np.max(np.abs(want))
        sim.close()


# ------------------------------------------------------------------ Strang steps vs oracle

def test_c1_full(mods):
    snref, Oracle, inputs, sn = mods
    cfg = inputs.CONFIGS["C1"]
    got, want, sim = run_pair(mods, cfg, cfg.steps)
    assert_state(got, want)
    d = sim.diagnostics()
    assert abs(d["norm"] - 1.0) < TOL_NORM
    sim.close()


STEP_CASES = [
    # name, dims, L, steps  (resampled grids keep the recipe, seed and constants of the config)
    ("C2", (256, 256), 25.0, 400),
    ("C2", (1024, 1024), 100.0, 40),      # full size, prefix of the 1000 steps
    ("C3", (512, 512), 50.0, 150),        # C = -1 screened case, h as in the config
    ("C3", (4096, 64), 50.0, 20),         # the 4096-point line kernels
    ("C3", (2048, 128), 50.0, 20),        # 2048-point strided lines: 32-byte rows, SWIZZLE_32B boxes
    ("C4", (64, 2048, 64), 16.0, 4),      # 2048-point lines along axis 1 of a 3D grid
    ("C4", (64, 64, 4096), 16.0, 3),      # 4096-point contiguous lines in 3D
    ("C4", (64, 64, 64), 16.0, 100),
    ("C5_64", (64, 64, 64), 128.0, 100),  # full config
    ("C5_128", (128, 128, 128), 128.0, 10),
    ("C4", (64, 128, 256), 32.0, 10),     # rectangular 3D, three different line lengths
    ("C5_256", (256, 256, 256), 128.0, 2),  # many tiles per pass
    ("C2", (384, 96), 25.0, 100),           # 6*4^a line lengths on both axes
    ("C5_384", (96, 96, 96), 128.0, 20),    # the sweep's 3*2^7 family, coarse
    ("C5_384", (384, 64, 128), 128.0, 4),   # 384-point strided lines next to pipelined axes
    ("C5_384", (64, 128, 384), 128.0, 4),   # 384-point contiguous lines
    ("C2", (192, 768), 25.0, 60),           # 12*4^a line lengths (leading radix-2 stage) on both axes
    ("C5_384", (192, 192, 192), 128.0, 6),  # 192^3
    ("C3", (3072, 64), 50.0, 12),           # 3072-point strided lines
    ("C4", (64, 768, 192), 16.0, 6),
    ("C2", (32, 32), 6.25, 200),            # 32-point lines (first-path kernels only), both axes
    ("C4", (32, 32, 32), 8.0, 100),
    ("C4", (32, 256, 32), 16.0, 10),        # 32-point axis-0 and contiguous lines around a pipelined axis
    ("C3", (512, 32), 25.0, 40),
    # full-size grids of every BASELINE.json config (prefixes of the configured step count where the oracle needs
    # minutes for the whole run; the whole runs are the `heavy` cases below)
    ("C2", (1024, 1024), 100.0, 1000),    # C2 in full
    ("C3", (4096, 4096), 400.0, 5),
    ("C4", (256, 256, 256), 64.0, 5),
    ("C5_128", (128, 128, 128), 128.0, 100),  # sweep point in full
    ("C5_384", (384, 384, 384), 128.0, 1),
    ("C5_512", (512, 512, 512), 128.0, 1),    # the bench's own kernel instantiations: 512-point lines on all three axes
    ("C5_512", (64, 512, 128), 128.0, 4),     # 512-point strided lines along axis 1 (S_KIN, S_FFT on the half spectrum)
    ("C5_512", (128, 512, 512), 128.0, 2),
]

# C > 0 lying BETWEEN grid modes: 1/(C - k^2) changes sign inside the spectrum and is large next to C; the
# hi/lo denominator of the Helmholtz pass keeps those modes accurate in fp32.  name, dims, L, C, steps
POSITIVE_C_CASES = [
    ("C2", (128, 128), 12.5, 3.3, 60),
    ("C2", (512, 64), 25.0, 1.7, 30),          # pipelined 512-point passes
    ("C4", (64, 64, 64), 16.0, 7.7, 30),       # 1.4e-3 (relative) from the mode k^2 = 7.711
    ("C4", (64, 128, 256), 32.0, 2.05, 8),
]


@pytest.mark.parametrize("name,dims,L,C,steps", POSITIVE_C_CASES)
def test_steps_match_oracle_with_positive_c(mods, name, dims, L, C, steps):
    import dataclasses
    snref, Oracle, inputs, sn = mods
    cfg = dataclasses.replace(inputs.scaled(inputs.CONFIGS[name], dims, L=L, steps=steps), C=C)
    got, want, sim = run_pair(mods, cfg, steps)
    d = sim.diagnostics()
    sim.close()
    assert_state(got, want)
    assert np.isfinite(d["e_total"])


@pytest.mark.parametrize("name,dims,L,steps", STEP_CASES)
def test_steps_match_oracle(mods, name, dims, L, steps):
    snref, Oracle, inputs, sn = mods
    cfg = inputs.scaled(inputs.CONFIGS[name], dims, L=L, steps=steps)
    got, want, sim = run_pair(mods, cfg, steps)
    sim.close()
    assert_state(got, want)


# The whole configured runs that take the oracle minutes each (C3 7 min, C4 4 min, 256^3 1.5 min, 384^3 5 min,
# 512^3 x 20 steps 2.5 min on 16 host cores).  Deselected (not skipped) unless SN_HEAVY=1 -- tests/conftest.py; the
# log of the last SN_HEAVY=1 run on a B200 is profiles/r02_full_configs.md.
HEAVY_CASES = [("C3", None), ("C4", None), ("C5_256", None), ("C5_384", None), ("C5_512", 20)]


@pytest.mark.heavy
@pytest.mark.parametrize("name,steps", HEAVY_CASES)
def test_full_configured_runs_vs_oracle(mods, name, steps):
    snref, Oracle, inputs, sn = mods
    cfg = inputs.CONFIGS[name]
    steps = steps or cfg.steps
    psi0 = cfg.initial_state()
    sim = sn.Simulation.from_config(cfg)
    sim.set_state(psi0)
    d0 = sim.diagnostics()
    sim.step(steps)
    got = sim.get_state()
    d1 = sim.diagnostics()
    sim.close()
    orc = Oracle.from_config(cfg)
    orc.set_state(psi0.astype(np.complex128))
    del psi0
    orc.step(steps)
    want = orc.get_state()
    orc.close()
    e2, em = rel(got, want), maxrel(got, want)
    drift = abs(d1["norm"] - d0["norm"]) / d0["norm"]
    print(f"FULL {name} {'x'.join(map(str, cfg.dims))} steps={steps}: rel-L2 {e2:.3e} max-rel {em:.3e} norm drift {drift:.3e}")
    assert e2 < TOL_STATE and em < 10 * TOL_STATE and drift < TOL_NORM


def test_split_calls_equal_one_call(mods):
    """sn_step(5) merges half kinetics; sn_step(2)+sn_step(3) does not across the call boundary."""
    snref, Oracle, inputs, sn = mods
    cfg = inputs.scaled(inputs.CONFIGS["C2"], (128, 128), L=12.5, steps=5)
    a, want, s1 = run_pair(mods, cfg, 5)
    b, _, s2 = run_pair(mods, cfg, 5, split=(2, 3))
    s1.close()
    s2.close()
    assert rel(a, want) < TOL_STATE and rel(b, want) < TOL_STATE
    assert rel(a, b) < 5e-6


def test_counter_scheduled_axis0_kernel_over_many_launches(mods):
    """512 tiles along axis 0 (> 2 per CTA): the pipelined axis-0 kernel takes its tiles from the device-wide counter
    (DESIGN.md 4.2), which the last CTA rewinds; consecutive launches and separate calls must all start from zero."""
    snref, Oracle, inputs, sn = mods
    cfg = inputs.scaled(inputs.CONFIGS["C4"], (256, 64, 256), L=32.0, steps=6)
    a, want, s1 = run_pair(mods, cfg, 6)
    b, _, s2 = run_pair(mods, cfg, 6, split=(1, 2, 3))
    s1.close()
    s2.close()
    assert rel(a, want) < TOL_STATE and rel(b, want) < TOL_STATE
    assert rel(a, b) < 5e-6


# ------------------------------------------------------------------ full-size properties

def plane_wave(inputs, dims, L, mode, amp):
    """a exp(i q.x) as complex64, built from its 1D factors (cheap at 512^3); returns (psi0, |q|^2)."""
    q = 2 * np.pi / L * np.asarray(mode, dtype=np.float64)
    f = [np.exp(1j * qa * inputs.coords(n, L)) for qa, n in zip(q, dims)]
    psi = np.asarray(amp * f[0], dtype=np.complex128)
    for fa in f[1:]:
        psi = (psi[..., None] * fa).astype(np.complex64 if fa is f[-1] else np.complex128)
    return np.ascontiguousarray(psi, dtype=np.complex64), float(q @ q)


@pytest.mark.parametrize("dims,C", [((512, 512, 512), 0.0), ((4096, 4096), -1.0), ((256, 256, 256), -1.0),
                                    ((1024, 1024), 0.0)])
def test_plane_wave_exact_solution_full_size(mods, dims, C):
    """psi0 = a e^{iq.x}, q on the k-lattice, solves the full system and every sub-step exactly:
    psi(tau) = psi0 exp(i (A|q|^2 - B phi0 - G(a^2)) tau), phi0 = 0 if C == 0 else D a^2/C  [pin V2]."""
    snref, Oracle, inputs, sn = mods
    L, A, B, D, g, dtau, steps, amp = 32.0, -0.5, 1.3, 0.9, (0.2, 0.05), 5e-3, 20, 0.8
    mode = (3, -2, 5)[: len(dims)]
    psi0, q2 = plane_wave(inputs, dims, L, mode, amp)
    sim = sn.Simulation(dims, L, A, B, C, D, g, dtau)
    sim.set_state(psi0)
    sim.step(steps)
    got = sim.get_state()
    a2 = amp * amp
    phi0 = 0.0 if C == 0 else D * a2 / C
    omega = A * q2 - B * phi0 - (g[0] * a2 + g[1] * a2 * a2)
    rot = np.complex64(np.exp(1j * omega * dtau * steps))
    sim.close()
    # chunked ||got - psi0*rot|| / ||psi0|| in float64 (keeps the 512^3 case at a few GB)
    num = den = 0.0
    g1, p1 = got.reshape(-1), psi0.reshape(-1)
    for i in range(0, g1.size, 1 << 24):
        w = p1[i:i + (1 << 24)].astype(np.complex128) * complex(rot)
        num += float(np.sum(np.abs(g1[i:i + (1 << 24)] - w) ** 2))
        den += float(np.sum(np.abs(w) ** 2))
    assert np.sqrt(num / den) < 2e-5


@pytest.mark.parametrize("name", ["C2", "C3", "C4", "C5_512"])
def test_norm_drift_over_configured_steps(mods, name):
    """Full config, full step count, GPU only: |N_end - N_0|/N_0 <= 1e-5 (unitarity of every sub-step)."""
    snref, Oracle, inputs, sn = mods
    cfg = inputs.CONFIGS[name]
    sim = sn.Simulation.from_config(cfg)
    sim.set_state(cfg.initial_state())
    d0 = sim.diagnostics()
    sim.step(cfg.steps)
    d1 = sim.diagnostics()
    sim.close()
    assert abs(d1["norm"] - d0["norm"]) / d0["norm"] < TOL_NORM
    # the Hamiltonian is conserved up to the O(dtau^2) splitting error (reading Q10)
    assert abs(d1["e_total"] - d0["e_total"]) < 2e-3 * (abs(d0["e_kin"]) + abs(d0["e_nonlocal"]) + abs(d0["e_local"]))


def test_time_reversal(mods):
    snref, Oracle, inputs, sn = mods
    cfg = inputs.CONFIGS["C5_128"]
    psi0 = cfg.initial_state()
    sim = sn.Simulation.from_config(cfg)
    sim.set_state(psi0)
    sim.step(20)
    sim.set_dtau(-cfg.dtau)
    sim.step(20)
    back = sim.get_state()
    sim.close()
    assert rel(back, psi0) < 2e-5


# ------------------------------------------------------------------ diagnostics and edge cases

@pytest.mark.parametrize("name,dims,L", [("C2", (128, 256), 20.0), ("C4", (64, 128, 64), 16.0),
                                         ("C5_384", (96, 64, 384), 128.0), ("C5_384", (384, 96, 64), 128.0)])
def test_diagnostics_match_oracle(mods, name, dims, L):
    snref, Oracle, inputs, sn = mods
    cfg = inputs.scaled(inputs.CONFIGS[name], dims, L=L)
    psi0 = cfg.initial_state()
    sim = sn.Simulation.from_config(cfg)
    sim.set_state(psi0)
    orc = Oracle.from_config(cfg)
    orc.set_state(psi0.astype(np.complex128))
    d, r = sim.diagnostics(), orc.diagnostics()
    sim.close()
    orc.close()
    scale = abs(r["e_kin"]) + abs(r["e_nonlocal"]) + abs(r["e_local"])
    assert abs(d["norm"] - r["norm"]) < 1e-6 * r["norm"]
    for k in ("e_kin", "e_nonlocal", "e_local", "e_total"):
        assert abs(d[k] - r[k]) < 2e-6 * scale, k


def test_edge_cases(mods):
    snref, Oracle, inputs, sn = mods
    dims = (64, 64)
    x = inputs.white_noise(dims, 3)
    sim = sn.Simulation(dims, 10.0, -0.5, 1.0, 0.0, 1.0, (0.1,), 1e-3)
    with pytest.raises(sn.SnError) as e:
        sim.step(1)                       # no state yet
    assert e.value.code == -6
    sim.set_state(x)
    sim.step(0)                           # no-op
    assert np.array_equal(sim.get_state(), x)
    with pytest.raises(sn.SnError) as e:
        sim.step(-1)
    assert e.value.code == -3
    sim.set_state(np.zeros(dims, np.complex64))
    sim.step(3)                           # zero state stays zero, no NaN
    assert np.array_equal(sim.get_state(), np.zeros(dims, np.complex64))
    sim.set_dtau(0.0)                     # dtau = 0: every sub-step is the identity (to a round trip)
    sim.set_state(x)
    sim.step(2)
    assert rel(sim.get_state(), x) < 4 * TOL_ROUNDTRIP
    sim.close()


def test_device_state_round_trip_and_launch_count(mods):
    import torch
    snref, Oracle, inputs, sn = mods
    dims = (64, 64, 64)
    x = torch.from_numpy(inputs.white_noise(dims, 5)).cuda()
    sim = sn.Simulation(dims, 10.0, -0.5, 1.0, 0.0, 1.0, (0.1,), 1e-3)
    sim.set_state(x)
    out = torch.empty_like(x)
    sim.get_state(out)
    assert torch.equal(out, x)
    n0 = sim.launch_count()
    sim.step(4)
    # 3D: 3 kinetic passes + 4 steps x (r2c, y fwd, x Poisson, y inv + 3 kinetic passes)
    assert sim.launch_count() - n0 == 3 + 4 * 7
    sim.close()


@pytest.mark.parametrize("dims,L,name", [((512, 128), 50.0, "C3"), ((64, 256, 128), 32.0, "C4")])
def test_first_path_and_pipelined_kernels_agree(mods, dims, L, name):
    """sn_set_option(SN_OPT_DISPATCH, 1) routes every pass to the first-path kernels of sn_kernels.cu, 2 to the
    TMA-pipelined kernels of sn_pipe.cu wherever they are instantiated.  Same arithmetic order inside a line, so the
    two agree to a few ulp, and both meet the oracle tolerance."""
    snref, Oracle, inputs, sn = mods
    cfg = inputs.scaled(inputs.CONFIGS[name], dims, L=L, steps=6)
    psi0 = cfg.initial_state()
    out = {}
    for mode in ("0", "1"):
        sim = sn.Simulation.from_config(cfg)
        sim.set_option(sn.OPT_DISPATCH, sn.DISPATCH_FIRST_PATH if mode == "1" else sn.DISPATCH_PIPELINED)
        sim.set_state(psi0)
        sim.step(cfg.steps)
        out[mode] = sim.get_state()
        sim.close()
    orc = Oracle.from_config(cfg)
    orc.set_state(psi0.astype(np.complex128))
    orc.step(cfg.steps)
    want = orc.get_state()
    orc.close()
    assert rel(out["0"], want) < TOL_STATE and rel(out["1"], want) < TOL_STATE
    assert rel(out["0"], out["1"]) < 5e-6


@pytest.mark.parametrize("name,dims,L,steps", [("C2", (256, 128), 25.0, 50), ("C4", (64, 128, 256), 32.0, 10),
                                               ("C5_64", (64, 64, 64), 128.0, 20), ("C2", (1024, 64), 25.0, 10)])
def test_steps_match_oracle_all_pipelined(mods, name, dims, L, steps):
    """The default dispatch uses the pipelined kernels only where they are faster (axis-0 nonlinear pass always,
    the others at N = 512 and N >= 2048); SN_OPT_DISPATCH = 2 forces them for every kind and length."""
    snref, Oracle, inputs, sn = mods
    cfg = inputs.scaled(inputs.CONFIGS[name], dims, L=L, steps=steps)
    got, want, sim = run_pair(mods, cfg, steps, dispatch=sn.DISPATCH_PIPELINED)
    sim.close()
    assert_state(got, want)


def test_graph_replay_is_bitwise_the_stream_launch_path(mods):
    """sn_step(n >= 4) on grids of <= 2^24 cells replays a captured CUDA graph of the interior step; the kernels and
    their order are the same as with plain stream launches (SN_OPT_GRAPH = 0), so the states must agree bit for bit, also
    after sn_set_dtau (which drops the graph) and across split calls."""
    snref, Oracle, inputs, sn = mods
    cfg = inputs.scaled(inputs.CONFIGS["C4"], (64, 64, 128), L=16.0, steps=12)
    psi0 = cfg.initial_state()
    out = {}
    for mode, (graph, per_graph) in {"plain": (0, 1), "graph1": (1, 1), "graph3": (1, 3), "graph5": (1, 5)}.items():
        sim = sn.Simulation.from_config(cfg)
        sim.set_option(sn.OPT_GRAPH, graph)
        sim.set_option(sn.OPT_GRAPH_STEPS, per_graph)   # interior steps per replayed graph; the remainder replays a one-step graph
        sim.set_state(psi0)
        n0 = sim.launch_count()
        sim.step(7)
        sim.set_dtau(0.5 * cfg.dtau)
        sim.step(5)
        sim.step(2)                                   # below the graph threshold: plain launches in every mode
        out[mode] = (sim.get_state(), sim.launch_count() - n0)
        sim.close()
    for mode in ("graph1", "graph3", "graph5"):
        assert np.array_equal(out["plain"][0], out[mode][0]), mode
        assert out["plain"][1] == out[mode][1], mode  # the launch counter counts the kernels inside the graph too


def test_runs_on_a_side_stream(mods):
    """All device work goes to the cudaStream_t given to sn_create: run on a non-default torch stream (graph replay
    included) and compare with the default-stream result bit for bit."""
    import torch
    snref, Oracle, inputs, sn = mods
    cfg = inputs.scaled(inputs.CONFIGS["C4"], (64, 128, 64), L=16.0, steps=9)
    psi0 = cfg.initial_state()
    ref = sn.Simulation.from_config(cfg)
    ref.set_state(psi0)
    ref.step(9)
    want = ref.get_state()
    ref.close()
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        sim = sn.Simulation.from_config(cfg, stream=side)
        dev = torch.from_numpy(psi0).to("cuda:0", non_blocking=True)
        side.synchronize()
        sim.set_state(dev)
        sim.step(9)
        out = torch.empty_like(dev)
        sim.get_state(out)
        side.synchronize()
        got = out.cpu().numpy()
        sim.close()
    assert np.array_equal(got, want)


def _two_gpus():
    try:
        import torch
        return torch.cuda.is_available() and torch.cuda.device_count() >= 2
    except Exception:
        return False


if _two_gpus():   # defined only on a multi-GPU box (a skip would show up in the single-GPU report)
    def test_context_on_a_device_that_is_not_current(mods):
        """The library runs every call on the device that owns the workspace (sn.h): a context on cuda:1 driven while
        cuda:0 is current gives the same bits as one on cuda:0."""
        import torch
        snref, Oracle, inputs, sn = mods
        cfg = inputs.scaled(inputs.CONFIGS["C4"], (64, 64, 64), L=16.0, steps=6)
        psi0 = cfg.initial_state()
        out = []
        for dev in ("cuda:0", "cuda:1"):
            torch.cuda.set_device(0)
            sim = sn.Simulation.from_config(cfg, device=dev)
            sim.set_state(psi0)
            sim.step(6)
            sim.diagnostics()
            out.append(sim.get_state())
            sim.close()
            assert torch.cuda.current_device() == 0
        assert np.array_equal(out[0], out[1])

"""The allocation-free entry point sn_norm_static (include/sn.h; csrc/sn_static.cu) against the existing paths.

Collected last on purpose (file name): the suite runs with `pytest -x`, and a failure here must not hide other tests.
sn_norm_static computes norm = dV sum |psi|^2 with its scratch in a static device array of the library (no context,
no workspace, no cudaMalloc).  Checked here, on two calls in a row that need different numbers of scratch slots:
  * against the existing diagnostics path (sn_diagnostics of a context: sum of rho in the axis-0 kernel, fp64 atomics
    into workspace scratch) within the tolerance tests/test_gpu_parity.py uses for the norm (1e-6 relative),
  * against the existing k_norm path (sn_mc_norms of a one-component coupled context) at the same tolerance,
  * against the float64 sum of the same complex64 values taken on the host,
  * the second, smaller call must not see the first call's stale partial sums, a repeat of the first call must
    reproduce its result bit for bit (fixed summation order), sizes beyond the stated maximum are rejected with
    SN_ERR_TOO_LARGE before anything is launched, and device memory in use does not change across a call.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL_NORM_DIAG = 1e-6   # tests/test_gpu_parity.py::test_diagnostics_match_oracle: |norm - ref| < 1e-6 ref


@pytest.fixture(scope="module")
def mods():
    import torch
    from paper_1909_08354_b200 import inputs, sn
    return torch, inputs, sn


def existing_norms(sn, cfg, psi0):
    """(norm of sn_diagnostics, norm of sn_mc_norms) for the state psi0 of config cfg: the two existing paths."""
    sim = sn.Simulation.from_config(cfg)
    sim.set_state(psi0)
    d = sim.diagnostics()["norm"]
    sim.close()
    mc = sn.CoupledSimulation(cfg.dims, cfg.L, (cfg.A,), (cfg.B,), cfg.C, cfg.D, (1.0,), [[0.0]], cfg.dtau)
    mc.set_state(psi0[None])
    k = float(mc.norms()[0])
    mc.close()
    return d, k


def test_norm_static_matches_existing_paths_on_two_calls_in_a_row(mods):
    torch, inputs, sn = mods
    big = inputs.scaled(inputs.CONFIGS["C5_128"], (128, 128, 128))          # 2^21 cells: 256 scratch slots
    small = inputs.scaled(inputs.CONFIGS["C2"], (96, 128), L=25.0)           # 12288 cells: 2 slots, the last one half full
    odd = inputs.scaled(inputs.CONFIGS["C2"], (96, 192), L=25.0)             # 18432 cells: 3 slots, the last one a quarter full
    want = {}
    states = {}
    for name, cfg in (("big", big), ("small", small), ("odd", odd)):
        psi0 = cfg.initial_state()
        states[name] = (cfg, psi0, torch.from_numpy(psi0).cuda())
        want[name] = existing_norms(sn, cfg, psi0)
    out = torch.full((4,), float("nan"), dtype=torch.float64, device="cuda")
    got = {}
    # two calls in a row on one stream, then a third with a ragged last block; results read after all were enqueued
    for slot, name in enumerate(("big", "small", "odd")):
        cfg, psi0, dev = states[name]
        dv = float(np.prod([cfg.L / n for n in cfg.dims]))
        sn.norm_static(dev, dv, out[slot:slot + 1])
    cfg, psi0, dev = states["big"]
    sn.norm_static(dev, float(np.prod([cfg.L / n for n in cfg.dims])), out[3:4])     # repeat of the first call
    torch.cuda.synchronize()
    res = out.cpu().numpy()
    for slot, name in enumerate(("big", "small", "odd")):
        cfg, psi0, dev = states[name]
        dv = float(np.prod([cfg.L / n for n in cfg.dims]))
        got[name] = float(res[slot])
        host = float(np.sum(np.abs(psi0.astype(np.complex128)) ** 2)) * dv
        d, k = want[name]
        assert abs(got[name] - d) < TOL_NORM_DIAG * d, (name, got[name], d)         # vs sn_diagnostics
        assert abs(got[name] - k) < TOL_NORM_DIAG * k, (name, got[name], k)         # vs k_norm (sn_mc_norms)
        assert abs(got[name] - host) < 1e-7 * host, (name, got[name], host)         # fp32 squares, fp64 sums
    assert res[3] == res[0]                                                          # fixed order: bitwise reproducible


def test_norm_static_edge_cases_and_limit(mods):
    torch, inputs, sn = mods
    x = torch.from_numpy(inputs.white_noise((64, 64), 3)).cuda()
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    sn.norm_static(x, 0.5, out, n_cells=0)                                          # empty input: 0
    torch.cuda.synchronize()
    assert float(out[0]) == 0.0
    sn.norm_static(x, 2.0, out, n_cells=1)                                          # one cell
    torch.cuda.synchronize()
    v = x.reshape(-1)[0].item()
    assert abs(float(out[0]) - 2.0 * abs(v) ** 2) < 1e-6 * 2.0 * abs(v) ** 2
    out.fill_(-7.0)
    with pytest.raises(sn.SnError) as e:                                            # beyond the stated maximum: rejected,
        sn.norm_static(x, 1.0, out, n_cells=sn.STATIC_NORM_MAX_CELLS + 1)           # nothing launched (x is far smaller)
    assert e.value.code == -10 and "SN_STATIC_NORM_MAX_CELLS" in str(e.value)
    torch.cuda.synchronize()
    assert float(out[0]) == -7.0
    with pytest.raises(sn.SnError) as e:
        sn.norm_static(x, 1.0, out, n_cells=-1)
    assert e.value.code == -3


def test_norm_static_allocates_nothing_and_runs_on_a_side_stream(mods):
    torch, inputs, sn = mods
    x = torch.from_numpy(inputs.white_noise((256, 256), 5)).cuda()
    out = torch.zeros(2, dtype=torch.float64, device="cuda")
    side = torch.cuda.Stream()
    sn.norm_static(x, 1.0, out[0:1])                                                # first use on this device: symbol address, module load
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        sn.norm_static(x, 1.0, out[1:2], stream=side)
    side.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0                                                           # no device memory taken or returned
    assert float(out[0]) == float(out[1])
    host = float(np.sum(np.abs(x.cpu().numpy().astype(np.complex128)) ** 2))
    assert abs(float(out[0]) - host) < 1e-7 * host

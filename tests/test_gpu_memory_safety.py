"""Memory-safety and race checks that do not need compute-sanitizer (closed on this GPU pool: runs under it left GPUs
needing a reset -- the tool's own message; B200_PROFILING.md says to use bounds checks of one's own instead).

* Guard zones: the context's workspace is the middle of a larger buffer filled with a poison byte; after every kind of
  call (steps on all three dispatches, diagnostics, both test hooks, the NEXT-1 setters, order-4 steps) the zones before
  and after the workspace must still hold the poison -- an out-of-bounds store of any kernel, TMA box or copy lands there.
* Determinism: the same call sequence twice must give bit-identical states.  The pipelined kernels exchange in place inside
  TMA tiles with warp-level ordering only in places (csrc/sn_pipe.cu); a race there shows up as run-to-run differences,
  the tile schedule of the axis-0 kernel being dynamic (atomic counter) on top.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

GUARD = 1 << 20
POISON = 0xA5


@pytest.fixture(scope="module")
def mods():
    from paper_1909_08354_b200 import inputs, sn
    return inputs, sn


def guarded(sn, dims, **kw):
    import torch
    n = sn.workspace_bytes(dims, batch=kw.get("batch") or 1, features=kw.get("features", 0), dtype=kw.get("dtype", "complex64"))
    buf = torch.full((n + 2 * GUARD,), POISON, dtype=torch.uint8, device="cuda:0")
    sim = sn.Simulation(dims, 12.0, -0.5, 1.0, -0.3, 0.9, (0.1, 0.02), 2e-3, workspace=buf[GUARD:GUARD + n], **kw)
    return sim, buf, n


def guards_intact(buf, n):
    import torch
    torch.cuda.synchronize()
    return bool((buf[:GUARD] == POISON).all()) and bool((buf[GUARD + n:] == POISON).all())


CASES = [((64, 64), {}), ((128, 96), {}), ((512, 64), {}), ((64, 4096), {}), ((2048, 32), {}),
         ((64, 64, 64), {}), ((32, 64, 96), {}), ((64, 512, 64), {}), ((512, 32, 64), {}), ((96, 64, 384), {}),
         ((64, 64), {"batch": 3}), ((64, 32, 64), {"batch": 2}),
         ((64, 128), {"dtype": "complex128"}), ((96, 64, 64), {"dtype": "complex128"}), ((64, 512, 32), {"dtype": "complex128"})]


@pytest.mark.parametrize("dims,kw", CASES)
def test_no_kernel_writes_outside_the_workspace(mods, dims, kw):
    inputs, sn = mods
    c128 = kw.get("dtype") == "complex128"
    sim, buf, n = guarded(sn, dims, features=0 if c128 else sn.FEAT_ALL, **kw)
    shape = sim.dims
    x = inputs.white_noise(shape, 9)
    x = (0.3 * x).astype(np.complex128 if c128 else np.complex64)
    for dispatch in ((sn.DISPATCH_DEFAULT,) if c128 else (sn.DISPATCH_DEFAULT, sn.DISPATCH_FIRST_PATH, sn.DISPATCH_PIPELINED)):
        sim.set_option(sn.OPT_DISPATCH, dispatch)
        sim.set_state(x)
        sim.step(5)                      # graph replay for small grids (n >= 4)
        sim.step(2)
        sim.step_order4(1)
        sim.diagnostics()
        sim.debug_potential()
        sim.debug_fft(+1)
        sim.debug_fft(-1)
        if not c128:
            v = np.cos(np.arange(int(np.prod(shape)), dtype=np.float32)).reshape(shape)
            sim.set_external_potential(v)
            sim.set_source_tables(0.1 * v, 1.0 + 0.1 * v)
            sim.set_local_terms(0.01, 1e-9, 0.02, 0.5)
            sim.set_bohm(0.05, 1e-3)
            sim.step(2)
            sim.diagnostics()
            sim.set_external_potential(None)
            sim.set_source_tables(None, None)
            sim.set_local_terms(0.0, 1e-9, 0.0, 1.0)
            sim.set_bohm(0.0, 1e-3)
        assert np.isfinite(sim.get_state()).all()
        assert guards_intact(buf, n), dispatch
    sim.close()


@pytest.mark.parametrize("dims,steps", [((128, 128), 30), ((1024, 64), 10), ((64, 64, 64), 12), ((256, 64, 256), 4),
                                        ((64, 512, 128), 4), ((512, 64, 64), 6), ((96, 96, 96), 6)])
def test_repeated_runs_are_bitwise_identical(mods, dims, steps):
    inputs, sn = mods
    x = (0.3 * inputs.white_noise(dims, 4)).astype(np.complex64)
    for dispatch in (sn.DISPATCH_DEFAULT, sn.DISPATCH_PIPELINED):
        outs = []
        for rep in range(3):
            sim = sn.Simulation(dims, 12.0, -0.5, 1.0, 0.0, 0.9, (0.1,), 2e-3)
            sim.set_option(sn.OPT_DISPATCH, dispatch)
            sim.set_state(x)
            sim.step(steps)
            outs.append(sim.get_state())
            sim.close()
        assert np.array_equal(outs[0], outs[1]) and np.array_equal(outs[0], outs[2]), dispatch

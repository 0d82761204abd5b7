"""NEXT-2 on one GPU: the slab-decomposed step run as R virtual ranks (R contexts on one device, blocks moved by
sn_slab_exchange_local), against the single-context step and the float64 oracle."""
import numpy as np
import pytest

from _parity import TOL_NORM, assert_state, rel

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def mods():
    from oracle.snref import Oracle
    from paper_1909_08354_b200 import inputs, slab, sn
    return Oracle, inputs, slab, sn


CASES = [
    # recipe, dims, L, ranks, steps, C
    ("C4", (64, 64, 64), 16.0, 1, 6, 0.0),       # one rank: views coincide, no exchange
    ("C4", (64, 64, 64), 16.0, 2, 12, 0.0),
    ("C4", (64, 64, 64), 16.0, 4, 12, -0.7),
    ("C4", (128, 64, 128), 32.0, 8, 6, 0.0),     # 8 ranks: 16-row z-slabs, 8 x 128 columns per y-slab
    ("C4", (64, 128, 256), 32.0, 2, 6, 0.0),     # three different line lengths
    ("C5_512", (512, 64, 64), 128.0, 4, 3, 0.0), # 512-point lines along axis 0: the pipelined axis-0 kernels on view B
    ("C5_512", (64, 512, 128), 128.0, 2, 3, 0.0),  # 512-point strided lines along axis 1 on view A
    ("C5_384", (96, 96, 64), 128.0, 3, 8, 0.0),  # 3*2^a lengths, three ranks
]


@pytest.mark.parametrize("name,dims,L,R,steps,C", CASES)
def test_virtual_rank_step_matches_single_context_and_oracle(mods, name, dims, L, R, steps, C):
    Oracle, inputs, slab, sn = mods
    cfg = inputs.scaled(inputs.CONFIGS[name], dims, L=L, steps=steps)
    psi0 = cfg.initial_state()
    one = sn.Simulation(dims, L, cfg.A, cfg.B, C, cfg.D, cfg.g, cfg.dtau)
    one.set_state(psi0)
    n_one = one.diagnostics()["norm"]
    one.step(steps)
    a = one.get_state()
    one.close()
    grp = slab.LocalSlabGroup(dims, L, cfg.A, cfg.B, C, cfg.D, cfg.g, cfg.dtau, R)
    grp.set_state(psi0)
    n0 = grp.norm()
    grp.step(steps // 2)
    grp.step(steps - steps // 2)                 # split calls: psi is back in view A between them
    b = grp.get_state()
    n1 = grp.norm()
    moved = grp.exchanged_elems
    grp.close()
    orc = Oracle(dims, L, cfg.A, cfg.B, C, cfg.D, cfg.g, cfg.dtau)
    orc.set_state(psi0.astype(np.complex128))
    orc.step(steps)
    want = orc.get_state()
    orc.close()
    assert_state(a, want)
    assert_state(b, want)
    assert rel(a, b) < 5e-6                      # same kernels on the same lines; only the merged-half-step boundary differs
    assert abs(n0 - n_one) < 1e-6 * n_one and abs(n1 - n0) < TOL_NORM * n0
    # bytes on the links: per step psi twice and the half spectrum twice (one psi exchange saved per call)
    # (a call of n steps: 1 + n + (n - 1) = 2n psi exchanges and 2n half-spectrum exchanges)
    cells, hs = int(np.prod(dims)), (dims[0] // 2 + 1) * dims[1] * dims[2]
    assert moved == 2 * steps * cells + 2 * steps * hs


def test_slab_contract(mods):
    Oracle, inputs, slab, sn = mods
    dims = (64, 64, 64)
    assert slab._lib().sn_slab_workspace_bytes((__import__("ctypes").c_int64 * 3)(*dims), 3, 0) == 0      # 64 % 3
    assert slab._lib().sn_slab_workspace_bytes((__import__("ctypes").c_int64 * 3)(64, 64, 8), 8, 0) == 0  # 8 x 8 columns < 32
    r = slab.SlabRank(dims, 10.0, -0.5, 1.0, 0.0, 1.0, (0.1,), 1e-3, 2, 1)
    with pytest.raises(sn.SnError) as e:
        r.stage(slab.KIN_A, True)                # no state yet
    assert e.value.code == -6
    r.set_state(np.zeros((32, 64, 64), np.complex64))
    with pytest.raises(sn.SnError) as e:
        r.step(1)                                # whole-grid call on a slab context
    assert e.value.code == -9
    assert r.buffer(slab.PSI_B).numel() == 32 * 64 * 64 and r.buffer(slab.HS_A).numel() == 17 * 64 * 64
    assert r.buffer(slab.HS_B).numel() == 33 * 32 * 64
    r.close()

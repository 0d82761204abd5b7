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


DIST_WORKER = r"""
import json, os, sys
sys.path.insert(0, %r)
import numpy as np, torch, torch.distributed as dist
from paper_1909_08354_b200 import inputs, slab
rank, R = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo", rank=rank, world_size=R)
torch.cuda.set_device(0)
dims, L, steps = tuple(json.loads(os.environ["SLAB_DIMS"])), float(os.environ["SLAB_L"]), int(os.environ["SLAB_STEPS"])
cfg = inputs.scaled(inputs.CONFIGS["C4"], dims, L=L, steps=steps)
psi0 = cfg.initial_state()
rows = dims[0] // R
sim = slab.DistributedSlab(dims, L, cfg.A, cfg.B, cfg.C, cfg.D, cfg.g, cfg.dtau, device="cuda:0")
sim.ctx.set_state(np.ascontiguousarray(psi0[rank * rows:(rank + 1) * rows]))
n0 = sim.norm()
sim.step(steps // 2)
sim.step(steps - steps // 2)
n1 = sim.norm()
np.save(os.environ["SLAB_OUT"] + ".%%d.npy" %% rank, sim.ctx.get_state())
print(json.dumps({"rank": rank, "n0": n0, "n1": n1}))
dist.barrier()
sim.ctx.close()
dist.destroy_process_group()
"""


@pytest.mark.parametrize("dims,R,steps", [((64, 64, 64), 2, 6), ((128, 64, 128), 4, 4)])
def test_distributed_driver_as_rank_processes_on_one_gpu(mods, tmp_path, dims, R, steps):
    """The one-process-per-rank driver (DistributedSlab: sn_slab_pack -> all_to_all_single -> unpack) run as R rank
    PROCESSES that share this one GPU, over the gloo backend with host staging (nccl refuses two ranks on one device).
    No kernel waits on another process: every exchange synchronises its stream and goes through the host.  Same
    result as the single-context step."""
    import json
    import os
    import socket
    import subprocess
    import sys
    Oracle, inputs, slab, sn = mods
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    script = tmp_path / "worker.py"
    script.write_text(DIST_WORKER % root)
    with socket.socket() as so:
        so.bind(("127.0.0.1", 0))
        port = str(so.getsockname()[1])
    L = 16.0
    procs = []
    for r in range(R):
        env = dict(os.environ, RANK=str(r), WORLD_SIZE=str(R), LOCAL_RANK=str(r), MASTER_ADDR="127.0.0.1", MASTER_PORT=port,
                   SLAB_DIMS=json.dumps(list(dims)), SLAB_L=str(L), SLAB_STEPS=str(steps), SLAB_OUT=str(tmp_path / "out"))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE,
                                      text=True))
    norms = []
    for p in procs:
        o, e = p.communicate(timeout=600)
        assert p.returncode == 0, e[-2000:]
        norms.append(json.loads(o.strip().splitlines()[-1]))
    got = np.concatenate([np.load(str(tmp_path / "out") + ".%d.npy" % r) for r in range(R)], axis=0)
    cfg = inputs.scaled(inputs.CONFIGS["C4"], dims, L=L, steps=steps)
    one = sn.Simulation.from_config(cfg)
    one.set_state(cfg.initial_state())
    d0 = one.diagnostics()
    one.step(steps)
    want = one.get_state()
    one.close()
    assert rel(got, want) < 5e-6
    for n in norms:                                   # the all-reduced norm is the global one on every rank, and conserved
        assert abs(n["n0"] - d0["norm"]) < 1e-6 * d0["norm"] and abs(n["n1"] - n["n0"]) < TOL_NORM * n["n0"]

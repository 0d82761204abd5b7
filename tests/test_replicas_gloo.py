"""world_size-2 gloo test of the replica bookkeeping bench.py uses for --gpus N."""
import os
import socket
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = textwrap.dedent("""
    import os, sys, json
    sys.path.insert(0, %r)
    import torch.distributed as dist
    from paper_1909_08354_b200 import replicas
    rank, world, local = replicas.rank_world()
    dist.init_process_group("gloo", rank=rank, world_size=world)
    # each rank "measures" a different time; the job figure must use the slowest one
    ms_local = [10.0, 14.0][rank]
    e2e_local = [30.0, 25.0][rank]
    dist.barrier()
    ms, e2e = replicas.max_over_ranks([ms_local, e2e_local])
    rate = replicas.whole_job_rate(1000, 7, world, ms)
    print(json.dumps({"rank": rank, "world": world, "ms": ms, "e2e": e2e, "rate": rate}))
    dist.barrier()
    dist.destroy_process_group()
""") % ROOT


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_two_rank_gloo_max_and_rate(tmp_path):
    import json
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    port = str(_free_port())
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), WORLD_SIZE="2", LOCAL_RANK=str(r), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=port)
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        o, e = p.communicate(timeout=180)
        assert p.returncode == 0, e
        outs.append(json.loads(o.strip().splitlines()[-1]))
    for o in outs:
        assert o["world"] == 2
        assert o["ms"] == 14.0 and o["e2e"] == 30.0          # MAX over ranks on every rank
        assert abs(o["rate"] - 2 * 1000 * 7 / 14e-3) < 1e-6   # both replicas' work / slowest time


def test_single_process_is_identity():
    from paper_1909_08354_b200 import replicas
    assert replicas.rank_world()[1] >= 1
    assert replicas.max_over_ranks([3.0, 4.0]) == [3.0, 4.0]
    assert replicas.whole_job_rate(10, 2, 1, 1.0) == 20000.0

"""world_size-2 (and 3) gloo test of the slab exchange plumbing (paper_1909_08354_b200/slab.py: exchange_plan,
all_to_all, run_schedule) on CPU tensors -- no kernels, no GPU.  Every rank builds its view-A and view-B buffers from
one known global array, runs the exchange, and must end up with exactly the other view's slab of that array: the psi
exchange (equal blocks) and the half-spectrum exchange (the Nyquist row makes the last rank's blocks one row taller),
in both directions."""
import json
import os
import socket
import subprocess
import sys
import textwrap

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = textwrap.dedent("""
    import json, os, sys
    sys.path.insert(0, %r)
    import numpy as np, torch, torch.distributed as dist
    from paper_1909_08354_b200 import slab
    rank, R = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
    dist.init_process_group("gloo", rank=rank, world_size=R)
    dims = (12 * R, 4 * R, 8)
    n0, n1, n2 = dims
    rng = np.random.default_rng(5)
    out = {"rank": rank}
    for what, name in ((slab.PSI_A, "psi"), (slab.HS_A, "hs")):
        rows_tot = n0 if what == slab.PSI_A else n0 // 2 + 1
        G = (rng.standard_normal((rows_tot, n1, n2)) + 1j * rng.standard_normal((rows_tot, n1, n2))).astype(np.complex64)
        lo, cnt = (rank * (n0 // R), n0 // R) if what == slab.PSI_A else slab.hs_rows(n0, R, rank)
        c0, c1 = rank * (n1 // R), (rank + 1) * (n1 // R)
        A_true = torch.from_numpy(np.ascontiguousarray(G[lo:lo + cnt]))          # [rows of this rank][n1][n2]
        B_true = torch.from_numpy(np.ascontiguousarray(G[:, c0:c1]))             # [all rows][n1/R][n2]
        staging = torch.zeros(A_true.numel(), dtype=torch.complex64)
        colsB = (n1 // R) * n2

        def make_pack(Abuf):
            # what sn_slab_pack does on the device: staging block s = columns of peer s of every local row
            def pack(unpack):
                a3 = Abuf.view(cnt, R, colsB)
                st = staging[: cnt * R * colsB].view(R, cnt, colsB)
                if unpack:
                    a3.copy_(st.permute(1, 0, 2))
                else:
                    st.copy_(a3.permute(1, 0, 2))
            return pack

        # view B -> view A
        A = torch.zeros_like(A_true).reshape(-1)
        B = B_true.clone().reshape(-1)
        slab.all_to_all(staging, B, dims, R, rank, what, True, make_pack(A))
        out[name + "_to_a"] = bool(torch.equal(A.view_as(A_true), A_true))
        # view A -> view B
        A = A_true.clone().reshape(-1)
        B = torch.zeros_like(B_true).reshape(-1)
        slab.all_to_all(staging, B, dims, R, rank, what, False, make_pack(A))
        out[name + "_to_b"] = bool(torch.equal(B.view_as(B_true), B_true))
        a_split, b_split = slab.exchange_plan(dims, R, rank, what)
        out[name + "_sizes"] = [sum(a_split), sum(b_split), int(A_true.numel()), int(B_true.numel())]
    # the schedule: every rank issues the same sequence, 2n psi and 2n half-spectrum exchanges for a call of n steps
    seq = []
    slab.run_schedule(3, lambda w, h: seq.append(("s", w, h)), lambda w, t: seq.append(("x", w, t)))
    out["psi_x"] = sum(1 for e in seq if e[0] == "x" and e[1] == slab.PSI_A)
    out["hs_x"] = sum(1 for e in seq if e[0] == "x" and e[1] == slab.HS_A)
    out["first_last"] = [seq[0], seq[-1]]
    print(json.dumps(out))
    dist.barrier()
    dist.destroy_process_group()
""") % ROOT


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


@pytest.mark.parametrize("world", [2, 3])
def test_slab_exchange_over_gloo(tmp_path, world):
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    port = str(_free_port())
    procs = []
    for r in range(world):
        env = dict(os.environ, RANK=str(r), WORLD_SIZE=str(world), LOCAL_RANK=str(r), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=port)
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    for p in procs:
        o, e = p.communicate(timeout=300)
        assert p.returncode == 0, e
        res = json.loads(o.strip().splitlines()[-1])
        for k in ("psi_to_a", "psi_to_b", "hs_to_a", "hs_to_b"):
            assert res[k], (res["rank"], k)
        for name in ("psi", "hs"):
            a, b, na, nb = res[name + "_sizes"]
            assert a == na and b == nb
        assert res["psi_x"] == 6 and res["hs_x"] == 6
        assert res["first_last"] == [["s", 0, True], ["s", 0, True]]    # KIN_A(half) opens and closes a call


def test_hs_rows_cover_the_half_spectrum():
    from paper_1909_08354_b200 import slab
    for n0, R in ((64, 1), (64, 2), (512, 8), (96, 3), (384, 4)):
        rows = [slab.hs_rows(n0, R, r) for r in range(R)]
        assert rows[0][0] == 0 and rows[-1][0] + rows[-1][1] == n0 // 2 + 1
        for (lo, cnt), (lo2, _) in zip(rows, rows[1:]):
            assert lo + cnt == lo2

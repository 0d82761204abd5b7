"""Slab-decomposed Strang step over R ranks (NEXT-2) -- the schedule and the exchanges.

Every arithmetic step runs in libsn.so's kernels (sn_slab_stage); this module only sequences the stages and moves
blocks between the z-slab view A = [N0/R][N1][N2] and the y-slab view B = [N0][N1/R][N2] (include/sn.h, "NEXT-2"):

    KIN_A(half) | psi A->B | KIN0_B(half)
    n times:  R2C_B | hs B->A | CHAIN_A | hs A->B | NLKIN_B | psi B->A | KIN_A | psi A->B   (last psi A->B dropped)

4 exchanges per step: psi twice (8 B/cell), the half spectrum twice (4 B/cell) = 24 B/cell-update over the links
against 88 B/cell-update over HBM.  Two drivers:

* ``LocalSlabGroup``: R contexts on ONE device and stream ("virtual ranks"), blocks copied device-to-device by
  sn_slab_exchange_local.  This is how the path is validated on a single GPU: parity with the single-context step
  and with the oracle.
* ``DistributedSlab``: one process per GPU; pack (sn_slab_pack) -> ``torch.distributed.all_to_all_single`` -> unpack.
  With the nccl backend the blocks travel over NVLink/NVSwitch.  NOT measured on hardware in this build (one GPU per
  call); its rank plumbing (split sizes, block order) is ``exchange_plan`` below, covered by a world_size-2 gloo test
  on CPU tensors.
"""
from __future__ import annotations

import ctypes
from typing import List, Sequence

import numpy as np

from . import sn

KIN_A, KIN0_B, R2C_B, CHAIN_A, NLKIN_B = 0, 1, 2, 3, 4
PSI_A, PSI_B, HS_A, HS_B, STAGING = 0, 1, 2, 3, 4


def hs_rows(n0: int, nranks: int, rank: int):
    """(first row, row count) of the n0/2+1 half-spectrum rows owned by `rank` in view A: (n0/2)/R each, the Nyquist
    row to the last rank (the rule of sn_slab_create)."""
    per = (n0 // 2) // nranks
    return per * rank, per + (1 if rank == nranks - 1 else 0)


def exchange_plan(dims: Sequence[int], nranks: int, rank: int, what: int):
    """Element counts of the all-to-all for `what` (PSI_A or HS_A), seen from `rank`.

    Returns (a_split, b_split): a_split[s] = elements of the view-A side's block exchanged with peer s (all equal: this
    rank's rows x peer's columns); b_split[r] = elements of the view-B side's block exchanged with peer r (peer's rows x
    this rank's columns; contiguous in the view-B buffer, in rank order).  B->A sends b_split and receives a_split;
    A->B the reverse."""
    n0, n1, n2 = (int(n) for n in dims)
    colsB = (n1 // nranks) * n2
    if what == PSI_A:
        rows = [n0 // nranks] * nranks
    else:
        rows = [hs_rows(n0, nranks, r)[1] for r in range(nranks)]
    return [rows[rank] * colsB] * nranks, [rows[r] * colsB for r in range(nranks)]


def _lib():
    L = sn.lib()
    if not getattr(L, "_slab_ready", False):
        vp, i64p, dp = ctypes.c_void_p, ctypes.POINTER(ctypes.c_int64), ctypes.POINTER(ctypes.c_double)
        L.sn_slab_workspace_bytes.argtypes = [i64p, ctypes.c_int, ctypes.c_int]
        L.sn_slab_workspace_bytes.restype = ctypes.c_size_t
        L.sn_slab_create.argtypes = [ctypes.POINTER(vp), i64p, dp, ctypes.c_double, ctypes.c_double, ctypes.c_double,
                                     ctypes.c_double, dp, ctypes.c_int, ctypes.c_double, ctypes.c_int, ctypes.c_int, vp,
                                     ctypes.c_size_t, vp]
        L.sn_slab_stage.argtypes = [vp, ctypes.c_int, ctypes.c_int]
        L.sn_slab_buffer.argtypes = [vp, ctypes.c_int, ctypes.POINTER(vp), i64p]
        L.sn_slab_pack.argtypes = [vp, ctypes.c_int, ctypes.c_int]
        L.sn_slab_exchange_local.argtypes = [ctypes.POINTER(vp), ctypes.c_int, ctypes.c_int, ctypes.c_int]
        L.sn_slab_local_norm.argtypes = [vp, dp]
        L._slab_ready = True
    return L


class SlabRank(sn.Simulation):
    """The context of one rank (sn_slab_create): local passes, buffers and pack/unpack; state shape (N0/R, N1, N2)."""

    def __init__(self, dims: Sequence[int], L, A, B, C, D, g, dtau, nranks: int, rank: int, device="cuda:0", stream=None):
        import torch

        if not torch.cuda.is_available():
            raise RuntimeError("paper_1909_08354_b200 needs a CUDA device (no CPU fallback)")
        gd = tuple(int(n) for n in dims)
        assert len(gd) == 3
        self.global_dims, self.nranks, self.rank = gd, int(nranks), int(rank)
        self.dims = (gd[0] // nranks, gd[1], gd[2])
        self.features = 0
        self.dtype, self.real_dtype = np.dtype(np.complex64), np.dtype(np.float32)
        Ls = [float(L)] * 3 if np.isscalar(L) else [float(v) for v in L]
        g = [float(v) for v in g]
        self.device = torch.device(device)
        c_dims = (ctypes.c_int64 * 3)(*gd)
        nbytes = int(_lib().sn_slab_workspace_bytes(c_dims, nranks, rank))
        if nbytes == 0:
            raise sn.SnError(-2, "sn_slab_workspace_bytes", sn.lib().sn_strerror(-2).decode())
        with torch.cuda.device(self.device):
            self._ws = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            self._stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self._h = ctypes.c_void_p()
        sn._chk(_lib().sn_slab_create(ctypes.byref(self._h), c_dims, (ctypes.c_double * 3)(*Ls), A, B, C, D,
                                      (ctypes.c_double * max(1, len(g)))(*(g or [0.0])), len(g), dtau, nranks, rank,
                                      ctypes.c_void_p(self._ws.data_ptr()), nbytes,
                                      ctypes.c_void_p(self._stream.cuda_stream)), "sn_slab_create")

    def stage(self, which: int, half: bool) -> None:
        sn._chk(_lib().sn_slab_stage(self._h, which, 1 if half else 0), "sn_slab_stage")

    def pack(self, what: int, unpack: bool) -> None:
        sn._chk(_lib().sn_slab_pack(self._h, what, 1 if unpack else 0), "sn_slab_pack")

    def buffer(self, which: int):
        """A flat complex64 torch view of one of the context's exchange buffers (inside the workspace tensor)."""
        import torch
        p, n = ctypes.c_void_p(), ctypes.c_int64()
        sn._chk(_lib().sn_slab_buffer(self._h, which, ctypes.byref(p), ctypes.byref(n)), "sn_slab_buffer")
        off = p.value - self._ws.data_ptr()
        return self._ws[off:off + 8 * n.value].view(torch.complex64)

    def local_norm(self) -> float:
        v = ctypes.c_double()
        sn._chk(_lib().sn_slab_local_norm(self._h, ctypes.byref(v)), "sn_slab_local_norm")
        return float(v.value)


def run_schedule(nsteps: int, stage, exchange) -> None:
    """The stage/exchange sequence of one call of nsteps Strang steps (merged half kinetics), psi in view A at both
    ends.  stage(which, half) runs a local stage on every rank this driver owns; exchange(what, to_a) moves psi
    (PSI_A) or the half spectrum (HS_A) between the views."""
    if nsteps <= 0:
        return
    stage(KIN_A, True)
    exchange(PSI_A, False)
    stage(KIN0_B, True)
    for i in range(1, nsteps + 1):
        last = i == nsteps
        stage(R2C_B, False)
        exchange(HS_A, True)
        stage(CHAIN_A, False)
        exchange(HS_A, False)
        stage(NLKIN_B, last)
        exchange(PSI_A, True)
        stage(KIN_A, last)
        if not last:
            exchange(PSI_A, False)


class LocalSlabGroup:
    """R virtual ranks on one device and stream: the whole decomposed step on a single GPU."""

    def __init__(self, dims, L, A, B, C, D, g, dtau, nranks: int, device="cuda:0"):
        self.dims, self.nranks = tuple(int(n) for n in dims), int(nranks)
        self.ranks: List[SlabRank] = [SlabRank(dims, L, A, B, C, D, g, dtau, nranks, r, device=device) for r in range(nranks)]
        self._arr = (ctypes.c_void_p * nranks)(*[r._h for r in self.ranks])
        self.exchanged_elems = 0

    def set_state(self, psi: np.ndarray) -> None:
        rows = self.dims[0] // self.nranks
        for r, ctx in enumerate(self.ranks):
            ctx.set_state(np.ascontiguousarray(psi[r * rows:(r + 1) * rows]))

    def get_state(self) -> np.ndarray:
        return np.concatenate([ctx.get_state() for ctx in self.ranks], axis=0)

    def _stage(self, which, half):
        for ctx in self.ranks:
            ctx.stage(which, half)

    def _exchange(self, what, to_a):
        sn._chk(_lib().sn_slab_exchange_local(self._arr, self.nranks, what, 1 if to_a else 0), "sn_slab_exchange_local")
        self.exchanged_elems += sum(sum(exchange_plan(self.dims, self.nranks, r, what)[0]) for r in range(self.nranks))

    def step(self, nsteps: int) -> None:
        run_schedule(int(nsteps), self._stage, self._exchange)

    def norm(self) -> float:
        return sum(ctx.local_norm() for ctx in self.ranks)

    def launch_count(self) -> int:
        return sum(ctx.launch_count() for ctx in self.ranks)

    def close(self) -> None:
        for ctx in self.ranks:
            ctx.close()


class DistributedSlab:
    """One process per GPU (torch.distributed initialised by the caller; nccl on GPUs): this rank's slab."""

    def __init__(self, dims, L, A, B, C, D, g, dtau, device=None, group=None):
        import torch.distributed as dist
        self.group = group
        self.nranks, self.rank = dist.get_world_size(group), dist.get_rank(group)
        self.dims = tuple(int(n) for n in dims)
        self.ctx = SlabRank(dims, L, A, B, C, D, g, dtau, self.nranks, self.rank,
                            device=device or f"cuda:{self.rank}")

    def _exchange(self, what, to_a):
        all_to_all(self.ctx.buffer(STAGING), self.ctx.buffer(PSI_B if what == PSI_A else HS_B), self.dims, self.nranks,
                   self.rank, what, to_a, lambda unpack: self.ctx.pack(what, unpack), self.group)

    def step(self, nsteps: int) -> None:
        run_schedule(int(nsteps), self.ctx.stage, self._exchange)

    def norm(self) -> float:
        import torch
        import torch.distributed as dist
        on_gpu = dist.get_backend(self.group) != "gloo"
        t = torch.tensor([self.ctx.local_norm()], dtype=torch.float64, device=self.ctx.device if on_gpu else "cpu")
        dist.all_reduce(t, group=self.group)
        return float(t[0])


def all_to_all(staging, b_buf, dims, nranks, rank, what, to_a, pack, group=None) -> None:
    """One exchange of a rank: `staging` = the view-A blocks in rank order (filled / drained by pack(unpack)),
    `b_buf` = the view-B buffer, whose blocks are contiguous in rank order already.  Works on any backend (the CPU
    test drives it with gloo and plain tensors)."""
    import torch
    import torch.distributed as dist
    a_split, b_split = exchange_plan(dims, nranks, rank, what)
    na, nb = sum(a_split), sum(b_split)
    if staging.is_complex():                            # move (re, im) pairs as floats: every backend takes those
        staging, b_buf = torch.view_as_real(staging).reshape(-1), torch.view_as_real(b_buf).reshape(-1)
        a_split, b_split, na, nb = [2 * v for v in a_split], [2 * v for v in b_split], 2 * na, 2 * nb
    def a2a(out, inp, out_split, in_split):
        if inp.is_cuda and dist.get_backend(group) == "gloo":
            # gloo moves host memory: stage through the CPU (the single-GPU validation of this driver runs two rank
            # processes on one device this way; nccl takes the device buffers directly)
            host_out = torch.empty(out.shape, dtype=out.dtype)
            dist.all_to_all_single(host_out, inp.cpu(), output_split_sizes=out_split, input_split_sizes=in_split, group=group)
            out.copy_(host_out)
        else:
            dist.all_to_all_single(out, inp, output_split_sizes=out_split, input_split_sizes=in_split, group=group)

    if to_a:                                            # view B -> view A
        a2a(staging[:na], b_buf[:nb], a_split, b_split)
        pack(True)
    else:                                               # view A -> view B
        pack(False)
        a2a(b_buf[:nb], staging[:na], b_split, a_split)

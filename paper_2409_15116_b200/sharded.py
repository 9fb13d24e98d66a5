"""Row-sharded two-body kernel over several GPUs (SURVEY 8(f) #3; PAPER.md:148, :156 and Fig. 2).

One process per GPU.  The N_v output rows (orbitals of A_s) are block-distributed over the ranks, u and phi are replicated
(P_c needs every orbital).  Per application:
  1. the all-gather of the trial blocks a (each rank holds its rows of every block, PW coefficients on H) is STARTED on a side
     stream, one collective per trial block so that it is chunked ("initiated in a non-blocking fashion");
  2. meanwhile K1e runs on the local rows: the Hartree potential of the local share of the transition density
     (bse_k1e_hartree_partial), one all-reduce of B * N_pw_h coefficients (the sum over occupied states of eq. 4), the
     products and P_c for the local rows (bse_k1e_from_hartree);
  3. the gather is waited for ("we enforce the completion of the communication before evaluating the K1d term") and
     bse_apply_k1x runs on a handle restricted to the local rows by bse_set_rows: tau only for the pairs that touch them.
This file is plumbing (torch.distributed collectives, buffers, streams): every numeric step is a call into libbse_b200.
The pure partition / collective helpers work on CPU tensors with the gloo backend (tests/test_sharded_gloo.py).
"""
from __future__ import annotations

import os

import numpy as np


def row_blocks(Nv: int, world: int):
    """Block distribution of Fig. 2: contiguous row ranges, the first Nv % world ranks hold one row more."""
    base, extra = divmod(Nv, world)
    out, v0 = [], 0
    for r in range(world):
        n = base + (1 if r < extra else 0)
        out.append((v0, v0 + n))
        v0 += n
    return out


def start_gather(a_local, blocks, rank, dist, group=None):
    """All-gather of the trial blocks, one collective per block b.  a_local: [B][nloc][K] (this rank's rows), any device.
    Returns (a_full [B][Nv][K], finish): finish() waits for the collectives and, when the row blocks are uneven, moves the
    padded pieces into place.  With equal blocks every collective writes straight into a_full[b] (ranks' rows are adjacent)."""
    import torch
    B, nloc, K = a_local.shape
    world = len(blocks)
    Nv = blocks[-1][1]
    assert blocks[rank][1] - blocks[rank][0] == nloc
    a_full = torch.empty((B, Nv, K), dtype=a_local.dtype, device=a_local.device)
    if world == 1:
        a_full.copy_(a_local)
        return a_full, (lambda: a_full)
    nmax = max(v1 - v0 for v0, v1 in blocks)
    even = all(v1 - v0 == nmax for v0, v1 in blocks)
    works = []
    if even:
        for b in range(B):
            works.append(dist.all_gather_into_tensor(a_full[b], a_local[b].contiguous(), group=group, async_op=True))
        pad = None
    else:
        pad = torch.zeros((B, world, nmax, K), dtype=a_local.dtype, device=a_local.device)
        mine = torch.zeros((B, nmax, K), dtype=a_local.dtype, device=a_local.device)
        mine[:, :nloc] = a_local
        for b in range(B):
            works.append(dist.all_gather_into_tensor(pad[b].view(world * nmax, K), mine[b], group=group, async_op=True))

    def finish():
        for w in works:
            w.wait()
        if pad is not None:
            for r, (v0, v1) in enumerate(blocks):
                a_full[:, v0:v1] = pad[:, r, :v1 - v0]
        return a_full
    return a_full, finish


def allreduce_sum(x, dist, group=None):
    if dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(x, op=dist.ReduceOp.SUM, group=group)
    return x


class ShardedBSE:
    """One rank's share: a handle restricted to its row block, buffers, the side stream of the gather."""

    def __init__(self, grid, cell, ecut, Nv, u, Npdep, phi, lam, eta, tau_flag, rank, world, dist, device):
        import torch
        from . import bse
        self.bse, self.dist, self.torch = bse, dist, torch
        self.rank, self.world, self.device, self.Nv = rank, world, device, Nv
        self.blocks = row_blocks(Nv, world)
        self.v0, self.v1 = self.blocks[rank]
        self.stream = torch.cuda.current_stream(device)
        self.side = torch.cuda.Stream(device)
        self.h = bse.bse_create(grid, cell, ecut, Nv, u, Npdep, phi, lam, eta, tau_flag | bse.BSE_VEC_PW, self.stream.cuda_stream)
        bse.bse_set_rows(self.h, self.v0, self.v1)
        self.npw_h = bse.bse_npw_half(self.h)

    def build(self):
        self.bse.bse_build_tau(self.h)

    def apply(self, a_local, out_e, out_x):
        """a_local, out_e, out_x: [B][nloc][npw_h][2] on the device.  out_e = K1e rows, out_x = K1x rows (eq. 4, 5); the caller
        combines them with the signs of eq. 1."""
        torch, bse, dist = self.torch, self.bse, self.dist
        B = a_local.shape[0]
        nloc = self.v1 - self.v0
        flat = a_local.reshape(B, nloc, self.npw_h * 2)
        self.side.wait_stream(self.stream)                       # a_local is ready on the main stream
        with torch.cuda.stream(self.side):
            a_full, finish = start_gather(flat, self.blocks, self.rank, dist)
        vG = torch.empty((B, self.npw_h, 2), dtype=torch.float64, device=self.device)
        bse.bse_k1e_hartree_partial(self.h, a_local, self.v0, self.v1, B, vG)
        allreduce_sum(vG, dist)
        bse.bse_k1e_from_hartree(self.h, vG, self.v0, self.v1, B, out_e)
        with torch.cuda.stream(self.side):
            finish()
        self.stream.wait_stream(self.side)                       # the gather is complete before K1d
        bse.bse_apply_k1x(self.h, a_full, out_x, B)
        return a_full

    def close(self):
        self.bse.bse_destroy(self.h)


def bench_main(args, rank, local_rank, world):
    """bench.py --mode sharded: strong scaling of one two-body application (K1e + K1d) over the ranks; the workload is the
    config's, the rows are block-distributed.  value = K1 applies / s of the whole job (max over ranks)."""
    import json
    import torch
    import torch.distributed as dist
    from . import bse, workloads as wl
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    os.environ.setdefault("MASTER_PORT", "29533")
    if not dist.is_initialized():
        dist.init_process_group("nccl", rank=rank, world_size=world, device_id=dev)
    cfg = args.config
    tau = args.tau or {1: "pw", 2: "pw", 3: "pw", 4: "pw", 5: "stream"}[cfg]
    flag = {"pw": bse.BSE_TAU_PW, "stream": bse.BSE_TAU_STREAM}[tau]
    w = wl.make_device(cfg, dev)
    Nv, B = w.Nv, w.a_pw.shape[0]
    phi_d = torch.view_as_real(w.phi).contiguous()
    sh = ShardedBSE([w.n] * 3, w.cell, w.ecut, Nv, w.u, w.phi.shape[0], phi_d, w.lam, w.eta, flag, rank, world, dist, dev)
    a_local = torch.view_as_real(w.a_pw[:, sh.v0:sh.v1]).contiguous()
    w.a_pw = None
    w.u_pw = None
    torch.cuda.empty_cache()
    out_e, out_x = torch.empty_like(a_local), torch.empty_like(a_local)
    steps, warm = args.steps, max(args.warmup, 3)
    tb, ta = [], []
    for i in range(warm + steps):
        e0, e1, e2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
        dist.barrier()
        torch.cuda.synchronize()
        e0.record()
        sh.build()
        e1.record()
        sh.apply(a_local, out_e, out_x)
        e2.record()
        e2.synchronize()
        if i >= warm:
            tb.append(e0.elapsed_time(e1))
            ta.append(e1.elapsed_time(e2))
    t = torch.tensor([float(np.mean(tb)), float(np.mean(ta))], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    P = bse.bse_num_pairs(sh.h)
    sh.close()
    if rank == 0:
        tb_ms, ta_ms = t.tolist()
        line = {"metric": "K1 (K1e + K1d) applies/s, rows sharded over the GPUs (SURVEY 8(f) #3), fp64", "value": B / (ta_ms * 1e-3),
                "unit": "applies/s", "n_gpus": world, "steps": steps, "warmup": warm, "ms_per_step": tb_ms + ta_ms,
                "build_ms": tb_ms, "apply_ms": ta_ms, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
                "dtype": "f64", "data": "synthetic", "pairs": P,
                "config": {"workload": f"BASELINE.json configs[{cfg - 1}] (cfg{cfg}): grid {w.n}^3, Nv={Nv}, B={B}, P={P}",
                           "tau_storage": tau, "vec_layout": "pw", "parallelism": f"rows/{world}",
                           "collectives": "all-gather of a (per block, side stream) overlapped with K1e; all-reduce of v_c n(G)"}}
        print(json.dumps(line))
    dist.destroy_process_group()

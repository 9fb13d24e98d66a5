"""Row-sharded two-body kernel (paper_2409_15116_b200/sharded.py): the N > 1 host logic on CPU.

World sizes 2 and 3 over gloo: block distribution of the rows (Fig. 2), the per-block all-gather of the trial
blocks (even and uneven row blocks), the all-reduce of the Hartree shares.  The numeric steps a rank would run on its GPU are
stood in for by the ORACLE here (this is a test: it checks that partition + collectives reproduce the single-rank oracle
result; the GPU path of the same partition is tests/test_gpu_parity.py::test_row_sharded_*)."""
import os
import sys

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.multiprocessing as mp          # noqa: E402

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_row_blocks_cover_every_row_once():
    sys.path.insert(0, ROOT)
    from paper_2409_15116_b200.sharded import row_blocks
    for Nv, world in ((8, 2), (9, 2), (10, 3), (5, 8), (1024, 8), (7, 1)):
        blocks = row_blocks(Nv, world)
        assert len(blocks) == world and blocks[0][0] == 0 and blocks[-1][1] == Nv
        assert all(blocks[r][1] == blocks[r + 1][0] for r in range(world - 1))
        sizes = [v1 - v0 for v0, v1 in blocks]
        assert max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)


def _worker(rank, world, port, Nv, q):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    from oracle import bse_oracle as orc
    from paper_2409_15116_b200 import workloads as wl
    from paper_2409_15116_b200.sharded import allreduce_sum, row_blocks, start_gather
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        cfg = wl.Config("shard", 9.0, 12, Nv, 7, 3.0, 1.3, 0.8, 3.0, 0.05, 2, "random", seed=910 + Nv)
        w = wl.make(cfg=cfg)                                        # every rank generates the same seeded inputs (u, phi replicated)
        tab = orc.Tables(w.n, w.L, w.ecut)
        blocks = row_blocks(Nv, world)
        v0, v1 = blocks[rank]
        B = w.a_pw.shape[0]
        # ---- 1. all-gather of the trial blocks from the ranks' row blocks
        a_local = torch.from_numpy(np.ascontiguousarray(w.a_pw[:, v0:v1]).view(np.float64).reshape(B, v1 - v0, -1))
        a_full_t, finish = start_gather(a_local, blocks, rank, dist)
        a_full = finish().numpy().reshape(B, Nv, -1, 2).view(np.complex128)[..., 0]
        assert np.array_equal(a_full, w.a_pw)
        # ---- 2. K1e: local share of v_c n(G), all-reduce, local rows
        uS = np.array([tab.to_G(w.u[x]) for x in range(Nv)])
        share = np.zeros((B, tab.npw), dtype=np.complex128)
        for b in range(B):
            n_r = np.zeros(tab.N)
            for v in range(v0, v1):
                n_r += w.u[v] * tab.to_r(tab.expand_H_to_S(w.a_pw[b, v]))
            share[b] = tab.vc12 * tab.vc12 * tab.to_G(n_r)
        tot = torch.from_numpy(share.view(np.float64).copy())
        allreduce_sum(tot, dist)
        vG = tot.numpy().view(np.complex128)
        out_e = np.empty((B, v1 - v0, tab.npw_h), dtype=np.complex128)
        for b in range(B):
            vH = tab.to_r(vG[b])
            for v in range(v0, v1):
                out_e[b, v - v0] = orc.S_to_H(tab, orc.p_c_pw(tab, uS, tab.to_G(2.0 * w.u[v] * vH)))
        # ---- 3. K1d on the local rows with the pairs that touch them
        pairs, _ = orc.screen_pairs(w.u, w.eta)
        mine = [(int(v), int(x)) for v, x in pairs if v0 <= v < v1 or v0 <= x < v1]
        tau = {vx: orc.tau_r(tab, w.u[vx[0]], w.u[vx[1]], tab.expand_H_to_S(w.phi), w.lam) for vx in mine}
        a_r = {(b, x): tab.to_r(tab.expand_H_to_S(a_full[b, x])) for b in range(B) for x in range(Nv)}
        out_x = np.empty_like(out_e)
        for b in range(B):
            for v in range(v0, v1):
                acc = np.zeros(tab.N)
                for (p, x) in mine:
                    if p == v:
                        acc += tau[(p, x)] * a_r[(b, x)]
                    elif x == v:
                        acc += tau[(p, x)] * a_r[(b, p)]
                out_x[b, v - v0] = orc.S_to_H(tab, orc.p_c_pw(tab, uS, tab.to_G(acc)))
        q.put((rank, v0, v1, out_e, out_x, len(mine), len(pairs)))
        dist.barrier()
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world,Nv", [(2, 6), (3, 7)])
def test_sharded_partition_reproduces_the_single_rank_oracle(world, Nv):
    sys.path.insert(0, ROOT)
    from oracle import bse_oracle as orc
    from paper_2409_15116_b200 import workloads as wl
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + ((os.getpid() * 7 + world) % 2000)
    procs = [ctx.Process(target=_worker, args=(r, world, port, Nv, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = sorted((q.get(timeout=300) for _ in range(world)), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    cfg = wl.Config("shard", 9.0, 12, Nv, 7, 3.0, 1.3, 0.8, 3.0, 0.05, 2, "random", seed=910 + Nv)
    w = wl.make(cfg=cfg)
    tab = orc.Tables(w.n, w.L, w.ecut)
    pairs, _ = orc.screen_pairs(w.u, w.eta)
    tau = orc.build_tau(tab, w.u, w.phi, w.lam, pairs, want="r")
    ref_x = orc.apply_k1x_pw(tab, w.u, pairs, tau, w.a_pw)
    ref_e = orc.apply_k1e_pw(tab, w.u, w.a_pw)
    out_e = np.concatenate([g[3] for g in got], axis=1)
    out_x = np.concatenate([g[4] for g in got], axis=1)
    assert np.linalg.norm(out_e - ref_e) <= 1e-12 * np.linalg.norm(ref_e)
    assert np.linalg.norm(out_x - ref_x) <= 1e-12 * np.linalg.norm(ref_x)
    # a pair that straddles two owners is held by both; together the ranks hold every pair at least once
    assert sum(g[5] for g in got) >= len(pairs) and all(g[6] == len(pairs) for g in got)

#!/usr/bin/env python
"""bench.py - throughput of the screened-exchange hot path on B200 (one line of JSON on stdout).

A "step" = one pass of the whole hot path over one synthetic workload: bse_build_tau (screen, pair list, tau for every
surviving pair) followed by bse_apply_k1x on the config's B trial blocks.  Default workload = BASELINE.json configs[4]
(cfg 5, the largest single-GPU configuration: tau streamed, trial blocks in the plane-wave layout); `--config C` picks
another one.
  value  = screened pair integrals / s = P / device time spent producing them (screen + pair list + the fill of the tau
           store: inside bse_build_tau for tau storage real / pw, inside the apply for `stream`, where it is timed by the
           library's own CUDA events), inputs resident in HBM
  k1x    = K1x applies / s = B / device time of bse_apply_k1x (for `stream` the call includes the tau rebuild: that is
           what one apply costs in that mode)
  e2e    = the same two through the C ABI with HOST buffers (pinned): H2D of u, phi, a and D2H of out inside the timed region
  roofline     = the stage with the largest share of the step against the measured HBM / FP64 peak; `frac` uses the
                 algorithmic bytes of SURVEY.md 8(d) (8N per field for a plane pass, 16 N_pw_h per field for a stick pass: the
                 stick-plane hand-off Z is not credited), `frac_with_handoff` the library's own model that also counts Z
  cpu_baseline = the CPU oracle (oracle/bse_oracle.py, as it stands) on a bounded sample of the same workload

`--impl reference` times the oracle alone on the host cores (rank 0 only).
Multi-GPU: `--mode replicas` (default; the hot path of north_star has no exchange step: every rank runs an independent
replica, value = pairs of all ranks / max-over-ranks time, "weak") or `--mode sharded` (output rows
block-distributed over the ranks, all-gather of the trial blocks, "strong").
"""
from __future__ import annotations

import argparse
import csv
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "screened pair integrals/s (tau build incl. screen; K1x applies/s beside it), fp64, B200"
TRAFFIC_FILE = os.path.join(ROOT, "profiles", "ncu_traffic.csv")


def max_over_ranks(values, dist=None, device=None):
    """Element-wise MAX over the ranks of the default process group (every rank gets the result).
    Multi-GPU = independent replicas: the step time of the job is the slowest replica's."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return [float(v) for v in values]
    import torch
    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return t.tolist()


def load_traffic(config, tau, vec):
    """DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum) of the kernel behind each stage, from committed
    `ncu --set full` captures: profiles/ncu_traffic.csv (columns config,tau,vec,stage,dram_bytes_per_launch,source).
    Constants of those captures, not measured by this run; {} when the file has no row for this launch configuration."""
    out = {}
    if os.path.exists(TRAFFIC_FILE):
        with open(TRAFFIC_FILE) as f:
            for row in csv.DictReader(f):
                if int(row["config"]) == config and row["tau"] == tau and row["vec"] == vec:
                    out[row["stage"]] = (float(row["dram_bytes_per_launch"]), row["source"])
    return out


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""

    def __init__(self, index=0):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        self.t.join(timeout=2)
        sm = [float(r[0]) for r in self.rows if len(r) >= 7 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 7 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({names[i] for r in self.rows if len(r) >= 7 for i in range(4) if r[3 + i] == "Active"})
        pw = [float(r[2]) for r in self.rows if len(r) >= 7 and r[2].replace(".", "").isdigit()]
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "sm_mhz_min": min(sm) if sm else None, "sm_mhz_p10": float(np.percentile(sm, 10)) if sm else None,
                "power_w_max": max(pw) if pw else None, "reasons": reasons, "samples": len(sm)}


BOUND = {"screen_syrk": "tensor", "pair_list": "hbm", "fwd_plane": "hbm", "fwd_stick": "hbm", "pdep_project": "tensor",
         "pdep_backproject": "tensor", "inv_stick": "hbm", "inv_plane": "hbm", "k1x_accumulate": "hbm",
         "pc_overlap": "tensor", "pc_update": "tensor", "k1e_density": "hbm", "k1e_product": "hbm"}


def workload_string(cfg_id, n, Nv, n_pdep, npw_h, eta, P, B):
    return (f"BASELINE.json configs[{cfg_id - 1}] (cfg{cfg_id}): grid {n}^3, Nv={Nv}, Npdep={n_pdep}, Npw_h={npw_h}, "
            f"eta={eta}, P={P} surviving pairs, B={B}")


# ------------------------------------------------------------------------------------------------ the CPU oracle, sampled
def oracle_sample(get_u, n, L, ecut, Nv, phi_host, lam, pairs, n_pairs, n_rows, n_cols, seconds_cap=25.0):
    """The oracle, as it stands, on a bounded sample of the workload: `n_rows` x `n_cols` entries of the eq. 16 overlap
    matrix in long double (extrapolated to the N_v x N_v entries the oracle's screen forms) and tau for `n_pairs` of the
    surviving pairs (extrapolated to all P).  get_u(v) returns orbital v as a float64 host array."""
    import psutil
    from oracle import bse_oracle as orc
    proc = psutil.Process()
    c0 = proc.cpu_times()
    t0 = time.perf_counter()
    rng = np.random.default_rng(11)
    tab = orc.Tables(n, L, ecut)
    cols = sorted(rng.choice(Nv, size=min(n_cols, Nv), replace=False).tolist())
    k = min(n_rows, len(cols))
    t1 = time.perf_counter()
    orc.overlap_rows(lambda i: get_u(cols[i]), len(cols), list(range(k)))      # rows = the first k sampled orbitals
    t_entries = time.perf_counter() - t1
    n_entries = k * len(cols)
    phiS = tab.expand_H_to_S(phi_host)
    P = len(pairs)
    sel = rng.choice(P, size=min(n_pairs, P), replace=False)
    t2 = time.perf_counter()
    done = 0
    for p in sel:
        v, x = pairs[p]
        orc.tau_r(tab, get_u(int(v)), get_u(int(x)), phiS, lam)
        done += 1
        if time.perf_counter() - t2 > seconds_cap:
            break
    t_tau = time.perf_counter() - t2
    wall = time.perf_counter() - t0
    c1 = proc.cpu_times()
    cores = max(1, int(round(((c1.user - c0.user) + (c1.system - c0.system)) / wall)))
    per_entry = t_entries / max(n_entries, 1)
    per_pair = t_tau / max(done, 1)
    screen_s = per_entry * Nv * Nv
    return dict(pairs_per_s=P / (screen_s + per_pair * P), per_pair_s=per_pair, per_entry_s=per_entry, screen_s=screen_s,
                sampled_pairs=done, sampled_entries=n_entries, P=P, cores=cores)


def run_reference(args, rank):
    """The oracle, as it stands, on the host cores (rank 0 only).  One step = a bounded sample of the workload: a few entries
    of the eq. 16 overlap matrix (long double) and tau for one or two surviving pairs, each extrapolated to the whole workload
    (N_v^2 entries, P pairs).  Which pairs survive comes from one untimed set-up screen: the oracle's own for cfg 1-2; for
    cfg 3-5, whose full long-double screen takes hours, an fp64 torch.matmul of the squared orbitals (set-up only: it picks
    the sample and P, nothing of it is timed)."""
    if rank != 0:
        return
    import psutil
    from oracle import bse_oracle as orc
    from paper_2409_15116_b200 import workloads as wl
    cfg_id = args.config
    large = cfg_id >= 3
    if large:
        import torch
        dev = "cuda:0" if torch.cuda.is_available() else "cpu"
        w = wl.make_device(cfg_id, dev)
        q = w.u * w.u
        M = q @ q.T
        d = torch.sqrt(torch.diagonal(M))
        O = (M / (d[:, None] * d[None, :])).cpu().numpy()
        del q, M
        iu = np.triu_indices(w.Nv)
        keep = (O[iu] >= w.eta) | (iu[0] == iu[1])
        pairs = np.stack([iu[0][keep], iu[1][keep]], axis=1)
        phi_host = w.phi.cpu().numpy()
        n_pdep, B = w.phi.shape[0], w.a_pw.shape[0]
        cache = {}

        def get_u(v):
            if v not in cache:
                cache[v] = w.u[v].cpu().numpy()
            return cache[v]
        n_pairs, n_ent = 1, 8
    else:
        w = wl.make(cfg_id)
        pairs, _ = orc.screen_pairs(w.u, w.eta)
        phi_host = w.phi
        n_pdep, B = w.phi.shape[0], w.a_pw.shape[0]

        def get_u(v):
            return w.u[v]
        n_pairs, n_ent = 2, 4 * w.Nv
    tab = orc.Tables(w.n, w.L, w.ecut)
    P = len(pairs)
    phiS = tab.expand_H_to_S(phi_host)
    rng = np.random.default_rng(12)
    proc = psutil.Process()
    vals, cores = [], 1
    for i in range(args.warmup + args.steps):
        c0, t0 = proc.cpu_times(), time.perf_counter()
        v = int(rng.integers(w.Nv))
        cols = rng.choice(w.Nv, size=min(n_ent, w.Nv), replace=False).tolist()
        qv = (get_u(v) ** 2).astype(np.longdouble)
        for x in cols:                                             # eq. 16 numerators, as overlap_rows forms them
            (qv * (get_u(int(x)) ** 2).astype(np.longdouble)).sum()
        t1 = time.perf_counter()
        for p in rng.choice(P, size=min(n_pairs, P), replace=False):
            orc.tau_r(tab, get_u(int(pairs[p][0])), get_u(int(pairs[p][1])), phiS, w.lam)
        t2 = time.perf_counter()
        c1 = proc.cpu_times()
        est = (t1 - t0) * w.Nv * w.Nv / len(cols) + (t2 - t1) * P / min(n_pairs, P)
        cores = max(1, int(round(((c1.user - c0.user) + (c1.system - c0.system)) / (t2 - t0))))
        if i >= args.warmup:
            vals.append(P / est)
    v = float(np.mean(vals))
    sample = (f"per step: {min(n_ent, w.Nv)} entries of the eq.16 overlap matrix (long double; extrapolated to Nv^2 = "
              f"{w.Nv * w.Nv}) + tau for {min(n_pairs, P)} of {P} surviving pairs (extrapolated to all)")
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": "pairs/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * P / v, "ms_per_step_is": "extrapolated",
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_string(cfg_id, w.n, w.Nv, n_pdep, w.mill.shape[0], w.eta, P, B),
                       "tau_storage": "oracle", "vec_layout": "real", "parallelism": "host cores"},
            "cpu_baseline": {"value": v, "unit": "pairs/s", "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": v, "unit": "pairs/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def pinned_copy(t):
    import torch
    h = torch.empty(t.shape, dtype=t.dtype, pin_memory=True)
    h.copy_(t)
    return h


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=5, help="BASELINE.json config number (1-based); 5 = configs[4], the largest")
    ap.add_argument("--tau", default=None, choices=["real", "pw", "stream"],
                    help="tau storage; default per config: 1-2 real, 3-4 pw, 5 stream (SURVEY.md 8(d) item 7)")
    ap.add_argument("--vec", default=None, choices=["real", "pw"], help="layout of a/out; default: 1-3 real, 4-5 pw")
    ap.add_argument("--mode", default="replicas", choices=["replicas", "sharded"])
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-k1e", action="store_true")
    ap.add_argument("--tau-f32", action="store_true", help="mixed-precision variant: tau(G) kept as complex64 (BSE_TAU_F32); "
                    "not the headline (the 1e-10 parity bar applies to the double store)")
    ap.add_argument("--reduce", default=None, metavar="Nv,Npdep,B",
                    help="profiling only: the chosen config's grid, cell and sphere with fewer orbitals / PDEP vectors / blocks "
                         "(cfg 3-5; ncu --set full saves and restores the whole device memory around every replay); the line "
                         "is marked REDUCED and is not a bench value")
    ap.add_argument("--knob", action="append", default=[], help="key=value for bse_debug_set (tuning / A-B runs), repeatable")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, rank)
        return
    if args.mode == "sharded":
        from paper_2409_15116_b200 import sharded
        sharded.bench_main(args, rank, local_rank, world)
        return
    args.warmup = max(args.warmup, 3)
    if args.reduce:
        args.no_e2e = args.no_cpu_baseline = True

    import psutil
    import torch
    import torch.distributed as dist
    from paper_2409_15116_b200 import bse, workloads as wl

    # cfg 5 end to end keeps u, phi, a and out in pinned host memory (103 GB): without that much host memory fall back to
    # cfg 4 (never to a small config) and say so
    fallback = None
    if args.config == 5 and not args.no_e2e:
        need = 103e9 * max(1, world if world <= 8 else 8)
        avail = psutil.virtual_memory().available
        if avail < need + 24e9:
            fallback = f"cfg5 e2e needs {need / 1e9:.0f} GB of pinned host memory, {avail / 1e9:.0f} GB available: ran cfg4"
            args.config = 4
    if args.tau is None:
        args.tau = {1: "real", 2: "real", 3: "pw", 4: "pw", 5: "stream"}[args.config]
    if args.vec is None:
        args.vec = "pw" if args.config >= 4 else "real"
    large = args.config >= 3

    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=dev)

    t_gen0 = time.perf_counter()
    u_host = phi_host = a_host = out_host = None
    if large:
        if args.reduce:
            r_nv, r_npdep, r_b = (int(x) for x in args.reduce.split(","))
            w = wl.make_device(args.config, dev, Nv=r_nv, Npdep=r_npdep, B=r_b)
        else:
            w = wl.make_device(args.config, dev)
        B = w.a_pw.shape[0]
        u_d = w.u
        phi_d = torch.view_as_real(w.phi).contiguous()
        if args.vec == "pw":
            a_d = torch.view_as_real(w.a_pw).contiguous()
        else:
            a_d = wl.device_a_real(w)
        w.a_pw = None
        w.u_pw = None
        w.phi = None
        torch.cuda.empty_cache()
        if not args.no_e2e:
            u_host, phi_host, a_host = pinned_copy(u_d), pinned_copy(phi_d), pinned_copy(a_d)
            out_host = torch.empty(a_d.shape, dtype=a_d.dtype, pin_memory=True)
    else:
        w = wl.make(args.config)
        B = w.a_pw.shape[0]
        a_np = w.a_real() if args.vec == "real" else np.ascontiguousarray(w.a_pw).view(np.float64)
        a_host = torch.from_numpy(np.ascontiguousarray(a_np)).pin_memory()
        u_host = torch.from_numpy(w.u).pin_memory()
        phi_host = torch.from_numpy(np.ascontiguousarray(w.phi).view(np.float64)).pin_memory()
        out_host = torch.empty_like(a_host).pin_memory()
        u_d, phi_d, a_d = u_host.to(dev), phi_host.to(dev), a_host.to(dev)
    n_pdep = phi_d.shape[0]
    Nv = w.Nv
    t_gen = time.perf_counter() - t_gen0
    out_d = torch.empty_like(a_d)
    flags = {"real": bse.BSE_TAU_REAL, "pw": bse.BSE_TAU_PW, "stream": bse.BSE_TAU_STREAM}[args.tau]
    flags |= bse.BSE_VEC_PW if args.vec == "pw" else bse.BSE_VEC_REAL
    if args.tau_f32:
        flags |= bse.BSE_TAU_F32
    stream = torch.cuda.current_stream().cuda_stream
    h = bse.bse_create([w.n] * 3, w.cell, w.ecut, Nv, u_d, n_pdep, phi_d, w.lam, w.eta, flags, stream)
    for kv in args.knob:
        key, val = kv.split("=")
        bse.bse_debug_set(h, key, int(val))
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev)     # > 126 MB L2

    def step(timed):
        flush.fill_(1)                                                  # L2 flush, outside the timed events
        e0, e1, e2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
        e0.record()
        bse.bse_build_tau(h)
        e1.record()
        bse.bse_apply_k1x(h, a_d, out_d, B)
        e2.record()
        if timed:
            e2.synchronize()
            return e0.elapsed_time(e1), e1.elapsed_time(e2), bse.bse_last_tau_fill_ms(h)
        return None

    for _ in range(args.warmup):
        step(False)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    bse.bse_profile_reset(h)
    t_build, t_apply, t_fill = [], [], []
    torch.cuda.profiler.start()          # `ncu --profile-from-start off` then lists the kernels of the timed steps only
    wall0 = time.perf_counter()
    for _ in range(args.steps):
        tb, ta, tf = step(True)
        t_build.append(tb)
        t_apply.append(ta)
        t_fill.append(tf)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    wall = time.perf_counter() - wall0
    torch.cuda.profiler.stop()
    clocks = sampler.stop() if rank == 0 else None
    prof_counts = bse.bse_profile_get(h)
    P = bse.bse_num_pairs(h)
    pairs_host = bse.bse_get_pairs(h)
    tb_ms, ta_ms, tf_ms = float(np.mean(t_build)), float(np.mean(t_apply)), float(np.mean(t_fill))
    tb_ms, ta_ms, tf_ms = max_over_ranks([tb_ms, ta_ms, tf_ms], dist if world > 1 else None, dev)
    # time spent producing the pair integrals: the whole build call, plus the in-apply fill in the streamed mode
    t_pairs_ms = tb_ms + (tf_ms if args.tau == "stream" else 0.0)
    launches = sum(prof_counts[s][1] * k for s, k in zip(bse.STAGES, bse.KERNELS_PER_STAGE)) / max(args.steps, 1)

    # ---- per-stage device times (CUDA events on the library's stream, one extra profiled pass per step) ----
    bse.bse_profile_enable(h, True)
    bse.bse_profile_reset(h)
    nprof = 1 if large else max(3, min(args.steps, 5))
    for _ in range(nprof):
        step(False)
    torch.cuda.synchronize()
    prof = bse.bse_profile_get(h)
    work = bse.bse_profile_model(h)      # algorithmic flops / HBM bytes of those launches by SURVEY 8(d)
    hand = bse.bse_profile_handoff(h)    # + the stick-plane hand-off Z (implementation traffic)
    bse.bse_profile_enable(h, False)
    npw_h = bse.bse_npw_half(h)
    model = {s_: dict(flops=work[s_][0] / nprof, bytes=work[s_][1] / nprof, handoff=hand[s_] / nprof, bound=BOUND[s_])
             for s_ in bse.STAGES}
    hbm_gbs, peak_src = load_peaks()
    dmma_tf, dfma_tf = bse.bse_probe_fp64_peak(stream)
    traffic = load_traffic(args.config, args.tau, args.vec)
    stages = {}
    for s in bse.STAGES:
        ms = prof[s][0] / nprof
        m = model[s]
        t_f = m["flops"] / (dmma_tf * 1e12 if m["bound"] == "tensor" else dfma_tf * 1e12)
        t_b = m["bytes"] / (hbm_gbs * 1e9)
        t_bh = (m["bytes"] + m["handoff"]) / (hbm_gbs * 1e9)
        stages[s] = {"ms": round(ms, 4), "launches_per_step": prof[s][1] / nprof * bse.KERNELS_PER_STAGE[bse.STAGES.index(s)],
                     "gflop": round(m["flops"] / 1e9, 3), "mbytes": round(m["bytes"] / 1e6, 2),
                     "mbytes_handoff": round(m["handoff"] / 1e6, 2),
                     "roof_ms": round(1e3 * max(t_f, t_b), 4),
                     "frac": round(max(t_f, t_b) * 1e3 / ms, 4) if ms > 0 else None,
                     "frac_with_handoff": round(max(t_f, t_bh) * 1e3 / ms, 4) if ms > 0 else None}
    top = max(bse.STAGES, key=lambda s: stages[s]["ms"])
    mt = model[top]
    ms_top = stages[top]["ms"]
    n_launch_top = max(1.0, prof[top][1] / nprof)
    t_f = mt["flops"] / (dmma_tf * 1e12)
    t_b = mt["bytes"] / (hbm_gbs * 1e9)
    if mt["bound"] == "tensor" and t_f >= t_b:
        roof = {"bound": "tensor", "achieved": mt["flops"] / (ms_top * 1e-3) / 1e12, "peak": dmma_tf, "unit": "TFLOP/s",
                "peak_source": "fp64 DMMA chain measured live by bse_probe_fp64_peak (bf16-derived alternative in DESIGN.md)"}
    else:
        roof = {"bound": "hbm", "achieved": mt["bytes"] / (ms_top * 1e-3) / 1e9, "peak": hbm_gbs, "unit": "GB/s",
                "peak_source": peak_src,
                "frac_with_handoff": (mt["bytes"] + mt["handoff"]) / (ms_top * 1e-3) / 1e9 / hbm_gbs}
    roof["frac"] = roof["achieved"] / roof["peak"]
    roof["kernel"] = top
    roof["launches_per_step"] = n_launch_top
    roof["ms_per_launch"] = ms_top / n_launch_top
    roof["traffic"] = traffic[top][0] if top in traffic else None
    roof["traffic_source"] = (traffic[top][1] + " (constant of that committed ncu --set full capture, not measured by this run)"
                              if top in traffic else None)
    roof["algorithmic_bytes_per_launch"] = mt["bytes"] / n_launch_top
    roof["algorithmic_bytes_are"] = "SURVEY 8(d): 8N per field (plane pass), 16 N_pw_h per field (stick pass), operands once (GEMM)"
    tot_f = sum(m["flops"] for m in model.values())
    tot_b = sum(m["bytes"] for m in model.values())
    tot_bh = tot_b + sum(m["handoff"] for m in model.values())
    pipe_roof_ms = 1e3 * max(tot_f / (dmma_tf * 1e12), tot_b / (hbm_gbs * 1e9))
    pipe_roof_h_ms = 1e3 * max(tot_f / (dmma_tf * 1e12), tot_bh / (hbm_gbs * 1e9))
    pipeline = {"roof_ms": round(pipe_roof_ms, 4), "measured_ms": round(tb_ms + ta_ms, 4),
                "frac": round(pipe_roof_ms / (tb_ms + ta_ms), 4), "frac_with_handoff": round(pipe_roof_h_ms / (tb_ms + ta_ms), 4),
                "gflop": round(tot_f / 1e9, 2), "mbytes": round(tot_b / 1e6, 1), "mbytes_with_handoff": round(tot_bh / 1e6, 1),
                "fp64_dmma_tflops": round(dmma_tf, 2), "fp64_dfma_tflops": round(dfma_tf, 2)}

    # ---- K1e (eq. 4) timed beside the step: not part of `value` ----
    k1e_ms = k1_ms = None
    if not args.no_k1e and (not large or args.vec == "pw"):
        reps = 1 if large else 10
        for _ in range(1 if large else 2):
            bse.bse_apply_k1e(h, a_d, out_d, B)
        torch.cuda.synchronize()
        ke0, ke1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ke0.record()
        for _ in range(reps):
            bse.bse_apply_k1e(h, a_d, out_d, B)
        ke1.record()
        ke1.synchronize()
        k1e_ms = ke0.elapsed_time(ke1) / reps
        for _ in range(1 if large else 2):
            bse.bse_apply_k1(h, a_d, out_d, B, 1.0, -1.0)     # eq. 1: K1e - K1d with one P_c
        torch.cuda.synchronize()
        ke0.record()
        for _ in range(reps):
            bse.bse_apply_k1(h, a_d, out_d, B, 1.0, -1.0)
        ke1.record()
        ke1.synchronize()
        k1_ms = ke0.elapsed_time(ke1) / reps

    bse.bse_destroy(h)

    # ---- end to end through the C ABI with host (pinned) buffers ----
    def run_e2e(flags_e, a_h, out_h, reps):
        hh = bse.bse_create([w.n] * 3, w.cell, w.ecut, Nv, u_host, n_pdep, phi_host, w.lam, w.eta,
                            flags_e | bse.BSE_PTR_HOST, stream)
        eb, ea, ef = [], [], []
        for i in range(1 + reps):
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            bse.bse_set_inputs_host(hh, u_host, phi_host)        # this step's orbitals and PDEP vectors: H2D, no realloc
            bse.bse_build_tau(hh)
            torch.cuda.synchronize()
            t1 = time.perf_counter()
            bse.bse_apply_k1x_host(hh, a_h, out_h, B)            # H2D a, apply, D2H out
            t2 = time.perf_counter()
            if i >= 1:
                eb.append(t1 - t0)
                ea.append(t2 - t1)
                ef.append(bse.bse_last_tau_fill_ms(hh) * 1e-3)
        bse.bse_destroy(hh)
        e_b, e_a, e_f = float(np.mean(eb)), float(np.mean(ea)), float(np.mean(ef))
        e_b, e_a, e_f = max_over_ranks([e_b, e_a, e_f], dist if world > 1 else None, dev)
        t_pairs = e_b + (e_f if args.tau == "stream" else 0.0)
        h2d = u_host.numel() * 8 + phi_host.numel() * 8 + a_h.numel() * 8
        d2h = out_h.numel() * 8 + 8
        return {"value": world * P / t_pairs, "unit": "pairs/s", "k1x_applies_per_s": world * B / e_a,
                "build_ms": 1e3 * e_b, "apply_ms": 1e3 * e_a, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                "what": "per step: bse_set_inputs_host (H2D of u, phi into the handle's buffers) + bse_build_tau, then "
                        "bse_apply_k1x_host (H2D a, apply, D2H out); pinned host buffers, host wall clock"
                        + ("; value = P / (build call + the tau fill inside the apply)" if args.tau == "stream" else "")}

    e2e = e2e_pw = None
    if not args.no_e2e:
        del out_d, a_d, u_d, phi_d                       # the host-pointer handle owns its own device copies
        if large:
            w.u = None
        torch.cuda.empty_cache()
        e2e = run_e2e(flags, a_host, out_host, 2 if large else 5)
        e2e["vec_layout"] = args.vec
        if not large and args.vec == "real":             # the paper's representation beside it: 16x fewer bytes
            a_pw_h = torch.from_numpy(np.ascontiguousarray(w.a_pw).view(np.float64)).pin_memory()
            out_pw_h = torch.empty_like(a_pw_h).pin_memory()
            e2e_pw = run_e2e((flags & ~bse.BSE_VEC_PW) | bse.BSE_VEC_PW, a_pw_h, out_pw_h, 5)
            e2e_pw["vec_layout"] = "pw"

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    cpu = None
    if not args.no_cpu_baseline and world == 1:
        if large:
            if u_host is not None:
                phi_np = phi_host.numpy().view(np.complex128)[..., 0]
                info = oracle_sample(lambda v: u_host[v].numpy(), w.n, w.L, w.ecut, Nv, phi_np, w.lam, pairs_host,
                                     n_pairs=2, n_rows=1, n_cols=24)
            else:                                         # --no-e2e: the inputs are still on the device
                phi_np = phi_d.cpu().numpy().view(np.complex128)[..., 0]
                info = oracle_sample(lambda v: u_d[v].cpu().numpy(), w.n, w.L, w.ecut, Nv, phi_np, w.lam, pairs_host,
                                     n_pairs=2, n_rows=1, n_cols=24)
        else:
            info = oracle_sample(lambda v: w.u[v], w.n, w.L, w.ecut, Nv, w.phi, w.lam, pairs_host,
                                 n_pairs=40, n_rows=8, n_cols=Nv, seconds_cap=15.0)
        if info:
            cpu = {"value": info["pairs_per_s"], "unit": "pairs/s", "cores": info["cores"], "kind": "oracle",
                   "sample": f"{info['sampled_entries']} entries of the eq.16 overlap matrix in long double ({info['per_entry_s']:.4f} s "
                             f"each, extrapolated to Nv^2 = {Nv * Nv}: {info['screen_s']:.0f} s) + tau for {info['sampled_pairs']} "
                             f"of {info['P']} surviving pairs ({info['per_pair_s']:.3f} s/pair, extrapolated to all pairs); the pairs "
                             f"are drawn from the list this run produced"}

    line = {
        "metric": METRIC, "value": world * P / (t_pairs_ms * 1e-3), "unit": "pairs/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": tb_ms + ta_ms, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": ("REDUCED for profiling, not a bench value: " if args.reduce else "")
                               + workload_string(args.config, w.n, Nv, n_pdep, npw_h, w.eta, P, B),
                   "tau_storage": args.tau + (" (kept as complex64: mixed-precision variant)" if args.tau_f32 else ""),
                   "vec_layout": args.vec, "parallelism": "replicas" if world > 1 else "1gpu",
                   "l2": "512 MB buffer written between timed steps (L2 flush); inputs also exceed L2",
                   "fallback": fallback},
        "value_is": "P / (bse_build_tau" + (" + the tau fill inside bse_apply_k1x, timed by the library's CUDA events" if args.tau == "stream" else "") + ")",
        "k1x_applies_per_s": world * B / (ta_ms * 1e-3),
        "k1e_applies_per_s": (world * B / (k1e_ms * 1e-3)) if k1e_ms else None, "k1e_ms": k1e_ms,
        "k1_combined_ms": k1_ms, "k1_combined_applies_per_s": (world * B / (k1_ms * 1e-3)) if k1_ms else None,
        "build_ms": tb_ms, "apply_ms": ta_ms, "tau_fill_ms": tf_ms, "pairs": P,
        "gpu_launches": int(round(launches * args.steps)), "gpu_launches_per_step": launches,
        "wall_s_timed_region": wall, "input_generation_s": t_gen,
        "clocks": clocks,
        "e2e": e2e, "e2e_pw_layout": e2e_pw,
        "roofline": roof, "pipeline_roofline": pipeline, "stages": stages, "cpu_baseline": cpu,
    }
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

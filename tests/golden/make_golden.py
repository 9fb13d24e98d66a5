"""Writes tests/golden/cfg1_golden.txt from the CPU oracle ONLY (never from the CUDA path).

The paper prints no worked numerical example for this path (PAPER.md has no tabulated tau or K1x value), so the stored
values are the oracle's evaluation of eq. 16, eq. 6/9/11 and eq. 5 on the seeded
config-1 workload.  They pin the oracle against silent changes (tests/test_golden.py, CPU) and give the CUDA path a
stored target that no GPU code produced (same file, -m gpu).

Run:  python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

from oracle import bse_oracle as orc                      # noqa: E402
from paper_2409_15116_b200 import workloads as wl         # noqa: E402


def main():
    w = wl.make(1)
    tab = orc.Tables(w.n, w.L, w.ecut)
    pairs, O = orc.screen_pairs(w.u, w.eta)
    tau = orc.build_tau(tab, w.u, w.phi, w.lam, pairs, want="r")
    a = w.a_real()
    out = orc.apply_k1x_real(tab, w.u, pairs, tau, a)
    out_pw = orc.apply_k1x_pw(tab, w.u, pairs, tau, w.a_pw)
    rng = np.random.default_rng(20240915)
    lines = ["# written by tests/golden/make_golden.py from oracle/bse_oracle.py only; config 1, seed 151161",
             "# eq. 16 (PAPER.md:135-140), eq. 6/9/11 (PAPER.md:71, :85-102), eq. 5 (PAPER.md:64-67)",
             f"npairs {len(pairs)}"]
    for v, x in [(0, 1), (2, 5), (3, 7), (6, 6)]:
        lines.append(f"O {v} {x} {float(O[v, x])!r}")
    for _ in range(12):
        p, r = int(rng.integers(len(pairs))), int(rng.integers(tab.N))
        lines.append(f"tau {p} {r} {float(tau[p, r])!r}")
    for p in (0, 17, 35):
        lines.append(f"tau_norm {p} {float(np.linalg.norm(tau[p]))!r}")
    for _ in range(12):
        b, v, r = int(rng.integers(a.shape[0])), int(rng.integers(w.Nv)), int(rng.integers(tab.N))
        lines.append(f"out {b} {v} {r} {float(out[b, v, r])!r}")
    lines.append(f"out_norm {float(np.linalg.norm(out))!r}")
    for _ in range(8):
        b, v, g = int(rng.integers(a.shape[0])), int(rng.integers(w.Nv)), int(rng.integers(tab.npw_h))
        lines.append(f"out_pw {b} {v} {g} {float(out_pw[b, v, g].real)!r} {float(out_pw[b, v, g].imag)!r}")
    open(os.path.join(HERE, "cfg1_golden.txt"), "w").write("\n".join(lines) + "\n")


if __name__ == "__main__":
    main()

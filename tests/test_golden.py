"""Stored oracle values (tests/golden/cfg1_golden.txt, written by tests/golden/make_golden.py from oracle/ only):
the oracle must still reproduce them (CPU), and the CUDA path must match them (GPU) to the parity bar."""
import os

import numpy as np
import pytest

from oracle import bse_oracle as orc
from paper_2409_15116_b200 import workloads as wl

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "cfg1_golden.txt")


def _load():
    rows = [ln.split() for ln in open(GOLD) if ln.strip() and not ln.startswith("#")]
    return rows


def _check(rows, npairs, O, tau, out, out_pw, tol):
    for r in rows:
        k = r[0]
        if k == "npairs":
            assert npairs == int(r[1])
        elif k == "O":
            assert abs(O[int(r[1]), int(r[2])] - float(r[3])) <= 1e-12
        elif k == "tau":
            ref = float(r[3])
            assert abs(tau[int(r[1]), int(r[2])] - ref) <= tol * max(abs(ref), np.abs(tau[int(r[1])]).max())
        elif k == "tau_norm":
            assert abs(np.linalg.norm(tau[int(r[1])]) - float(r[2])) <= tol * float(r[2])
        elif k == "out":
            ref = float(r[4])
            assert abs(out[int(r[1]), int(r[2]), int(r[3])] - ref) <= tol * np.abs(out).max()
        elif k == "out_norm":
            assert abs(np.linalg.norm(out) - float(r[1])) <= tol * float(r[1])
        elif k == "out_pw":
            ref = complex(float(r[4]), float(r[5]))
            assert abs(out_pw[int(r[1]), int(r[2]), int(r[3])] - ref) <= tol * np.abs(out_pw).max()


def test_oracle_reproduces_golden():
    w = wl.make(1)
    tab = orc.Tables(w.n, w.L, w.ecut)
    pairs, O = orc.screen_pairs(w.u, w.eta)
    tau = orc.build_tau(tab, w.u, w.phi, w.lam, pairs, want="r")
    out = orc.apply_k1x_real(tab, w.u, pairs, tau, w.a_real())
    out_pw = orc.apply_k1x_pw(tab, w.u, pairs, tau, w.a_pw)
    _check(_load(), len(pairs), O, tau, out, out_pw, 1e-13)


@pytest.mark.gpu
def test_cuda_path_matches_golden():
    torch = pytest.importorskip("torch")
    from paper_2409_15116_b200 import bse
    w = wl.make(1)
    dev = torch.device("cuda:0")
    u = torch.from_numpy(w.u).to(dev)
    phi = torch.from_numpy(np.ascontiguousarray(w.phi).view(np.float64)).to(dev)
    res = {}
    for vec in (bse.BSE_VEC_REAL, bse.BSE_VEC_PW):
        h = bse.bse_create([w.n] * 3, w.cell, w.ecut, w.Nv, u, w.phi.shape[0], phi, w.lam, w.eta, bse.BSE_TAU_PW | vec)
        try:
            bse.bse_build_tau(h)
            P = bse.bse_num_pairs(h)
            if vec == bse.BSE_VEC_REAL:
                res["O"] = bse.bse_get_overlap(h, w.Nv)
                t = torch.empty((P, w.N), dtype=torch.float64, device=dev)
                bse.bse_get_tau(h, 0, P, t, bse.BSE_TAU_REAL)
                res["tau"] = t.cpu().numpy()
                a = torch.from_numpy(np.ascontiguousarray(w.a_real())).to(dev)
            else:
                a = torch.from_numpy(np.ascontiguousarray(w.a_pw).view(np.float64)).to(dev)
            out = torch.empty_like(a)
            bse.bse_apply_k1x(h, a, out, w.a_pw.shape[0])
            torch.cuda.synchronize()
            if vec == bse.BSE_VEC_REAL:
                res["out"] = out.cpu().numpy()
            else:
                res["out_pw"] = out.cpu().numpy().view(np.complex128).reshape(w.a_pw.shape)
            res["P"] = P
        finally:
            bse.bse_destroy(h)
    _check(_load(), res["P"], res["O"], res["tau"], res["out"], res["out_pw"], 1e-10)

"""Pins of the JADE localisation oracle (oracle/jade_oracle.py; eq. 12-15).  CPU only."""
import math

import numpy as np

from oracle import jade_oracle as jo
from paper_2409_15116_b200 import workloads as wl


def _sym(rng, K, n):
    A = rng.normal(size=(K, n, n))
    return A + A.transpose(0, 2, 1)


def test_pj1_pair_angle_minimises_the_pair_off_diagonal_sum():
    rng = np.random.default_rng(1)
    for _ in range(20):
        app, aqq, apq = rng.normal(size=(3, 6))
        c, s = jo.givens_angle(app, aqq, apq)
        assert abs(c * c + s * s - 1.0) < 1e-15 and c >= math.cos(math.pi / 4) - 1e-15      # inner rotation |theta| <= pi/4

        def off(th):
            return float((((math.cos(2 * th)) * apq - 0.5 * math.sin(2 * th) * (app - aqq)) ** 2).sum())
        best = min(off(t) for t in np.linspace(-math.pi / 2, math.pi / 2, 20001))
        assert off(math.atan2(s, c)) <= best + 1e-9 * (1.0 + best)
        # and the formula for a'_pq used in off() is what the rotation does to an explicit 2 x 2 matrix
        R = np.array([[c, -s], [s, c]])
        for n in range(6):
            M = np.array([[app[n], apq[n]], [apq[n], aqq[n]]])
            th = math.atan2(s, c)
            assert abs((R.T @ M @ R)[0, 1] - (math.cos(2 * th) * apq[n] - 0.5 * math.sin(2 * th) * (app[n] - aqq[n]))) < 1e-13


def test_pj6_round_robin_rounds_are_disjoint_and_cover_every_pair_once():
    for Nv in (2, 3, 5, 8, 13, 64):
        rounds = jo.round_robin(Nv)
        seen = set()
        for pairs in rounds:
            idx = [i for pq in pairs for i in pq]
            assert len(idx) == len(set(idx))                       # disjoint: the rotations of a round are independent
            for pq in pairs:
                assert pq[0] < pq[1] < Nv and pq not in seen
                seen.add(pq)
        assert len(seen) == Nv * (Nv - 1) // 2


def test_pj2_commuting_matrices_are_diagonalised_exactly():
    rng = np.random.default_rng(2)
    for Nv, init in ((7, "identity"), (12, "eig"), (12, "identity")):
        Q, _ = np.linalg.qr(rng.normal(size=(Nv, Nv)))
        D = rng.normal(size=(6, Nv))
        A = np.array([Q @ np.diag(d) @ Q.T for d in D])
        V, Ad = jo.jade(A, init=init)
        assert np.abs(V.T @ V - np.eye(Nv)).max() < 1e-13
        assert jo.off_sum(Ad) < 1e-24 * sum((a * a).sum() for a in A)
        for n in range(6):
            assert np.abs(V.T @ A[n] @ V - Ad[n]).max() < 1e-12
        # V = Q up to the order and sign of its columns
        M = np.abs(Q.T @ V)
        assert np.abs(M.max(axis=0) - 1.0).max() < 1e-10 and np.abs(M.max(axis=1) - 1.0).max() < 1e-10


def test_pj3_one_matrix_reduces_to_the_symmetric_eigenproblem():
    rng = np.random.default_rng(3)
    A = _sym(rng, 1, 9)
    V, Ad = jo.jade(A, init="identity")                            # classic cyclic Jacobi in round-robin order
    assert np.abs(np.sort(np.diag(Ad[0])) - np.linalg.eigvalsh(A[0])).max() < 1e-12
    assert jo.off_sum(Ad) < 1e-24


def test_pj4_off_diagonal_sum_never_increases_and_spread_follows():
    cfg = wl.Config("jade", 10.0, 24, 8, 8, 8.0, 1.2, 0.8, 3.0, 0.0, 1, "random", seed=31)
    w = wl.make(cfg=cfg)
    rng = np.random.default_rng(4)
    Q, _ = np.linalg.qr(rng.normal(size=(w.Nv, w.Nv)))
    psi = Q @ w.u                                                  # delocalised orthonormal orbitals
    A, B = jo.position_matrices(psi, w.n, w.L, squares=True)
    assert np.abs(A - A.transpose(0, 2, 1)).max() < 1e-14
    # cos^2 + sin^2 = 1 and orthonormal orbitals: the B of one axis sum to the identity, so sum_n Tr B = 3 N_v
    assert abs(sum(np.trace(b) for b in B) - 3.0 * w.Nv) < 1e-10
    for init in ("identity", "eig"):
        hist = []
        V, Ad = jo.jade(A, init=init, history=hist)
        assert all(hist[i + 1] <= hist[i] * (1 + 1e-13) + 1e-18 for i in range(len(hist) - 1))
        Bd = np.array([V.T @ b @ V for b in B])
        # eq. 14 differs from the off-diagonal sum by a constant: sigma^2 = sum Tr B - sum ||A||_F^2 + off_sum
        const = sum(np.trace(b) for b in B) - sum((a * a).sum() for a in A)
        assert abs(jo.spread(Ad, Bd) - (const + jo.off_sum(Ad))) < 1e-10
        assert jo.spread(Ad, Bd) < jo.spread(A, B)
    # the localised orbitals are at least as compact as the ones the mixing started from
    U, loc = jo.localise(psi, w.n, w.L)
    A0, B0 = jo.position_matrices(w.u, w.n, w.L, squares=True)
    A1, B1 = jo.position_matrices(loc, w.n, w.L, squares=True)
    assert np.abs(U @ U.T - np.eye(w.Nv)).max() < 1e-13
    assert jo.spread(A1, B1) <= jo.spread(A0, B0) * (1 + 1e-9)
    assert jo.spread(A1, B1) < 0.8 * jo.spread(A, B)


def test_pj5_position_matrices_of_gaussians_closed_form():
    n, L, sig = 36, 12.0, 0.9
    ax = np.arange(n) * (L / n)
    centres = np.array([[3.1, 7.7, 5.2], [8.4, 2.3, 9.9]])
    dV = (L / n) ** 3
    u = []
    for c in centres:
        d = [(ax - c[k] + L / 2) % L - L / 2 for k in range(3)]
        g = np.exp(-0.5 * (d[0][:, None, None] ** 2 + d[1][None, :, None] ** 2 + d[2][None, None, :] ** 2) / sig ** 2)
        u.append((g / math.sqrt(dV * (g * g).sum())).ravel())
    A = jo.position_matrices(np.array(u), n, L)
    damp = math.exp(-(math.pi * sig / L) ** 2)
    for v, c in enumerate(centres):
        for axis in range(3):
            ang = 2.0 * math.pi * c[axis] / L
            assert abs(A[2 * axis, v, v] - damp * math.cos(ang)) < 1e-12
            assert abs(A[2 * axis + 1, v, v] - damp * math.sin(ang)) < 1e-12
            # the centre read back from the two diagonal entries
            x0 = (L / (2 * math.pi)) * math.atan2(A[2 * axis + 1, v, v], A[2 * axis, v, v]) % L
            assert abs(x0 - c[axis]) < 1e-10

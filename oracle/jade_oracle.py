"""CPU ORACLE for the localisation step that produces U (JADE; eq. 12-15).  TEST INFRASTRUCTURE ONLY.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference` leg may import this file.  It shares no
code with the CUDA path.  fp64 throughout, plain loops, each function citing its passage.

What the paper fixes:
  * six real symmetric matrices A^(n)_{vv'} = <psi_v| M^(n) |psi_v'>, M^(1..6) = cos / sin of (2 pi / L) x, y, z  (eq. 13, 15);
  * U minimises the spread sigma^2(U) = sum_n [ Tr(U^T B^(n) U) - sum_v |(U^T A^(n) U)_vv|^2 ]  (eq. 14), which is the same as
    minimising the off-diagonal elements of the rotated A^(n);
  * U is initialised with the eigenvectors of A^(1) (not the identity);
  * "a concurrent loop on 2x2 Givens rotations": the rotations of one such loop are independent (disjoint index pairs), are all
    determined from the matrices as they stand when the loop starts, and are applied together at its end.
What it leaves open (readings, listed in DESIGN.md):
  J1  the Givens angle of one pair: the closed form of the joint-diagonalisation algorithm of the paper's refs. 68-69 for real
      symmetric matrices - with h_n = (a^(n)_pp - a^(n)_qq, 2 a^(n)_pq) and G = sum_n h_n h_n^T, ton = G_11 - G_22,
      toff = 2 G_12, theta = atan2(toff, ton + sqrt(ton^2 + toff^2)) / 2 - which is the exact minimiser of the pair's
      off-diagonal sum sum_n (a'^(n)_pq)^2;
  J2  which disjoint pairs form one concurrent loop: the round-robin tournament ("circle method"): with m = N_v rounded up to
      even, round r = 0..m-2 holds the pairs (m-1, r) and ((r+k) mod (m-1), (r-k) mod (m-1)), k = 1..m/2-1; a pair that contains
      the padding index N_v (odd N_v) is skipped.  One sweep = m-1 rounds = every pair once;
  J3  stopping: sweeps until the largest |sin theta| of a sweep is below `tol` (default 1e-14) or `max_sweeps` is reached;
  J4  the orientation of eq. 12: psi~_v = sum_v' U_vv' psi_v' with U = V^T, V the accumulated column rotations (A' = V^T A V).

Pins (tests/test_jade_pins.py): PJ1 the one-pair angle minimises the pair's off-diagonal sum (brute-force scan over theta);
PJ2 six commuting matrices Q D_n Q^T are diagonalised exactly and V = Q up to order and sign; PJ3 one matrix: the result is
the symmetric eigen-decomposition (numpy.linalg.eigvalsh); PJ4 the off-diagonal sum never increases from round to round and
sigma^2 of eq. 14 (with B) decreases by the same amount; PJ5 A^(n) of shifted periodised Gaussians against the closed form
exp(-(pi sigma / L)^2) cos / sin (2 pi x0 / L) and the resulting centres; PJ6 round-robin rounds are disjoint and cover every
pair exactly once.  No function here is "parity unpinned".
"""
from __future__ import annotations

import math

import numpy as np


def position_matrices(u: np.ndarray, n: int, L: float, squares: bool = False):
    """A^(k)_{vw} = dV sum_r u_v(r) M^(k)(r) u_w(r), k = 0..5 for cos x, sin x, cos y, sin y, cos z, sin z of 2 pi r / L
    (eq. 13, 15; cubic cell, real orbitals u [Nv][n^3], r = (L/n) i, linear index (i1 n + i2) n + i3).
    squares=True returns B^(k) (the same with (M^(k))^2) as well."""
    Nv = u.shape[0]
    dV = L ** 3 / n ** 3
    ax = 2.0 * np.pi * np.arange(n) / n                      # (2 pi / L) * (L / n) i
    f = u.reshape(Nv, n, n, n)
    A = np.empty((6, Nv, Nv))
    B = np.empty((6, Nv, Nv)) if squares else None
    for axis in range(3):
        shape = [1, 1, 1, 1]
        shape[1 + axis] = n
        for k, fn in ((2 * axis, np.cos), (2 * axis + 1, np.sin)):
            m = fn(ax).reshape(shape)
            A[k] = dV * np.einsum("vijk,wijk->vw", f * m, f)
            if squares:
                B[k] = dV * np.einsum("vijk,wijk->vw", f * (m * m), f)
    return (A, B) if squares else A


def round_robin(Nv: int):
    """Reading J2: list of rounds, each a list of disjoint pairs (p < q); every pair p < q < Nv appears exactly once."""
    m = Nv + (Nv & 1)
    rounds = []
    for r in range(m - 1):
        pairs = [(m - 1, r)]
        for k in range(1, m // 2):
            pairs.append(((r + k) % (m - 1), (r - k) % (m - 1)))
        rounds.append(sorted((min(p, q), max(p, q)) for p, q in pairs if max(p, q) < Nv))
    return rounds


def givens_angle(app: np.ndarray, aqq: np.ndarray, apq: np.ndarray):
    """Reading J1: (c, s) of the rotation of the index pair (p, q) that minimises sum_n (a'^(n)_pq)^2, given the diagonal and
    off-diagonal entries of the pair in every matrix (arrays over n)."""
    h1 = app - aqq
    h2 = 2.0 * apq
    ton = float(np.dot(h1, h1) - np.dot(h2, h2))
    toff = float(2.0 * np.dot(h1, h2))
    theta = 0.5 * math.atan2(toff, ton + math.sqrt(ton * ton + toff * toff))
    return math.cos(theta), math.sin(theta)


def off_sum(A: np.ndarray) -> float:
    """sum_n sum_{v != w} (A^(n)_vw)^2 - what eq. 14 minimises up to a constant."""
    return float(sum(((a - np.diag(np.diag(a))) ** 2).sum() for a in A))


def spread(A: np.ndarray, B: np.ndarray) -> float:
    """sigma^2 of eq. 14 for matrices that already carry the rotation: sum_n [ Tr B^(n) - sum_v (A^(n)_vv)^2 ]."""
    return float(sum(np.trace(b) - (np.diag(a) ** 2).sum() for a, b in zip(A, B)))


def jade(A_in: np.ndarray, init: str = "eig", tol: float = 1e-14, max_sweeps: int = 60, history: list | None = None):
    """Joint approximate diagonalisation of the real symmetric matrices A_in [K][Nv][Nv].
    Returns (V, A'): V orthogonal with A'^(n) = V^T A^(n) V as diagonal as possible; the U of eq. 12 is V^T (J4).
    init = "eig": V starts from the eigenvectors of A^(1) (the paper's choice); "identity": the original algorithm.
    history (optional list) receives off_sum after every round."""
    A = np.array(A_in, dtype=np.float64, copy=True)
    K, Nv, _ = A.shape
    if init == "eig":
        _, V = np.linalg.eigh(A[0])                          # library eigensolver as one step
        for n in range(K):
            A[n] = V.T @ A[n] @ V
    else:
        V = np.eye(Nv)
    rounds = round_robin(Nv)
    for _sweep in range(max_sweeps):
        smax = 0.0
        for pairs in rounds:
            # the concurrent loop: every angle from the matrices as they stand now ...
            cs = [givens_angle(A[:, p, p], A[:, q, q], A[:, p, q]) for (p, q) in pairs]
            # ... then all rotations applied together: A <- R^T A R, V <- V R, R = product of the disjoint rotations
            for (p, q), (c, s) in zip(pairs, cs):
                smax = max(smax, abs(s))
                for n in range(K):
                    colp, colq = A[n][:, p].copy(), A[n][:, q].copy()
                    A[n][:, p] = c * colp + s * colq
                    A[n][:, q] = -s * colp + c * colq
                vp, vq = V[:, p].copy(), V[:, q].copy()
                V[:, p] = c * vp + s * vq
                V[:, q] = -s * vp + c * vq
            for (p, q), (c, s) in zip(pairs, cs):
                for n in range(K):
                    rowp, rowq = A[n][p, :].copy(), A[n][q, :].copy()
                    A[n][p, :] = c * rowp + s * rowq
                    A[n][q, :] = -s * rowp + c * rowq
            if history is not None:
                history.append(off_sum(A))
        if smax < tol:
            break
    return V, A


def localise(u: np.ndarray, n: int, L: float, **kw):
    """eq. 12: psi~ = U psi with U = V^T from jade() on the six position matrices of u.  Returns (U, psi~)."""
    A = position_matrices(u, n, L)
    V, _ = jade(A, **kw)
    U = V.T.copy()
    return U, U @ u

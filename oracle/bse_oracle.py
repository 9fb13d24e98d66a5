"""CPU ORACLE for the screened-exchange hot path (tau build + K1x apply).  TEST INFRASTRUCTURE ONLY.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference` leg may
import this file.  It shares no code with the CUDA path (`paper_2409_15116_b200/csrc/`, `bse.py`):
own FFT, own sphere tables, own loops.  fp64 / complex128 throughout.  Plain and slow on purpose:
every function is the paper's definition written out, in the paper's order, with the passage cited.

What the path computes is *defined* (not approximated) by PAPER.md eq. 5, 6, 9, 10, 11, 16 once the
conventions below are fixed, so this oracle is "the definition evaluated slowly".

Conventions / readings (S1..S20):
  * Gamma point, real orbitals, no spin.  psi_v psi*_v' = u_v u_v'.
  * Hartree atomic units.  v_c(G) = 4 pi / |G|^2 (v_c = 1/|r-r'|), v_c(0) := 0.
  * f(r) = sum_G f(G) e^{+iG.r};  f(G) = (1/N) sum_r f(r) e^{-iG.r}.
  * everything in reciprocal space is truncated to the sphere S: |G|^2/2 <= ecut.
  * eq. 11 with Xi = 0 and phi normalised sum_S |phi_a(G)|^2 = 1: the 1/Omega is absorbed, the
    operator acts on coefficients as (chi g)(G) = sum_a phi_a(G) f_a sum_G' conj(phi_a(G')) g(G').
  * K1x := + P_c sum_v' tau_vv' a_v'   (eq. 5, no prefactor; the minus sign of eq. 1 is the caller's).

Pins (tests/test_oracle_pins.py, all `-m "not gpu"`): P1 brute-force DFT, P2 Parseval, P3 analytic
Gaussian Hartree potential at lambda = 0, P4 dense real-space operator on a tiny grid, P5 rank-1
closed form, P6 complete-basis closed form, P7 W symmetric, P8 sum_r tau = 0, P9 P_c idempotent,
P10 K symmetric, P11 analytic Gaussian overlap for eq. 16, P12 PW layout == gather(FFT(REAL)), P18 the single-precision
store: every component representable in binary32 and within half an ulp (2^-24 relative) of the double value.
No function here is "parity unpinned".
"""
from __future__ import annotations

import math

import numpy as np


# =============================================================================== own FFT
def _fft_last(x: np.ndarray, sign: int) -> np.ndarray:
    """Unnormalised DFT along the last axis: X[k] = sum_j x[j] exp(sign 2 pi i j k / n).

    Naive recursive decimation-in-time, radix 2, 3 or 5 (whichever divides n first); a length with
    no such factor is done by the O(n^2) definition.  Textbook Cooley-Tukey:
        X[k] = sum_{q<r} w_n^{qk} * X_q[k mod m],   X_q = DFT_m of x[q::r],  m = n / r.
    """
    n = x.shape[-1]
    if n == 1:
        return x.astype(np.complex128)
    r = 0
    for cand in (2, 3, 5):
        if n % cand == 0:
            r = cand
            break
    k = np.arange(n)
    if r == 0:
        W = np.exp(sign * 2j * np.pi * np.outer(k, k) / n)      # W[k][j]
        return np.einsum("kj,...j->...k", W, x.astype(np.complex128))
    m = n // r
    out = np.zeros(x.shape, dtype=np.complex128)
    for q in range(r):
        Xq = _fft_last(x[..., q::r], sign)                       # [..., m]
        out += np.exp(sign * 2j * np.pi * q * k / n) * Xq[..., k % m]
    return out


def fft3(f: np.ndarray, sign: int) -> np.ndarray:
    """Unnormalised 3-D DFT of f[n1][n2][n3] with kernel exp(sign i G.r), one axis at a time."""
    g = np.asarray(f, dtype=np.complex128)
    for ax in range(3):
        g = np.moveaxis(_fft_last(np.ascontiguousarray(np.moveaxis(g, ax, -1)), sign), -1, ax)
    return g


# ========================================================================== O0: tables
class Tables:
    """Sphere S, half sphere H, |G|, v_c^{1/2}(G); cubic cell of edge L, grid n^3."""

    def __init__(self, n: int, L: float, ecut: float):
        self.n, self.L = n, L
        self.N = n ** 3
        self.Omega = L ** 3
        self.dV = self.Omega / self.N
        msq_max = int(math.floor(2.0 * ecut * (L / (2.0 * math.pi)) ** 2 * (1.0 + 1e-12)))
        S = []
        H = []
        R = int(math.isqrt(msq_max))
        if 2 * R >= n:
            raise ValueError("sphere does not fit in the grid")
        for m1 in range(-R, R + 1):
            for m2 in range(-R, R + 1):
                for m3 in range(-R, R + 1):
                    if m1 * m1 + m2 * m2 + m3 * m3 <= msq_max:
                        S.append((m1, m2, m3))
                        if m3 > 0 or (m3 == 0 and m2 > 0) or (m3 == 0 and m2 == 0 and m1 >= 0):
                            H.append((m1, m2, m3))
        H.sort(key=lambda m: ((m[0] % n) * n + (m[1] % n)) * n + (m[2] % n))
        self.S = np.array(S, dtype=np.int64)                    # [Npw][3]
        self.H = np.array(H, dtype=np.int64)                    # [Npw_h][3]
        self.npw, self.npw_h = len(S), len(H)
        hidx = {m: i for i, m in enumerate(H)}
        # for every G in S: index of +G or of -G in H, and whether to conjugate
        self.S_h = np.empty(self.npw, dtype=np.int64)
        self.S_conj = np.zeros(self.npw, dtype=bool)
        for i, m in enumerate(S):
            if m in hidx:
                self.S_h[i] = hidx[m]
            else:
                self.S_h[i] = hidx[(-m[0], -m[1], -m[2])]
                self.S_conj[i] = True
        self.S_grid = (self.S[:, 0] % n, self.S[:, 1] % n, self.S[:, 2] % n)
        g2 = (2.0 * np.pi / L) ** 2 * (self.S ** 2).sum(1).astype(np.float64)
        self.vc12 = np.zeros(self.npw)                          # sqrt(4 pi)/|G|, 0 at G = 0  (S2, S4)
        nz = g2 > 0
        self.vc12[nz] = np.sqrt(4.0 * np.pi) / np.sqrt(g2[nz])

    def expand_H_to_S(self, cH: np.ndarray) -> np.ndarray:
        """[..., Npw_h] coefficients on H -> [..., Npw] on the full sphere, c(-G) = conj c(G)."""
        c = cH[..., self.S_h]
        return np.where(self.S_conj, np.conj(c), c)

    def to_G(self, f_real: np.ndarray) -> np.ndarray:
        """f(G) = (1/N) sum_r f(r) e^{-iG.r}, read on S only (components outside S discarded)."""
        F = fft3(f_real.reshape(self.n, self.n, self.n), -1) / self.N
        return F[self.S_grid]

    def to_r(self, cS: np.ndarray) -> np.ndarray:
        """f(r) = sum_{G in S} c(G) e^{+iG.r}; result must be real for Hermitian c."""
        F = np.zeros((self.n, self.n, self.n), dtype=np.complex128)
        F[self.S_grid] = cS
        f = fft3(F, +1)
        assert np.abs(f.imag).max() <= 1e-9 * max(np.abs(f.real).max(), 1e-300), "non-Hermitian input"
        return f.real.ravel().copy()


# ============================================================= O1: overlap screen, eq. 16
def overlap_matrix(u: np.ndarray) -> np.ndarray:
    """O_vw = sum_r u_v^2 u_w^2 / sqrt(sum_r u_v^4 sum_r u_w^4)   (eq. 16).
    dV cancels.  Accumulated in extended precision (long double) row by row."""
    Nv = u.shape[0]
    q = (u.astype(np.float64) ** 2).astype(np.longdouble)
    M = np.empty((Nv, Nv), dtype=np.longdouble)
    for v in range(Nv):
        M[v] = (q * q[v]).sum(axis=1)
    d = np.sqrt(np.diag(M))
    return (M / (d[:, None] * d[None, :]))


def overlap_rows(get_u, Nv: int, rows):
    """Rows of O (eq. 16) without holding all of u in extended precision: O[v, :] for v in `rows`.
    get_u(w) returns orbital w as a float64 [N] array (so the caller may stream it from anywhere).
    Same sums as overlap_matrix, one (v, w) pair at a time.  Used for the sampled screen check at the full size of
    configs 4-5, where the N_v x N_v x N long-double SYRK of overlap_matrix would take hours."""
    qrows = {v: (get_u(v) ** 2).astype(np.longdouble) for v in rows}
    M = np.empty((len(rows), Nv), dtype=np.longdouble)
    d = np.empty(Nv, dtype=np.longdouble)
    for w in range(Nv):
        qw = (get_u(w) ** 2).astype(np.longdouble)
        d[w] = (qw * qw).sum()
        for i, v in enumerate(rows):
            M[i, w] = (qrows[v] * qw).sum()
    dd = np.sqrt(d)
    return np.asarray(M / (dd[list(rows)][:, None] * dd[None, :]), dtype=np.float64)


def screen_pairs(u: np.ndarray, eta: float):
    """Surviving unordered pairs v <= w with O_vw >= eta, lexicographic (tau := 0 if O is
    *smaller than* the threshold; diagonal always kept).  Returns (pairs [P][2] int32, O float64)."""
    O = overlap_matrix(u)
    Nv = u.shape[0]
    pairs = [(v, w) for v in range(Nv) for w in range(v, Nv) if (v == w or O[v, w] >= eta)]
    return np.array(pairs, dtype=np.int32).reshape(-1, 2), np.asarray(O, dtype=np.float64)


def screen_margin(O: np.ndarray, eta: float) -> float:
    """min_{v<w} |O_vw - eta| / eta  (guard band S10); inf when eta = 0."""
    if eta <= 0:
        return math.inf
    iu = np.triu_indices(O.shape[0], 1)
    return float(np.min(np.abs(O[iu] - eta)) / eta)


# ===================================================== O2..O7: one screened pair integral
def tau_G(tab: Tables, uv: np.ndarray, uw: np.ndarray, phiS: np.ndarray, lam: np.ndarray) -> np.ndarray:
    """tau_vw(G) on the full sphere S (eq. 6 via eq. 9-11).
    phiS: [Npdep][Npw] PDEP vectors on the full sphere."""
    rho = uv * uw                                   # O2: psi_v psi*_v' (real orbitals)
    rhoG = tab.to_G(rho)                            # O3
    x = tab.vc12 * rhoG                             # O4: v_c^{1/2} rho, x(0) = 0
    f = lam / (1.0 - lam)                           # eq. 11: lambda_a / (1 - lambda_a)
    c = np.conj(phiS) @ x                           # O5: <phi_a | x>, full-sphere sum
    y = (f * c) @ phiS                              # O6: sum_a phi_a f_a c_a
    return tab.vc12 * (x + y)                       # O7: v_c rho + v_c^{1/2} chibar v_c^{1/2} rho


def tau_G_f32(tab: Tables, uv, uw, phiS, lam) -> np.ndarray:
    """Mixed-precision variant of the tau build ("experimenting with the use of single precision"; reading:
    the pair integral is evaluated in fp64 and KEPT in single precision): tau_G rounded once, component by component, to
    IEEE binary32 (round to nearest even), returned widened back to complex128."""
    return tau_G(tab, uv, uw, phiS, lam).astype(np.complex64).astype(np.complex128)


def tau_r(tab: Tables, uv, uw, phiS, lam) -> np.ndarray:
    """tau_vw(r) = sum_{G in S} tau_vw(G) e^{iG.r}, real [N]."""
    return tab.to_r(tau_G(tab, uv, uw, phiS, lam))


def S_to_H(tab: Tables, cS: np.ndarray) -> np.ndarray:
    """Pick the H entries of a full-sphere coefficient vector."""
    out = np.empty(tab.npw_h, dtype=np.complex128)
    sel = ~tab.S_conj
    out[tab.S_h[sel]] = cS[sel]
    return out


def build_tau(tab: Tables, u, phiH, lam, pairs, want="r"):
    """All listed pairs.  want = "r": [P][N] real;  "G": [P][Npw_h] complex on H."""
    phiS = tab.expand_H_to_S(phiH)
    out = []
    for (v, w) in pairs:
        tG = tau_G(tab, u[v], u[w], phiS, lam)
        out.append(tab.to_r(tG) if want == "r" else S_to_H(tab, tG))
    return np.array(out)


# ===================================================================== O8: K1x, eq. 5
def p_c_real(tab: Tables, u: np.ndarray, x: np.ndarray) -> np.ndarray:
    """P_c x = x - sum_w u_w <u_w|x>, <f|g> = dV sum_r f g."""
    ov = tab.dV * (u @ x)                           # [w]
    return x - ov @ u


def apply_k1x_real(tab: Tables, u, pairs, tau, a) -> np.ndarray:
    """out[b,v,:] = P_c sum_{w : (v,w) or (w,v) kept} tau_vw(r) a[b,w,r]  (eq. 5).
    tau: [P][N] real in the order of `pairs`; a: [B][Nv][N] real."""
    B, Nv, N = a.shape
    acc = np.zeros((B, Nv, N))
    for p, (v, w) in enumerate(pairs):
        for b in range(B):
            acc[b, v] += tau[p] * a[b, w]
            if w != v:
                acc[b, w] += tau[p] * a[b, v]       # tau_wv = tau_vw (real orbitals, symmetric W)
    out = np.empty_like(acc)
    for b in range(B):
        for v in range(Nv):
            out[b, v] = p_c_real(tab, u, acc[b, v])
    return out


def apply_k1x_pw(tab: Tables, u, pairs, tau, a_pw) -> np.ndarray:
    """PW layout (A_s "of length N_pw"): a_pw [B][Nv][Npw_h] on H.
    a(r) from coefficients; accumulate in real space; acc(G) = gather_H(FFT(acc)/N);
    P_c in PW with <f|g> = Omega sum_S conj f(G) g(G)."""
    B, Nv, _ = a_pw.shape
    a = np.empty((B, Nv, tab.N))
    for b in range(B):
        for v in range(Nv):
            a[b, v] = tab.to_r(tab.expand_H_to_S(a_pw[b, v]))
    acc = np.zeros((B, Nv, tab.N))
    for p, (v, w) in enumerate(pairs):
        for b in range(B):
            acc[b, v] += tau[p] * a[b, w]
            if w != v:
                acc[b, w] += tau[p] * a[b, v]
    uS = np.array([tab.to_G(u[w]) for w in range(Nv)])          # [Nv][Npw]
    out = np.empty((B, Nv, tab.npw_h), dtype=np.complex128)
    for b in range(B):
        for v in range(Nv):
            out[b, v] = S_to_H(tab, p_c_pw(tab, uS, tab.to_G(acc[b, v])))
    return out


def p_c_pw(tab: Tables, uS: np.ndarray, accS: np.ndarray) -> np.ndarray:
    """P_c in PW on the full sphere: x - sum_w u_w <u_w|x>, <f|g> = Omega sum_{G in S} conj f(G) g(G).
    uS: [Nv][Npw] orbital coefficients on S; accS: [Npw]."""
    ov = tab.Omega * (np.conj(uS) @ accS)                        # <u_w|acc>, real up to rounding
    return accS - ov.real @ uS


# ===================================================================== K1e, eq. 4 (the bare exchange-like Hartree term)
def hartree_r(tab: Tables, n_r: np.ndarray) -> np.ndarray:
    """v_H(r) = int v_c(r, r') n(r') dr' = sum_{G in S} v_c(G) n(G) e^{iG.r},  v_c(G) = 4 pi / |G|^2 = vc12^2, v_c(0) := 0
    (readings S2, S4, S5: the density is truncated to S like every reciprocal-space object)."""
    return tab.to_r(tab.vc12 * tab.vc12 * tab.to_G(n_r))


def apply_k1e_real(tab: Tables, u: np.ndarray, a: np.ndarray) -> np.ndarray:
    """K1e a = { 2 P_c [ psi_v(r) * int v_c(r, r') sum_v' psi_v'(r') a_v'(r') dr' ] : v }   (eq. 4; real orbitals).
    a: [B][Nv][N] real; returns [B][Nv][N]."""
    B, Nv, N = a.shape
    out = np.empty_like(a)
    for b in range(B):
        n_r = np.zeros(N)
        for v in range(Nv):
            n_r += u[v] * a[b, v]                    # sum_v' psi*_v' a_v'
        vH = hartree_r(tab, n_r)
        for v in range(Nv):
            out[b, v] = p_c_real(tab, u, 2.0 * u[v] * vH)
    return out


def apply_k1e_pw(tab: Tables, u: np.ndarray, a_pw: np.ndarray) -> np.ndarray:
    """PW layout of K1e: a_pw [B][Nv][Npw_h] on H; psi_v * v_H is truncated to S before P_c (S15)."""
    B, Nv, _ = a_pw.shape
    uS = np.array([tab.to_G(u[w]) for w in range(Nv)])
    out = np.empty((B, Nv, tab.npw_h), dtype=np.complex128)
    for b in range(B):
        n_r = np.zeros(tab.N)
        for v in range(Nv):
            n_r += u[v] * tab.to_r(tab.expand_H_to_S(a_pw[b, v]))
        vH = hartree_r(tab, n_r)
        for v in range(Nv):
            out[b, v] = S_to_H(tab, p_c_pw(tab, uS, tab.to_G(2.0 * u[v] * vH)))
    return out


# ===================================================== KS <-> localised representation, eq. 12
def rotate(U: np.ndarray, x: np.ndarray, transpose: bool = False) -> np.ndarray:
    """y[b, v, :] = sum_v' U[v, v'] x[b, v', :]  (eq. 12 applied to the orbitals of A_s), or with U^T (the way back;
    U is real orthogonal at the Gamma point).  x: [B][Nv][K], any K (real-space points or PW coefficients)."""
    M = U.T if transpose else U
    out = np.zeros_like(x)
    for b in range(x.shape[0]):
        for v in range(M.shape[0]):
            for w in range(M.shape[1]):
                out[b, v] += M[v, w] * x[b, w]
    return out

"""Pins of the CPU oracle against things that are NOT the oracle.

Each pin is a closed form, an invariant, a brute-force definition or a dense-matrix construction;
none calls the oracle to produce its own expected value.  All run without a GPU.
"""
import math

import numpy as np
import pytest

from oracle import bse_oracle as orc
from paper_2409_15116_b200 import workloads as wl

TWO_PI = 2.0 * math.pi


def _small_cfg(n=12, L=9.0, ecut=3.0, Nv=4, Npdep=6, B=2, sigma=1.3, eta=0.0, seed=7):
    return wl.Config("tiny", L, n, Nv, Npdep, ecut, sigma, 0.8, 3.0, eta, B, "random", seed=seed)


# ------------------------------------------------------------------ P1: FFT vs brute-force DFT
@pytest.mark.parametrize("shape", [(4, 4, 4), (6, 6, 6), (10, 10, 10), (12, 12, 12), (15, 15, 15), (7, 6, 5)])
@pytest.mark.parametrize("sign", [-1, +1])
def test_P1_fft_vs_bruteforce_dft(shape, sign):
    rng = np.random.default_rng(1)
    f = rng.normal(size=shape) + 1j * rng.normal(size=shape)
    n1, n2, n3 = shape
    # brute force: X[m] = sum_r f[r] exp(sign 2 pi i (m1 r1/n1 + m2 r2/n2 + m3 r3/n3)), O(N^2)
    r1, r2, r3 = np.meshgrid(np.arange(n1), np.arange(n2), np.arange(n3), indexing="ij")
    ref = np.empty(shape, dtype=np.complex128)
    for m1 in range(n1):
        for m2 in range(n2):
            for m3 in range(n3):
                ph = sign * TWO_PI * (m1 * r1 / n1 + m2 * r2 / n2 + m3 * r3 / n3)
                ref[m1, m2, m3] = np.sum(f * np.exp(1j * ph))
    got = orc.fft3(f, sign)
    assert np.linalg.norm(got - ref) <= 1e-12 * np.linalg.norm(ref)


def test_P1b_fft_single_mode_and_roundtrip():
    # a single plane wave e^{+iG.r} must land on exactly one coefficient
    n = 12
    i = np.arange(n)
    m = (2, -3, 5)
    f = np.exp(1j * TWO_PI * (m[0] * i[:, None, None] + m[1] * i[None, :, None] + m[2] * i[None, None, :]) / n)
    F = orc.fft3(f, -1) / n ** 3
    want = np.zeros((n, n, n), complex)
    want[m[0] % n, m[1] % n, m[2] % n] = 1.0
    assert np.abs(F - want).max() < 1e-13
    g = orc.fft3(F, +1)
    assert np.abs(g - f).max() < 1e-12


# ------------------------------------------------------------------ tables / H ordering
def test_tables_half_sphere_matches_generator_rule():
    for (n, L, ecut) in [(12, 9.0, 3.0), (24, 10.0, 8.0)]:
        tab = orc.Tables(n, L, ecut)
        mill = wl.half_sphere(n, L, ecut)
        assert tab.npw_h == mill.shape[0] and tab.npw == 2 * tab.npw_h - 1
        assert np.array_equal(tab.H, mill.astype(np.int64))
    tab = orc.Tables(24, 10.0, 8.0)
    assert (tab.npw, tab.npw_h) == (1045, 523)          # SURVEY Table S, config 1


# ------------------------------------------------------------------ P2: Parseval
def test_P2_parseval_band_limited():
    w = wl.make(cfg=_small_cfg())
    tab = orc.Tables(w.n, w.L, w.ecut)
    for v in range(w.Nv):
        c = tab.to_G(w.u[v])
        lhs = tab.dV * np.sum(w.u[v] ** 2)
        rhs = tab.Omega * np.sum(np.abs(c) ** 2)
        assert abs(lhs - rhs) < 1e-12 and abs(lhs - 1.0) < 1e-12
        # and the round trip through S is exact because u is band-limited
        assert np.abs(tab.to_r(c) - w.u[v]).max() < 1e-12


# ------------------------------------------------------------------ P3: lambda=0 -> analytic Hartree
def test_P3_bare_limit_is_analytic_gaussian_hartree():
    n, L, ecut, sig = 32, 16.0, 6.0, 1.3
    tab = orc.Tables(n, L, ecut)
    R1 = np.array([7.3, 8.1, 7.9])
    R2 = np.array([8.6, 7.4, 8.8])
    ax = np.arange(n) * (L / n)

    def gauss(R):
        e = [np.exp(-0.5 * ((ax - R[k]) / sig) ** 2) for k in range(3)]   # no images needed: L >= 12 sigma
        return (e[0][:, None, None] * e[1][None, :, None] * e[2][None, None, :]).ravel()

    g1, g2 = gauss(R1), gauss(R2)
    phiS = np.zeros((1, tab.npw), complex)
    got = orc.tau_G(tab, g1, g2, phiS, np.zeros(1))
    # closed form: g1 g2 = A exp(-|r-Rc|^2/sig^2), A = exp(-|R1-R2|^2/(4 sig^2)), Rc = midpoint
    # rho(G) = (A/Omega) (pi sig^2)^{3/2} exp(-G^2 sig^2/4) exp(-iG.Rc);  tau(G) = 4 pi rho(G)/G^2
    A = math.exp(-np.sum((R1 - R2) ** 2) / (4 * sig ** 2))
    Rc = 0.5 * (R1 + R2)
    G = (TWO_PI / L) * tab.S.astype(float)
    G2 = (G ** 2).sum(1)
    rho = (A / tab.Omega) * (math.pi * sig ** 2) ** 1.5 * np.exp(-G2 * sig ** 2 / 4) * np.exp(-1j * G @ Rc)
    want = np.zeros(tab.npw, complex)
    nz = G2 > 0
    want[nz] = 4 * math.pi * rho[nz] / G2[nz]
    assert np.linalg.norm(got - want) <= 1e-10 * np.linalg.norm(want)
    assert got[~nz] == 0


# ------------------------------------------------------------------ P4: dense operator, tiny grid
def test_P4_dense_real_space_operator_tiny_grid():
    cfg = _small_cfg(n=6, L=5.0, ecut=2.5, Nv=3, Npdep=4, B=2, sigma=1.1)
    w = wl.make(cfg=cfg)
    n, N, L = w.n, w.N, w.L
    Omega, dV = L ** 3, L ** 3 / N
    # full-sphere list built here, independently: all m with |m|^2 <= msq_max
    mx = wl.msq_max(L, w.ecut)
    rng_m = range(-n // 2, n // 2)
    S = [(a, b, c) for a in rng_m for b in rng_m for c in rng_m if a * a + b * b + c * c <= mx]
    idx = {tuple(m): i for i, m in enumerate(w.mill.tolist())}
    r = np.stack(np.meshgrid(*(np.arange(n),) * 3, indexing="ij"), -1).reshape(-1, 3)
    E = np.array([np.exp(1j * TWO_PI * (r @ np.array(m)) / n) for m in S])       # E[G][r] = e^{iG.r}
    vc = np.array([0.0 if m == (0, 0, 0) else 4 * math.pi / ((TWO_PI / L) ** 2 * (m[0] ** 2 + m[1] ** 2 + m[2] ** 2)) for m in S])
    phi_full = np.array([[w.phi[a, idx[m]] if m in idx else np.conj(w.phi[a, idx[(-m[0], -m[1], -m[2])]]) for m in S]
                         for a in range(w.phi.shape[0])])
    f = w.lam / (1 - w.lam)
    # W(G,G') = vc^{1/2} (delta + sum_a phi_a f_a phi_a^*) vc^{1/2};  W(r,r') = (1/Omega) sum E W E^*
    Wg = np.diag(vc) + (np.sqrt(vc)[:, None] * (phi_full.T * f) @ np.conj(phi_full)) * np.sqrt(vc)[None, :]
    Wr = (E.T @ Wg @ np.conj(E)) / Omega
    assert np.abs(Wr.imag).max() < 1e-12 and np.abs(Wr - Wr.T).max() < 1e-12
    Wr = Wr.real
    tab = orc.Tables(n, L, w.ecut)
    pairs, _ = orc.screen_pairs(w.u, 0.0)
    tau = orc.build_tau(tab, w.u, w.phi, w.lam, pairs, want="r")
    for p, (v, x) in enumerate(pairs):
        want = dV * (Wr @ (w.u[v] * w.u[x]))                    # tau(r) = int W(r,r') rho(r') dr'  (eq. 6)
        assert np.linalg.norm(tau[p] - want) <= 1e-11 * np.linalg.norm(want)
    # K1x by four nested loops with the dense operator
    a = w.a_real()
    got = orc.apply_k1x_real(tab, w.u, pairs, tau, a)
    Pc = np.eye(N) - dV * (w.u.T @ w.u)
    for b in range(a.shape[0]):
        for v in range(w.Nv):
            acc = np.zeros(N)
            for x in range(w.Nv):
                acc += dV * (Wr @ (w.u[v] * w.u[x])) * a[b, x]
            want = Pc @ acc
            assert np.linalg.norm(got[b, v] - want) <= 1e-11 * np.linalg.norm(want)


# ------------------------------------------------------------------ P5 / P6: closed forms
def test_P5_rank1_closed_form():
    w = wl.make(cfg=_small_cfg(Npdep=1))
    tab = orc.Tables(w.n, w.L, w.ecut)
    none = np.zeros((1, tab.npw), complex)
    bare = orc.tau_G(tab, w.u[0], w.u[1], none, np.zeros(1))
    x = np.zeros(tab.npw)
    nz = tab.vc12 > 0
    xS = np.zeros(tab.npw, complex)
    xS[nz] = bare[nz] / tab.vc12[nz]                             # x = vc^{1/2} rho
    phi1 = (xS / np.linalg.norm(xS))[None, :]
    lam = np.array([-0.7])
    got = orc.tau_G(tab, w.u[0], w.u[1], phi1, lam)
    assert np.linalg.norm(got - bare / (1 - lam[0])) <= 1e-12 * np.linalg.norm(bare)


def test_P6_complete_basis_closed_form():
    cfg = _small_cfg(n=8, L=6.0, ecut=2.0, Nv=3, Npdep=2, sigma=1.2)
    npw_h = wl.half_sphere(cfg.n, cfg.L, cfg.ecut).shape[0]
    cfg.Npdep = 2 * (npw_h - 1)
    w = wl.make(cfg=cfg)
    tab = orc.Tables(w.n, w.L, w.ecut)
    lam = np.full(cfg.Npdep, -0.45)
    pairs, _ = orc.screen_pairs(w.u, 0.0)
    full = orc.build_tau(tab, w.u, w.phi, lam, pairs, want="G")
    bare = orc.build_tau(tab, w.u, w.phi, np.zeros_like(lam), pairs, want="G")
    assert np.linalg.norm(full - bare / (1 + 0.45)) <= 1e-11 * np.linalg.norm(bare)


# ------------------------------------------------------------------ P7 / P8: W symmetric, G=0 removed
def test_P7_P8_W_symmetric_and_zero_mean():
    w = wl.make(cfg=_small_cfg())
    tab = orc.Tables(w.n, w.L, w.ecut)
    pairs, _ = orc.screen_pairs(w.u, 0.0)
    assert len(pairs) == w.Nv * (w.Nv + 1) // 2
    tau = orc.build_tau(tab, w.u, w.phi, w.lam, pairs, want="r")
    rho = np.array([w.u[v] * w.u[x] for v, x in pairs])
    Mx = rho @ tau.T                                            # <rho_p | W rho_q>
    assert np.abs(Mx - Mx.T).max() <= 1e-12 * np.abs(Mx).max()
    assert np.abs(tau.sum(axis=1)).max() <= 1e-10 * np.abs(tau).max() * tab.N ** 0.5
    # and the screened integral differs from the bare one (lambda is doing something)
    bare = orc.build_tau(tab, w.u, w.phi, 0 * w.lam, pairs, want="r")
    assert np.linalg.norm(tau - bare) > 1e-3 * np.linalg.norm(bare)


# ------------------------------------------------------------------ P9 / P10: projector, K symmetric
def test_P9_P10_projector_and_K_symmetry():
    w = wl.make(cfg=_small_cfg(eta=0.05))
    tab = orc.Tables(w.n, w.L, w.ecut)
    pairs, O = orc.screen_pairs(w.u, w.eta)
    assert 0 < len(pairs) < w.Nv * (w.Nv + 1) // 2 + 1
    tau = orc.build_tau(tab, w.u, w.phi, w.lam, pairs, want="r")
    a = w.a_real()
    out = orc.apply_k1x_real(tab, w.u, pairs, tau, a)
    ov = tab.dV * np.einsum("wr,bvr->bvw", w.u, out)
    assert np.abs(ov).max() < 1e-12 * np.abs(out).max() * tab.N ** 0.5
    again = np.array([[orc.p_c_real(tab, w.u, out[b, v]) for v in range(w.Nv)] for b in range(a.shape[0])])
    assert np.linalg.norm(again - out) <= 1e-12 * np.linalg.norm(out)
    x = rng_vec = np.random.default_rng(3).normal(size=tab.N)
    px = orc.p_c_real(tab, w.u, x)
    assert np.linalg.norm(orc.p_c_real(tab, w.u, px) - px) <= 1e-12 * np.linalg.norm(px)
    assert np.linalg.norm(px - x) > 1e-3                        # it does remove something
    # K symmetric on projected blocks: sum_v <b_v|(K a)_v> = sum_v <a_v|(K b)_v>
    lhs = tab.dV * np.sum(a[1] * out[0])
    rhs = tab.dV * np.sum(a[0] * out[1])
    assert abs(lhs - rhs) <= 1e-12 * max(abs(lhs), abs(rhs))


# ------------------------------------------------------------------ P11: eq. 16 analytic
def test_P11_overlap_analytic_gaussians():
    n, L, sig = 48, 20.0, 1.4
    ax = np.arange(n) * (L / n)
    R = np.array([[9.0, 10.0, 10.5], [10.4, 10.9, 9.6], [12.5, 8.0, 11.0]])

    def gauss(Rv):
        e = [np.exp(-0.5 * ((ax - Rv[k]) / sig) ** 2) for k in range(3)]
        return (e[0][:, None, None] * e[1][None, :, None] * e[2][None, None, :]).ravel()

    u = np.array([gauss(Rv) for Rv in R])
    O = np.asarray(orc.overlap_matrix(u), dtype=float)
    for v in range(3):
        for x in range(3):
            d2 = np.sum((R[v] - R[x]) ** 2)
            assert abs(O[v, x] - math.exp(-d2 / (2 * sig ** 2))) < 1e-10      # O = exp(-d^2 / 2 sigma^2)
    assert np.allclose(np.diag(O), 1.0) and np.abs(O - O.T).max() == 0 and O.min() >= 0 and O.max() <= 1 + 1e-15
    thr = 0.5 * (O[0, 1] + O[0, 2])
    pairs, _ = orc.screen_pairs(u, thr)
    want = [(v, x) for v in range(3) for x in range(v, 3) if v == x or math.exp(-np.sum((R[v] - R[x]) ** 2) / (2 * sig ** 2)) >= thr]
    assert [tuple(p) for p in pairs.tolist()] == want


# ------------------------------------------------------------------ P12: PW layout vs REAL layout
def test_P12_pw_equals_gathered_real():
    w = wl.make(cfg=_small_cfg(eta=0.02))
    tab = orc.Tables(w.n, w.L, w.ecut)
    pairs, _ = orc.screen_pairs(w.u, w.eta)
    tau = orc.build_tau(tab, w.u, w.phi, w.lam, pairs, want="r")
    out_r = orc.apply_k1x_real(tab, w.u, pairs, tau, w.a_real())
    out_g = orc.apply_k1x_pw(tab, w.u, pairs, tau, w.a_pw)
    for b in range(out_r.shape[0]):
        for v in range(w.Nv):
            # independent gather: numpy's FFT, generator's H order
            want = wl.real_to_pw(out_r[b, v].reshape(w.n, w.n, w.n), w.mill, w.n)
            assert np.linalg.norm(out_g[b, v] - want) <= 1e-11 * np.linalg.norm(want)
    # tau in G form is the gather of tau in r form
    tg = orc.build_tau(tab, w.u, w.phi, w.lam, pairs[:2], want="G")
    for p in range(2):
        want = wl.real_to_pw(tau[p].reshape(w.n, w.n, w.n), w.mill, w.n)
        assert np.linalg.norm(tg[p] - want) <= 1e-11 * np.linalg.norm(want)


# ------------------------------------------------------------------ workload sanity (inputs only)
def test_workload_cfg1_inputs():
    w = wl.make(1)
    assert w.u.shape == (8, 24 ** 3) and w.phi.shape == (32, 523) and w.a_pw.shape == (2, 8, 523)
    dV = w.L ** 3 / w.N
    assert np.abs(dV * (w.u @ w.u.T) - np.eye(8)).max() < 1e-12
    G = 2 * np.real(np.conj(w.phi) @ w.phi.T)
    assert np.abs(G - np.eye(32)).max() < 1e-12 and np.all(w.phi[:, 0] == 0)
    assert np.all(w.lam < 0) and abs(w.lam[0] + 0.8) < 1e-15
    pairs, O = orc.screen_pairs(w.u, w.eta)
    assert len(pairs) == 36                                       # config 1: "all 36 pairs"


def test_P11b_overlap_rows_equals_overlap_matrix_rows():
    """overlap_rows (streamed form used for the sampled screen check at cfg 4-5) gives the rows of overlap_matrix."""
    w = wl.make(1)
    O = np.asarray(orc.overlap_matrix(w.u), dtype=np.float64)
    rows = [0, 5, 7]
    Or = orc.overlap_rows(lambda v: w.u[v], w.Nv, rows)
    assert np.abs(Or - O[rows]).max() < 1e-15


# ------------------------------------------------------------------ P13-P16: K1e (eq. 4)
def test_P13_k1e_dense_coulomb_operator_tiny_grid():
    """K1e from a dense real-space Coulomb matrix built from brute-force plane waves, by loops (eq. 4 written out)."""
    cfg = _small_cfg(n=6, L=5.0, ecut=2.5, Nv=3, Npdep=4, B=2, sigma=1.1)
    w = wl.make(cfg=cfg)
    n, N, L = w.n, w.N, w.L
    Omega, dV = L ** 3, L ** 3 / N
    mx = wl.msq_max(L, w.ecut)
    rng_m = range(-n // 2, n // 2)
    S = [(a, b, c) for a in rng_m for b in rng_m for c in rng_m if a * a + b * b + c * c <= mx]
    r = np.stack(np.meshgrid(*(np.arange(n),) * 3, indexing="ij"), -1).reshape(-1, 3)
    E = np.array([np.exp(1j * TWO_PI * (r @ np.array(m)) / n) for m in S])
    vc = np.array([0.0 if m == (0, 0, 0) else 4 * math.pi / ((TWO_PI / L) ** 2 * (m[0] ** 2 + m[1] ** 2 + m[2] ** 2)) for m in S])
    Vr = ((E.T * vc) @ np.conj(E)).real / Omega                  # v_c(r, r') restricted to S
    tab = orc.Tables(n, L, w.ecut)
    a = w.a_real()
    got = orc.apply_k1e_real(tab, w.u, a)
    Pc = np.eye(N) - dV * (w.u.T @ w.u)
    for b in range(a.shape[0]):
        dens = sum(w.u[x] * a[b, x] for x in range(w.Nv))
        vH = dV * (Vr @ dens)
        for v in range(w.Nv):
            want = Pc @ (2.0 * w.u[v] * vH)
            assert np.linalg.norm(got[b, v] - want) <= 1e-11 * np.linalg.norm(want)


def test_P14_hartree_of_gaussian_density_is_analytic():
    """v_H(G) = 4 pi n(G) / G^2 for a periodised Gaussian density given analytically in reciprocal space."""
    n, L, ecut, sig = 20, 12.0, 4.0, 1.4
    tab = orc.Tables(n, L, ecut)
    Rc = np.array([5.3, 6.1, 6.8])
    G = (TWO_PI / L) * tab.S.astype(float)
    G2 = (G ** 2).sum(1)
    nG = (2 * math.pi * sig ** 2) ** 1.5 / L ** 3 * np.exp(-0.5 * sig ** 2 * G2) * np.exp(-1j * (G @ Rc))
    n_r = tab.to_r(nG)                                            # band-limited density on the grid
    got = tab.to_G(orc.hartree_r(tab, n_r))
    want = np.zeros(tab.npw, complex)
    nz = G2 > 0
    want[nz] = 4 * math.pi * nG[nz] / G2[nz]
    assert np.linalg.norm(got - want) <= 1e-12 * np.linalg.norm(want)


def test_P15_k1e_symmetric_and_projected():
    w = wl.make(cfg=_small_cfg(n=12, Nv=4, B=2))
    tab = orc.Tables(w.n, w.L, w.ecut)
    a = w.a_real()
    out = orc.apply_k1e_real(tab, w.u, a)
    ov = tab.dV * np.einsum("wr,bvr->bvw", w.u, out)
    assert np.abs(ov).max() < 1e-12                               # P_c: <u_w|out> = 0
    A, Bv = a[0], a[1]
    KA, KB = out[0], out[1]
    lhs = tab.dV * np.sum(Bv * KA)
    rhs = tab.dV * np.sum(A * KB)
    assert abs(lhs - rhs) <= 1e-12 * max(abs(lhs), abs(rhs), 1e-30)   # K1e symmetric on the projected space
    # positive semi-definite (Coulomb energy of the transition density): <a|K1e a> = 2 int n v_H >= 0
    assert tab.dV * np.sum(A * KA) > 0


def test_P16_k1e_pw_equals_gathered_real():
    w = wl.make(cfg=_small_cfg(n=12, Nv=4, B=2))
    tab = orc.Tables(w.n, w.L, w.ecut)
    real = orc.apply_k1e_real(tab, w.u, w.a_real())
    pw = orc.apply_k1e_pw(tab, w.u, w.a_pw)
    for b in range(real.shape[0]):
        for v in range(w.Nv):
            want = orc.S_to_H(tab, tab.to_G(real[b, v]))
            assert np.linalg.norm(pw[b, v] - want) <= 1e-11 * np.linalg.norm(want)


# ------------------------------------------------------------------ P17: rotation of the representation (eq. 12)
def test_P17_rotation_covariance_of_k1x_and_k1e():
    """With every pair kept (eta = 0), K1x and K1e are covariant under an orthogonal mixing of the occupied orbitals:
    K(U u, U a) = U K(u, a).  Pins `rotate` (index order, transpose) through the whole chain, not against itself."""
    w = wl.make(cfg=_small_cfg(n=12, Nv=4, Npdep=6, B=2, eta=0.0))
    tab = orc.Tables(w.n, w.L, w.ecut)
    rng = np.random.default_rng(5)
    U, _ = np.linalg.qr(rng.normal(size=(w.Nv, w.Nv)))
    a = w.a_real()
    u2 = U @ w.u
    a2 = orc.rotate(U, a)
    assert np.allclose(orc.rotate(U, a2, transpose=True), a, atol=1e-14)
    assert np.allclose(a2, np.einsum("vw,bwr->bvr", U, a), atol=1e-14)
    pairs, _ = orc.screen_pairs(w.u, 0.0)
    pairs2, _ = orc.screen_pairs(u2, 0.0)
    k = orc.apply_k1x_real(tab, w.u, pairs, orc.build_tau(tab, w.u, w.phi, w.lam, pairs), a)
    k2 = orc.apply_k1x_real(tab, u2, pairs2, orc.build_tau(tab, u2, w.phi, w.lam, pairs2), a2)
    assert np.linalg.norm(k2 - orc.rotate(U, k)) <= 1e-11 * np.linalg.norm(k)
    e = orc.apply_k1e_real(tab, w.u, a)
    e2 = orc.apply_k1e_real(tab, u2, a2)
    assert np.linalg.norm(e2 - orc.rotate(U, e)) <= 1e-11 * np.linalg.norm(e)


def test_p18_single_precision_store_is_one_rounding_of_the_double_value():
    """tau_G_f32 (PAPER.md:279 reading): each component is an exactly representable binary32 number and differs from the fp64
    pair integral by at most half a unit in the last place of binary32 (relative 2^-24)."""
    w = wl.make(1)
    tab = orc.Tables(w.n, w.L, w.ecut)
    phiS = tab.expand_H_to_S(w.phi)
    t64 = orc.tau_G(tab, w.u[0], w.u[3], phiS, w.lam)
    t32 = orc.tau_G_f32(tab, w.u[0], w.u[3], phiS, w.lam)
    for a, b in ((t64.real, t32.real), (t64.imag, t32.imag)):
        assert np.array_equal(b.astype(np.float32).astype(np.float64), b)
        nz = np.abs(a) > 1e-30
        assert np.all(np.abs(a[nz] - b[nz]) <= 2.0 ** -24 * np.abs(a[nz]) * (1 + 1e-12))
        assert np.any(a[nz] != b[nz])

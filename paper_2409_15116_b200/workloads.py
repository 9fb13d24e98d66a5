"""Seeded synthetic workloads (inputs only) for the screened-exchange hot path.

This module serves BOTH the CPU oracle (`oracle/`) and the CUDA library: it makes the
inputs (u, phi, lambda, eta, trial blocks a) and nothing else.  It holds none of the
method's arithmetic (no screen, no pair integral, no K1x, no P_c): those live, written
independently, in `oracle/bse_oracle.py` and in `paper_2409_15116_b200/csrc/`.  It uses
`numpy.fft` only to band-limit and orthonormalise the raw orbitals, which is input
preparation, not a step of the path.

The paper's data sets (QE wave-functions, PDEP files) are not available;
these workloads stand in for them and take their shape and structure from
BASELINE.json `configs` (localised orbitals in a cubic supercell, N_pdep ~ N_v..2N_v,
overlap threshold 1e-3..1e-4, a line defect).  Recipe: SURVEY.md section 8(d).

Conventions (normative, restated in include/bse.h):
  grid n x n x n, linear index (i1*n + i2)*n + i3, r = (L/n) i
  G = (2 pi / L) m,  sphere S = { m : |m|^2 <= msq_max },
      msq_max = floor(2 ecut (L / 2 pi)^2 (1 + 1e-12))
  half sphere H = { m in S : m3>0 } + { m3=0, m2>0 } + { m3=m2=0, m1>=0 },
      sorted by ascending ((m1 mod n) n + (m2 mod n)) n + (m3 mod n)
  f(r) = sum_{G in S} c(G) exp(+i G.r), c(-G) = conj c(G); PW arrays hold c on H.
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

SEEDS = {1: 151161, 2: 151162, 3: 151163, 4: 151164, 5: 151165}


@dataclasses.dataclass
class Config:
    name: str
    L: float
    n: int
    Nv: int
    Npdep: int
    ecut: float
    sigma: float
    lam_c: float
    lam_k: float
    eta: float
    B: int
    sites: str          # "random" | "bcc" | "diamond_line"
    poly: bool = False
    seed: int = 0


CONFIGS = {
    1: Config("cfg1", 10.0, 24, 8, 32, 8.0, 1.2, 0.8, 3.0, 0.0, 2, "random", seed=SEEDS[1]),
    2: Config("cfg2", 20.0, 64, 64, 256, 12.0, 1.5, 0.9, 4.0, 1e-3, 4, "random", seed=SEEDS[2]),
    3: Config("cfg3", 30.0, 96, 256, 512, 12.0, 2.25, 0.9, 4.0, 1e-3, 8, "random", poly=True, seed=SEEDS[3]),
    4: Config("cfg4", 45.0, 144, 1024, 1024, 12.0, 1.8, 0.95, 5.0, 1e-4, 8, "bcc", seed=SEEDS[4]),
    5: Config("cfg5", 50.0, 160, 1024, 2048, 12.0, 1.8, 0.95, 5.0, 1e-4, 16, "diamond_line", seed=SEEDS[5]),
}


def msq_max(L: float, ecut: float) -> int:
    return int(math.floor(2.0 * ecut * (L / (2.0 * math.pi)) ** 2 * (1.0 + 1e-12)))


def half_sphere(n: int, L: float, ecut: float) -> np.ndarray:
    """Miller indices of H in the normative order, int32 [Npw_h][3]."""
    mx = msq_max(L, ecut)
    R = int(math.isqrt(mx))
    if 2 * R >= n:
        raise ValueError("sphere does not fit the grid (R >= n/2)")
    r = np.arange(-R, R + 1)
    m1, m2, m3 = np.meshgrid(r, r, r, indexing="ij")
    m1, m2, m3 = m1.ravel(), m2.ravel(), m3.ravel()
    ins = (m1 * m1 + m2 * m2 + m3 * m3) <= mx
    half = (m3 > 0) | ((m3 == 0) & (m2 > 0)) | ((m3 == 0) & (m2 == 0) & (m1 >= 0))
    keep = ins & half
    m1, m2, m3 = m1[keep], m2[keep], m3[keep]
    key = ((m1 % n) * n + (m2 % n)) * n + (m3 % n)
    order = np.argsort(key, kind="stable")
    return np.stack([m1[order], m2[order], m3[order]], axis=1).astype(np.int32)


# ----------------------------------------------------------------------------- sites
def _min_image(d, L):
    return d - L * np.round(d / L)


def _sites_random(rng, Nv, L, dmin):
    pts = []
    while len(pts) < Nv:
        c = rng.uniform(0.0, L, size=3)
        ok = True
        for p in pts:
            if np.linalg.norm(_min_image(c - p, L)) < dmin:
                ok = False
                break
        if ok:
            pts.append(c)
    return np.array(pts)


def _sites_bcc(rng, Nv, L):
    m = round((Nv / 2) ** (1.0 / 3.0))
    assert 2 * m ** 3 == Nv, "bcc lattice needs Nv = 2 m^3"
    a = L / m
    base = np.array([[0.0, 0.0, 0.0], [0.5, 0.5, 0.5]])
    ijk = np.stack(np.meshgrid(*(np.arange(m),) * 3, indexing="ij"), -1).reshape(-1, 3)
    pts = (ijk[:, None, :] + base[None, :, :]).reshape(-1, 3) * a + 0.25 * a
    pts = pts + rng.normal(0.0, 0.05 * a, size=pts.shape)
    return np.mod(pts, L)


def _sites_diamond_line(rng, Nv, L, sigma):
    m = 1
    while 8 * (m + 1) ** 3 <= Nv:
        m += 1
    nlat = 8 * m ** 3
    nline = Nv - nlat
    a = L / m
    fcc = np.array([[0, 0, 0], [0, .5, .5], [.5, 0, .5], [.5, .5, 0]])
    base = np.concatenate([fcc, fcc + 0.25])
    ijk = np.stack(np.meshgrid(*(np.arange(m),) * 3, indexing="ij"), -1).reshape(-1, 3)
    lat = (ijk[:, None, :] + base[None, :, :]).reshape(-1, 3) * a + 0.125 * a
    lat = np.mod(lat + rng.normal(0.0, 0.03 * a, size=lat.shape), L)
    if nline == 0:
        return lat
    for _ in range(1000):
        y0, z0 = rng.uniform(0.0, L, size=2)
        x = (np.arange(nline) + 0.5) * (L / nline)
        sgn = np.where(np.arange(nline) % 2 == 0, 1.0, -1.0)
        line = np.stack([x, np.full(nline, y0) + 1.5 * sgn, np.full(nline, z0)], axis=1)
        line = np.mod(line, L)
        d = _min_image(line[:, None, :] - lat[None, :, :], L)
        if np.sqrt((d ** 2).sum(-1)).min() >= sigma:
            return np.concatenate([lat, line])
    raise RuntimeError("could not place the line-defect row")


# -------------------------------------------------------------------------- orbitals
_POLY = ("x", "y", "z", "xy", "yz", "xz", "x2-y2", "2z2-x2-y2")


def _raw_orbital(n, L, sigma, R, coef):
    """g(r) = p((r-R)/sigma) exp(-|r-R|^2 / 2 sigma^2), minimum-image distances."""
    ax = np.arange(n) * (L / n)
    d = [_min_image(ax - R[k], L) / sigma for k in range(3)]
    e = [np.exp(-0.5 * dk * dk) for dk in d]
    g = e[0][:, None, None] * e[1][None, :, None] * e[2][None, None, :]
    if coef is not None:
        x, y, z = d[0][:, None, None], d[1][None, :, None], d[2][None, None, :]
        p = (1.0 + coef[0] * x + coef[1] * y + coef[2] * z + coef[3] * x * y + coef[4] * y * z
             + coef[5] * x * z + coef[6] * (x * x - y * y) + coef[7] * (2 * z * z - x * x - y * y))
        g = g * p
    return g


def _gather_H(F_half, mill, n):
    """rfftn-layout array [n][n][n/2+1] -> coefficients on H."""
    return F_half[mill[:, 0] % n, mill[:, 1] % n, mill[:, 2]]


def _scatter_H(c, mill, n):
    """coefficients on H -> rfftn-layout array (m3 = 0 plane filled with both +-G)."""
    F = np.zeros((n, n, n // 2 + 1), dtype=np.complex128)
    F[mill[:, 0] % n, mill[:, 1] % n, mill[:, 2]] = c
    z = mill[:, 2] == 0
    F[(-mill[z, 0]) % n, (-mill[z, 1]) % n, 0] = np.conj(c[z])
    if mill[0, 0] == 0 and mill[0, 1] == 0 and mill[0, 2] == 0:
        F[0, 0, 0] = c[0].real
    return F


def pw_to_real(c, mill, n):
    """f(r) = sum_{G in S} c(G) e^{iG.r} for one coefficient vector on H (input prep only)."""
    return np.fft.irfftn(_scatter_H(c, mill, n), s=(n, n, n), axes=(0, 1, 2)) * float(n) ** 3


def real_to_pw(f, mill, n):
    return _gather_H(np.fft.rfftn(f, axes=(0, 1, 2)), mill, n) / float(n) ** 3


def _hdot(a, b, g0):
    """sum over the full sphere of conj(a) b for Hermitian coefficient sets stored on H.
    a: [..., Npw_h], b: [..., Npw_h]; g0 = index of G=0 in H (always 0)."""
    full = 2.0 * np.real(np.conj(a) @ b.T)
    full -= np.real(np.conj(a[:, g0:g0 + 1]) @ b[:, g0:g0 + 1].T)
    return full


@dataclasses.dataclass
class Workload:
    cfg: Config
    n: int
    L: float
    ecut: float
    eta: float
    mill: np.ndarray        # [Npw_h][3] int32
    u: np.ndarray           # [Nv][N] float64, orthonormal (dV sum u_v u_w = delta), band-limited to S
    u_pw: np.ndarray        # [Nv][Npw_h] complex128 (same functions, coefficients on H)
    phi: np.ndarray         # [Npdep][Npw_h] complex128
    lam: np.ndarray         # [Npdep]
    a_pw: np.ndarray        # [B][Nv][Npw_h] complex128 trial blocks
    sites: np.ndarray

    @property
    def N(self):
        return self.n ** 3

    @property
    def Nv(self):
        return self.u.shape[0]

    @property
    def cell(self):
        return np.diag([self.L] * 3).astype(np.float64)

    def a_real(self):
        """[B][Nv][N] real-space trial blocks (inverse transform of a_pw)."""
        B, Nv, _ = self.a_pw.shape
        out = np.empty((B, Nv, self.N))
        for b in range(B):
            for v in range(Nv):
                out[b, v] = pw_to_real(self.a_pw[b, v], self.mill, self.n).ravel()
        return out


def make(cfg_id=None, *, cfg: Config | None = None, Nv=None, Npdep=None, B=None, seed=None,
         lam_zero=False) -> Workload:
    """Build a workload.  `Nv`, `Npdep`, `B` override the config (reduced cases for tests)."""
    c = dataclasses.replace(CONFIGS[cfg_id] if cfg is None else cfg)
    if Nv is not None:
        c.Nv = Nv
    if Npdep is not None:
        c.Npdep = Npdep
    if B is not None:
        c.B = B
    if seed is not None:
        c.seed = seed
    rng = np.random.default_rng(c.seed)
    n, L = c.n, c.L
    Omega = L ** 3
    mill = half_sphere(n, L, c.ecut)
    npw_h = mill.shape[0]
    assert tuple(mill[0]) == (0, 0, 0)

    if c.sites == "random":
        sites = _sites_random(rng, c.Nv, L, c.sigma)
    elif c.sites == "bcc":
        sites = _sites_bcc(rng, c.Nv, L)
    else:
        sites = _sites_diamond_line(rng, c.Nv, L, c.sigma)
    coefs = rng.normal(0.0, 0.35, size=(c.Nv, len(_POLY))) if c.poly else None

    # raw orbitals -> coefficients on H (band-limit to S)
    g_pw = np.empty((c.Nv, npw_h), dtype=np.complex128)
    for v in range(c.Nv):
        g = _raw_orbital(n, L, c.sigma, sites[v], None if coefs is None else coefs[v])
        g_pw[v] = real_to_pw(g, mill, n)
    # Loewdin: S_vw = Omega sum_S conj(g_v) g_w ; u = S^{-1/2} g
    S = Omega * _hdot(g_pw, g_pw, 0)
    w, V = np.linalg.eigh(0.5 * (S + S.T))
    assert w.min() > 1e-10 * w.max(), "raw orbitals are linearly dependent"
    Sm12 = (V / np.sqrt(w)) @ V.T
    u_pw = Sm12 @ g_pw
    u_pw[:, 0] = u_pw[:, 0].real
    u = np.empty((c.Nv, n ** 3))
    for v in range(c.Nv):
        u[v] = pw_to_real(u_pw[v], mill, n).ravel()

    # PDEP basis: random, phi(0)=0, orthonormal under <p|q> = 2 sum_{H\0} Re(conj p q)
    npd = c.Npdep
    assert npd <= 2 * (npw_h - 1)
    A = rng.normal(size=(2 * (npw_h - 1), npd))
    Q, _ = np.linalg.qr(A)
    Q = Q / math.sqrt(2.0)
    phi = np.zeros((npd, npw_h), dtype=np.complex128)
    phi[:, 1:] = (Q[0::2, :] + 1j * Q[1::2, :]).T
    i = np.arange(npd)
    lam = -c.lam_c * np.exp(-c.lam_k * i / npd)
    if lam_zero:
        lam = np.zeros(npd)

    # trial blocks: random Hermitian PW coefficients, made orthogonal to every u_w, normalised
    a_pw = rng.normal(size=(c.B, c.Nv, npw_h)) + 1j * rng.normal(size=(c.B, c.Nv, npw_h))
    a_pw[:, :, 0] = a_pw[:, :, 0].real
    for b in range(c.B):
        ov = Omega * _hdot(u_pw, a_pw[b], 0)          # [w][v] = <u_w|a_v>
        a_pw[b] = a_pw[b] - ov.T @ u_pw
        a_pw[b, :, 0] = a_pw[b, :, 0].real
        nrm = Omega * np.trace(_hdot(a_pw[b], a_pw[b], 0))
        a_pw[b] /= math.sqrt(nrm)

    return Workload(cfg=c, n=n, L=L, ecut=c.ecut, eta=c.eta, mill=mill, u=u, u_pw=u_pw,
                    phi=phi, lam=lam, a_pw=a_pw, sites=sites)


# =============================================================================================================
# Device generator for the large configurations (cfg 3-5): the same recipe executed with torch on a given device
# (the GPU when there is one), because at 144^3 / 160^3 with 1024 orbitals the arrays are tens of GB and the numpy
# path above takes tens of minutes.  Still inputs only: torch.fft / torch.linalg are used to band-limit,
# orthonormalise and transform the INPUT functions; none of the method's steps (screen, pair integral, K1x, P_c of
# the accumulated result) is evaluated here.  Differences from `make`: non-polynomial raw orbitals are the periodised
# Gaussians given analytically in reciprocal space, g_v(G) ~ exp(-|G|^2 sigma^2 / 2) exp(-i G.R_v) (identical to the
# minimum-image Gaussian up to exp(-(L/2)^2 / 2 sigma^2) < 1e-30 at cfg 4-5); phi and a are drawn from a seeded
# torch.Generator on the device (so the draws differ from `make`, and depend on the device type, not on the run).
@dataclasses.dataclass
class DeviceWorkload:
    cfg: Config
    n: int
    L: float
    ecut: float
    eta: float
    mill: np.ndarray        # host [Npw_h][3] int32
    u: "object"             # torch [Nv][N] float64 on the device
    u_pw: "object"          # torch [Nv][Npw_h] complex128
    phi: "object"           # torch [Npdep][Npw_h] complex128
    lam: np.ndarray         # host [Npdep]
    a_pw: "object"          # torch [B][Nv][Npw_h] complex128
    sites: np.ndarray

    @property
    def N(self):
        return self.n ** 3

    @property
    def Nv(self):
        return self.u.shape[0]

    @property
    def cell(self):
        return np.diag([self.L] * 3).astype(np.float64)


def make_device(cfg_id=None, device="cuda:0", *, cfg: Config | None = None, Nv=None, Npdep=None, B=None,
                seed=None) -> DeviceWorkload:
    import torch
    c = dataclasses.replace(CONFIGS[cfg_id] if cfg is None else cfg)
    if Nv is not None:
        c.Nv = Nv
    if Npdep is not None:
        c.Npdep = Npdep
    if B is not None:
        c.B = B
    if seed is not None:
        c.seed = seed
    dev = torch.device(device)
    rng = np.random.default_rng(c.seed)
    gen = torch.Generator(device=dev)
    gen.manual_seed(c.seed)
    n, L = c.n, c.L
    N = n ** 3
    Omega = L ** 3
    mill = half_sphere(n, L, c.ecut)
    npw_h = mill.shape[0]
    assert tuple(mill[0]) == (0, 0, 0)
    if c.sites == "random":
        sites = _sites_random(rng, c.Nv, L, c.sigma)
    elif c.sites == "bcc":
        sites = _sites_bcc(rng, c.Nv, L)
    else:
        sites = _sites_diamond_line(rng, c.Nv, L, c.sigma)
    coefs = rng.normal(0.0, 0.35, size=(c.Nv, len(_POLY))) if c.poly else None

    m_t = torch.from_numpy(mill.astype(np.int64)).to(dev)
    i1, i2, i3 = m_t[:, 0] % n, m_t[:, 1] % n, m_t[:, 2]
    z0 = m_t[:, 2] == 0
    j1, j2 = (-m_t[z0, 0]) % n, (-m_t[z0, 1]) % n

    def to_real(cH):                       # [k][Npw_h] complex -> [k][N] real (input prep, as pw_to_real)
        k = cH.shape[0]
        F = torch.zeros((k, n, n, n // 2 + 1), dtype=torch.complex128, device=dev)
        F[:, i1, i2, i3] = cH
        F[:, j1, j2, 0] = torch.conj(cH[:, z0])
        F[:, 0, 0, 0] = cH[:, 0].real.to(torch.complex128)
        return (torch.fft.irfftn(F, s=(n, n, n), dim=(1, 2, 3)) * float(N)).reshape(k, N)

    def hdot(a, b):                        # full-sphere sum of conj(a) b for Hermitian sets stored on H
        return 2.0 * (torch.conj(a) @ b.T).real - (torch.conj(a[:, :1]) @ b[:, :1].T).real

    # raw orbitals -> coefficients on H
    if coefs is None:
        G = (2.0 * math.pi / L) * m_t.to(torch.float64)                    # [Npw_h][3]
        R_t = torch.from_numpy(sites).to(dev)
        ph = G @ R_t.T                                                     # [Npw_h][Nv]
        env = torch.exp(-0.5 * c.sigma ** 2 * (G * G).sum(1))
        g_pw = (env[:, None] * torch.polar(torch.ones_like(ph), -ph)).T.contiguous()
        del ph
    else:
        g_pw = torch.empty((c.Nv, npw_h), dtype=torch.complex128, device=dev)
        for v in range(c.Nv):
            g = torch.from_numpy(_raw_orbital(n, L, c.sigma, sites[v], coefs[v])).to(dev)
            g_pw[v] = torch.fft.rfftn(g, dim=(0, 1, 2))[i1, i2, i3] / float(N)
    # Loewdin in PW
    S = Omega * hdot(g_pw, g_pw)
    w, V = torch.linalg.eigh(0.5 * (S + S.T))
    assert float(w.min()) > 1e-10 * float(w.max()), "raw orbitals are linearly dependent"
    Sm12 = ((V / torch.sqrt(w)) @ V.T).to(torch.complex128)
    u_pw = Sm12 @ g_pw
    del g_pw
    u_pw[:, 0] = u_pw[:, 0].real.to(torch.complex128)
    u = torch.empty((c.Nv, N), dtype=torch.float64, device=dev)
    step = max(1, min(16, (1 << 28) // N))
    for v0 in range(0, c.Nv, step):
        u[v0:v0 + step] = to_real(u_pw[v0:v0 + step])

    # PDEP basis
    npd = c.Npdep
    assert npd <= 2 * (npw_h - 1)
    A = torch.randn((2 * (npw_h - 1), npd), dtype=torch.float64, device=dev, generator=gen)
    Q, _ = torch.linalg.qr(A, mode="reduced")
    del A
    Q = Q / math.sqrt(2.0)
    phi = torch.zeros((npd, npw_h), dtype=torch.complex128, device=dev)
    phi[:, 1:] = torch.complex(Q[0::2, :], Q[1::2, :]).T
    del Q
    lam = -c.lam_c * np.exp(-c.lam_k * np.arange(npd) / npd)

    # trial blocks
    a_pw = torch.empty((c.B, c.Nv, npw_h), dtype=torch.complex128, device=dev)
    for b in range(c.B):
        ab = torch.complex(torch.randn((c.Nv, npw_h), dtype=torch.float64, device=dev, generator=gen),
                           torch.randn((c.Nv, npw_h), dtype=torch.float64, device=dev, generator=gen))
        ab[:, 0] = ab[:, 0].real.to(torch.complex128)
        ov = Omega * hdot(u_pw, ab)                                        # [w][v] = <u_w|a_v>
        ab = ab - ov.T.to(torch.complex128) @ u_pw
        ab[:, 0] = ab[:, 0].real.to(torch.complex128)
        nrm = Omega * float(torch.trace(hdot(ab, ab)))
        a_pw[b] = ab / math.sqrt(nrm)
        del ab
    if dev.type == "cuda":
        torch.cuda.synchronize(dev)
        torch.cuda.empty_cache()           # the library allocates with cudaMalloc: give the cached blocks back
    return DeviceWorkload(cfg=c, n=n, L=L, ecut=c.ecut, eta=c.eta, mill=mill, u=u, u_pw=u_pw, phi=phi, lam=lam,
                          a_pw=a_pw, sites=sites)


def device_a_real(w: DeviceWorkload):
    """[B][Nv][N] real-space trial blocks of a DeviceWorkload (inverse transform of a_pw; input preparation)."""
    import torch
    n, dev = w.n, w.a_pw.device
    m = torch.from_numpy(w.mill.astype(np.int64)).to(dev)
    i1, i2, i3 = m[:, 0] % n, m[:, 1] % n, m[:, 2]
    z0 = m[:, 2] == 0
    j1, j2 = (-m[z0, 0]) % n, (-m[z0, 1]) % n
    B, Nv, _ = w.a_pw.shape
    out = torch.empty((B, Nv, n ** 3), dtype=torch.float64, device=dev)
    step = max(1, min(16, (1 << 28) // n ** 3))
    for b in range(B):
        for v0 in range(0, Nv, step):
            cH = w.a_pw[b, v0:v0 + step]
            F = torch.zeros((cH.shape[0], n, n, n // 2 + 1), dtype=torch.complex128, device=dev)
            F[:, i1, i2, i3] = cH
            F[:, j1, j2, 0] = torch.conj(cH[:, z0])
            F[:, 0, 0, 0] = cH[:, 0].real.to(torch.complex128)
            out[b, v0:v0 + step] = (torch.fft.irfftn(F, s=(n, n, n), dim=(1, 2, 3)) * float(n) ** 3).reshape(cH.shape[0], -1)
    return out

"""GPU parity of the JADE localisation (bse_jade; eq. 12-15) against oracle/jade_oracle.py.

U is unique up to the sign of each row (the eigenvectors that initialise it are): rows are compared after fixing the sign
of their largest entry; the spread of eq. 14 and the localised orbitals' screen are compared as they are."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle import bse_oracle as orc                      # noqa: E402
from oracle import jade_oracle as jo                      # noqa: E402
from paper_2409_15116_b200 import workloads as wl         # noqa: E402


def _fix_signs(U):
    U = np.array(U, copy=True)
    for v in range(U.shape[0]):
        if U[v, np.argmax(np.abs(U[v]))] < 0:
            U[v] = -U[v]
    return U


@pytest.mark.parametrize("Nv,n,init_eig", [(8, 24, True), (7, 20, True), (12, 24, False)])
def test_jade_matches_the_oracle(Nv, n, init_eig):
    from paper_2409_15116_b200 import bse
    cfg = wl.Config("jade", 10.0, n, Nv, 8, 4.0 if n == 20 else 8.0, 1.2, 0.8, 3.0, 0.0, 1, "random", seed=500 + Nv)
    w = wl.make(cfg=cfg)
    rng = np.random.default_rng(5)
    Q, _ = np.linalg.qr(rng.normal(size=(Nv, Nv)))
    psi = np.ascontiguousarray(Q @ w.u)                        # delocalised orthonormal orbitals
    A, B = jo.position_matrices(psi, w.n, w.L, squares=True)
    V, Ad = jo.jade(A, init="eig" if init_eig else "identity")
    U_ref = V.T
    Bd = np.array([V.T @ b @ V for b in B])
    psi_d = torch.from_numpy(psi).cuda()
    U_d = torch.empty((Nv, Nv), dtype=torch.float64, device="cuda:0")
    loc_d = torch.empty_like(psi_d)
    sweeps, s0, s1 = bse.bse_jade([w.n] * 3, w.cell, Nv, psi_d, U_d, loc_d, init_eig=init_eig)
    torch.cuda.synchronize()
    U = U_d.cpu().numpy()
    assert 1 <= sweeps < 60
    assert np.abs(U @ U.T - np.eye(Nv)).max() < 1e-13
    assert abs(s0 - jo.spread(A, B)) < 1e-10 and abs(s1 - jo.spread(Ad, Bd)) < 1e-10
    assert np.abs(_fix_signs(U) - _fix_signs(U_ref)).max() < 1e-9
    loc = loc_d.cpu().numpy()
    assert np.abs(loc - U @ psi).max() < 1e-12 * np.abs(psi).max() * Nv
    # the localised orbitals are the compact ones again: same spread as the Loewdin Gaussians the mixing started from (or lower)
    A0, B0 = jo.position_matrices(w.u, w.n, w.L, squares=True)
    assert s1 <= jo.spread(A0, B0) * (1 + 1e-9) and s1 < 0.8 * s0


def test_jade_makes_the_screen_effective():
    """eq. 12 -> eq. 16: on delocalised orbitals nearly every pair survives the screen, on the JADE-localised ones the list
    is the short one again, and the library's list on them is the oracle's."""
    from paper_2409_15116_b200 import bse
    cfg = wl.Config("jscr", 14.0, 30, 10, 8, 5.0, 1.1, 0.8, 3.0, 0.02, 1, "random", seed=612)
    w = wl.make(cfg=cfg)
    Nv = w.Nv
    rng = np.random.default_rng(6)
    Q, _ = np.linalg.qr(rng.normal(size=(Nv, Nv)))
    psi_d = torch.from_numpy(np.ascontiguousarray(Q @ w.u)).cuda()
    U_d = torch.empty((Nv, Nv), dtype=torch.float64, device="cuda:0")
    loc_d = torch.empty_like(psi_d)
    bse.bse_jade([w.n] * 3, w.cell, Nv, psi_d, U_d, loc_d)
    torch.cuda.synchronize()
    phi_d = torch.from_numpy(np.ascontiguousarray(w.phi).view(np.float64)).cuda()
    counts = []
    for orb in (psi_d, loc_d):
        h = bse.bse_create([w.n] * 3, w.cell, w.ecut, Nv, orb, w.phi.shape[0], phi_d, w.lam, w.eta, 0)
        try:
            bse.bse_build_tau(h)
            pairs = bse.bse_get_pairs(h)
            ref, O = orc.screen_pairs(orb.cpu().numpy(), w.eta)
            if orc.screen_margin(O, w.eta) > 1e-9:
                assert np.array_equal(pairs, ref)
            counts.append(len(pairs))
        finally:
            bse.bse_destroy(h)
    assert counts[1] < counts[0] and counts[1] <= len(orc.screen_pairs(w.u, w.eta)[0]) + 2


def test_jade_many_orbitals_two_sweeps():
    """N_v = 520 (> 512: the round kernels run over several CTAs, 519 rounds of 260 pairs per sweep): two sweeps from the
    identity against the oracle's two sweeps, element by element (no sign freedom without the eigenvector start)."""
    from paper_2409_15116_b200 import bse
    Nv, n, L = 520, 24, 10.0
    rng = np.random.default_rng(77)
    Q, _ = np.linalg.qr(rng.normal(size=(n ** 3, Nv)))
    psi = np.ascontiguousarray(Q.T) / np.sqrt(L ** 3 / n ** 3)            # orthonormal: dV sum_r psi_v psi_w = delta
    A = jo.position_matrices(psi, n, L)
    V, Ad = jo.jade(A, init="identity", tol=0.0, max_sweeps=2)
    psi_d = torch.from_numpy(psi).cuda()
    U_d = torch.empty((Nv, Nv), dtype=torch.float64, device="cuda:0")
    sweeps, s0, s1 = bse.bse_jade([n] * 3, np.eye(3) * L, Nv, psi_d, U_d, None, tol=0.0, max_sweeps=2, init_eig=False)
    torch.cuda.synchronize()
    U = U_d.cpu().numpy()
    assert sweeps == 2
    assert np.abs(U - V.T).max() < 1e-10
    assert np.abs(U @ U.T - np.eye(Nv)).max() < 1e-12
    const = 3.0 * Nv - sum((a * a).sum() for a in A)
    assert abs(s0 - (const + jo.off_sum(A))) < 1e-8 and abs(s1 - (const + jo.off_sum(Ad))) < 1e-8 and s1 < s0

"""GPU parity: CUDA path (through the C ABI) vs the CPU oracle, element by element, same seeded inputs.

Bar (BASELINE.json north_star): surviving-pair list bit-exact; tau and K1x output within 1e-10 relative L2.
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from oracle import bse_oracle as orc                      # noqa: E402
from paper_2409_15116_b200 import workloads as wl         # noqa: E402

TOL = 1e-10


def _bse():
    from paper_2409_15116_b200 import bse
    return bse


def rel(a, b):
    return float(np.linalg.norm(np.asarray(a) - np.asarray(b)) / np.linalg.norm(np.asarray(b)))


class Gpu:
    """Device-resident inputs + handle for one workload."""

    def __init__(self, w, flags=0, knobs=None):
        bse = _bse()
        self.bse, self.w = bse, w
        dev = torch.device("cuda:0")
        self.u = torch.from_numpy(w.u).to(dev)
        phi = np.ascontiguousarray(w.phi).view(np.float64)          # interleaved (re, im)
        self.phi = torch.from_numpy(phi).to(dev)
        self.h = bse.bse_create([w.n] * 3, w.cell, w.ecut, w.Nv, self.u, w.phi.shape[0], self.phi, w.lam, w.eta, flags)
        for key, value in (knobs or {}).items():           # test knobs of the handle (include/bse.h: bse_debug_set)
            bse.bse_debug_set(self.h, key, value)

    def build(self):
        self.bse.bse_build_tau(self.h)
        torch.cuda.synchronize()
        return self.bse.bse_get_pairs(self.h)

    def tau_r(self, first, count):
        dst = torch.empty((count, self.w.N), dtype=torch.float64, device="cuda:0")
        self.bse.bse_get_tau(self.h, first, count, dst, self.bse.BSE_TAU_REAL)
        torch.cuda.synchronize()
        return dst.cpu().numpy()

    def tau_g(self, first, count):
        npw_h = self.bse.bse_npw_half(self.h)
        dst = torch.empty((count, npw_h, 2), dtype=torch.float64, device="cuda:0")
        self.bse.bse_get_tau(self.h, first, count, dst, self.bse.BSE_TAU_PW)
        torch.cuda.synchronize()
        return dst.cpu().numpy().view(np.complex128)[..., 0]

    def apply(self, a):
        a_d = torch.from_numpy(np.ascontiguousarray(a)).to("cuda:0")
        out = torch.empty_like(a_d)
        self.bse.bse_apply_k1x(self.h, a_d, out, a.shape[0])
        torch.cuda.synchronize()
        return out.cpu().numpy()

    def close(self):
        self.bse.bse_destroy(self.h)


def _check_full(w, flags=0, check_g=True, knobs=None, tau_ref=None):
    tab = orc.Tables(w.n, w.L, w.ecut)
    pairs_ref, O = orc.screen_pairs(w.u, w.eta)
    assert orc.screen_margin(O, w.eta) > 1e-9, "workload violates the screen guard band (S10)"
    g = Gpu(w, flags, knobs)
    try:
        assert np.array_equal(g.bse.bse_gvectors(g.h), w.mill)
        pairs = g.build()
        assert pairs.dtype == np.int32 and np.array_equal(pairs, pairs_ref)          # bit-exact list
        O_gpu = g.bse.bse_get_overlap(g.h, w.Nv)
        assert np.abs(O_gpu - O).max() < 1e-12
        if tau_ref is None:
            tau_ref = orc.build_tau(tab, w.u, w.phi, w.lam, pairs_ref, want="r")
        tau = g.tau_r(0, len(pairs))
        assert rel(tau, tau_ref) <= TOL
        worst = max(rel(tau[p], tau_ref[p]) for p in range(len(pairs)))
        assert worst <= 10 * TOL
        if check_g:
            tg_ref = orc.build_tau(tab, w.u, w.phi, w.lam, pairs_ref, want="G")
            assert rel(g.tau_g(0, len(pairs)), tg_ref) <= TOL
        a = w.a_real()
        out_ref = orc.apply_k1x_real(tab, w.u, pairs_ref, tau_ref, a)
        out = g.apply(a)
        assert rel(out, out_ref) <= TOL
        # P_c did its job on the GPU result: <u_w|out> = 0
        ov = tab.dV * np.einsum("wr,bvr->bvw", w.u, out)
        assert np.abs(ov).max() < 1e-11 * np.abs(out).max() * tab.N ** 0.5
        return out
    finally:
        g.close()


def _check_pw(w, flags=0, knobs=None):
    """PW layout (a12): a, out on the half sphere H; reference = oracle apply_k1x_pw (O8 'K1x PW')."""
    bse = _bse()
    tab = orc.Tables(w.n, w.L, w.ecut)
    pairs_ref, _ = orc.screen_pairs(w.u, w.eta)
    g = Gpu(w, flags | bse.BSE_VEC_PW, knobs)
    try:
        pairs = g.build()
        assert np.array_equal(pairs, pairs_ref)
        tau_ref = orc.build_tau(tab, w.u, w.phi, w.lam, pairs_ref, want="r")
        ref = orc.apply_k1x_pw(tab, w.u, pairs_ref, tau_ref, w.a_pw)
        a_d = torch.from_numpy(np.ascontiguousarray(w.a_pw).view(np.float64)).to("cuda:0")
        out = torch.empty_like(a_d)
        bse.bse_apply_k1x(g.h, a_d, out, w.a_pw.shape[0])
        torch.cuda.synchronize()
        got = out.cpu().numpy().view(np.complex128).reshape(ref.shape)
        wt = np.full(tab.npw_h, 2.0)
        wt[0] = 1.0                                   # S18: PW norm with weight 2 on G != 0
        err = np.sqrt((wt * np.abs(got - ref) ** 2).sum() / (wt * np.abs(ref) ** 2).sum())
        assert err <= TOL, err
        # second call reuses the staging buffers and gives the same bits
        out2 = torch.empty_like(a_d)
        bse.bse_apply_k1x(g.h, a_d, out2, w.a_pw.shape[0])
        torch.cuda.synchronize()
        assert torch.equal(out, out2)
        return got
    finally:
        g.close()


def test_pw_layout_all_tau_modes():
    bse = _bse()
    w = wl.make(1)
    o = [_check_pw(w, f) for f in (bse.BSE_TAU_REAL, bse.BSE_TAU_PW, bse.BSE_TAU_STREAM)]
    assert rel(o[1], o[0]) < 1e-12 and rel(o[2], o[0]) < 1e-12
    cfg = wl.Config("edge", 9.0, 12, 5, 7, 3.0, 1.3, 0.8, 3.0, 0.05, 3, "random", seed=112)
    _check_pw(wl.make(cfg=cfg))
    _check_pw(wl.make(2, Nv=12, Npdep=40, B=2), bse.BSE_TAU_PW)


def test_several_groups_and_row_batches():
    """Small case forced through the large-config machinery: trial blocks in groups of 2 (B = 5: ragged last group) and
    row batches of at most 7 pairs (several batches, pairs shared between batches re-inverted)."""
    bse = _bse()
    knobs = {"max_group": 2, "max_batch": 7}
    cfg = wl.Config("grp", 10.0, 24, 9, 20, 8.0, 1.2, 0.8, 3.0, 0.02, 5, "random", seed=77)
    w = wl.make(cfg=cfg)
    o1 = _check_pw(w, bse.BSE_TAU_PW, knobs)
    o2 = _check_pw(w, bse.BSE_TAU_STREAM, knobs)
    assert rel(o2, o1) < 1e-12
    _check_full(w, bse.BSE_TAU_PW, check_g=False, knobs=knobs)
    o3 = _check_pw(w, bse.BSE_TAU_PW)
    assert rel(o3, o1) < 1e-12


def test_seventeen_trial_blocks():
    """B = 17: the accumulate stage takes the two whole groups of 8 blocks side by side in one launch (the grouped kernel
    variant, otherwise only reached by cfg 5's B = 16) and the last block through the row kernel; slab path, group /
    row-batch path and the REAL layout with tau on H."""
    bse = _bse()
    w = wl.make(cfg=wl.Config("b17", 10.0, 20, 7, 10, 6.0, 1.2, 0.8, 3.0, 0.02, 17, "random", seed=1717))
    for tau in (bse.BSE_TAU_PW, bse.BSE_TAU_STREAM):
        o_slab = _check_pw(w, tau, {"slab_rows": 3, "slab_planes": 5})
        o_grp = _check_pw(w, tau, {"slab_rows": -1, "max_batch": 6})
        assert rel(o_grp, o_slab) < 1e-12
    _check_full(w, bse.BSE_TAU_PW, check_g=False, knobs={"max_batch": 5})


def test_cfg1_full_all_modes():
    w = wl.make(1)
    bse = _bse()
    o0 = _check_full(w, bse.BSE_TAU_REAL)
    o1 = _check_full(w, bse.BSE_TAU_PW, check_g=False)
    o2 = _check_full(w, bse.BSE_TAU_STREAM, check_g=False)
    assert rel(o1, o0) < 1e-12 and rel(o2, o0) < 1e-12


@pytest.mark.parametrize("n,L,ecut,Nv,Npdep,B,eta", [
    (12, 9.0, 3.0, 5, 7, 3, 0.05),        # odd Nv / Npdep / B, radix 4*3, screened
    (20, 12.0, 4.0, 6, 9, 1, 0.0),        # radix 5
    (30, 14.0, 5.0, 4, 16, 2, 0.02),      # radices 2,3,5
    (24, 10.0, 8.0, 9, 33, 16, 0.9),      # big threshold: (nearly) only diagonal pairs, B = 16
])
def test_small_shapes_and_edges(n, L, ecut, Nv, Npdep, B, eta):
    cfg = wl.Config("edge", L, n, Nv, Npdep, ecut, 1.3, 0.8, 3.0, eta, B, "random", seed=100 + n)
    w = wl.make(cfg=cfg)
    _check_full(w)


def test_cfg2_reduced_full_check():
    # config-2 grid and sphere (64^3, 15895 PWs, several GEMM tiles and a ragged K tail), fewer orbitals
    w = wl.make(2, Nv=12, Npdep=40, B=2)
    for flags in (0, _bse().BSE_TAU_PW, _bse().BSE_TAU_STREAM):
        _check_full(w, flags, check_g=(flags == 0))


_W2 = {}


def _w_tau_pair(vx):
    return orc.tau_r(_W2["tab"], _W2["u"][vx[0]], _W2["u"][vx[1]], _W2["phiS"], _W2["lam"])


def test_cfg2_full_size_in_full():
    """BASELINE config 2 at full size IN FULL: the whole list, all 234 tau, all 64 x 4 output rows.  The oracle's pair integrals
    (independent calls of orc.tau_r, as it stands) are spread over forked worker processes by the harness."""
    import multiprocessing as mp
    import os
    w = wl.make(2)
    tab = orc.Tables(w.n, w.L, w.ecut)
    pairs_ref, _ = orc.screen_pairs(w.u, w.eta)
    assert 64 <= len(pairs_ref) < 2080
    _W2.update(tab=tab, u=w.u, phiS=tab.expand_H_to_S(w.phi), lam=w.lam)
    with mp.get_context("fork").Pool(min(12, os.cpu_count() or 4)) as pool:
        tau_ref = np.array(pool.map(_w_tau_pair, [(int(v), int(x)) for v, x in pairs_ref], chunksize=4))
    _W2.clear()
    _check_full(w, 0, check_g=False, tau_ref=tau_ref)
    _check_full(w, _bse().BSE_TAU_PW, check_g=False, tau_ref=tau_ref)


def test_error_paths():
    bse = _bse()
    w = wl.make(cfg=wl.Config("e", 9.0, 12, 4, 6, 3.0, 1.3, 0.8, 3.0, 0.0, 2, "random", seed=3))
    g = Gpu(w)
    try:
        a = torch.zeros((1, w.Nv, w.N), dtype=torch.float64, device="cuda:0")
        with pytest.raises(bse.BseError) as e:
            bse.bse_apply_k1x(g.h, a, torch.empty_like(a), 1)
        assert e.value.code == bse.BSE_ESTATE
        g.build()
        with pytest.raises(bse.BseError) as e:
            bse.bse_apply_k1x(g.h, a, a, 1)
        assert e.value.code == bse.BSE_EINVAL
    finally:
        g.close()
    lam_bad = w.lam.copy()
    lam_bad[0] = 1.0
    u = torch.from_numpy(w.u).cuda()
    phi = torch.from_numpy(np.ascontiguousarray(w.phi).view(np.float64)).cuda()
    for kwargs, code in [
        (dict(lam=lam_bad), bse.BSE_EINVAL),
        (dict(ecut=40.0), bse.BSE_EINVAL),                 # sphere does not fit
        (dict(eta=-1.0), bse.BSE_EINVAL),
        (dict(grid=[12, 12, 10]), bse.BSE_EUNSUPPORTED),
        (dict(flags=3), bse.BSE_EINVAL),                   # bad tau storage flag
    ]:
        args = dict(grid=[w.n] * 3, ecut=w.ecut, lam=w.lam, eta=0.0, flags=0)
        args.update(kwargs)
        with pytest.raises(bse.BseError) as e:
            bse.bse_create(args["grid"], w.cell, args["ecut"], w.Nv, u, w.phi.shape[0], phi, args["lam"], args["eta"], args["flags"])
        assert e.value.code == code


def test_host_pointer_entry_points():
    bse = _bse()
    w = wl.make(cfg=wl.Config("h", 9.0, 12, 4, 6, 3.0, 1.3, 0.8, 3.0, 0.0, 2, "random", seed=4))
    tab = orc.Tables(w.n, w.L, w.ecut)
    phi = np.ascontiguousarray(w.phi).view(np.float64)
    h = bse.bse_create([w.n] * 3, w.cell, w.ecut, w.Nv, w.u, w.phi.shape[0], phi, w.lam, w.eta, bse.BSE_PTR_HOST)
    try:
        bse.bse_build_tau(h)
        pairs = bse.bse_get_pairs(h)
        a = np.ascontiguousarray(w.a_real())
        out = np.empty_like(a)
        bse.bse_apply_k1x_host(h, a, out, a.shape[0])
        tau_ref = orc.build_tau(tab, w.u, w.phi, w.lam, pairs, want="r")
        assert rel(out, orc.apply_k1x_real(tab, w.u, pairs, tau_ref, a)) <= TOL       # B = 2: the pipelined path
        # new inputs into the same handle: tau is invalidated, a rebuild gives the new problem's result
        w2 = wl.make(cfg=wl.Config("h", 9.0, 12, 4, 6, 3.0, 1.3, 0.8, 3.0, 0.0, 2, "random", seed=5))
        phi2 = np.ascontiguousarray(w2.phi).view(np.float64)
        bse.bse_set_inputs_host(h, np.ascontiguousarray(w2.u), phi2)
        with pytest.raises(bse.BseError) as e:
            bse.bse_apply_k1x_host(h, a, out, a.shape[0])
        assert e.value.code == bse.BSE_ESTATE
        bse.bse_build_tau(h)
        pairs2 = bse.bse_get_pairs(h)
        a2 = np.ascontiguousarray(w2.a_real())
        bse.bse_apply_k1x_host(h, a2, out, a2.shape[0])
        tau2 = orc.build_tau(tab, w2.u, w2.phi, w2.lam, pairs2, want="r")
        assert rel(out, orc.apply_k1x_real(tab, w2.u, pairs2, tau2, a2)) <= TOL
    finally:
        bse.bse_destroy(h)
    u_d = torch.from_numpy(w.u).cuda()
    phi_d = torch.from_numpy(phi).cuda()
    hb = bse.bse_create([w.n] * 3, w.cell, w.ecut, w.Nv, u_d, w.phi.shape[0], phi_d, w.lam, w.eta, 0)
    try:
        with pytest.raises(bse.BseError) as e:
            bse.bse_set_inputs_host(hb, w.u, phi)
        assert e.value.code == bse.BSE_ESTATE                  # borrowed device arrays: nothing to copy into
    finally:
        bse.bse_destroy(hb)


@pytest.mark.parametrize("cfg", [
    None,                                                                        # BASELINE config 1
    wl.Config("k1e", 9.0, 12, 5, 7, 3.0, 1.3, 0.8, 3.0, 0.05, 3, "random", seed=112),     # odd Nv, B; apply grid = grid
    wl.Config("k1e", 12.0, 20, 6, 9, 4.0, 1.3, 0.8, 3.0, 0.0, 1, "random", seed=120),     # radix 5
])
def test_k1e_real_and_pw_layouts(cfg):
    """K1e (eq. 4) against the oracle in both layouts; needs no pair list."""
    bse = _bse()
    w = wl.make(1) if cfg is None else wl.make(cfg=cfg)
    tab = orc.Tables(w.n, w.L, w.ecut)
    B = w.a_pw.shape[0]
    g = Gpu(w, bse.BSE_TAU_PW)
    try:
        a = w.a_real()
        ref = orc.apply_k1e_real(tab, w.u, a)
        a_d = torch.from_numpy(np.ascontiguousarray(a)).to("cuda:0")
        out = torch.empty_like(a_d)
        bse.bse_apply_k1e(g.h, a_d, out, B)                     # before bse_build_tau: allowed
        torch.cuda.synchronize()
        assert rel(out.cpu().numpy(), ref) <= TOL
    finally:
        g.close()
    g = Gpu(w, bse.BSE_TAU_PW | bse.BSE_VEC_PW)
    try:
        ref = orc.apply_k1e_pw(tab, w.u, w.a_pw)
        a_d = torch.from_numpy(np.ascontiguousarray(w.a_pw).view(np.float64)).to("cuda:0")
        out = torch.empty_like(a_d)
        bse.bse_apply_k1e(g.h, a_d, out, B)
        torch.cuda.synchronize()
        got = out.cpu().numpy().view(np.complex128).reshape(ref.shape)
        wt = np.full(tab.npw_h, 2.0)
        wt[0] = 1.0
        err = np.sqrt((wt * np.abs(got - ref) ** 2).sum() / (wt * np.abs(ref) ** 2).sum())
        assert err <= TOL, err
        # K1x on the same handle afterwards still matches (shared workspaces)
        g.build()
        pairs_ref, _ = orc.screen_pairs(w.u, w.eta)
        tau_ref = orc.build_tau(tab, w.u, w.phi, w.lam, pairs_ref, want="r")
        refx = orc.apply_k1x_pw(tab, w.u, pairs_ref, tau_ref, w.a_pw)
        bse.bse_apply_k1x(g.h, a_d, out, B)
        torch.cuda.synchronize()
        gotx = out.cpu().numpy().view(np.complex128).reshape(refx.shape)
        assert np.sqrt((wt * np.abs(gotx - refx) ** 2).sum() / (wt * np.abs(refx) ** 2).sum()) <= TOL
    finally:
        g.close()


@pytest.mark.parametrize("Nv", [5, 8])
def test_rotate_between_representations(Nv):
    """bse_rotate (eq. 12) against the oracle's triple loop, both directions, both layouts; then the
    covariance K(U u, U a) = U K(u, a) of K1x and K1e with every pair kept, end to end on the GPU."""
    bse = _bse()
    cfg = wl.Config("rot", 9.0, 12, Nv, 7, 3.0, 1.3, 0.8, 3.0, 0.0, 2, "random", seed=200 + Nv)
    w = wl.make(cfg=cfg)
    rng = np.random.default_rng(9)
    U, _ = np.linalg.qr(rng.normal(size=(Nv, Nv)))
    U_d = torch.from_numpy(np.ascontiguousarray(U)).to("cuda:0")
    B = w.a_pw.shape[0]
    for vec, x in ((bse.BSE_VEC_REAL, w.a_real()), (bse.BSE_VEC_PW, np.ascontiguousarray(w.a_pw).view(np.float64))):
        g = Gpu(w, vec)
        try:
            x_d = torch.from_numpy(np.ascontiguousarray(x)).to("cuda:0")
            y_d = torch.empty_like(x_d)
            for tr in (False, True):
                bse.bse_rotate(g.h, U_d, x_d, y_d, B, transpose=tr)
                torch.cuda.synchronize()
                ref = orc.rotate(U, x.reshape(B, Nv, -1), transpose=tr)
                assert rel(y_d.cpu().numpy().reshape(ref.shape), ref) <= 1e-13
        finally:
            g.close()
    # covariance on the GPU (REAL layout): handle 1 = (u, a), handle 2 = (U u, U a)
    a = w.a_real()
    outs = []
    for uu, aa in ((w.u, a), (U @ w.u, orc.rotate(U, a))):
        u_d = torch.from_numpy(np.ascontiguousarray(uu)).to("cuda:0")
        phi_d = torch.from_numpy(np.ascontiguousarray(w.phi).view(np.float64)).to("cuda:0")
        h = bse.bse_create([w.n] * 3, w.cell, w.ecut, Nv, u_d, w.phi.shape[0], phi_d, w.lam, 0.0, 0)
        try:
            bse.bse_build_tau(h)
            a_d = torch.from_numpy(np.ascontiguousarray(aa)).to("cuda:0")
            kx, ke = torch.empty_like(a_d), torch.empty_like(a_d)
            bse.bse_apply_k1x(h, a_d, kx, B)
            bse.bse_apply_k1e(h, a_d, ke, B)
            torch.cuda.synchronize()
            outs.append((kx.cpu().numpy(), ke.cpu().numpy()))
        finally:
            bse.bse_destroy(h)
    assert rel(outs[1][0], orc.rotate(U, outs[0][0])) <= 1e-10
    assert rel(outs[1][1], orc.rotate(U, outs[0][1])) <= 1e-10


@pytest.mark.parametrize("tau", ["real", "pw", "stream"])
def test_combined_two_body_call(tau):
    """bse_apply_k1 = ce * K1e + cd * K1x with one P_c (eq. 1), against the oracle's two terms, both layouts, every tau mode;
    the PW case is also forced through several block groups and row batches."""
    bse = _bse()
    flag = {"real": bse.BSE_TAU_REAL, "pw": bse.BSE_TAU_PW, "stream": bse.BSE_TAU_STREAM}[tau]
    cfg = wl.Config("k1", 10.0, 24, 9, 20, 8.0, 1.2, 0.8, 3.0, 0.02, 3, "random", seed=78)
    w = wl.make(cfg=cfg)
    tab = orc.Tables(w.n, w.L, w.ecut)
    B = w.a_pw.shape[0]
    pairs, _ = orc.screen_pairs(w.u, w.eta)
    tau_ref = orc.build_tau(tab, w.u, w.phi, w.lam, pairs, want="r")
    ce, cd = 1.0, -1.0
    a = w.a_real()
    ref_r = ce * orc.apply_k1e_real(tab, w.u, a) + cd * orc.apply_k1x_real(tab, w.u, pairs, tau_ref, a)
    ref_g = ce * orc.apply_k1e_pw(tab, w.u, w.a_pw) + cd * orc.apply_k1x_pw(tab, w.u, pairs, tau_ref, w.a_pw)
    g = Gpu(w, flag)
    try:
        g.build()
        a_d = torch.from_numpy(np.ascontiguousarray(a)).to("cuda:0")
        out = torch.empty_like(a_d)
        bse.bse_apply_k1(g.h, a_d, out, B, ce, cd)
        torch.cuda.synchronize()
        assert rel(out.cpu().numpy(), ref_r) <= TOL
    finally:
        g.close()
    wt = np.full(tab.npw_h, 2.0)
    wt[0] = 1.0
    for forced in (False, True):
        g = Gpu(w, flag | bse.BSE_VEC_PW, {"max_group": 2, "max_batch": 7} if forced else None)
        try:
            g.build()
            a_d = torch.from_numpy(np.ascontiguousarray(w.a_pw).view(np.float64)).to("cuda:0")
            out = torch.empty_like(a_d)
            bse.bse_apply_k1(g.h, a_d, out, B, ce, cd)
            torch.cuda.synchronize()
            got = out.cpu().numpy().view(np.complex128).reshape(ref_g.shape)
            err = np.sqrt((wt * np.abs(got - ref_g) ** 2).sum() / (wt * np.abs(ref_g) ** 2).sum())
            assert err <= TOL, (forced, err)
        finally:
            g.close()


def test_block_count_grows_and_stream_real_batches():
    """One handle, PW layout: B = 1 first, then B = 3 (the apply plan is re-made for the larger group) - same rows both
    times.  Then the REAL layout with BSE_TAU_STREAM forced through several row batches."""
    bse = _bse()
    cfg = wl.Config("grow", 10.0, 24, 7, 12, 8.0, 1.2, 0.8, 3.0, 0.02, 3, "random", seed=79)
    w = wl.make(cfg=cfg)
    tab = orc.Tables(w.n, w.L, w.ecut)
    pairs, _ = orc.screen_pairs(w.u, w.eta)
    tau_ref = orc.build_tau(tab, w.u, w.phi, w.lam, pairs, want="r")
    ref = orc.apply_k1x_pw(tab, w.u, pairs, tau_ref, w.a_pw)
    wt = np.full(tab.npw_h, 2.0)
    wt[0] = 1.0
    g = Gpu(w, bse.BSE_TAU_PW | bse.BSE_VEC_PW)
    try:
        g.build()
        a_all = torch.from_numpy(np.ascontiguousarray(w.a_pw).view(np.float64)).to("cuda:0")
        for B in (1, 3, 2):
            out = torch.empty_like(a_all[:B])
            bse.bse_apply_k1x(g.h, a_all[:B].contiguous(), out, B)
            torch.cuda.synchronize()
            got = out.cpu().numpy().view(np.complex128).reshape(ref[:B].shape)
            err = np.sqrt((wt * np.abs(got - ref[:B]) ** 2).sum() / (wt * np.abs(ref[:B]) ** 2).sum())
            assert err <= TOL, (B, err)
        # tau(G) of a pair range straight from the store
        tg_ref = orc.build_tau(tab, w.u, w.phi, w.lam, pairs[2:5], want="G")
        assert rel(g.tau_g(2, 3), tg_ref) <= TOL
    finally:
        g.close()
    _check_full(w, bse.BSE_TAU_STREAM, check_g=True, knobs={"max_batch": 5})


def test_compact_inverse_plane_kernel_small_grids():
    """The compact inverse plane kernel (used by default only at n = 120, 144) forced on small grids: radices 4x6, 5x4, 5x6."""
    knobs = {"compact_inv": 2}
    for n, L, ecut, Nv, Npdep, B in ((24, 10.0, 8.0, 8, 16, 2), (20, 12.0, 4.0, 6, 9, 1), (30, 14.0, 5.0, 4, 16, 2)):
        cfg = wl.Config("cmp", L, n, Nv, Npdep, ecut, 1.3, 0.8, 3.0, 0.0, B, "random", seed=300 + n)
        w = wl.make(cfg=cfg)
        _check_full(w, knobs=knobs)
        _check_pw(w, _bse().BSE_TAU_PW, knobs)


def test_real_layout_with_orbitals_that_are_not_band_limited():
    """The REAL layout takes any u.  With band-limited u (every generated workload) the P_c overlaps go through the pruned FFT;
    with u that has components outside S the library must notice (Parseval check) and keep the real-space overlaps."""
    bse = _bse()
    cfg = wl.Config("nbl", 10.0, 24, 6, 12, 8.0, 1.2, 0.8, 3.0, 0.01, 2, "random", seed=81)
    w = wl.make(cfg=cfg)
    rng = np.random.default_rng(3)
    u = w.u + 0.02 * rng.normal(size=w.u.shape) * np.abs(w.u).max()                             # grid noise: not in S
    dV = w.L ** 3 / w.N
    ev, V = np.linalg.eigh(dV * (u @ u.T))
    w.u = np.ascontiguousarray(((V / np.sqrt(ev)) @ V.T) @ u)                                    # orthonormal again
    _check_full(w, bse.BSE_TAU_REAL, check_g=True)
    _check_full(w, bse.BSE_TAU_PW, check_g=False)


def test_rebuilt_list_with_the_same_pair_count_gets_a_new_plan():
    """new orbitals whose surviving-pair list has the SAME length but other pairs (the old orbitals, permuted)
    must not reuse the row batches / slots planned for the old list.  PW layout, tau on H, row batches forced small."""
    bse = _bse()
    cfg = wl.Config("perm", 10.0, 24, 10, 20, 8.0, 1.2, 0.8, 3.0, 0.05, 2, "random", seed=91)
    w = wl.make(cfg=cfg)
    tab = orc.Tables(w.n, w.L, w.ecut)
    phi = np.ascontiguousarray(w.phi).view(np.float64)
    wt = np.full(tab.npw_h, 2.0)
    wt[0] = 1.0
    rng = np.random.default_rng(4)
    h = bse.bse_create([w.n] * 3, w.cell, w.ecut, w.Nv, np.ascontiguousarray(w.u), w.phi.shape[0], phi, w.lam, w.eta,
                       bse.BSE_PTR_HOST | bse.BSE_TAU_PW | bse.BSE_VEC_PW)
    try:
        bse.bse_debug_set(h, "max_batch", 6)
        lists = []
        for trial in range(3):
            perm = np.arange(w.Nv) if trial == 0 else rng.permutation(w.Nv)
            u = np.ascontiguousarray(w.u[perm])
            a_pw = np.ascontiguousarray(w.a_pw[:, perm])
            bse.bse_set_inputs_host(h, u, None)
            bse.bse_build_tau(h)
            pairs = bse.bse_get_pairs(h)
            pairs_ref, _ = orc.screen_pairs(u, w.eta)
            assert np.array_equal(pairs, pairs_ref)
            lists.append(pairs)
            a = np.ascontiguousarray(a_pw).view(np.float64)
            out = np.empty_like(a)
            bse.bse_apply_k1x_host(h, a, out, a_pw.shape[0])
            tau_ref = orc.build_tau(tab, u, w.phi, w.lam, pairs_ref, want="r")
            ref = orc.apply_k1x_pw(tab, u, pairs_ref, tau_ref, a_pw)
            got = out.view(np.complex128).reshape(ref.shape)
            err = np.sqrt((wt * np.abs(got - ref) ** 2).sum() / (wt * np.abs(ref) ** 2).sum())
            assert err <= TOL, (trial, err)
        assert len(lists[0]) == len(lists[1]) == len(lists[2]) < w.Nv * (w.Nv + 1) // 2
        assert not np.array_equal(lists[0], lists[1])          # same P, other pairs: the case the old plan check missed
    finally:
        bse.bse_destroy(h)


@pytest.mark.parametrize("n", [16, 32, 36, 40, 60, 80, 100, 128])
def test_every_supported_grid_edge(n):
    """the grid edges no other test touches (each has its own Geo<R1,R2> instantiation), as the problem grid in
    the REAL layout and, tau on H, in the PW layout (which runs on whatever apply grid n_a >= 3R+1 the library picks)."""
    bse = _bse()
    R = max(2, n // 5)
    L = 10.0
    ecut = 0.5 * (2.0 * np.pi / L) ** 2 * (R * R + 0.5)
    cfg = wl.Config(f"n{n}", L, n, 3, 5, ecut, 1.6, 0.8, 3.0, 0.0, 1, "random", seed=400 + n)
    w = wl.make(cfg=cfg)
    _check_full(w, check_g=True)
    _check_pw(w, bse.BSE_TAU_PW)


@pytest.mark.parametrize("n", [12, 16, 20, 24, 30, 32, 36, 40, 48, 60, 64, 72, 80, 96, 100, 108, 120, 128, 144, 160])
def test_pipelined_plane_passes_every_grid_edge(n):
    """The pipelined plane passes (fft_pipe.cuh: persistent CTAs, cp.async.bulk staging on mbarriers, compact columns; the
    default only from n = 100 on) forced on every supported grid edge: pair densities + inverse pass in the REAL layout,
    single-field forward / slab inverse in the PW layout, with the slab height the launcher picks and with 3 lines per
    slab (several slabs, the last one ragged where 3 does not divide n / 2)."""
    bse = _bse()
    R = max(2, min(n // 5, 12))
    L = 10.0
    ecut = 0.5 * (2.0 * np.pi / L) ** 2 * (R * R + 0.5)
    big = n >= 120                               # the oracle's own FFT takes seconds per field there: fewer fields
    cfg = wl.Config(f"p{n}", L, n, 2 if big else 3, 5, ecut, 1.6, 0.8, 3.0, 0.0, 1 if big else 2, "random", seed=700 + n)
    w = wl.make(cfg=cfg)
    tab = orc.Tables(w.n, w.L, w.ecut)
    pairs_ref, _ = orc.screen_pairs(w.u, w.eta)
    tau_ref = orc.build_tau(tab, w.u, w.phi, w.lam, pairs_ref, want="r")
    o1 = _check_full(w, check_g=True, knobs={"pipe": 1}, tau_ref=tau_ref)
    if n < 96:                                   # (every oracle apply costs seconds from there on)
        o2 = _check_full(w, check_g=False, knobs={"pipe": 1, "pipe_lc": 3}, tau_ref=tau_ref)
        o0 = _check_full(w, check_g=False, knobs={"pipe": 0}, tau_ref=tau_ref)
        assert rel(o1, o0) < 1e-12 and rel(o2, o0) < 1e-12
        _check_pw(w, bse.BSE_TAU_PW, {"pipe": 1})
    _check_pw(w, bse.BSE_TAU_STREAM, {"pipe": 1, "pipe_lc": 3, "slab_planes": 2})


def test_compact_inverse_kernel_subtract_epilogue():
    """the SUB epilogue of the compact inverse plane kernel (P_c update of the REAL layout, taken from N_v >= 48
    with band-limited orbitals) forced on a small grid."""
    cfg = wl.Config("sub", 12.0, 24, 48, 24, 5.5, 1.3, 0.8, 3.0, 0.1, 2, "random", seed=95)
    w = wl.make(cfg=cfg)
    o1 = _check_full(w, check_g=False, knobs={"compact_inv": 2})
    o0 = _check_full(w, check_g=False, knobs={"compact_inv": 0})
    assert rel(o1, o0) < 1e-12


def test_plane_slab_apply_matches_the_group_path():
    """PW layout with tau on H: the plane-slab streaming apply (default: one slab of planes at a time, all blocks and all
    pairs resident, slab stick passes) against the oracle, with ragged row chunks, and against the group / row-batch path
    it replaces (knob slab_rows = -1).  Apply grids 20 / 24, 30 and 12, split into slabs of 6, 5, 4, 3 or 2 planes."""
    bse = _bse()
    for cfg in (wl.Config("slab", 10.0, 24, 9, 20, 8.0, 1.2, 0.8, 3.0, 0.02, 5, "random", seed=77),
                wl.Config("slab", 14.0, 30, 7, 16, 5.0, 1.3, 0.8, 3.0, 0.0, 3, "random", seed=311),
                wl.Config("slab", 9.0, 12, 5, 7, 3.0, 1.3, 0.8, 3.0, 0.05, 2, "random", seed=112)):
        w = wl.make(cfg=cfg)
        for tau in (bse.BSE_TAU_PW, bse.BSE_TAU_STREAM):
            o_def = _check_pw(w, tau)                                           # small grid: one slab holds every plane
            o_rag = _check_pw(w, tau, {"slab_rows": 4, "slab_planes": 6})      # several slabs, ragged row chunks
            o_thin = _check_pw(w, tau, {"slab_planes": 2})
            o_old = _check_pw(w, tau, {"slab_rows": -1})
            assert rel(o_rag, o_def) < 1e-12 and rel(o_thin, o_def) < 1e-12 and rel(o_old, o_def) < 1e-12


def test_row_sharded_handles_reproduce_the_full_apply():
    """SURVEY 8(f) #3 on one GPU: handles that own the row blocks [0, 4), [4, 7), [7, 9) (one after the other, nothing waits on
    anything) build tau only for the pairs that touch their rows and together reproduce the unsharded K1x output; the pieces
    are also compared with the oracle through the full result."""
    bse = _bse()
    cfg = wl.Config("shard", 10.0, 24, 9, 20, 8.0, 1.2, 0.8, 3.0, 0.02, 3, "random", seed=77)
    w = wl.make(cfg=cfg)
    for tau in (bse.BSE_TAU_PW, bse.BSE_TAU_STREAM):
        full = _check_pw(w, tau)                                              # [B][Nv][npw_h], checked against the oracle
        B, Nv, npw_h = full.shape
        a_d = torch.from_numpy(np.ascontiguousarray(w.a_pw).view(np.float64)).to("cuda:0")
        pieces = []
        for v0, v1 in ((0, 4), (4, 7), (7, 9)):
            g = Gpu(w, tau | bse.BSE_VEC_PW, {"slab_planes": 6})
            try:
                bse.bse_set_rows(g.h, v0, v1)
                g.build()
                out = torch.empty((B, v1 - v0, npw_h, 2), dtype=torch.float64, device="cuda:0")
                bse.bse_apply_k1x(g.h, a_d, out, B)
                torch.cuda.synchronize()
                pieces.append(out.cpu().numpy().view(np.complex128)[..., 0])
            finally:
                g.close()
        got = np.concatenate(pieces, axis=1)
        assert rel(got, full) < 1e-13
    g = Gpu(w, 0)
    try:
        with pytest.raises(bse.BseError) as e:
            bse.bse_set_rows(g.h, 0, 4)                                       # REAL layout: not supported
        assert e.value.code == bse.BSE_EUNSUPPORTED
    finally:
        g.close()


def test_k1e_split_over_row_blocks():
    """SURVEY 8(f) #3, K1e part: the Hartree shares of row blocks (bse_k1e_hartree_partial) summed - the all-reduce a
    multi-GPU run does - then bse_k1e_from_hartree on every block reproduce bse_apply_k1e and the oracle."""
    bse = _bse()
    cfg = wl.Config("k1es", 10.0, 24, 9, 20, 8.0, 1.2, 0.8, 3.0, 0.02, 3, "random", seed=78)
    w = wl.make(cfg=cfg)
    tab = orc.Tables(w.n, w.L, w.ecut)
    ref = orc.apply_k1e_pw(tab, w.u, w.a_pw)
    B, Nv, npw_h = ref.shape
    g = Gpu(w, bse.BSE_TAU_PW | bse.BSE_VEC_PW)
    try:
        blocks = ((0, 4), (4, 7), (7, 9))
        a_d = torch.from_numpy(np.ascontiguousarray(w.a_pw).view(np.float64)).to("cuda:0").reshape(B, Nv, npw_h, 2)
        vG = torch.zeros((B, npw_h, 2), dtype=torch.float64, device="cuda:0")
        for v0, v1 in blocks:
            share = torch.empty_like(vG)
            bse.bse_k1e_hartree_partial(g.h, a_d[:, v0:v1].contiguous(), v0, v1, B, share)
            vG += share                                                       # what the all-reduce does
        pieces = []
        for v0, v1 in blocks:
            out = torch.empty((B, v1 - v0, npw_h, 2), dtype=torch.float64, device="cuda:0")
            bse.bse_k1e_from_hartree(g.h, vG, v0, v1, B, out)
            torch.cuda.synchronize()
            pieces.append(out.cpu().numpy().view(np.complex128)[..., 0])
        got = np.concatenate(pieces, axis=1)
        wt = np.full(tab.npw_h, 2.0)
        wt[0] = 1.0
        err = np.sqrt((wt * np.abs(got - ref) ** 2).sum() / (wt * np.abs(ref) ** 2).sum())
        assert err <= TOL, err
    finally:
        g.close()


def test_sharded_driver_single_rank():
    """paper_2409_15116_b200/sharded.py end to end on one rank (world size 1, no collective to wait on): K1e and K1d rows
    against the oracle."""
    bse = _bse()
    from paper_2409_15116_b200 import sharded

    class _NoDist:
        @staticmethod
        def is_initialized():
            return False

    cfg = wl.Config("shd", 10.0, 24, 8, 16, 8.0, 1.2, 0.8, 3.0, 0.02, 2, "random", seed=83)
    w = wl.make(cfg=cfg)
    tab = orc.Tables(w.n, w.L, w.ecut)
    pairs, _ = orc.screen_pairs(w.u, w.eta)
    tau_ref = orc.build_tau(tab, w.u, w.phi, w.lam, pairs, want="r")
    ref_x = orc.apply_k1x_pw(tab, w.u, pairs, tau_ref, w.a_pw)
    ref_e = orc.apply_k1e_pw(tab, w.u, w.a_pw)
    dev = torch.device("cuda:0")
    u_d = torch.from_numpy(w.u).to(dev)
    phi_d = torch.from_numpy(np.ascontiguousarray(w.phi).view(np.float64)).to(dev)
    sh = sharded.ShardedBSE([w.n] * 3, w.cell, w.ecut, w.Nv, u_d, w.phi.shape[0], phi_d, w.lam, w.eta, bse.BSE_TAU_PW, 0, 1,
                            _NoDist, dev)
    try:
        sh.build()
        B, Nv, npw_h = ref_x.shape
        a_d = torch.from_numpy(np.ascontiguousarray(w.a_pw).view(np.float64)).to(dev).reshape(B, Nv, npw_h, 2)
        out_e, out_x = torch.empty_like(a_d), torch.empty_like(a_d)
        sh.apply(a_d, out_e, out_x)
        torch.cuda.synchronize()
        wt = np.full(tab.npw_h, 2.0)
        wt[0] = 1.0
        for got_d, ref in ((out_e, ref_e), (out_x, ref_x)):
            got = got_d.cpu().numpy().view(np.complex128)[..., 0]
            assert np.sqrt((wt * np.abs(got - ref) ** 2).sum() / (wt * np.abs(ref) ** 2).sum()) <= TOL
    finally:
        sh.close()


@pytest.mark.parametrize("tau", ["pw", "stream"])
def test_single_precision_tau_store(tau):
    """Mixed-precision variant (BSE_TAU_F32): tau(G) computed in fp64 and kept as complex64.  Against the oracle
    with the same single rounding (tau_G_f32) the K1x output agrees to ~1e-9 (the two sides may round a coefficient that sits
    on a binary32 tie differently: 2^-24 on that one coefficient); against the all-double oracle the error is the rounding
    itself, 2^-24 = 6e-8 relative per coefficient, i.e. between 1e-9 and 2e-7 in the L2 norm - derived from the arithmetic, not
    the 1e-10 bar of the double store.  Slab path and group path."""
    bse = _bse()
    flag = {"pw": bse.BSE_TAU_PW, "stream": bse.BSE_TAU_STREAM}[tau] | bse.BSE_TAU_F32 | bse.BSE_VEC_PW
    cfg = wl.Config("f32", 10.0, 24, 9, 20, 8.0, 1.2, 0.8, 3.0, 0.02, 3, "random", seed=77)
    w = wl.make(cfg=cfg)
    tab = orc.Tables(w.n, w.L, w.ecut)
    pairs, _ = orc.screen_pairs(w.u, w.eta)
    phiS = tab.expand_H_to_S(w.phi)
    tau32 = np.array([tab.to_r(orc.tau_G_f32(tab, w.u[v], w.u[x], phiS, w.lam)) for v, x in pairs])
    tau64 = orc.build_tau(tab, w.u, w.phi, w.lam, pairs, want="r")
    ref32 = orc.apply_k1x_pw(tab, w.u, pairs, tau32, w.a_pw)
    ref64 = orc.apply_k1x_pw(tab, w.u, pairs, tau64, w.a_pw)
    wt = np.full(tab.npw_h, 2.0)
    wt[0] = 1.0

    def err(got, ref):
        return float(np.sqrt((wt * np.abs(got - ref) ** 2).sum() / (wt * np.abs(ref) ** 2).sum()))
    assert 1e-9 < err(ref32, ref64) < 2e-7
    for knobs in (None, {"slab_planes": 6, "slab_rows": 4}):
        g = Gpu(w, flag, knobs)
        try:
            assert np.array_equal(g.build(), pairs)
            a_d = torch.from_numpy(np.ascontiguousarray(w.a_pw).view(np.float64)).to("cuda:0")
            out = torch.empty_like(a_d)
            bse.bse_apply_k1x(g.h, a_d, out, w.a_pw.shape[0])
            torch.cuda.synchronize()
            got = out.cpu().numpy().view(np.complex128).reshape(ref32.shape)
            assert err(got, ref32) <= 2e-9, err(got, ref32)
            assert 1e-9 < err(got, ref64) < 2e-7
            # bse_get_tau still hands out the double values
            assert rel(g.tau_g(0, 3), orc.build_tau(tab, w.u, w.phi, w.lam, pairs[:3], want="G")) <= TOL
        finally:
            g.close()
    u = torch.from_numpy(w.u).cuda()
    phi = torch.from_numpy(np.ascontiguousarray(w.phi).view(np.float64)).cuda()
    with pytest.raises(bse.BseError) as e:
        bse.bse_create([w.n] * 3, w.cell, w.ecut, w.Nv, u, w.phi.shape[0], phi, w.lam, w.eta, bse.BSE_TAU_REAL | bse.BSE_TAU_F32)
    assert e.value.code == bse.BSE_EINVAL


@pytest.mark.parametrize("tau", ["stream", "pw"])
def test_host_pointer_apply_with_overlapped_copies(tau):
    """bse_apply_k1x_host in the non-pipelined form: a is copied in while tau is rebuilt (STREAM), and P_c's row chunks
    (capped at 64 rows here: 3 chunks, the last one ragged) leave for the host one by one.  Same result as the device call."""
    bse = _bse()
    cfg = wl.Config("h2", 10.0, 24, 40, 20, 8.0, 1.2, 0.8, 3.0, 0.05, 4, "random", seed=93)
    w = wl.make(cfg=cfg)
    tab = orc.Tables(w.n, w.L, w.ecut)
    phi = np.ascontiguousarray(w.phi).view(np.float64)
    flag = {"stream": bse.BSE_TAU_STREAM, "pw": bse.BSE_TAU_PW}[tau]
    h = bse.bse_create([w.n] * 3, w.cell, w.ecut, w.Nv, np.ascontiguousarray(w.u), w.phi.shape[0], phi, w.lam, w.eta,
                       bse.BSE_PTR_HOST | flag | bse.BSE_VEC_PW)
    try:
        bse.bse_debug_set(h, "pc_rows", 64)
        bse.bse_debug_set(h, "in_chunks", 8)                     # u arrives in 7 column slabs (the last one ragged): the screen
        u_pin = torch.from_numpy(np.ascontiguousarray(w.u)).pin_memory()         # accumulates slab after slab behind the copy
        phi_pin = torch.from_numpy(phi).pin_memory()
        bse.bse_set_inputs_host(h, u_pin, phi_pin)
        bse.bse_build_tau(h)
        pairs = bse.bse_get_pairs(h)
        assert np.array_equal(pairs, orc.screen_pairs(w.u, w.eta)[0])
        a = torch.from_numpy(np.ascontiguousarray(w.a_pw).view(np.float64)).pin_memory()
        out = torch.full(a.shape, float("nan"), dtype=torch.float64).pin_memory()
        for _ in range(2):                                       # the second call reuses streams, events and staging
            out.fill_(float("nan"))
            bse.bse_apply_k1x_host(h, a, out, w.a_pw.shape[0])
            tau_ref = orc.build_tau(tab, w.u, w.phi, w.lam, pairs, want="r")
            ref = orc.apply_k1x_pw(tab, w.u, pairs, tau_ref, w.a_pw)
            got = out.numpy().view(np.complex128).reshape(ref.shape)
            wt = np.full(tab.npw_h, 2.0)
            wt[0] = 1.0
            err = np.sqrt((wt * np.abs(got - ref) ** 2).sum() / (wt * np.abs(ref) ** 2).sum())
            assert err <= TOL, err
    finally:
        bse.bse_destroy(h)

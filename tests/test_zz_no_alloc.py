"""bse_screen_overlap_static (include/bse.h): the allocation-free variant of the screen a1 (eq. 16) against the
existing path (bse_build_tau + bse_get_overlap), on two calls in a row that share the static scratch array.

Collected last on purpose (the suite runs with pytest -x): a failure here hides no other test.
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from paper_2409_15116_b200 import workloads as wl         # noqa: E402

TOL = 1e-10


def _bse():
    from paper_2409_15116_b200 import bse
    return bse


def _existing_overlap(bse, w):
    """Normalised overlap matrix of the existing path: handle, bse_build_tau, bse_get_overlap."""
    u = torch.from_numpy(np.ascontiguousarray(w.u)).cuda()
    phi = torch.from_numpy(np.ascontiguousarray(w.phi).view(np.float64)).cuda()
    h = bse.bse_create([w.n] * 3, w.cell, w.ecut, w.Nv, u, w.phi.shape[0], phi, w.lam, w.eta, 0)
    try:
        bse.bse_build_tau(h)
        return bse.bse_get_overlap(h, w.Nv)
    finally:
        bse.bse_destroy(h)


def _check(M_dev, w, O_ref):
    M = M_dev.cpu().numpy()
    Nv = w.Nv
    iu = np.triu_indices(Nv)
    d = np.sqrt(np.diag(M))
    O = M / np.outer(d, d)
    assert np.linalg.norm(O[iu] - O_ref[iu]) <= TOL * np.linalg.norm(O_ref[iu])       # against the existing path
    f2 = np.asarray(w.u, dtype=np.float64) ** 2
    M_np = f2 @ f2.T                                                                    # the definition, raw scale
    assert np.linalg.norm(M[iu] - M_np[iu]) <= TOL * np.linalg.norm(M_np[iu])


def test_static_scratch_screen_matches_the_existing_path_on_two_calls_in_a_row():
    bse = _bse()
    wa = wl.make(2)                                              # Nv = 64, N = 64^3: many split-K slices of the scratch
    wb = wl.make(cfg=wl.Config("na", 9.0, 12, 5, 6, 3.0, 1.3, 0.8, 3.0, 0.05, 1, "random", seed=77))   # Nv = 5: ragged tile
    Oa, Ob = _existing_overlap(bse, wa), _existing_overlap(bse, wb)
    ua = torch.from_numpy(np.ascontiguousarray(wa.u)).cuda()
    ub = torch.from_numpy(np.ascontiguousarray(wb.u)).cuda()
    Ma = torch.full((wa.Nv, wa.Nv), float("nan"), dtype=torch.float64, device="cuda")
    Mb = torch.full((wb.Nv, wb.Nv), float("nan"), dtype=torch.float64, device="cuda")
    Ma2 = torch.full_like(Ma, float("nan"))
    stream = torch.cuda.current_stream().cuda_stream
    bse.bse_screen_overlap_static(ua, wa.Nv, wa.u.shape[1], Ma, stream)          # first call (resolves the array's address)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    # two calls in a row on one stream, no synchronisation between them: the second starts from the first one's scratch
    bse.bse_screen_overlap_static(ub, wb.Nv, wb.u.shape[1], Mb, stream)
    bse.bse_screen_overlap_static(ua, wa.Nv, wa.u.shape[1], Ma2, stream)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0                 # nothing was allocated or freed on the device
    _check(Ma, wa, Oa)
    _check(Mb, wb, Ob)
    _check(Ma2, wa, Oa)
    assert torch.equal(torch.triu(Ma), torch.triu(Ma2))          # same inputs, same split: bit-identical


def test_static_scratch_screen_rejects_what_does_not_fit():
    bse = _bse()
    # the limit itself is accepted: Nv = 1024 fills the array with one set of partial sums (split-K factor 1)
    g = torch.Generator().manual_seed(5)
    ul = torch.randn(bse.BSE_SCREEN_STATIC_MAX_NV, 96, dtype=torch.float64, generator=g)
    Ml = torch.empty(ul.shape[0], ul.shape[0], dtype=torch.float64, device="cuda")
    ul_d = ul.cuda()
    bse.bse_screen_overlap_static(ul_d, ul.shape[0], ul.shape[1], Ml)
    torch.cuda.synchronize()
    f2 = ul.numpy() ** 2
    iu = np.triu_indices(ul.shape[0])
    ref = (f2 @ f2.T)[iu]
    assert np.linalg.norm(Ml.cpu().numpy()[iu] - ref) <= TOL * np.linalg.norm(ref)
    u = torch.zeros(64, dtype=torch.float64, device="cuda")
    M = torch.zeros(64, dtype=torch.float64, device="cuda")
    with pytest.raises(bse.BseError) as e:
        bse.bse_screen_overlap_static(u, bse.BSE_SCREEN_STATIC_MAX_NV + 1, 2, M)
    assert e.value.code == bse.BSE_EINVAL and "static array holds" in str(e.value)
    with pytest.raises(bse.BseError) as e:
        bse.bse_screen_overlap_static(u, 4, 3, M)                # odd N: rows would not be 16-byte aligned
    assert e.value.code == bse.BSE_EINVAL
    with pytest.raises(bse.BseError) as e:
        bse.bse_screen_overlap_static(None, 4, 4, M)
    assert e.value.code == bse.BSE_EINVAL

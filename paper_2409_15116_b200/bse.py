"""Thin ctypes binding of libbse_b200 (include/bse.h): argument marshalling only.

Every step of the path runs in the CUDA kernels of the shared library; there is no CPU fallback and
no torch compute here.  torch is used by callers for device memory and streams.  Importing this
module fails loudly if the library has not been built (`python -m paper_2409_15116_b200.build`).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libbse_b200.so")
if not os.path.exists(LIB_PATH):
    raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2409_15116_b200.build` "
                      "(there is no CPU fallback)")
lib = C.CDLL(LIB_PATH)

BSE_OK, BSE_EINVAL, BSE_ENOMEM, BSE_ECUDA, BSE_ESTATE, BSE_EUNSUPPORTED = 0, -1, -2, -3, -4, -5
BSE_TAU_REAL, BSE_TAU_PW, BSE_TAU_STREAM = 0x0, 0x1, 0x2
BSE_VEC_REAL, BSE_VEC_PW, BSE_PTR_HOST, BSE_TAU_F32 = 0x0, 0x4, 0x8, 0x10
STAGES = ["screen_syrk", "pair_list", "fwd_plane", "fwd_stick", "pdep_project", "pdep_backproject",
          "inv_stick", "inv_plane", "k1x_accumulate", "pc_overlap", "pc_update", "k1e_density", "k1e_product"]
# kernels launched per stage invocation (bse_api.cu): split-K GEMMs launch GEMM + reduce, pair list 1 kernel
KERNELS_PER_STAGE = [2, 1, 1, 1, 2, 1, 1, 1, 1, 2, 1, 1, 1]

_vp, _i, _d, _u, _ll = C.c_void_p, C.c_int, C.c_double, C.c_uint, C.c_longlong
_sig = {
    "bse_create": [C.POINTER(_vp), C.POINTER(_i), C.POINTER(_d), _d, _i, _vp, _i, _vp, C.POINTER(_d), _d, _u, _vp],
    "bse_build_tau": [_vp],
    "bse_apply_k1x": [_vp, _vp, _vp, _i],
    "bse_apply_k1x_host": [_vp, _vp, _vp, _i],
    "bse_apply_k1e": [_vp, _vp, _vp, _i],
    "bse_rotate": [_vp, _vp, _i, _vp, _vp, _i],
    "bse_apply_k1": [_vp, _vp, _vp, _i, _d, _d],
    "bse_set_inputs_host": [_vp, _vp, _vp],
    "bse_jade": [C.POINTER(_i), C.POINTER(_d), _i, _vp, _vp, _vp, _d, _i, _i, C.POINTER(_i), C.POINTER(_d), _vp],
    "bse_destroy": [_vp],
    "bse_npw_half": [_vp, C.POINTER(_ll)],
    "bse_gvectors": [_vp, _vp],
    "bse_num_pairs": [_vp, C.POINTER(_ll)],
    "bse_get_pairs": [_vp, _vp],
    "bse_get_overlap": [_vp, _vp],
    "bse_get_tau": [_vp, _ll, _ll, _vp, _u],
    "bse_debug_set": [_vp, C.c_char_p, _ll],
    "bse_set_rows": [_vp, _i, _i],
    "bse_k1e_hartree_partial": [_vp, _vp, _i, _i, _i, _vp],
    "bse_k1e_from_hartree": [_vp, _vp, _i, _i, _i, _vp],
    "bse_last_tau_fill_ms": [_vp, C.POINTER(_d)],
    "bse_profile_enable": [_vp, _i],
    "bse_profile_reset": [_vp],
    "bse_profile_get": [_vp, C.POINTER(_d), C.POINTER(_ll)],
    "bse_profile_model": [_vp, C.POINTER(_d), C.POINTER(_d)],
    "bse_profile_handoff": [_vp, C.POINTER(_d)],
    "bse_probe_fp64_peak": [C.POINTER(_d), C.POINTER(_d), _vp],
    "bse_screen_overlap_static": [_vp, _i, _ll, _vp, _vp],
}
for _name, _args in _sig.items():
    getattr(lib, _name).argtypes = _args
    getattr(lib, _name).restype = _i
lib.bse_last_error.restype = C.c_char_p
lib.bse_version.restype = C.c_char_p
lib.bse_stage_name.restype = C.c_char_p
lib.bse_stage_name.argtypes = [_i]
EXPORTS = list(_sig) + ["bse_last_error", "bse_version", "bse_stage_name"]


class BseError(RuntimeError):
    def __init__(self, code, where):
        self.code = code
        super().__init__(f"{where} failed with status {code}: {lib.bse_last_error().decode()}")


def _check(code, where):
    if code != BSE_OK:
        raise BseError(code, where)


def _ptr(x):
    """Raw address of a torch tensor / numpy array / int."""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    if isinstance(x, np.ndarray):
        return x.ctypes.data
    return x.data_ptr()


def bse_create(grid, cell, ecut, Nv, u, Npdep, phi, lam, eta, flags=0, stream=None):
    h = _vp()
    g = (_i * 3)(*[int(v) for v in grid])
    c = (_d * 9)(*[float(v) for v in np.asarray(cell, dtype=np.float64).ravel()])
    lam = np.ascontiguousarray(lam, dtype=np.float64)
    _check(lib.bse_create(C.byref(h), g, c, float(ecut), int(Nv), _ptr(u), int(Npdep), _ptr(phi),
                          lam.ctypes.data_as(C.POINTER(_d)), float(eta), int(flags), _ptr(stream)), "bse_create")
    return h


def bse_build_tau(h):
    _check(lib.bse_build_tau(h), "bse_build_tau")


def bse_apply_k1x(h, a, out, B):
    _check(lib.bse_apply_k1x(h, _ptr(a), _ptr(out), int(B)), "bse_apply_k1x")


def bse_apply_k1e(h, a, out, B):
    _check(lib.bse_apply_k1e(h, _ptr(a), _ptr(out), int(B)), "bse_apply_k1e")


def bse_apply_k1(h, a, out, B, ce=1.0, cd=-1.0):
    _check(lib.bse_apply_k1(h, _ptr(a), _ptr(out), int(B), float(ce), float(cd)), "bse_apply_k1")


def bse_rotate(h, U, x, y, B, transpose=False):
    _check(lib.bse_rotate(h, _ptr(U), 1 if transpose else 0, _ptr(x), _ptr(y), int(B)), "bse_rotate")


def bse_jade(grid, cell, Nv, psi, U, psi_loc=None, tol=1e-14, max_sweeps=60, init_eig=True, stream=None):
    """Returns (sweeps done, sigma^2 before, sigma^2 after); U (and psi_loc) are written on the device."""
    g = (_i * 3)(*[int(v) for v in grid])
    c = (_d * 9)(*[float(v) for v in np.asarray(cell, dtype=np.float64).ravel()])
    sw = _i()
    sp = (_d * 2)()
    _check(lib.bse_jade(g, c, int(Nv), _ptr(psi), _ptr(U), _ptr(psi_loc), float(tol), int(max_sweeps), 1 if init_eig else 0,
                        C.byref(sw), sp, _ptr(stream)), "bse_jade")
    return sw.value, sp[0], sp[1]


def bse_apply_k1x_host(h, a_host, out_host, B):
    _check(lib.bse_apply_k1x_host(h, _ptr(a_host), _ptr(out_host), int(B)), "bse_apply_k1x_host")


def bse_set_inputs_host(h, u_host=None, phi_host=None):
    _check(lib.bse_set_inputs_host(h, _ptr(u_host), _ptr(phi_host)), "bse_set_inputs_host")


def bse_destroy(h):
    _check(lib.bse_destroy(h), "bse_destroy")


def bse_npw_half(h):
    v = _ll()
    _check(lib.bse_npw_half(h, C.byref(v)), "bse_npw_half")
    return v.value


def bse_gvectors(h):
    m = np.empty((bse_npw_half(h), 3), dtype=np.int32)
    _check(lib.bse_gvectors(h, m.ctypes.data), "bse_gvectors")
    return m


def bse_num_pairs(h):
    v = _ll()
    _check(lib.bse_num_pairs(h, C.byref(v)), "bse_num_pairs")
    return v.value


def bse_get_pairs(h):
    p = np.empty((bse_num_pairs(h), 2), dtype=np.int32)
    _check(lib.bse_get_pairs(h, p.ctypes.data), "bse_get_pairs")
    return p


def bse_get_overlap(h, Nv):
    o = np.empty((Nv, Nv), dtype=np.float64)
    _check(lib.bse_get_overlap(h, o.ctypes.data), "bse_get_overlap")
    return o


BSE_SCREEN_STATIC_BYTES, BSE_SCREEN_STATIC_MAX_NV = 8 << 20, 1024


def bse_screen_overlap_static(u, Nv, N, M, stream=None):
    """Allocation-free screen (include/bse.h): u DEVICE [Nv][N], M DEVICE [Nv][Nv] (v <= w defined); enqueued on `stream`."""
    _check(lib.bse_screen_overlap_static(_ptr(u), int(Nv), int(N), _ptr(M), _ptr(stream)), "bse_screen_overlap_static")


def bse_get_tau(h, first, count, dst, layout=BSE_TAU_REAL):
    _check(lib.bse_get_tau(h, int(first), int(count), _ptr(dst), int(layout)), "bse_get_tau")


def bse_set_rows(h, v0, v1):
    _check(lib.bse_set_rows(h, int(v0), int(v1)), "bse_set_rows")


def bse_k1e_hartree_partial(h, a_rows, v0, v1, B, vG):
    _check(lib.bse_k1e_hartree_partial(h, _ptr(a_rows), int(v0), int(v1), int(B), _ptr(vG)), "bse_k1e_hartree_partial")


def bse_k1e_from_hartree(h, vG, v0, v1, B, out_rows):
    _check(lib.bse_k1e_from_hartree(h, _ptr(vG), int(v0), int(v1), int(B), _ptr(out_rows)), "bse_k1e_from_hartree")


def bse_debug_set(h, key, value):
    _check(lib.bse_debug_set(h, str(key).encode(), int(value)), "bse_debug_set")


def bse_last_tau_fill_ms(h):
    v = _d()
    _check(lib.bse_last_tau_fill_ms(h, C.byref(v)), "bse_last_tau_fill_ms")
    return v.value


def bse_profile_enable(h, on=True):
    _check(lib.bse_profile_enable(h, 1 if on else 0), "bse_profile_enable")


def bse_profile_reset(h):
    _check(lib.bse_profile_reset(h), "bse_profile_reset")


def bse_profile_get(h):
    ms = (_d * len(STAGES))()
    ln = (_ll * len(STAGES))()
    _check(lib.bse_profile_get(h, ms, ln), "bse_profile_get")
    return {s: (ms[i], ln[i]) for i, s in enumerate(STAGES)}


def bse_profile_model(h):
    fl = (_d * len(STAGES))()
    by = (_d * len(STAGES))()
    _check(lib.bse_profile_model(h, fl, by), "bse_profile_model")
    return {s: (fl[i], by[i]) for i, s in enumerate(STAGES)}


def bse_profile_handoff(h):
    by = (_d * len(STAGES))()
    _check(lib.bse_profile_handoff(h, by), "bse_profile_handoff")
    return {s: by[i] for i, s in enumerate(STAGES)}


def bse_probe_fp64_peak(stream=None):
    a, b = _d(), _d()
    _check(lib.bse_probe_fp64_peak(C.byref(a), C.byref(b), _ptr(stream)), "bse_probe_fp64_peak")
    return a.value, b.value

"""Python binding of libhr (include/hr.h): the B200-native Wilson-Dirac hopping term Dphi for
higher-representation SU(N) fermions (arxiv 2405.19294 hot path; BASELINE.json:north_star).

Argument marshalling only: every step of the path runs in the CUDA kernels of libhr.so.  The
functions below carry the names of the C ABI (hr_ctx_create, hr_gauge_alloc, hr_represent_links,
hr_dphi_eo, hr_dirac, ...) and raise HrError on any non-zero hr_status.  `Lattice` is a small
convenience wrapper that owns the handles and uses torch only for device memory and streams.

There is NO CPU fallback: if libhr.so is missing, importing this package compiles it in-tree with
nvcc (paper_2405_19294_b200/build.py); if that fails the import raises, and on a box without a CUDA
device every compute call raises HrError(HR_ECUDA).
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libhr.so")

HR_OK, HR_EINVAL, HR_EUNSUPPORTED, HR_ECUDA, HR_ENOMEM = 0, -1, -2, -3, -4
HR_F64, HR_F32 = 0, 1
HR_REP_FUND, HR_REP_ADJ, HR_REP_SYM, HR_REP_ASYM = 0, 1, 2, 3
REP_NAMES = {"fund": HR_REP_FUND, "adj": HR_REP_ADJ, "sym": HR_REP_SYM, "asym": HR_REP_ASYM}
PREC_NAMES = {"f64": HR_F64, "f32": HR_F32}


class HrError(RuntimeError):
    def __init__(self, status: int, text: str):
        super().__init__(f"libhr status {status}: {text}")
        self.status = status


if not os.path.exists(LIB_PATH):
    from . import build as _build  # pure python; compiles csrc/*.cu with nvcc for sm_100a
    try:
        _build.build()
    except Exception as exc:  # no CPU fallback: without the CUDA library there is no product
        raise ImportError(
            f"{LIB_PATH} is missing and could not be built ({exc}); "
            "there is no CPU fallback for the CUDA path") from exc

_vp, _ci, _cd, _sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_size_t
_I4 = ctypes.c_int * 4
_D2 = ctypes.c_double * 2
_D2P = ctypes.POINTER(ctypes.c_double)

# every symbol include/hr.h declares: name -> (restype, argtypes)
_SIGNATURES = {
    "hr_version": (ctypes.c_char_p, []),
    "hr_last_error": (ctypes.c_char_p, []),
    "hr_ctx_create": (_ci, [ctypes.POINTER(_vp), _I4, _I4, _ci, _ci, _ci]),
    "hr_ctx_destroy": (None, [_vp]),
    "hr_rep_dim": (_ci, [_vp]),
    "hr_links_are_real": (_ci, [_vp]),
    "hr_half_volume": (_sz, [_vp]),
    "hr_gauge_bytes": (_sz, [_vp, _ci, _ci]),
    "hr_spinor_bytes": (_sz, [_vp, _ci]),
    "hr_gauge_alloc": (_ci, [_vp, _ci, _ci, _vp, ctypes.POINTER(_vp)]),
    "hr_gauge_free": (None, [_vp]),
    "hr_gauge_data": (_vp, [_vp]),
    "hr_gauge_import": (_ci, [_vp, _vp, _ci, _vp]),
    "hr_gauge_export": (_ci, [_vp, _vp, _ci, _vp]),
    "hr_spinor_import": (_ci, [_vp, _vp, _ci, _vp, _ci, _ci, _vp]),
    "hr_spinor_export": (_ci, [_vp, _vp, _ci, _vp, _ci, _ci, _vp]),
    "hr_represent_links": (_ci, [_vp, _vp, _vp]),
    "hr_gauge_compress": (_ci, [_vp, _vp, _vp]),
    "hr_dphi_eo": (_ci, [_vp, _vp, _vp, _ci, _vp]),
    "hr_dirac": (_ci, [_cd, _vp, _vp, _vp, _vp]),
    "hr_dphi_eo_host": (_ci, [_vp, _vp, _vp, _ci, _vp, _ci, _vp]),
    "hr_spinor_lincomb": (_ci, [_vp, _ci, _vp, _D2, _ci, _vp, _D2P, _vp, _vp]),
    "hr_spinor_copy": (_ci, [_vp, _ci, _vp, _vp, _vp]),
    "hr_spinor_g5": (_ci, [_vp, _ci, _vp, _vp, _vp]),
    "hr_spinor_mulc_add_assign": (_ci, [_vp, _ci, _vp, _cd, _cd, _vp, _vp]),
    "hr_spinor_g5_mulc_add_assign": (_ci, [_vp, _ci, _vp, _cd, _cd, _vp, _vp]),
    "hr_spinor_dot": (_ci, [_vp, _ci, _vp, _vp, _vp, _vp]),
    "hr_spinor_norm2": (_ci, [_vp, _ci, _vp, _vp, _vp]),
    "hr_spinor_dot_noalloc_max_bytes": (_sz, []),
    "hr_spinor_dot_noalloc": (_ci, [_vp, _ci, _vp, _vp, _vp, _vp]),
    "hr_dhat": (_ci, [_cd, _ci, _vp, _vp, _vp, _vp, _vp]),
    "hr_cg_workspace_bytes": (_sz, [_vp, _ci, _ci]),
    "hr_cg_dhat": (_ci, [_vp, _cd, _vp, _vp, _vp, _cd, _ci, _vp, ctypes.POINTER(_ci), ctypes.POINTER(_cd), _vp, _vp]),
    "hr_cg_dist_workspace_bytes": (_sz, [_vp, _ci]),
    "hr_cg_dhat_dist": (_ci, [_vp, _ci, _cd, _vp, _vp, _cd, _ci, _vp, _vp, _vp, _vp, ctypes.POINTER(_ci), ctypes.POINTER(_cd), _vp]),
    "hr_bicgstab_workspace_bytes": (_sz, [_vp, _ci, _ci]),
    "hr_bicgstab_dhat": (_ci, [_vp, _cd, _vp, _vp, _vp, _cd, _ci, _vp, ctypes.POINTER(_ci), ctypes.POINTER(_cd), _vp, _vp]),
    "hr_qmr_workspace_bytes": (_sz, [_vp, _ci]),
    "hr_qmr_dhat": (_ci, [_vp, _cd, _vp, _vp, _vp, _cd, _ci, _vp, ctypes.POINTER(_ci), ctypes.POINTER(_cd), _vp, _vp]),
    "hr_dirac_solve": (_ci, [_vp, _cd, _vp, _vp, _vp, _cd, _ci, _vp, ctypes.POINTER(_ci), ctypes.POINTER(_cd), _vp]),
    "hr_halo_bytes": (_sz, [_vp, _ci]),
    "hr_face_bytes": (_sz, [_vp, _ci, _ci]),
    "hr_dphi_eo_face_pack": (_ci, [_ci, _vp, _vp, _vp, _vp, _ci, _vp]),
    "hr_dphi_eo_faces_pack": (_ci, [_ci, ctypes.POINTER(_vp), ctypes.POINTER(_vp), _vp, _vp, _ci, _vp]),
    "hr_dphi_eo_faces_apply": (_ci, [_ci, _vp, ctypes.POINTER(_vp), ctypes.POINTER(_vp), _vp, _ci, _ci, _ci, _vp]),
    "hr_dphi_eo_interior_mask": (_ci, [_vp, _vp, _vp, _ci, _ci, _vp]),
    "hr_dphi_eo_face_apply": (_ci, [_ci, _vp, _vp, _vp, _vp, _ci, _ci, _ci, _vp]),
    "hr_halo_buffers_alloc": (_ci, [_vp, _ci, ctypes.POINTER(_vp)]),
    "hr_face_buffers_alloc": (_ci, [_vp, _ci, _ci, ctypes.POINTER(_vp)]),
    "hr_halo_buffers_free": (None, [_vp, _vp]),
    "hr_ipc_export": (_ci, [_vp, _vp, ctypes.c_char_p]),
    "hr_ipc_open": (_ci, [_vp, ctypes.c_char_p, ctypes.POINTER(_vp)]),
    "hr_ipc_close": (_ci, [_vp, _vp]),
    "hr_dphi_eo_halo_pack": (_ci, [_vp, _vp, _vp, _vp, _ci, _vp]),
    "hr_dphi_eo_interior": (_ci, [_vp, _vp, _vp, _ci, _vp]),
    "hr_dphi_eo_halo_apply": (_ci, [_vp, _vp, _vp, _vp, _ci, _ci, _ci, _vp]),
    "hr_clover_bytes": (_sz, [_vp, _ci]),
    "hr_clover_build": (_ci, [_vp, _vp, _cd, _vp]),
    "hr_clover_exp": (_ci, [_vp, _ci, _vp, _cd, _vp]),
    "hr_dirac_clover": (_ci, [_cd, _vp, _vp, _vp, _vp, _vp]),
    "hr_clover_finalize": (_ci, [_vp, _ci, _vp, _vp, _cd, _vp]),
    "hr_dhat_clover": (_ci, [_vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp]),
    "hr_clover_solve_workspace_bytes": (_sz, [_vp, _ci, _ci]),
    "hr_dirac_clover_solve": (_ci, [_vp, _vp, _vp, _vp, _vp, _vp, _cd, _ci, _vp, ctypes.POINTER(_ci), ctypes.POINTER(_cd), _vp]),
    "hr_dirac_solve_bicgstab": (_ci, [_vp, _cd, _vp, _vp, _vp, _cd, _ci, _vp, ctypes.POINTER(_ci), ctypes.POINTER(_cd), _vp]),
    "hr_mixed_workspace_bytes": (_sz, [_vp, _ci]),
    "hr_bicgstab_dhat_mixed": (_ci, [_vp, _cd, _vp, _vp, _vp, _vp, _cd, _cd, _ci, _vp, ctypes.POINTER(_ci), ctypes.POINTER(_ci), ctypes.POINTER(_cd), _vp]),
    "hr_ctx_set_tuning": (_ci, [_vp, ctypes.c_char_p, _ci]),
    "hr_dphi_variant_name": (ctypes.c_char_p, [_vp, _ci]),
    "hr_launch_count": (ctypes.c_ulonglong, []),
}


def _bind():
    lib = ctypes.CDLL(LIB_PATH)
    for name, (res, args) in _SIGNATURES.items():
        f = getattr(lib, name)  # AttributeError here = the library does not export the header's symbol
        f.restype = res
        f.argtypes = args
    return lib


def _exports_all() -> bool:
    blob = open(LIB_PATH, "rb").read()
    return all(name.encode() + b"\0" in blob for name in _SIGNATURES)


if not _exports_all():
    # a libhr.so older than include/hr.h (left over from an earlier checkout): rebuild BEFORE loading it
    from . import build as _build
    _build.build(force=True)
_lib = _bind()


def _check(status: int) -> None:
    if status != HR_OK:
        raise HrError(status, _lib.hr_last_error().decode())


def _ptr(x) -> int:
    """Raw address of a torch tensor / numpy array / int / None."""
    if x is None:
        return 0
    if isinstance(x, int):
        return x
    if isinstance(x, np.ndarray):
        if not x.flags.c_contiguous:
            raise ValueError("numpy buffer must be C-contiguous")
        return x.ctypes.data
    if hasattr(x, "data_ptr"):
        if not x.is_contiguous():
            raise ValueError("tensor must be contiguous")
        return x.data_ptr()
    raise TypeError(f"cannot take the address of {type(x)}")


# ---- the C ABI, same names --------------------------------------------------------------------

def hr_version() -> str:
    return _lib.hr_version().decode()


def hr_last_error() -> str:
    return _lib.hr_last_error().decode()


def hr_launch_count() -> int:
    return int(_lib.hr_launch_count())


def hr_ctx_create(dims, bc, N: int, rep: int, device: int = 0) -> int:
    h = _vp()
    _check(_lib.hr_ctx_create(ctypes.byref(h), _I4(*[int(v) for v in dims]), _I4(*[int(v) for v in bc]), N, rep, device))
    return h.value


def hr_ctx_destroy(ctx: int) -> None:
    _lib.hr_ctx_destroy(ctx)


def hr_rep_dim(ctx: int) -> int:
    return _lib.hr_rep_dim(ctx)


def hr_links_are_real(ctx: int) -> int:
    return _lib.hr_links_are_real(ctx)


def hr_half_volume(ctx: int) -> int:
    return _lib.hr_half_volume(ctx)


def hr_gauge_bytes(ctx: int, represented: int, prec: int) -> int:
    return _lib.hr_gauge_bytes(ctx, represented, prec)


def hr_spinor_bytes(ctx: int, prec: int) -> int:
    return _lib.hr_spinor_bytes(ctx, prec)


def hr_gauge_alloc(ctx: int, represented: int, prec: int, dev_mem=None) -> int:
    g = _vp()
    _check(_lib.hr_gauge_alloc(ctx, represented, prec, _ptr(dev_mem), ctypes.byref(g)))
    return g.value


def hr_gauge_free(g: int) -> None:
    _lib.hr_gauge_free(g)


def hr_gauge_data(g: int) -> int:
    return _lib.hr_gauge_data(g) or 0


def hr_gauge_import(g: int, canon, canon_prec: int, stream: int = 0) -> None:
    _check(_lib.hr_gauge_import(g, _ptr(canon), canon_prec, stream))


def hr_gauge_export(g: int, canon, canon_prec: int, stream: int = 0) -> None:
    _check(_lib.hr_gauge_export(g, _ptr(canon), canon_prec, stream))


def hr_spinor_import(ctx: int, dst_dev, prec: int, canon, canon_prec: int, parity: int, stream: int = 0) -> None:
    _check(_lib.hr_spinor_import(ctx, _ptr(dst_dev), prec, _ptr(canon), canon_prec, parity, stream))


def hr_spinor_export(ctx: int, src_dev, prec: int, canon, canon_prec: int, parity: int, stream: int = 0) -> None:
    _check(_lib.hr_spinor_export(ctx, _ptr(src_dev), prec, _ptr(canon), canon_prec, parity, stream))


def hr_gauge_compress(rows_out: int, fund_in: int, stream: int = 0) -> None:
    _check(_lib.hr_gauge_compress(rows_out, fund_in, stream))


def hr_represent_links(repr_out: int, fund_in: int, stream: int = 0) -> None:
    _check(_lib.hr_represent_links(repr_out, fund_in, stream))


def hr_dphi_eo(out, inp, links: int, parity: int, stream: int = 0) -> None:
    _check(_lib.hr_dphi_eo(_ptr(out), _ptr(inp), links, parity, stream))


def hr_dirac(m0: float, out_full, in_full, links: int, stream: int = 0) -> None:
    _check(_lib.hr_dirac(float(m0), _ptr(out_full), _ptr(in_full), links, stream))


def hr_dphi_eo_host(ctx: int, out_canon, in_canon, canon_prec: int, links: int, parity: int, stream: int = 0) -> None:
    _check(_lib.hr_dphi_eo_host(ctx, _ptr(out_canon), _ptr(in_canon), canon_prec, links, parity, stream))


def hr_spinor_lincomb(ctx: int, prec: int, out, ca: complex, g5: int, x, cb: complex = 0j, y=None, stream: int = 0) -> None:
    ca, cb = complex(ca), complex(cb)
    cbp = ctypes.cast(_D2(cb.real, cb.imag), _D2P) if y is not None else None
    _check(_lib.hr_spinor_lincomb(ctx, prec, _ptr(out), _D2(ca.real, ca.imag), int(g5), _ptr(x), cbp, _ptr(y), stream))


def hr_spinor_copy(ctx: int, prec: int, out, inp, stream: int = 0) -> None:
    _check(_lib.hr_spinor_copy(ctx, prec, _ptr(out), _ptr(inp), stream))


def hr_spinor_g5(ctx: int, prec: int, out, inp, stream: int = 0) -> None:
    _check(_lib.hr_spinor_g5(ctx, prec, _ptr(out), _ptr(inp), stream))


def hr_spinor_mulc_add_assign(ctx: int, prec: int, out, c: complex, inp, stream: int = 0) -> None:
    c = complex(c)
    _check(_lib.hr_spinor_mulc_add_assign(ctx, prec, _ptr(out), c.real, c.imag, _ptr(inp), stream))


def hr_spinor_g5_mulc_add_assign(ctx: int, prec: int, out, c: complex, inp, stream: int = 0) -> None:
    c = complex(c)
    _check(_lib.hr_spinor_g5_mulc_add_assign(ctx, prec, _ptr(out), c.real, c.imag, _ptr(inp), stream))


def hr_spinor_dot(ctx: int, prec: int, x, y, stream: int = 0, result=None):
    """<x, y>; result=None: returned as a Python complex (host result, synchronises); else a device buffer."""
    if result is not None:
        _check(_lib.hr_spinor_dot(ctx, prec, _ptr(x), _ptr(y), _ptr(result), stream))
        return None
    r = _D2()
    _check(_lib.hr_spinor_dot(ctx, prec, _ptr(x), _ptr(y), ctypes.addressof(r), stream))
    return complex(r[0], r[1])


def hr_spinor_dot_noalloc_max_bytes() -> int:
    return _lib.hr_spinor_dot_noalloc_max_bytes()


def hr_spinor_dot_noalloc(ctx: int, prec: int, x, y, result, stream: int = 0) -> None:
    """<x, y> into the device buffer `result` (2 doubles); allocates nothing, does not synchronise (include/hr.h)."""
    _check(_lib.hr_spinor_dot_noalloc(ctx, prec, _ptr(x), _ptr(y), _ptr(result), stream))


def hr_spinor_norm2(ctx: int, prec: int, x, stream: int = 0, result=None):
    if result is not None:
        _check(_lib.hr_spinor_norm2(ctx, prec, _ptr(x), _ptr(result), stream))
        return None
    r = _cd()
    _check(_lib.hr_spinor_norm2(ctx, prec, _ptr(x), ctypes.addressof(r), stream))
    return float(r.value)


def hr_dhat(m0: float, g5: int, out_e, in_e, tmp_o, links: int, stream: int = 0) -> None:
    _check(_lib.hr_dhat(float(m0), int(g5), _ptr(out_e), _ptr(in_e), _ptr(tmp_o), links, stream))


def hr_cg_workspace_bytes(ctx: int, prec: int, maxiter: int) -> int:
    return _lib.hr_cg_workspace_bytes(ctx, prec, maxiter)


def hr_cg_dhat(ctx: int, m0: float, x_e, b_e, links: int, tol: float, maxiter: int, workspace, stream: int = 0, want_hist: bool = False):
    """Returns (iterations, |r|^2/|rhs|^2, history or None)."""
    it, res = _ci(0), _cd(0.0)
    hist = np.zeros(maxiter + 1, dtype=np.float64) if want_hist else None
    _check(_lib.hr_cg_dhat(ctx, float(m0), _ptr(x_e), _ptr(b_e), links, float(tol), int(maxiter), _ptr(workspace),
                           ctypes.byref(it), ctypes.byref(res), _ptr(hist), stream))
    return it.value, res.value, (hist[:it.value + 1] if want_hist else None)


_DPHI_FN = ctypes.CFUNCTYPE(_ci, _vp, _vp, _vp, _ci)
_ALLSUM_FN = ctypes.CFUNCTYPE(_ci, _vp, ctypes.POINTER(_cd), _ci)


def hr_cg_dist_workspace_bytes(ctx: int, prec: int) -> int:
    return int(_lib.hr_cg_dist_workspace_bytes(ctx, prec))


def hr_cg_dhat_dist(ctx: int, prec: int, m0: float, x_e, b_e, tol: float, maxiter: int, workspace, dphi, allsum=None, stream: int = 0):
    """CG on a distributed lattice, every step in libhr; `dphi(out_ptr, in_ptr, parity)` runs the caller's distributed
    Dphi_eo on `stream`, `allsum(list of floats) -> list of floats` sums over the ranks (None: one rank).
    Returns (iterations, [|r_k|^2 / |rhs|^2])."""
    err = []

    def _dphi(user, out, inp, parity):
        try:
            dphi(int(out), int(inp), int(parity))
            return 0
        except Exception as exc:  # an exception must not cross the C frames
            err.append(exc)
            return 1

    def _allsum(user, vals, n):
        try:
            res = allsum([vals[i] for i in range(n)])
            for i in range(n):
                vals[i] = res[i]
            return 0
        except Exception as exc:
            err.append(exc)
            return 1

    cb_d = _DPHI_FN(_dphi)
    cb_a = _ALLSUM_FN(_allsum) if allsum is not None else None
    iters = _ci(0)
    hist = (_cd * (maxiter + 1))()
    rc = _lib.hr_cg_dhat_dist(ctx, prec, m0, _ptr(x_e), _ptr(b_e), tol, maxiter, _ptr(workspace), ctypes.cast(cb_d, _vp),
                              ctypes.cast(cb_a, _vp) if cb_a is not None else None, None, ctypes.byref(iters), hist, stream)
    if err:
        raise err[0]
    _check(rc)
    return iters.value, [hist[i] for i in range(iters.value + 1)]


def hr_bicgstab_workspace_bytes(ctx: int, prec: int, maxiter: int) -> int:
    return _lib.hr_bicgstab_workspace_bytes(ctx, prec, maxiter)


def hr_bicgstab_dhat(ctx: int, m0: float, x_e, b_e, links: int, tol: float, maxiter: int, workspace, stream: int = 0, want_hist: bool = False):
    """Returns (iterations, |r|^2/|b|^2, history or None)."""
    it, res = _ci(0), _cd(0.0)
    hist = np.zeros(maxiter + 1, dtype=np.float64) if want_hist else None
    _check(_lib.hr_bicgstab_dhat(ctx, float(m0), _ptr(x_e), _ptr(b_e), links, float(tol), int(maxiter), _ptr(workspace),
                                 ctypes.byref(it), ctypes.byref(res), _ptr(hist), stream))
    return it.value, res.value, (hist[:it.value + 1] if want_hist else None)


def hr_qmr_workspace_bytes(ctx: int, prec: int) -> int:
    return _lib.hr_qmr_workspace_bytes(ctx, prec)


def hr_qmr_dhat(ctx: int, m0: float, x_e, b_e, links: int, tol: float, maxiter: int, workspace, stream: int = 0, want_hist: bool = False):
    """Returns (iterations, true |b - Dhat x|^2/|b|^2, history of |eta_k|/|b| or None)."""
    it, res = _ci(0), _cd(0.0)
    hist = np.zeros(maxiter + 1, dtype=np.float64) if want_hist else None
    _check(_lib.hr_qmr_dhat(ctx, float(m0), _ptr(x_e), _ptr(b_e), links, float(tol), int(maxiter), _ptr(workspace),
                            ctypes.byref(it), ctypes.byref(res), _ptr(hist), stream))
    return it.value, res.value, (hist[:it.value + 1] if want_hist else None)


def hr_dirac_solve(ctx: int, m0: float, x_full, b_full, links: int, tol: float, maxiter: int, workspace, stream: int = 0):
    """Returns (iterations, |r|^2/|rhs|^2 of the preconditioned normal equations)."""
    it, res = _ci(0), _cd(0.0)
    _check(_lib.hr_dirac_solve(ctx, float(m0), _ptr(x_full), _ptr(b_full), links, float(tol), int(maxiter), _ptr(workspace),
                               ctypes.byref(it), ctypes.byref(res), stream))
    return it.value, res.value


def hr_halo_bytes(ctx: int, prec: int) -> int:
    return _lib.hr_halo_bytes(ctx, prec)


def hr_face_bytes(ctx: int, prec: int, mu: int) -> int:
    return _lib.hr_face_bytes(ctx, prec, mu)


def hr_dphi_eo_face_pack(mu: int, send_up, send_dn, inp, links: int, parity: int, stream: int = 0) -> None:
    _check(_lib.hr_dphi_eo_face_pack(mu, _ptr(send_up), _ptr(send_dn), _ptr(inp), links, parity, stream))


def hr_dphi_eo_faces_pack(split_mask: int, send_up: dict, send_dn: dict, inp, links: int, parity: int, stream: int = 0) -> None:
    """send_up / send_dn: {mu: buffer} for the split directions (bits of split_mask)."""
    up, dn = (_vp * 4)(), (_vp * 4)()
    for mu in range(4):
        up[mu] = _ptr(send_up.get(mu)) or None
        dn[mu] = _ptr(send_dn.get(mu)) or None
    _check(_lib.hr_dphi_eo_faces_pack(split_mask, up, dn, _ptr(inp), links, parity, stream))


def hr_dphi_eo_interior_mask(out, inp, links: int, parity: int, split_mask: int, stream: int = 0) -> None:
    _check(_lib.hr_dphi_eo_interior_mask(_ptr(out), _ptr(inp), links, parity, split_mask, stream))


def hr_dphi_eo_face_apply(mu: int, out, recv_prev, recv_next, links: int, parity: int, first_rank: int, last_rank: int,
                          stream: int = 0) -> None:
    _check(_lib.hr_dphi_eo_face_apply(mu, _ptr(out), _ptr(recv_prev), _ptr(recv_next), links, parity, int(first_rank),
                                      int(last_rank), stream))


def hr_dphi_eo_faces_apply(split_mask: int, out, recv_prev: dict, recv_next: dict, links: int, parity: int, first_mask: int,
                           last_mask: int, stream: int = 0) -> None:
    """recv_prev / recv_next: {mu: buffer} for the split directions; first_mask / last_mask: bit mu = first / last rank along mu."""
    rp, rn = (_vp * 4)(), (_vp * 4)()
    for mu in range(4):
        rp[mu] = _ptr(recv_prev.get(mu)) or None
        rn[mu] = _ptr(recv_next.get(mu)) or None
    _check(_lib.hr_dphi_eo_faces_apply(split_mask, _ptr(out), rp, rn, links, parity, int(first_mask), int(last_mask), stream))


def hr_halo_buffers_alloc(ctx: int, prec: int) -> int:
    p = _vp()
    _check(_lib.hr_halo_buffers_alloc(ctx, prec, ctypes.byref(p)))
    return p.value


def hr_face_buffers_alloc(ctx: int, prec: int, mu: int) -> int:
    p = _vp()
    _check(_lib.hr_face_buffers_alloc(ctx, prec, mu, ctypes.byref(p)))
    return p.value


def hr_halo_buffers_free(ctx: int, base: int) -> None:
    _lib.hr_halo_buffers_free(ctx, base)


def hr_ipc_export(ctx: int, base: int) -> bytes:
    buf = ctypes.create_string_buffer(64)
    _check(_lib.hr_ipc_export(ctx, base, buf))
    return buf.raw


def hr_ipc_open(ctx: int, handle: bytes) -> int:
    p = _vp()
    _check(_lib.hr_ipc_open(ctx, ctypes.create_string_buffer(bytes(handle), 64), ctypes.byref(p)))
    return p.value


def hr_ipc_close(ctx: int, peer_base: int) -> None:
    _check(_lib.hr_ipc_close(ctx, peer_base))


def hr_dphi_eo_halo_pack(send_up, send_dn, inp, links: int, parity: int, stream: int = 0) -> None:
    _check(_lib.hr_dphi_eo_halo_pack(_ptr(send_up), _ptr(send_dn), _ptr(inp), links, parity, stream))


def hr_dphi_eo_interior(out, inp, links: int, parity: int, stream: int = 0) -> None:
    _check(_lib.hr_dphi_eo_interior(_ptr(out), _ptr(inp), links, parity, stream))


def hr_dphi_eo_halo_apply(out, recv_prev, recv_next, links: int, parity: int, first_rank: bool, last_rank: bool,
                          stream: int = 0) -> None:
    _check(_lib.hr_dphi_eo_halo_apply(_ptr(out), _ptr(recv_prev), _ptr(recv_next), links, parity, int(first_rank),
                                      int(last_rank), stream))


def hr_clover_bytes(ctx: int, prec: int) -> int:
    return _lib.hr_clover_bytes(ctx, prec)


def hr_clover_build(clover, links: int, csw: float, stream: int = 0) -> None:
    _check(_lib.hr_clover_build(_ptr(clover), links, float(csw), stream))


def hr_clover_exp(ctx: int, prec: int, clover, m0: float, stream: int = 0) -> None:
    _check(_lib.hr_clover_exp(ctx, prec, _ptr(clover), float(m0), stream))


def hr_dirac_clover(m0: float, out_full, in_full, links: int, clover, stream: int = 0) -> None:
    _check(_lib.hr_dirac_clover(float(m0), _ptr(out_full), _ptr(in_full), links, _ptr(clover), stream))


def hr_dirac_solve_bicgstab(ctx: int, m0: float, x_full, b_full, links: int, tol: float, maxiter: int, workspace, stream: int = 0):
    """Returns (iterations, |r|^2/|bhat|^2 of the preconditioned system)."""
    it, res = _ci(0), _cd(0.0)
    _check(_lib.hr_dirac_solve_bicgstab(ctx, float(m0), _ptr(x_full), _ptr(b_full), links, float(tol), int(maxiter),
                                        _ptr(workspace), ctypes.byref(it), ctypes.byref(res), stream))
    return it.value, res.value


def hr_mixed_workspace_bytes(ctx: int, maxiter: int) -> int:
    return _lib.hr_mixed_workspace_bytes(ctx, maxiter)


def hr_bicgstab_dhat_mixed(ctx: int, m0: float, x_e, b_e, links64: int, links32: int, tol: float, inner_tol: float, maxiter: int,
                           workspace, stream: int = 0):
    """Returns (inner iterations in total, outer steps, true |r|^2/|b|^2)."""
    it, outer, res = _ci(0), _ci(0), _cd(0.0)
    _check(_lib.hr_bicgstab_dhat_mixed(ctx, float(m0), _ptr(x_e), _ptr(b_e), links64, links32, float(tol), float(inner_tol),
                                       int(maxiter), _ptr(workspace), ctypes.byref(it), ctypes.byref(outer), ctypes.byref(res), stream))
    return it.value, outer.value, res.value


def hr_clover_finalize(ctx: int, prec: int, site_term, site_inverse, m0: float, stream: int = 0) -> None:
    _check(_lib.hr_clover_finalize(ctx, prec, _ptr(site_term), _ptr(site_inverse), float(m0), stream))


def hr_dhat_clover(out_e, in_e, tmp_o, tmp2_o, links: int, site_term, site_inverse, stream: int = 0) -> None:
    _check(_lib.hr_dhat_clover(_ptr(out_e), _ptr(in_e), _ptr(tmp_o), _ptr(tmp2_o), links, _ptr(site_term), _ptr(site_inverse), stream))


def hr_clover_solve_workspace_bytes(ctx: int, prec: int, maxiter: int) -> int:
    return _lib.hr_clover_solve_workspace_bytes(ctx, prec, maxiter)


def hr_dirac_clover_solve(ctx: int, x_full, b_full, links: int, site_term, site_inverse, tol: float, maxiter: int, workspace, stream: int = 0):
    """Returns (iterations, |r|^2/|bhat|^2 of the preconditioned system)."""
    it, res = _ci(0), _cd(0.0)
    _check(_lib.hr_dirac_clover_solve(ctx, _ptr(x_full), _ptr(b_full), links, _ptr(site_term), _ptr(site_inverse), float(tol),
                                      int(maxiter), _ptr(workspace), ctypes.byref(it), ctypes.byref(res), stream))
    return it.value, res.value


def hr_ctx_set_tuning(ctx: int, key: str, value: int) -> None:
    _check(_lib.hr_ctx_set_tuning(ctx, key.encode(), int(value)))


def hr_dphi_variant_name(ctx: int, prec: int) -> str:
    return _lib.hr_dphi_variant_name(ctx, prec).decode()


# ---- convenience wrapper (handles + torch device memory; no arithmetic) ------------------------

_NP_REAL = {HR_F64: np.float64, HR_F32: np.float32}
_NP_CPLX = {HR_F64: np.complex128, HR_F32: np.complex64}


class Lattice:
    """Owns an hr_ctx and its gauge handles; spinors are torch uint8 tensors in the internal layout."""

    def __init__(self, dims, bc=(-1, 1, 1, 1), N: int = 3, rep="fund", device: int = 0):
        import torch  # device memory and streams only

        self._torch = torch
        self.dims = tuple(int(v) for v in dims)
        self.bc = tuple(int(v) for v in bc)
        self.N = N
        self.rep = REP_NAMES[rep] if isinstance(rep, str) else int(rep)
        self.device = device
        self.ctx = hr_ctx_create(self.dims, self.bc, N, self.rep, device)
        self.d = hr_rep_dim(self.ctx)
        self.real_links = bool(hr_links_are_real(self.ctx))
        self.vh = hr_half_volume(self.ctx)
        self._gauges = []

    # -- plumbing
    def stream(self) -> int:
        return int(self._torch.cuda.current_stream(self.device).cuda_stream)

    def close(self) -> None:
        for g in self._gauges:
            hr_gauge_free(g["handle"])
        self._gauges = []
        if self.ctx:
            hr_ctx_destroy(self.ctx)
            self.ctx = 0

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- fields
    def gauge(self, represented, prec: int) -> int:
        """hr_gauge_alloc on torch-owned device memory; returns the handle.  represented: False/0 fundamental,
        True/1 represented, 2 fundamental stored as N-1 rows (fill with compress_links)."""
        nbytes = hr_gauge_bytes(self.ctx, int(represented), prec)
        mem = self._torch.empty(nbytes, dtype=self._torch.uint8, device=f"cuda:{self.device}")
        h = hr_gauge_alloc(self.ctx, int(represented), prec, mem)
        self._gauges.append({"handle": h, "mem": mem})
        return h

    def spinor(self, prec: int, full: bool = False):
        nbytes = hr_spinor_bytes(self.ctx, prec) * (2 if full else 1)
        return self._torch.empty(nbytes, dtype=self._torch.uint8, device=f"cuda:{self.device}")

    def import_gauge(self, g: int, canon: np.ndarray) -> None:
        prec = HR_F64 if canon.dtype in (np.complex128, np.float64) else HR_F32
        hr_gauge_import(g, np.ascontiguousarray(canon), prec, self.stream())

    def export_gauge(self, g: int, represented: bool, prec: int = HR_F64) -> np.ndarray:
        V = 2 * self.vh
        if represented and self.real_links:
            out = np.empty((V, 4, self.d, self.d), dtype=_NP_REAL[prec])
        else:
            n = self.d if represented else self.N
            out = np.empty((V, 4, n, n), dtype=_NP_CPLX[prec])
        hr_gauge_export(g, out, prec, self.stream())
        return out

    def import_spinor(self, dst, prec: int, canon: np.ndarray, parity: int) -> None:
        cprec = HR_F64 if canon.dtype == np.complex128 else HR_F32
        hr_spinor_import(self.ctx, dst, prec, np.ascontiguousarray(canon), cprec, parity, self.stream())

    def export_spinor(self, src, prec: int, parity: int, out_prec: int = HR_F64) -> np.ndarray:
        out = np.empty((self.vh, 4, self.d), dtype=_NP_CPLX[out_prec])
        hr_spinor_export(self.ctx, src, prec, out, out_prec, parity, self.stream())
        return out

    # -- the hot path
    def compress_links(self, rows_out: int, fund_in: int) -> None:
        hr_gauge_compress(rows_out, fund_in, self.stream())

    def represent_links(self, repr_out: int, fund_in: int) -> None:
        hr_represent_links(repr_out, fund_in, self.stream())

    def dphi_eo(self, out, inp, links: int, parity: int) -> None:
        hr_dphi_eo(out, inp, links, parity, self.stream())

    def dirac(self, m0: float, out_full, in_full, links: int) -> None:
        hr_dirac(m0, out_full, in_full, links, self.stream())

    # -- NEXT-1: linear algebra, preconditioned operator, solver
    def cg_workspace(self, prec: int, maxiter: int):
        n = hr_cg_workspace_bytes(self.ctx, prec, maxiter)
        return self._torch.empty(n, dtype=self._torch.uint8, device=f"cuda:{self.device}")

    def dhat(self, m0: float, g5: bool, out_e, in_e, tmp_o, links: int) -> None:
        hr_dhat(m0, int(g5), out_e, in_e, tmp_o, links, self.stream())

    def cg_dhat(self, m0, x_e, b_e, links, tol, maxiter, workspace, want_hist=False):
        return hr_cg_dhat(self.ctx, m0, x_e, b_e, links, tol, maxiter, workspace, self.stream(), want_hist)

    def dirac_solve(self, m0, x_full, b_full, links, tol, maxiter, workspace):
        return hr_dirac_solve(self.ctx, m0, x_full, b_full, links, tol, maxiter, workspace, self.stream())

    def set_tuning(self, key: str, value: int) -> None:
        hr_ctx_set_tuning(self.ctx, key, value)

    def variant_name(self, prec: int) -> str:
        return hr_dphi_variant_name(self.ctx, prec)

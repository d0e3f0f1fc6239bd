"""CPU oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

ctypes front end of oracle.c (plain fp64 C, the definition written out) plus `oracle.dense`
(numpy brute-force dense assembly used to pin oracle.c).  Only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this package; it imports nothing from
paper_2405_19294_b200 and shares no code with it.  See the header of oracle.c for citations and pins.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liboracle.so")
_SRC = os.path.join(_HERE, "oracle.c")

REP_FUND, REP_ADJ, REP_SYM, REP_ASYM = 0, 1, 2, 3
REP_NAMES = {"fund": REP_FUND, "adj": REP_ADJ, "sym": REP_SYM, "asym": REP_ASYM}


def build(force: bool = False) -> str:
    """Compile oracle.c as it stands (-O2 -fopenmp); never tuned."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(
            ["gcc", "-O2", "-fopenmp", "-std=c99", "-shared", "-fPIC", "-o", _SO, _SRC, "-lm"]
        )
    return _SO


_lib = None
_I4 = ctypes.c_int * 4


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_SO)
        vp, ci, cl, cd = ctypes.c_void_p, ctypes.c_int, ctypes.c_long, ctypes.c_double
        lib.oracle_gamma.argtypes = [ci, vp]
        lib.oracle_gamma.restype = None
        lib.oracle_rep_dim.argtypes = [ci, ci]
        lib.oracle_rep_dim.restype = ci
        lib.oracle_represent.argtypes = [ci, ci, vp, vp, vp]
        lib.oracle_represent.restype = ci
        lib.oracle_represent_field.argtypes = [ci, ci, cl, vp, vp]
        lib.oracle_represent_field.restype = cd
        lib.oracle_dphi_lex.argtypes = [_I4, _I4, ci, vp, vp, vp]
        lib.oracle_dphi_lex.restype = ci
        lib.oracle_dphi_eo.argtypes = [_I4, _I4, ci, vp, ci, vp, vp]
        lib.oracle_dphi_eo.restype = ci
        lib.oracle_dphi_eo_sites.argtypes = [_I4, _I4, ci, vp, ci, vp, cl, vp, vp]
        lib.oracle_dphi_eo_sites.restype = ci
        lib.oracle_dirac.argtypes = [_I4, _I4, ci, vp, cd, vp, vp]
        lib.oracle_dirac.restype = ci
        lib.oracle_num_threads.argtypes = []
        lib.oracle_num_threads.restype = ci
        _lib = lib
    return _lib


def _c128(a) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=np.complex128)
    return a


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def gamma(mu: int) -> np.ndarray:
    """gamma_mu (mu = 0..3) or gamma_5 (mu = 5), 4x4 complex128 (reading C1)."""
    out = np.empty((4, 4), dtype=np.complex128)
    _load().oracle_gamma(mu, out.ctypes.data)
    return out


def rep_dim(N: int, rep: int) -> int:
    return int(_load().oracle_rep_dim(N, rep))


def represent(N: int, rep: int, U) -> np.ndarray:
    """R(U) for links U[..., N, N] -> [..., d, d] complex128, from the trace definitions."""
    U = _c128(U)
    d = rep_dim(N, rep)
    n = U.size // (N * N)
    R = np.empty(U.shape[:-2] + (d, d), dtype=np.complex128)
    worst = _load().oracle_represent_field(N, rep, n, U.ctypes.data, R.ctypes.data)
    if worst < 0:
        raise ValueError("unsupported N/rep")
    if rep == REP_ADJ and worst > 1e-13:
        raise AssertionError(f"adjoint not real: max |Im| = {worst}")  # reading C7
    return R


def _dims(dims, bc):
    return _I4(*[int(v) for v in dims]), _I4(*[int(v) for v in bc])


def dphi_lex(dims, bc, links_R, psi) -> np.ndarray:
    """Dphi on all sites. links_R [V][4][d][d], psi [V][4][d] lexicographic."""
    links_R, psi = _c128(links_R), _c128(psi)
    d = links_R.shape[-1]
    out = np.empty_like(psi)
    cd, cb = _dims(dims, bc)
    rc = _load().oracle_dphi_lex(cd, cb, d, links_R.ctypes.data, psi.ctypes.data, out.ctypes.data)
    if rc:
        raise ValueError("oracle_dphi_lex: bad arguments")
    return out


def dphi_eo(dims, bc, links_R, parity: int, psi_half) -> np.ndarray:
    """Dphi_eo: output on parity-`parity` sites [V/2][4][d], psi_half on parity 1-parity."""
    links_R, psi_half = _c128(links_R), _c128(psi_half)
    d = links_R.shape[-1]
    out = np.empty_like(psi_half)
    cd, cb = _dims(dims, bc)
    rc = _load().oracle_dphi_eo(cd, cb, d, links_R.ctypes.data, parity, psi_half.ctypes.data, out.ctypes.data)
    if rc:
        raise ValueError("oracle_dphi_eo: bad arguments")
    return out


def dphi_eo_sites(dims, bc, links_R, parity: int, psi_half, half_index) -> np.ndarray:
    """Dphi_eo at the listed output sites (half indices) only: [n][4][d]."""
    links_R, psi_half = _c128(links_R), _c128(psi_half)
    hi = np.ascontiguousarray(half_index, dtype=np.int64)
    d = links_R.shape[-1]
    out = np.empty((hi.size, 4, d), dtype=np.complex128)
    cd, cb = _dims(dims, bc)
    rc = _load().oracle_dphi_eo_sites(cd, cb, d, links_R.ctypes.data, parity, psi_half.ctypes.data,
                                      hi.size, hi.ctypes.data, out.ctypes.data)
    if rc:
        raise ValueError("oracle_dphi_eo_sites: bad arguments")
    return out


def dirac(dims, bc, links_R, m0: float, psi_eo) -> np.ndarray:
    """D = (4+m0) + Dphi on an eo full field [even half | odd half] of shape [V][4][d]."""
    links_R, psi_eo = _c128(links_R), _c128(psi_eo)
    d = links_R.shape[-1]
    out = np.empty_like(psi_eo)
    cd, cb = _dims(dims, bc)
    rc = _load().oracle_dirac(cd, cb, d, links_R.ctypes.data, float(m0), psi_eo.ctypes.data, out.ctypes.data)
    if rc:
        raise ValueError("oracle_dirac: bad arguments")
    return out


# -- canonical layout helpers (pure permutations, reading C4) ------------------------------------

def lex_to_eo(dims, field_lex: np.ndarray) -> np.ndarray:
    """[V]... lexicographic -> [even half | odd half]."""
    t, x, y, z = (int(v) for v in dims)
    tt, xx, yy, zz = np.meshgrid(np.arange(t), np.arange(x), np.arange(y), np.arange(z), indexing="ij")
    par = ((tt + xx + yy + zz) & 1).reshape(-1)
    return np.concatenate([field_lex[par == 0], field_lex[par == 1]], axis=0)


def eo_to_lex(dims, field_eo: np.ndarray) -> np.ndarray:
    t, x, y, z = (int(v) for v in dims)
    tt, xx, yy, zz = np.meshgrid(np.arange(t), np.arange(x), np.arange(y), np.arange(z), indexing="ij")
    par = ((tt + xx + yy + zz) & 1).reshape(-1)
    out = np.empty_like(field_eo)
    vh = field_eo.shape[0] // 2
    out[par == 0] = field_eo[:vh]
    out[par == 1] = field_eo[vh:]
    return out

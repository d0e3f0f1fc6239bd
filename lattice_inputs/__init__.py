"""Seeded synthetic inputs (canonical layout) for the tests, the oracle legs and bench.py.

Holds none of the method's arithmetic -- see gen.c.  The recipes are the ones BASELINE.json:configs
prescribes (Haar SU(N) links, near-identity exp(i eps H) links, unit-Gaussian spinors); DESIGN.md
"Input recipe" states them.  Everything is generated in fp64 and rounded once by the consumer for
fp32 runs (reading C13).

Streams: 0 = spinor, 1 = links, 2 = gauge transformation.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libgen.so")
_SRC = os.path.join(_HERE, "gen.c")

STREAM_SPINOR, STREAM_LINKS, STREAM_GAUGE = 0, 1, 2


def build(force: bool = False) -> str:
    """Compile gen.c into libgen.so (gcc, OpenMP)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(
            ["gcc", "-O2", "-fopenmp", "-std=c99", "-shared", "-fPIC", "-o", _SO, _SRC, "-lm"]
        )
    return _SO


_lib = None


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_SO)
        lib.gen_gaussian_complex.argtypes = [
            ctypes.c_uint64, ctypes.c_uint32, ctypes.c_int64, ctypes.c_int64, ctypes.c_void_p]
        lib.gen_gaussian_complex.restype = None
        lib.gen_sun.argtypes = [
            ctypes.c_uint64, ctypes.c_uint32, ctypes.c_int, ctypes.c_double, ctypes.c_int,
            ctypes.c_int64, ctypes.c_int64, ctypes.c_void_p]
        lib.gen_sun.restype = ctypes.c_int
        _lib = lib
    return _lib


def volume(dims) -> int:
    t, x, y, z = (int(v) for v in dims)
    return t * x * y * z


def gaussian_spinor(seed: int, nsites: int, d: int, first_site: int = 0, out=None) -> np.ndarray:
    """[nsites][4][d] complex128, every re/im ~ N(0,1) i.i.d.; sites first_site.. of the stream."""
    per = 4 * d
    if out is None:
        out = np.empty((nsites, 4, d), dtype=np.complex128)
    assert out.dtype == np.complex128 and out.flags.c_contiguous and out.size == nsites * per
    _load().gen_gaussian_complex(seed, STREAM_SPINOR, first_site * per, nsites * per, out.ctypes.data)
    return out


def _sun(seed, stream, kind, eps, N, first, count, out=None):
    if out is None:
        out = np.empty((count, N, N), dtype=np.complex128)
    assert out.dtype == np.complex128 and out.flags.c_contiguous and out.size == count * N * N
    rc = _load().gen_sun(seed, stream, kind, float(eps), N, first, count, out.ctypes.data)
    if rc != 0:
        raise ValueError("gen_sun: unsupported N")
    return out


def haar_links(seed: int, N: int, dims, out=None, first_site: int = 0, nsites=None) -> np.ndarray:
    """Haar-random SU(N) fundamental links, canonical [V][4][N][N] complex128 (or the nsites sites from first_site on of
    that field: the generator is counter-based, any slice is reproducible on its own)."""
    V = volume(dims) if nsites is None else int(nsites)
    if out is None:
        out = np.empty((V, 4, N, N), dtype=np.complex128)
    _sun(seed, STREAM_LINKS, 0, 0.0, N, 4 * first_site, 4 * V, out)
    return out


def near_identity_links(seed: int, N: int, dims, eps: float = 0.3, out=None, first_site: int = 0, nsites=None) -> np.ndarray:
    """U = exp(i eps H), H Gaussian Hermitian traceless; canonical [V][4][N][N] complex128 (or a slice, as haar_links)."""
    V = volume(dims) if nsites is None else int(nsites)
    if out is None:
        out = np.empty((V, 4, N, N), dtype=np.complex128)
    _sun(seed, STREAM_LINKS, 1, eps, N, 4 * first_site, 4 * V, out)
    return out


def unit_links(N: int, dims) -> np.ndarray:
    V = volume(dims)
    out = np.zeros((V, 4, N, N), dtype=np.complex128)
    out[..., range(N), range(N)] = 1.0
    return out


def haar_matrices(seed: int, N: int, count: int, stream: int = STREAM_GAUGE) -> np.ndarray:
    """count Haar SU(N) matrices (e.g. one gauge-transformation matrix per site)."""
    return _sun(seed, stream, 0, 0.0, N, 0, count)


def parity_mask(dims) -> np.ndarray:
    """parity (t+x+y+z)&1 of every lexicographic site, shape [V]."""
    t, x, y, z = (int(v) for v in dims)
    tt, xx, yy, zz = np.meshgrid(np.arange(t), np.arange(x), np.arange(y), np.arange(z), indexing="ij")
    return ((tt + xx + yy + zz) & 1).reshape(-1).astype(np.int8)

"""Python face of the CPU oracle (TEST INFRASTRUCTURE, NOT THE PRODUCT).

Thin ctypes marshalling around oracle/debye_oracle.c (plain C, fp64, Eq. 2 of PAPER.md:41-42 written out),
plus closed forms that follow from Eq. (2) by grouping equal distances.  Nothing here is imported by
paper_1306_2258_b200/ and nothing here imports it.
"""
from __future__ import annotations

import ctypes as C
import math

import numpy as np

from . import build as _build

_lib = None


def _L():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        fp, ip, dp = C.POINTER(C.c_float), C.POINTER(C.c_int32), C.POINTER(C.c_double)
        _lib.oracle_debye_full.argtypes = [fp, ip, C.c_int32, fp, C.c_int32, fp, C.c_int32, dp, dp]
        _lib.oracle_debye_full.restype = None
        _lib.oracle_debye_sym.argtypes = [fp, ip, C.c_int32, fp, C.c_int32, fp, C.c_int32, C.c_int32, C.c_int32,
                                          C.c_int32, dp, dp]
        _lib.oracle_debye_sym.restype = C.c_int32
        _lib.oracle_debye_full_w.argtypes = [fp, ip, fp, C.c_int32, fp, C.c_int32, fp, C.c_int32, dp, dp]
        _lib.oracle_debye_full_w.restype = None
        _lib.oracle_debye_sym_w.argtypes = [fp, ip, fp, C.c_int32, fp, C.c_int32, fp, C.c_int32, C.c_int32, C.c_int32,
                                            C.c_int32, dp, dp]
        _lib.oracle_debye_sym_w.restype = C.c_int32
        _lib.oracle_debye_peratom.argtypes = [fp, fp, C.c_int32, fp, C.c_int32, C.c_int32, dp, dp]
        _lib.oracle_debye_peratom.restype = None
        _lib.oracle_eq1_quadrature.argtypes = [dp, dp, C.c_int32, C.c_double, dp, dp, C.c_int32]
        _lib.oracle_eq1_quadrature.restype = C.c_double
    return _lib


def _prep(xyz, typ, fftab, q):
    xyz = np.ascontiguousarray(xyz, dtype=np.float32)
    typ = np.ascontiguousarray(typ, dtype=np.int32)
    fftab = np.ascontiguousarray(fftab, dtype=np.float32)
    q = np.ascontiguousarray(q, dtype=np.float32)
    assert xyz.ndim == 2 and xyz.shape[1] == 3 and typ.shape == (xyz.shape[0],)
    assert fftab.ndim == 2 and fftab.shape[1] == q.shape[0]
    assert typ.min() >= 0 and typ.max() < fftab.shape[0]
    return xyz, typ, fftab, q


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t))


def _w(weight, N):
    if weight is None:
        return None
    weight = np.ascontiguousarray(weight, dtype=np.float32)
    assert weight.shape == (N,)
    return weight


def debye_full(xyz, typ, fftab, q, return_abs=False, weight=None):
    """Eq. (2) literally (N x N loop including j == k), single thread.  PAPER.md:41-42.
    weight[N] (optional): f_j(q) = weight[j] * fftab[type[j]] (reading R10w)."""
    xyz, typ, fftab, q = _prep(xyz, typ, fftab, q)
    M = q.shape[0]
    I, A = np.zeros(M), np.zeros(M)
    w = _w(weight, xyz.shape[0])
    if w is None:
        _L().oracle_debye_full(_p(xyz, C.c_float), _p(typ, C.c_int32), xyz.shape[0], _p(fftab, C.c_float),
                               fftab.shape[0], _p(q, C.c_float), M, _p(I, C.c_double), _p(A, C.c_double))
    else:
        _L().oracle_debye_full_w(_p(xyz, C.c_float), _p(typ, C.c_int32), _p(w, C.c_float), xyz.shape[0],
                                 _p(fftab, C.c_float), fftab.shape[0], _p(q, C.c_float), M, _p(I, C.c_double),
                                 _p(A, C.c_double))
    return (I, A) if return_abs else I


def debye_sym(xyz, typ, fftab, q, rows=None, threads=0, return_abs=False, return_threads=False, weight=None):
    """I = sum_k f_k (f_k + 2 sum_{j>k} f_j sinc) (PAPER.md:88 'only j <= k'), OpenMP over rows.
    rows=(r0, r1) restricts the outer sum to a row slab (used for timing a bounded sample)."""
    xyz, typ, fftab, q = _prep(xyz, typ, fftab, q)
    M, N = q.shape[0], xyz.shape[0]
    r0, r1 = (0, N) if rows is None else rows
    I, A = np.zeros(M), np.zeros(M)
    w = _w(weight, N)
    if w is None:
        nthr = _L().oracle_debye_sym(_p(xyz, C.c_float), _p(typ, C.c_int32), N, _p(fftab, C.c_float), fftab.shape[0],
                                     _p(q, C.c_float), M, r0, r1, threads, _p(I, C.c_double), _p(A, C.c_double))
    else:
        nthr = _L().oracle_debye_sym_w(_p(xyz, C.c_float), _p(typ, C.c_int32), _p(w, C.c_float), N,
                                       _p(fftab, C.c_float), fftab.shape[0], _p(q, C.c_float), M, r0, r1, threads,
                                       _p(I, C.c_double), _p(A, C.c_double))
    out = [I]
    if return_abs:
        out.append(A)
    if return_threads:
        out.append(nthr)
    return out[0] if len(out) == 1 else tuple(out)


def debye_batch(xyz_b, typ, fftab, q, threads=0, weight=None):
    """Eq. (2) for each conformer of xyz_b[B][N][3] (shared type / fftab / q / weight)."""
    return np.stack([debye_sym(x, typ, fftab, q, threads=threads, weight=weight) for x in xyz_b])


def debye_peratom(xyz, ff, q, sym=True, return_abs=False):
    """Eq. (2) with per-ATOM form factors ff[N][M] (reading R10p).  sym=False: the full N x N loop,
    single thread; sym=True: sum_k f_k (f_k + 2 sum_{j>k} f_j sinc), OpenMP over rows."""
    xyz = np.ascontiguousarray(xyz, dtype=np.float32)
    ff = np.ascontiguousarray(ff, dtype=np.float32)
    q = np.ascontiguousarray(q, dtype=np.float32)
    assert xyz.ndim == 2 and xyz.shape[1] == 3 and ff.shape == (xyz.shape[0], q.shape[0])
    M = q.shape[0]
    I, A = np.zeros(M), np.zeros(M)
    _L().oracle_debye_peratom(_p(xyz, C.c_float), _p(ff, C.c_float), xyz.shape[0], _p(q, C.c_float), M, 1 if sym else 0,
                              _p(I, C.c_double), _p(A, C.c_double))
    return (I, A) if return_abs else I


def eq1_quadrature(x, f, qval, n=None):
    """Eq. (1): orientational average of |sum_j f_j exp(i q.r_j)|^2 by Gauss-Legendre (cos
    theta) x midpoint (phi) quadrature with n x 2n nodes; n defaults to max(32, ceil(q D / 2) + 16)."""
    x = np.ascontiguousarray(x, dtype=np.float64)
    f = np.ascontiguousarray(f, dtype=np.float64)
    if n is None:
        D = float(np.sqrt(((x[:, None, :] - x[None, :, :]) ** 2).sum(-1)).max()) if len(x) > 1 else 0.0
        n = max(32, int(math.ceil(qval * D / 2)) + 16)
    mu, w = np.polynomial.legendre.leggauss(n)
    mu = np.ascontiguousarray(mu); w = np.ascontiguousarray(w)
    return _L().oracle_eq1_quadrature(_p(x, C.c_double), _p(f, C.c_double), x.shape[0], float(qval),
                                      _p(mu, C.c_double), _p(w, C.c_double), n)


# ---- closed forms: exact consequences of Eq. (2) obtained by grouping equal distances ---------------
def _sinc(u):
    u = np.asarray(u, dtype=np.float64)
    return np.where(u == 0.0, 1.0, np.sin(u) / np.where(u == 0.0, 1.0, u))


def chain_closed_form(n, d, q):
    """n unit scatterers on a line, spacing d:  I = n + 2 sum_{m=1}^{n-1} (n-m) sinc(q m d)."""
    q = np.asarray(q, dtype=np.float64)
    m = np.arange(1, n, dtype=np.float64)
    return n + 2.0 * ((n - m)[None, :] * _sinc(q[:, None] * m[None, :] * d)).sum(axis=1)


def lattice_closed_form(nx, ny, nz, a, q, fa=1.0, fb=None, return_abs=False):
    """nx x ny x nz simple cubic lattice, spacing a.  Unit (or fa) form factors:
    I = fa^2 sum_{alpha,beta,gamma} (nx-|alpha|)(ny-|beta|)(nz-|gamma|) sinc(q a sqrt(alpha^2+beta^2+gamma^2)).
    With fb given, sites with odd (x+y+z) carry fb: the multiplicity of each displacement splits by parity."""
    q = np.asarray(q, dtype=np.float64)
    al = np.arange(-(nx - 1), nx); be = np.arange(-(ny - 1), ny); ga = np.arange(-(nz - 1), nz)
    A, Bm, G = np.meshgrid(al, be, ga, indexing="ij")
    r = a * np.sqrt((A * A + Bm * Bm + G * G).astype(np.float64)).ravel()
    if fb is None:
        mult = ((nx - np.abs(A)) * (ny - np.abs(Bm)) * (nz - np.abs(G))).astype(np.float64).ravel() * fa * fa
    else:
        # count start sites s with s and s+disp inside the box, split by parity of s; per axis, the start
        # coordinates form an interval of length n-|d|; count even and odd members.
        def eo(n, d):
            lo = np.maximum(0, -d); hi = n - 1 - np.maximum(0, d)          # inclusive range of start coord
            cnt = hi - lo + 1
            ev = (hi // 2) - ((lo + 1) // 2) + 1                            # evens in [lo, hi]
            return ev, cnt - ev
        ex, ox = eo(nx, A); ey, oy = eo(ny, Bm); ez, oz = eo(nz, G)
        even = ex * ey * ez + ex * oy * oz + ox * ey * oz + ox * oy * ez   # parity of sum even
        odd = ox * oy * oz + ox * ey * ez + ex * oy * ez + ex * ey * oz
        flip = ((A + Bm + G) % 2 != 0)
        f_even_start = np.where(flip, fa * fb, fa * fa)                     # even start site carries fa
        f_odd_start = np.where(flip, fb * fa, fb * fb)
        mult = (even * f_even_start + odd * f_odd_start).astype(np.float64).ravel()
    ru, inv = np.unique(r, return_inverse=True)
    mu = np.bincount(inv, weights=mult)
    out = np.empty(q.shape[0])
    ab = np.empty(q.shape[0])
    for i, qq in enumerate(q):
        t = mu * _sinc(qq * ru)
        out[i] = float(t.sum())
        ab[i] = float(np.abs(t).sum())
    return (out, ab) if return_abs else out

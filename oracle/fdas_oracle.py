"""ctypes loader for the CPU oracle (``fdas_oracle.c``).  TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this module.  It never imports the CUDA binding and the CUDA
binding never imports it.  All arithmetic lives in ``fdas_oracle.c``; this file only builds the
shared object with gcc, marshals numpy arrays and strings the oracle steps O1..O6 together
(``Oracle.run``) in the order of SURVEY.md 8(c) / DESIGN.md.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "fdas_oracle.c")
_LIB = os.path.join(_HERE, "libfdas_oracle.so")


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp -> oracle/libfdas_oracle.so (rebuilt when the source is newer)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-fno-fast-math",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None

_d = C.POINTER(C.c_double)
_f = C.POINTER(C.c_float)
_i64 = C.POINTER(C.c_int64)
_i32 = C.POINTER(C.c_int32)


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.orc_num_threads.restype = C.c_int
        L.orc_dft.argtypes = [_d, _d, C.c_int64, C.c_int]
        L.orc_fft.argtypes = [_d, C.c_int64, C.c_int]
        L.orc_spectrum.argtypes = [_f, C.c_int64, _d]
        L.orc_whiten_nblocks.argtypes = [C.c_int64]
        L.orc_whiten_nblocks.restype = C.c_int64
        L.orc_whiten.argtypes = [_d, C.c_int64, _d, _d, _d]
        L.orc_gauss_legendre.argtypes = [C.c_int, _d, _d]
        L.orc_halfwidth.argtypes = [C.c_double]
        L.orc_template.argtypes = [C.c_double, C.c_int, _d, C.c_int]
        L.orc_template_bank.argtypes = [C.c_double, C.c_double, C.c_int, C.c_int, _d]
        L.orc_plane.argtypes = [_d, C.c_int64, _d, C.c_int, C.c_int, C.c_int64, C.c_int64, _d]
        L.orc_plane_points.argtypes = [_d, C.c_int64, _d, C.c_int, C.c_int, _i64, _i32, C.c_int64, _d]
        L.orc_plane_ols_dft.argtypes = [_d, C.c_int64, _d, C.c_int, C.c_int, C.c_int, _d]
        L.orc_harmonic_sums_at.argtypes = [_d, C.c_int64, C.c_int, C.c_int, C.c_int64, C.c_int, _d]
        L.orc_harmonic_sums_sampled.argtypes = [_d, C.c_int64, _d, C.c_int, C.c_int, C.c_int, _i64, _i32,
                                                C.c_int64, _d, _i32]
        L.orc_candidates.argtypes = [_d, C.c_int64, C.c_int, C.c_int, _d, C.c_int64,
                                     _i64, _i32, _i32, _d, _i32, C.c_int64]
        L.orc_candidates.restype = C.c_int64
        L.orc_harmonic_sums_nbr_at.argtypes = [_d, C.c_int64, C.c_int, C.c_int, C.c_int64, C.c_int, _d]
        L.orc_candidates_nbr.argtypes = [_d, C.c_int64, C.c_int, C.c_int, _d, C.c_int64,
                                         _i64, _i32, _i32, _d, _i32, C.c_int64]
        L.orc_candidates_nbr.restype = C.c_int64
        L.orc_thresholds.argtypes = [C.c_int, C.c_double, _d]
        _lib = L
    return _lib


def _p(a, t):
    return a.ctypes.data_as(t)


def _c128(a):
    a = np.ascontiguousarray(a, dtype=np.complex128)
    return a, a.view(np.float64)


def num_threads() -> int:
    return int(lib().orc_num_threads())


def dft(x, sign=-1):
    x, xv = _c128(x)
    out = np.empty_like(x)
    lib().orc_dft(_p(xv, _d), _p(out.view(np.float64), _d), x.size, sign)
    return out


def fft(x, sign=-1):
    a = np.array(x, dtype=np.complex128, copy=True)
    rc = lib().orc_fft(_p(a.view(np.float64), _d), a.size, sign)
    if rc:
        raise ValueError("orc_fft: length must be a power of two")
    return a


def spectrum(x32, nfft):
    x32 = np.ascontiguousarray(x32[:nfft], dtype=np.float32)
    X = np.empty(nfft // 2, dtype=np.complex128)
    rc = lib().orc_spectrum(_p(x32, _f), nfft, _p(X.view(np.float64), _d))
    assert rc == 0
    return X


def whiten(X, want_blocks=False):
    X, Xv = _c128(X)
    nb = X.size
    w = np.empty(nb, dtype=np.complex128)
    nblk = int(lib().orc_whiten_nblocks(nb))
    med = np.empty(nblk)
    ctr = np.empty(nblk)
    rc = lib().orc_whiten(_p(Xv, _d), nb, _p(w.view(np.float64), _d), _p(med, _d), _p(ctr, _d))
    assert rc == 0
    return (w, med, ctr) if want_blocks else w


def gauss_legendre(n):
    x = np.empty(n)
    w = np.empty(n)
    lib().orc_gauss_legendre(n, _p(x, _d), _p(w, _d))
    return x, w


def halfwidth(zmax) -> int:
    return int(lib().orc_halfwidth(float(zmax)))


def template(z, h, normalise=True):
    T = np.empty(2 * h + 1, dtype=np.complex128)
    lib().orc_template(float(z), int(h), _p(T.view(np.float64), _d), int(bool(normalise)))
    return T


def template_bank(zmax, zstep, h=None):
    nz = int(round(2 * zmax / zstep)) + 1
    if h is None:
        h = halfwidth(zmax)
    bank = np.empty((nz, 2 * h + 1), dtype=np.complex128)
    lib().orc_template_bank(float(zmax), float(zstep), nz, h, _p(bank.view(np.float64), _d))
    return bank


def plane(w, bank, r0=0, r1=None):
    w, wv = _c128(w)
    bank, bv = _c128(bank)
    nz, taps = bank.shape
    h = (taps - 1) // 2
    nb = w.size
    if r1 is None:
        r1 = nb
    P = np.empty((nz, r1 - r0), dtype=np.float64)
    rc = lib().orc_plane(_p(wv, _d), nb, _p(bv, _d), nz, h, r0, r1, _p(P, _d))
    assert rc == 0
    return P


def plane_points(w, bank, rr, jj):
    w, wv = _c128(w)
    bank, bv = _c128(bank)
    nz, taps = bank.shape
    h = (taps - 1) // 2
    rr = np.ascontiguousarray(rr, dtype=np.int64)
    jj = np.ascontiguousarray(jj, dtype=np.int32)
    out = np.empty(rr.size, dtype=np.float64)
    lib().orc_plane_points(_p(wv, _d), w.size, _p(bv, _d), nz, h, _p(rr, _i64), _p(jj, _i32),
                           rr.size, _p(out, _d))
    return out


def plane_ols_dft(w, bank, seg_len):
    w, wv = _c128(w)
    bank, bv = _c128(bank)
    nz, taps = bank.shape
    h = (taps - 1) // 2
    P = np.zeros((nz, w.size), dtype=np.float64)
    rc = lib().orc_plane_ols_dft(_p(wv, _d), w.size, _p(bv, _d), nz, h, seg_len, _p(P, _d))
    assert rc == 0
    return P


def harmonic_sums_at(P, H, r, j):
    P = np.ascontiguousarray(P, dtype=np.float64)
    nz, nb = P.shape
    S = np.zeros(H)
    hmax = lib().orc_harmonic_sums_at(_p(P, _d), nb, nz, H, int(r), int(j), _p(S, _d))
    return S[:hmax]


def harmonic_sums_nbr_at(P, H, r, j):
    """Neighbour-maximised sums S'_1..S'_hmax at (r, j) (reading A24)."""
    P = np.ascontiguousarray(P, dtype=np.float64)
    nz, nb = P.shape
    S = np.zeros(H)
    hmax = lib().orc_harmonic_sums_nbr_at(_p(P, _d), nb, nz, H, int(r), int(j), _p(S, _d))
    return S[:hmax]


def harmonic_sums_sampled(w, bank, H, rr, jj):
    """S (npts x H, NaN where undefined) and hmax (npts) at sampled fundamentals, from w directly."""
    w, wv = _c128(w)
    bank, bv = _c128(bank)
    nz, taps = bank.shape
    h = (taps - 1) // 2
    rr = np.ascontiguousarray(rr, dtype=np.int64)
    jj = np.ascontiguousarray(jj, dtype=np.int32)
    S = np.full((rr.size, H), np.nan)
    hmax = np.zeros(rr.size, dtype=np.int32)
    lib().orc_harmonic_sums_sampled(_p(wv, _d), w.size, _p(bv, _d), nz, h, H, _p(rr, _i64),
                                    _p(jj, _i32), rr.size, _p(S, _d), _p(hmax, _i32))
    return S, hmax


def thresholds(H, nsigma):
    T = np.empty(H)
    lib().orc_thresholds(H, float(nsigma), _p(T, _d))
    return T


@dataclass
class Candidates:
    r: np.ndarray
    j: np.ndarray
    h: np.ndarray
    power: np.ndarray
    flag: np.ndarray
    count: int

    def triples(self):
        return set(zip(self.r.tolist(), self.j.tolist(), self.h.tolist()))

    def as_dict(self):
        return {(int(r), int(j), int(h)): (float(p), int(f))
                for r, j, h, p, f in zip(self.r, self.j, self.h, self.power, self.flag)}


def candidates(P, H, thr, r_lo, capacity=1 << 20, nbr=False):
    """Thresholded (r, j, h) triples of the plain sums (O6) or, nbr=True, of the neighbour-maximised
    sums (O5n)."""
    P = np.ascontiguousarray(P, dtype=np.float64)
    nz, nb = P.shape
    thr = np.ascontiguousarray(thr, dtype=np.float64)
    c_r = np.empty(capacity, dtype=np.int64)
    c_j = np.empty(capacity, dtype=np.int32)
    c_h = np.empty(capacity, dtype=np.int32)
    c_p = np.empty(capacity, dtype=np.float64)
    c_f = np.empty(capacity, dtype=np.int32)
    fn = lib().orc_candidates_nbr if nbr else lib().orc_candidates
    n = int(fn(_p(P, _d), nb, nz, H, _p(thr, _d), int(r_lo), _p(c_r, _i64),
               _p(c_j, _i32), _p(c_h, _i32), _p(c_p, _d), _p(c_f, _i32), capacity))
    m = min(n, capacity)
    return Candidates(c_r[:m].copy(), c_j[:m].copy(), c_h[:m].copy(), c_p[:m].copy(),
                      c_f[:m].copy(), n)


@dataclass
class OracleResult:
    X: np.ndarray
    w: np.ndarray
    bank: np.ndarray
    P: np.ndarray
    thr: np.ndarray
    cands: Candidates


def run(x32, nfft, zmax, zstep, H, nsigma, r_lo, want_candidates=True) -> OracleResult:
    """O1 -> O2 -> O3 -> O4 -> O5/O6 on one float32 time series (full plane in memory)."""
    X = spectrum(x32, nfft)
    w = whiten(X)
    bank = template_bank(zmax, zstep)
    P = plane(w, bank)
    thr = thresholds(H, nsigma)
    cands = candidates(P, H, thr, r_lo) if want_candidates else None
    return OracleResult(X, w, bank, P, thr, cands)

"""CPU oracle -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

ctypes binding over oracle/liboracle.so (oracle.cpp + oracle_bp.cpp, double
precision, no code shared with the CUDA path).  Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference arm may
import this package; the product package paper_2209_08450_b200 never does.

The stage arithmetic S1..S7, the exact and linear backprojections and the adjoint
pairs are in the C++ files; the wrappers of those only marshal numpy arrays.  Three
small functions do their arithmetic here in numpy (double precision), each citing
the reading it follows and pinned by its own test: `angle_weights` (trapezoid
weights, reading Q20, pin P11), `padded_size` and `recon_padded` (detector width not
a power of two, reading Q19, pin P10).  `recon_pre` only chains calls.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liboracle.so")
_SRC = [os.path.join(_HERE, "oracle.cpp"), os.path.join(_HERE, "oracle_bp.cpp"), os.path.join(_HERE, "oracle_pre.cpp")]

FILTERS = {"ramp": 0, "shepp": 1, "parzen": 2, "cosine": 3, "hann": 4, "hamming": 5}
METHODS = {"grid": 0, "exact": 1, "lin": 2}
DEFAULT_M = 4


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (building the checker is not using it)."""
    stale = force or not os.path.exists(_SO) or any(
        os.path.getmtime(s) > os.path.getmtime(_SO) for s in _SRC)
    if stale:
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-fopenmp", "-fPIC", "-shared",
                               "-o", _SO] + _SRC)
    return _SO


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_kernel_alpha.restype = C.c_double
        _lib.orc_kernel_alpha.argtypes = [C.c_int]
        _lib.orc_num_threads.restype = C.c_int
        _lib.orc_kernel_phi.restype = C.c_double
        _lib.orc_kernel_phi.argtypes = [C.c_int, C.c_double]
        _lib.orc_kernel_phihat.restype = C.c_double
        _lib.orc_kernel_phihat.argtypes = [C.c_int, C.c_double, C.c_int]
        _lib.orc_bessel_i0.restype = C.c_double
        _lib.orc_bessel_i0.argtypes = [C.c_double]
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _c128(a):
    return np.ascontiguousarray(a, dtype=np.complex128)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def num_threads() -> int:
    return int(lib().orc_num_threads())


def kernel_alpha(m: int = DEFAULT_M) -> float:
    return float(lib().orc_kernel_alpha(int(m)))


KB = 16     # kernel code = half-width m (Gaussian) or KB + m (Kaiser-Bessel window); every `m` argument below takes a code


def kernel_phi(code: int, t: float) -> float:
    """Interpolation weight phi(t) of the kernel `code` (0 outside the open box |t| < m)."""
    return float(lib().orc_kernel_phi(int(code), float(t)))


def kernel_phihat(code: int, x: float, M: int) -> float:
    """Continuous transform of phi at x / M cycles per grid cell (the deapodisation factor of image coordinate x)."""
    return float(lib().orc_kernel_phihat(int(code), float(x), int(M)))


def bessel_i0(z: float) -> float:
    return float(lib().orc_bessel_i0(float(z)))


def dft(x, sign=-1):
    x = _c128(x)
    X = np.empty_like(x)
    lib().orc_dft(_p(x), _p(X), C.c_int(x.size), C.c_int(sign))
    return X


def fft(x, sign=-1):
    x = _c128(x)
    X = np.empty_like(x)
    lib().orc_fft(_p(x), _p(X), C.c_int(x.size), C.c_int(sign))
    return X


def neglog(raw, flat, dark):
    """raw u16 [nproj][nz][n], flat/dark f32 [nz][n] -> p f64 [nz][nproj][n]  (S1+S2)."""
    raw = np.ascontiguousarray(raw, dtype=np.uint16)
    nproj, nz, n = raw.shape
    flat, dark = _f32(flat), _f32(dark)
    assert flat.shape == (nz, n) and dark.shape == (nz, n)
    p = np.empty((nz, nproj, n))
    lib().orc_neglog(_p(raw), _p(flat), _p(dark), C.c_int(nproj), C.c_int(nz), C.c_int(n), _p(p))
    return p


def filter_table(M, filt="ramp"):
    H = np.empty(M)
    lib().orc_filter(C.c_int(M), C.c_int(FILTERS[filt]), _p(H))
    return H


PADS = {"zero": 0, "edge": 1}


def filter_rows(p, filt="ramp", pad="zero"):
    """p [rows][n] -> q [rows][n]  (S3); pad: "zero" (default) or "edge"."""
    p = _f64(p)
    rows, n = p.shape
    q = np.empty_like(p)
    lib().orc_filter_rows_pad(_p(p), C.c_int(rows), C.c_int(n), C.c_int(FILTERS[filt]), C.c_int(PADS[pad]), _p(q))
    return q


def spectrum(q, center):
    """q [nproj][n] -> G complex [nproj][2n], FFT order  (S4)."""
    q = _f64(q)
    nproj, n = q.shape
    G = np.empty((nproj, 2 * n), dtype=np.complex128)
    lib().orc_spectrum(_p(q), C.c_int(nproj), C.c_int(n), C.c_double(center), _p(G))
    return G


def _bp(fn, G, theta, n, m=None):
    G = _c128(G)
    theta = _f32(theta)
    nproj = theta.size
    assert G.shape == (nproj, 2 * n)
    fre, fim = np.empty((n, n)), np.empty((n, n))
    if m is None:
        fn(_p(G), _p(theta), C.c_int(nproj), C.c_int(n), _p(fre), _p(fim))
    else:
        fn(_p(G), _p(theta), C.c_int(nproj), C.c_int(n), C.c_int(m), _p(fre), _p(fim))
    return fre + 1j * fim


def backproject_exact(G, theta, n):
    """B_exact: complex image [n][n] (real part = the slice; imag = packed second slice)."""
    return _bp(lib().orc_backproject_exact, G, theta, n)


def backproject_grid(G, theta, n, m=DEFAULT_M):
    """B_grid = S5 -> S6 -> S7: complex image [n][n]."""
    return _bp(lib().orc_backproject_grid, G, theta, n, m)


def backproject_lin(q, theta, center):
    q = _f64(q)
    theta = _f32(theta)
    nproj, n = q.shape
    f = np.empty((n, n))
    lib().orc_backproject_lin(_p(q), _p(theta), C.c_int(nproj), C.c_int(n), C.c_double(center), _p(f))
    return f


def project_lin_adjoint(f, theta, center):
    f = _f64(f)
    theta = _f32(theta)
    n = f.shape[0]
    q = np.empty((theta.size, n))
    lib().orc_project_lin_adjoint(_p(f), _p(theta), C.c_int(theta.size), C.c_int(n),
                                  C.c_double(center), _p(q))
    return q


def grid(G, theta, n, m=DEFAULT_M):
    """S5: G [nproj][2n] -> F [2n][2n] (FFT order, row = l2)."""
    G = _c128(G)
    theta = _f32(theta)
    F = np.empty((2 * n, 2 * n), dtype=np.complex128)
    lib().orc_grid(_p(G), _p(theta), C.c_int(theta.size), C.c_int(n), C.c_int(m), _p(F))
    return F


def grid_adjoint(F, theta, n, m=DEFAULT_M):
    F = _c128(F)
    theta = _f32(theta)
    G = np.empty((theta.size, 2 * n), dtype=np.complex128)
    lib().orc_grid_adjoint(_p(F), _p(theta), C.c_int(theta.size), C.c_int(n), C.c_int(m), _p(G))
    return G


def fft2(F, sign=+1):
    """S6 (sign=+1: unnormalised inverse; -1: forward)."""
    F = _c128(F)
    g = np.empty_like(F)
    lib().orc_fft2(_p(F), C.c_int(F.shape[0]), C.c_int(sign), _p(g))
    return g


def deapod_crop(g, n, m=DEFAULT_M):
    """S7: g [2n][2n] -> complex f [n][n]."""
    g = _c128(g)
    fre, fim = np.empty((n, n)), np.empty((n, n))
    lib().orc_deapod_crop(_p(g), C.c_int(n), C.c_int(m), _p(fre), _p(fim))
    return fre + 1j * fim


def deapod_crop_adjoint(f, n, m=DEFAULT_M):
    f = _c128(f)
    fre, fim = _f64(f.real), _f64(f.imag)
    g = np.empty((2 * n, 2 * n), dtype=np.complex128)
    lib().orc_deapod_crop_adjoint(_p(fre), _p(fim), C.c_int(n), C.c_int(m), _p(g))
    return g


def angle_weights(theta):
    """Quadrature weights of the backprojection integral over [0, pi) for angles that are NOT equally spaced
    (the Fourier-based method, unlike the log-polar one, applies to "non-equally spaced angles",
    e.g. interlaced scanning; reading Q20): the trapezoid (midpoint-cell) rule on the periodic
    angle axis, w_j = (theta_{j+1} - theta_{j-1}) / 2 with theta_nproj = theta_0 + pi and
    theta_{-1} = theta_{nproj-1} - pi, returned RELATIVE to the constant pi/nproj the default path uses
    (all ones for equispaced angles over a half turn).  theta float32, increasing, spanning less than pi;
    arithmetic in double from the float32 values."""
    t = _f32(theta).astype(np.float64)
    nxt = np.concatenate([t[1:], [t[0] + np.pi]])
    prv = np.concatenate([[t[-1] - np.pi], t[:-1]])
    return 0.5 * (nxt - prv) * t.size / np.pi


def fbp_from_sino(p, theta, center, filt="ramp", m=DEFAULT_M, method="grid", return_q=False, pad="zero", fused=False,
                  angle_weighted=False):
    """p f64 [nz][nproj][n] -> out f64 [nz][n][n] (S3..S7 or the two definitions).
    angle_weighted: projection j enters with weight angle_weights(theta)[j] * pi/nproj instead of pi/nproj
    (everything after S2 is linear in the projection, so the row of the sinogram is scaled)."""
    p = _f64(p)
    theta = _f32(theta)
    if angle_weighted:
        p = np.ascontiguousarray(p * angle_weights(theta)[None, :, None])
    nz, nproj, n = p.shape
    out = np.empty((nz, n, n))
    q = np.empty_like(p) if return_q else None
    lib().orc_fbp_from_sino_pad(_p(p), _p(theta), C.c_int(nproj), C.c_int(nz), C.c_int(n),
                            C.c_double(center), C.c_int(FILTERS[filt]), C.c_int(PADS[pad] | (2 if fused else 0)), C.c_int(m),
                            C.c_int(METHODS[method]), _p(out), _p(q) if return_q else None)
    return (out, q) if return_q else out


def recon(raw, flat, dark, theta, center, filt="ramp", m=DEFAULT_M, method="grid", pad="zero", fused=False,
          angle_weighted=False):
    """uint16 counts -> reconstruction, S1..S7.  raw [nproj][nz][n] -> out [nz][n][n]."""
    raw = np.ascontiguousarray(raw, dtype=np.uint16)
    nproj, nz, n = raw.shape
    flat, dark, theta = _f32(flat), _f32(dark), _f32(theta)
    if angle_weighted:
        return fbp_from_sino(neglog(raw, flat, dark), theta, center, filt=filt, m=m, method=method, pad=pad, fused=fused,
                             angle_weighted=True)
    out = np.empty((nz, n, n))
    lib().orc_recon_pad(_p(raw), _p(flat), _p(dark), _p(theta), C.c_int(nproj), C.c_int(nz), C.c_int(n),
                    C.c_double(center), C.c_int(FILTERS[filt]), C.c_int(PADS[pad] | (2 if fused else 0)), C.c_int(m), C.c_int(METHODS[method]),
                    _p(out))
    return out


def remove_zingers(p, dif):
    """orc_zinger (reading Q22): p f64 [nz][nproj][n] -> copy with every sample that lies more than `dif` below the
    median of its 3 x 3 (projection, pixel) neighbourhood replaced by that median."""
    p = _f64(p)
    nz, nproj, n = p.shape
    out = np.empty_like(p)
    lib().orc_zinger(_p(p), C.c_int(nz), C.c_int(nproj), C.c_int(n), C.c_double(dif), _p(out))
    return out


def remove_rings(p, alpha, return_r=False):
    """orc_ring_ti (reading Q23): p f64 [nz][nproj][n] -> p minus the per-pixel offsets r[nz][n] estimated from the
    angle-averaged profile by the closed-form Tikhonov formula (A + alpha I) r = A pbar, A = D2^T D2."""
    p = _f64(p)
    nz, nproj, n = p.shape
    out, r = np.empty_like(p), np.empty((nz, n))
    lib().orc_ring_ti(_p(p), C.c_int(nz), C.c_int(nproj), C.c_int(n), C.c_double(alpha), _p(out), _p(r))
    return (out, r) if return_r else out


def recon_pre(raw, flat, dark, theta, center, filt="ramp", m=DEFAULT_M, method="grid", zinger_dif=0.0, ring_alpha=0.0):
    """S1+S2, then the optional pre-processing steps in the order zingers, rings (each off when its parameter is 0),
    then S3..S7: the chain tcp_recon runs with TCP_PARAM_ZINGER_DIF / TCP_PARAM_RING_ALPHA set."""
    p = neglog(raw, _f32(flat), _f32(dark))
    if zinger_dif > 0:
        p = remove_zingers(p, zinger_dif)
    if ring_alpha > 0:
        p = remove_rings(p, ring_alpha)
    return fbp_from_sino(p, theta, center, filt=filt, m=m, method=method)


def padded_size(ndet: int) -> tuple[int, int]:
    """Detector of any width ndet -> (n, pad_l): n = the power of two >= max(ndet, 64) the FFTs run on
    ("16-bit data are additionally padded/unpadded to the power of 2 sizes"; DESIGN.md
    reading Q19 applies it to fp32 too), pad_l = ceil((n - ndet)/2) air samples (p = 0) on the left, so
    that output pixel ix sits at x = ix - floor(ndet/2)."""
    n = 64
    while n < ndet:
        n *= 2
    return n, (n - ndet + 1) // 2


def recon_padded(raw, flat, dark, theta, center, filt="ramp", m=DEFAULT_M, method="grid", pad="zero"):
    """Detector width ndet not a power of two: S1+S2 on the ndet samples,
    every sinogram row embedded at offset pad_l in a row of n zeros ("padded"), the rotation centre moved
    with it, S3..S7 (or a definition) at size n, and the central ndet x ndet pixels cut out ("unpadded").
    raw [nproj][nz][ndet] -> out [nz][ndet][ndet]."""
    raw = np.ascontiguousarray(raw, dtype=np.uint16)
    nproj, nz, ndet = raw.shape
    n, pad_l = padded_size(ndet)
    p = neglog(raw, flat, dark)                                   # [nz][nproj][ndet]
    pp = np.zeros((nz, nproj, n))
    pp[:, :, pad_l:pad_l + ndet] = p
    out = fbp_from_sino(pp, theta, float(center) + pad_l, filt=filt, m=m, method=method, pad=pad)
    return np.ascontiguousarray(out[:, pad_l:pad_l + ndet, pad_l:pad_l + ndet])

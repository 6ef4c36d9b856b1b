"""ctypes loader for oracle/blink_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs import
this.  It marshals numpy arrays into the C oracle; all arithmetic is in blink_oracle.c.
It imports nothing from paper_2505_15204_b200.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "blink_oracle.c")
_SO = os.path.join(_HERE, "liboracle.so")
_lib = None


def build(force: bool = False) -> str:
    """gcc -O2 the oracle (no tuning flags; -ffp-contract=off keeps the fp32 index multiply exact)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        tmp = _SO + f".{os.getpid()}.tmp"
        subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-pthread",
                               "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _SO)
    return _SO


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        c_f, c_d, c_i = ctypes.c_float, ctypes.c_double, ctypes.c_int
        vp = ctypes.c_void_p
        L.oracle_scale.restype = c_f
        L.oracle_scale.argtypes = [c_d, c_i, c_d]
        L.oracle_cell.restype = ctypes.c_int32
        L.oracle_cell.argtypes = [c_f, c_f, c_f, c_i]
        L.oracle_mirror_cell.restype = ctypes.c_int32
        L.oracle_mirror_cell.argtypes = [ctypes.c_int32, c_i]
        L.oracle_cells.restype = None
        L.oracle_cells.argtypes = [vp, vp, c_i, c_i, c_i, c_i, c_d, vp]
        L.oracle_grid_one.restype = c_d
        L.oracle_grid_one.argtypes = [vp, vp, c_d, c_i, c_i, c_d, c_i, vp, vp, vp]
        L.oracle_idft2_direct.restype = None
        L.oracle_idft2_direct.argtypes = [vp, c_i, vp]
        L.oracle_sparse_image.restype = None
        L.oracle_sparse_image.argtypes = [vp, c_i, c_d, vp, vp]
        L.oracle_ifft2_radix2.restype = None
        L.oracle_ifft2_radix2.argtypes = [vp, c_i, vp]
        L.oracle_image_one.restype = c_d
        L.oracle_image_one.argtypes = [vp, vp, c_d, c_i, c_i, c_d, c_i, vp, vp, vp, vp, vp]
        L.oracle_image_batch.restype = c_i
        L.oracle_image_batch.argtypes = [vp, vp, vp, c_i, c_i, c_i, c_i, c_i, c_d, c_i, vp, c_i, vp, vp, c_i]
        L.oracle_image_avg.restype = c_i
        L.oracle_image_avg.argtypes = [vp, vp, vp, c_i, c_i, c_i, c_i, c_i, c_d, c_i, c_i, vp]
        L.oracle_apply_gains.restype = None
        L.oracle_apply_gains.argtypes = [vp, vp, vp, c_i, c_i, c_i, c_i, c_i, vp]
        _lib = L
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _c64(a):
    a = np.ascontiguousarray(a, dtype=np.complex64)
    return a


def scale(f_hz: float, n_pix: int, pixscale_rad: float) -> np.float32:
    return np.float32(lib().oracle_scale(float(f_hz), int(n_pix), float(pixscale_rad)))


def cell(u_m, v_m, s, n_pix: int) -> int:
    return int(lib().oracle_cell(float(np.float32(u_m)), float(np.float32(v_m)), float(np.float32(s)), int(n_pix)))


def mirror_cell(cell_: int, n_pix: int) -> int:
    return int(lib().oracle_mirror_cell(int(cell_), int(n_pix)))


def cells(uvw_m, freqs_hz, n_pix: int, pixscale_rad: float) -> np.ndarray:
    """cell_idx[T][C][B] int32 for the whole batch."""
    uvw = np.ascontiguousarray(uvw_m, dtype=np.float32)
    fr = np.ascontiguousarray(freqs_hz, dtype=np.float64)
    T, B, _ = uvw.shape
    C = fr.shape[0]
    out = np.empty((T, C, B), dtype=np.int32)
    lib().oracle_cells(_p(uvw), _p(fr), T, C, B, int(n_pix), float(pixscale_rad), _p(out))
    return out


def grid_one(vis_b, uvw_t, f_hz: float, n_pix: int, pixscale_rad: float, weighting: int):
    """-> (grid complex128 [N][N] centred, cnt uint32 [N][N], W float, cell_idx int32 [B])"""
    v = _c64(vis_b)
    uvw = np.ascontiguousarray(uvw_t, dtype=np.float32)
    B = v.shape[0]
    grid = np.empty((n_pix, n_pix), dtype=np.complex128)
    cnt = np.empty((n_pix, n_pix), dtype=np.uint32)
    ci = np.empty(B, dtype=np.int32)
    W = lib().oracle_grid_one(_p(v), _p(uvw), float(f_hz), B, int(n_pix), float(pixscale_rad),
                              int(weighting), _p(grid), _p(cnt), _p(ci))
    return grid, cnt, W, ci


def idft2_direct(grid) -> np.ndarray:
    g = np.ascontiguousarray(grid, dtype=np.complex128)
    out = np.empty_like(g)
    lib().oracle_idft2_direct(_p(g), g.shape[0], _p(out))
    return out


def ifft2_radix2(grid) -> np.ndarray:
    g = np.ascontiguousarray(grid, dtype=np.complex128)
    out = np.empty_like(g)
    lib().oracle_ifft2_radix2(_p(g), g.shape[0], _p(out))
    return out


def sparse_image(grid, W: float, want_imag: bool = False):
    g = np.ascontiguousarray(grid, dtype=np.complex128)
    n = g.shape[0]
    img = np.empty((n, n), dtype=np.float64)
    im = np.empty((n, n), dtype=np.float64) if want_imag else None
    lib().oracle_sparse_image(_p(g), n, float(W), _p(img), _p(im))
    return (img, im) if want_imag else img


def image_one(vis_b, uvw_t, f_hz: float, n_pix: int, pixscale_rad: float, weighting: int,
              want_imag: bool = False):
    """-> dict(image float64 [N][N], imag (opt), grid, cnt, W, cell_idx)"""
    v = _c64(vis_b)
    uvw = np.ascontiguousarray(uvw_t, dtype=np.float32)
    B = v.shape[0]
    img = np.empty((n_pix, n_pix), dtype=np.float64)
    im = np.empty((n_pix, n_pix), dtype=np.float64) if want_imag else None
    grid = np.empty((n_pix, n_pix), dtype=np.complex128)
    cnt = np.empty((n_pix, n_pix), dtype=np.uint32)
    ci = np.empty(B, dtype=np.int32)
    W = lib().oracle_image_one(_p(v), _p(uvw), float(f_hz), B, int(n_pix), float(pixscale_rad),
                               int(weighting), _p(img), _p(im), _p(grid), _p(cnt), _p(ci))
    return dict(image=img, imag=im, grid=grid, cnt=cnt, W=W, cell_idx=ci)


def image_batch(vis, uvw_m, freqs_hz, n_pix: int, pixscale_rad: float, weighting: int,
                img_ids=None, nthreads: int = 1):
    """vis [T][C][P][B] complex64, uvw_m [T][B][3] -> (images float64 [n][N][N], wsum float64 [n])"""
    v = _c64(vis)
    uvw = np.ascontiguousarray(uvw_m, dtype=np.float32)
    fr = np.ascontiguousarray(freqs_hz, dtype=np.float64)
    T, C, P, B = v.shape
    if img_ids is None:
        img_ids = np.arange(T * C * P)
    ids = np.ascontiguousarray(img_ids, dtype=np.int64)
    images = np.empty((len(ids), n_pix, n_pix), dtype=np.float64)
    wsum = np.empty(len(ids), dtype=np.float64)
    rc = lib().oracle_image_batch(_p(v), _p(uvw), _p(fr), T, C, P, B, int(n_pix), float(pixscale_rad),
                                  int(weighting), _p(ids), len(ids), _p(images), _p(wsum), int(nthreads))
    if rc != 0:
        raise RuntimeError("oracle_image_batch failed")
    return images, wsum


def image_avg(vis, uvw_m, freqs_hz, n_pix: int, pixscale_rad: float, weighting: int, avg_time: bool = False):
    """Mean of the dirty images over channels (-> [T][P][N][N]) or over timesteps and channels (-> [P][N][N])."""
    v = _c64(vis)
    uvw = np.ascontiguousarray(uvw_m, dtype=np.float32)
    fr = np.ascontiguousarray(freqs_hz, dtype=np.float64)
    T, C, P, B = v.shape
    out = np.empty(((P,) if avg_time else (T, P)) + (n_pix, n_pix), dtype=np.float64)
    rc = lib().oracle_image_avg(_p(v), _p(uvw), _p(fr), T, C, P, B, int(n_pix), float(pixscale_rad),
                                int(weighting), int(bool(avg_time)), _p(out))
    if rc != 0:
        raise RuntimeError("oracle_image_avg failed")
    return out


def apply_gains(vis, gains, ant_pairs):
    """vis [T][C][P][B] complex64, gains [C][P][A] complex64, ant_pairs [B][2] int32 -> corrected vis (complex64)."""
    v = _c64(vis)
    g = _c64(gains)
    ap = np.ascontiguousarray(ant_pairs, dtype=np.int32)
    T, C, P, B = v.shape
    A = g.shape[2]
    assert g.shape[:2] == (C, P) and ap.shape == (B, 2) and ap.min() >= 0 and ap.max() < A
    out = np.empty_like(v)
    lib().oracle_apply_gains(_p(v), _p(g), _p(ap), T, C, P, B, A, _p(out))
    return out


def image_stokes_i(vis, uvw_m, freqs_hz, n_pix: int, pixscale_rad: float, weighting: int, tc_ids=None):
    """vis [T][C][P][B] (P = 2: XX, YY; P = 4: XX, XY, YX, YY) -> ((I_XX + I_YY) / 2 float64 [n][N][N], wsum [n]); tc = t*C + c."""
    v = _c64(vis)
    uvw = np.ascontiguousarray(uvw_m, dtype=np.float32)
    fr = np.ascontiguousarray(freqs_hz, dtype=np.float64)
    T, C, P, B = v.shape
    ids = np.ascontiguousarray(np.arange(T * C) if tc_ids is None else tc_ids, dtype=np.int64)
    L = lib()
    L.oracle_image_stokes_i.restype = ctypes.c_int
    L.oracle_image_stokes_i.argtypes = [ctypes.c_void_p] * 3 + [ctypes.c_int] * 5 + [ctypes.c_double, ctypes.c_int,
                                        ctypes.c_void_p, ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p]
    out = np.empty((len(ids), n_pix, n_pix), dtype=np.float64)
    wsum = np.empty(len(ids), dtype=np.float64)
    rc = L.oracle_image_stokes_i(_p(v), _p(uvw), _p(fr), T, C, P, B, int(n_pix), float(pixscale_rad), int(weighting),
                                 _p(ids), len(ids), _p(out), _p(wsum))
    if rc != 0:
        raise ValueError("oracle_image_stokes_i: P must be 2 or 4 and tc_ids inside the batch")
    return out, wsum


# ---- convolutional gridding (reading R16) ----------------------------------
def _conv_protos():
    L = lib()
    if getattr(L, "_conv_ready", False):
        return L
    c_f, c_d, c_i, vp = ctypes.c_float, ctypes.c_double, ctypes.c_int, ctypes.c_void_p
    L.oracle_bessel_i0.restype = c_d
    L.oracle_bessel_i0.argtypes = [c_d]
    L.oracle_kb.restype = c_d
    L.oracle_kb.argtypes = [c_d, c_i, c_d]
    L.oracle_conv_taps.restype = None
    L.oracle_conv_taps.argtypes = [c_d, c_i, c_d, vp]
    L.oracle_conv_taper.restype = c_d
    L.oracle_conv_taper.argtypes = [c_d, c_i, c_d]
    L.oracle_cell_conv.restype = ctypes.c_int32
    L.oracle_cell_conv.argtypes = [c_f, c_f, c_f, c_i, c_i, vp, vp]
    L.oracle_grid_conv_one.restype = c_d
    L.oracle_grid_conv_one.argtypes = [vp, vp, c_d, c_i, c_i, c_d, c_i, c_d, vp, vp]
    L.oracle_image_conv_one.restype = c_d
    L.oracle_image_conv_one.argtypes = [vp, vp, c_d, c_i, c_i, c_d, c_i, c_d, vp, vp, vp, vp]
    L.oracle_image_conv_batch.restype = c_i
    L.oracle_image_conv_batch.argtypes = [vp, vp, vp, c_i, c_i, c_i, c_i, c_i, c_d, c_i, c_d, vp, c_i, vp, vp, c_i]
    L._conv_ready = True
    return L


def bessel_i0(x: float) -> float:
    return float(_conv_protos().oracle_bessel_i0(float(x)))


def kb(d: float, support: int, beta: float) -> float:
    return float(_conv_protos().oracle_kb(float(d), int(support), float(beta)))


def conv_taps(f: float, support: int, beta: float) -> np.ndarray:
    w = np.empty(int(support), dtype=np.float64)
    _conv_protos().oracle_conv_taps(float(f), int(support), float(beta), _p(w))
    return w


def conv_taper(n_pix: int, support: int, beta: float) -> np.ndarray:
    """c((x - h)/N) for x = 0..N-1."""
    L = _conv_protos()
    h = n_pix // 2
    return np.array([L.oracle_conv_taper((x - h) / n_pix, int(support), float(beta)) for x in range(n_pix)])


def cell_conv(u_m, v_m, s, n_pix: int, support: int):
    """-> (cell or -1, fx, fy)"""
    fx, fy = ctypes.c_double(0.0), ctypes.c_double(0.0)
    c = _conv_protos().oracle_cell_conv(float(np.float32(u_m)), float(np.float32(v_m)), float(np.float32(s)),
                                        int(n_pix), int(support), ctypes.byref(fx), ctypes.byref(fy))
    return int(c), fx.value, fy.value


def grid_conv_one(vis_b, uvw_t, f_hz: float, n_pix: int, pixscale_rad: float, support: int, beta: float):
    """-> (grid complex128 [N][N] centred, W, cell_idx int32 [B])"""
    v = _c64(vis_b)
    uvw = np.ascontiguousarray(uvw_t, dtype=np.float32)
    B = v.shape[0]
    grid = np.empty((n_pix, n_pix), dtype=np.complex128)
    ci = np.empty(B, dtype=np.int32)
    W = _conv_protos().oracle_grid_conv_one(_p(v), _p(uvw), float(f_hz), B, int(n_pix), float(pixscale_rad),
                                            int(support), float(beta), _p(grid), _p(ci))
    return grid, W, ci


def image_conv_one(vis_b, uvw_t, f_hz: float, n_pix: int, pixscale_rad: float, support: int, beta: float,
                   want_imag: bool = False):
    v = _c64(vis_b)
    uvw = np.ascontiguousarray(uvw_t, dtype=np.float32)
    B = v.shape[0]
    img = np.empty((n_pix, n_pix), dtype=np.float64)
    im = np.empty((n_pix, n_pix), dtype=np.float64) if want_imag else None
    grid = np.empty((n_pix, n_pix), dtype=np.complex128)
    ci = np.empty(B, dtype=np.int32)
    W = _conv_protos().oracle_image_conv_one(_p(v), _p(uvw), float(f_hz), B, int(n_pix), float(pixscale_rad),
                                             int(support), float(beta), _p(img), _p(im), _p(grid), _p(ci))
    return dict(image=img, imag=im, grid=grid, W=W, cell_idx=ci)


def image_conv_batch(vis, uvw_m, freqs_hz, n_pix: int, pixscale_rad: float, support: int, beta: float,
                     img_ids=None, nthreads: int = 1):
    v = _c64(vis)
    uvw = np.ascontiguousarray(uvw_m, dtype=np.float32)
    fr = np.ascontiguousarray(freqs_hz, dtype=np.float64)
    T, C, P, B = v.shape
    if img_ids is None:
        img_ids = np.arange(T * C * P)
    ids = np.ascontiguousarray(img_ids, dtype=np.int64)
    images = np.empty((len(ids), n_pix, n_pix), dtype=np.float64)
    wsum = np.empty(len(ids), dtype=np.float64)
    rc = _conv_protos().oracle_image_conv_batch(_p(v), _p(uvw), _p(fr), T, C, P, B, int(n_pix), float(pixscale_rad),
                                                int(support), float(beta), _p(ids), len(ids), _p(images), _p(wsum),
                                                int(nthreads))
    if rc != 0:
        raise RuntimeError("oracle_image_conv_batch failed")
    return images, wsum


# ---- CMAC correlator (reading R17) -------------------------------------------
def correlate(volt, n_t: int, n_avg: int) -> np.ndarray:
    """volt [F][A][Ns][2] int8 -> vis [T][C][A(A+1)/2] complex64 (lower triangle, autos included)."""
    v = np.ascontiguousarray(volt, dtype=np.int8)
    F, A, Ns, two = v.shape
    assert two == 2
    L = lib()
    L.oracle_correlate.restype = ctypes.c_int
    L.oracle_correlate.argtypes = [ctypes.c_void_p] + [ctypes.c_int] * 5 + [ctypes.c_void_p]
    T, C = Ns // n_t, F // n_avg
    out = np.empty((T, C, A * (A + 1) // 2), dtype=np.complex64)
    rc = L.oracle_correlate(_p(v), F, A, Ns, int(n_t), int(n_avg), _p(out))
    if rc != 0:
        raise ValueError("oracle_correlate: Ns must be a multiple of n_t and F of n_avg")
    return out

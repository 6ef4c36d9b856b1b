"""Thin ctypes binding of libblinkimg (include/blinkimg.h): argument marshalling only.

PyTorch is used for device memory and streams; every step of the path runs in the library's CUDA
kernels.  There is no fallback: if the shared library is missing or a call fails, this raises.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libblinkimg.so")
_lib = None

W_NATURAL, W_UNIFORM = 0, 1
OP_GRID, OP_FFT2D, OP_IMAGE, OP_IMAGE_HOST, OP_IMAGE_AVG, OP_IMAGE_CONV, OP_IMAGE_STOKES_I, OP_IMAGE_CAL = 0, 1, 2, 3, 4, 5, 6, 7
OPT_IMAGE_PATH, OPT_FUSED_CTAS, OPT_GRID_CHUNK_B, OPT_AVG_WSUM, OPT_CORR_PATH, OPT_FUSED_TEAM = 0, 1, 2, 3, 4, 5

EXPORTS = ["blink_strerror", "blink_last_cuda_error", "blink_set_option", "blink_get_option",
           "blink_kernel_launches", "blink_workspace_bytes", "blink_grid", "blink_fft2d_inverse",
           "blink_image", "blink_image_host", "blink_image_avg", "blink_apply_gains", "blink_image_cal",
           "blink_image_conv", "blink_conv_taps_host", "blink_correlate", "blink_image_stokes_i",
           "blink_volt_out_of_range", "blink_static_scratch_bytes", "blink_image_static"]


class BlinkError(RuntimeError):
    pass


def lib_path() -> str:
    return _SO


def lib():
    """Loads libblinkimg.so (built in-tree by paper_2505_15204_b200/build.py).  Fails loudly if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(_SO):
            raise BlinkError(f"{_SO} not found: run `python -m paper_2505_15204_b200.build` (needs nvcc); "
                             "there is no CPU fallback")
        L = ctypes.CDLL(_SO)
        vp, i, d, sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_size_t
        L.blink_strerror.restype = ctypes.c_char_p
        L.blink_strerror.argtypes = [i]
        L.blink_last_cuda_error.restype = ctypes.c_char_p
        L.blink_last_cuda_error.argtypes = []
        L.blink_set_option.restype = i
        L.blink_set_option.argtypes = [i, i]
        L.blink_get_option.restype = i
        L.blink_get_option.argtypes = [i, ctypes.POINTER(i)]
        L.blink_kernel_launches.restype = ctypes.c_ulonglong
        L.blink_kernel_launches.argtypes = []
        L.blink_workspace_bytes.restype = i
        L.blink_workspace_bytes.argtypes = [i, i, i, i, i, i, i, ctypes.POINTER(sz), ctypes.POINTER(sz)]
        L.blink_grid.restype = i
        L.blink_grid.argtypes = [vp, vp, vp, i, i, i, i, i, d, i, vp, vp, vp, vp, vp, sz, vp]
        L.blink_fft2d_inverse.restype = i
        L.blink_fft2d_inverse.argtypes = [vp, i, i, vp, i, vp, vp, vp, sz, vp]
        L.blink_image.restype = i
        L.blink_image.argtypes = [vp, vp, vp, i, i, i, i, i, d, i, vp, vp, vp, vp, vp, sz, vp]
        L.blink_image_host.restype = i
        L.blink_image_host.argtypes = [vp, vp, vp, i, i, i, i, i, d, i, vp, vp, vp, sz]
        L.blink_image_avg.restype = i
        L.blink_image_avg.argtypes = [vp, vp, vp, i, i, i, i, i, d, i, i, vp, vp, vp, sz, vp]
        L.blink_apply_gains.restype = i
        L.blink_apply_gains.argtypes = [vp, vp, vp, i, i, i, i, i, vp]
        L.blink_image_cal.restype = i
        L.blink_image_cal.argtypes = [vp, vp, vp, vp, vp, i, i, i, i, i, i, d, i, vp, vp, vp, sz, vp]
        L.blink_image_conv.restype = i
        L.blink_image_conv.argtypes = [vp, vp, vp, i, i, i, i, i, d, i, d, vp, vp, vp, vp, sz, vp]
        L.blink_conv_taps_host.restype = i
        L.blink_conv_taps_host.argtypes = [d, i, d, vp, ctypes.POINTER(d)]
        L.blink_correlate.restype = i
        L.blink_correlate.argtypes = [vp, i, i, i, i, i, vp, vp]
        L.blink_image_stokes_i.restype = i
        L.blink_image_stokes_i.argtypes = [vp, vp, vp, i, i, i, i, i, d, i, vp, vp, vp, sz, vp]
        L.blink_volt_out_of_range.restype = i
        L.blink_volt_out_of_range.argtypes = [vp, sz, vp, vp]
        L.blink_static_scratch_bytes.restype = sz
        L.blink_static_scratch_bytes.argtypes = []
        L.blink_image_static.restype = i
        L.blink_image_static.argtypes = [vp, vp, vp, i, i, i, i, i, d, i, vp, vp, vp]
        _lib = L
    return _lib


def _check(rc: int, what: str) -> None:
    if rc != 0:
        L = lib()
        msg = L.blink_strerror(rc).decode()
        extra = L.blink_last_cuda_error().decode()
        raise BlinkError(f"{what} failed: {msg} ({rc})" + (f": {extra}" if extra else ""))


def _ptr(t: Optional[torch.Tensor]):
    return None if t is None else ctypes.c_void_p(t.data_ptr())


def _stream(device) -> ctypes.c_void_p:
    return ctypes.c_void_p(torch.cuda.current_stream(device).cuda_stream)


def _dev(t: torch.Tensor, dtype, name: str, shape=None, device=None) -> torch.Tensor:
    """Argument check only: contiguous CUDA tensor of the given dtype (and shape / device when stated)."""
    if not isinstance(t, torch.Tensor) or not t.is_cuda or t.dtype != dtype or not t.is_contiguous():
        raise BlinkError(f"{name} must be a contiguous CUDA tensor of dtype {dtype}")
    if shape is not None and tuple(t.shape) != tuple(shape):
        raise BlinkError(f"{name} must have shape {tuple(shape)}, got {tuple(t.shape)}")
    if device is not None and t.device != device:
        raise BlinkError(f"{name} is on {t.device}, expected {device}")
    return t


def _out(t: Optional[torch.Tensor], dtype, n_elems: int, name: str, device) -> None:
    """Caller-supplied output / workspace: right device and dtype, contiguous, at least n_elems elements."""
    if t is None:
        return
    if not t.is_cuda or t.device != device or t.dtype != dtype or not t.is_contiguous() or t.numel() < n_elems:
        raise BlinkError(f"{name} must be a contiguous {dtype} tensor on {device} with at least {n_elems} elements")


def _vis_uvw(vis: torch.Tensor, uvw_m: torch.Tensor, freqs_hz):
    """vis [T][C][P][B] complex64 and uvw_m [T][B][3] float32 on one device, len(freqs_hz) == C."""
    _dev(vis, torch.complex64, "vis")
    if vis.dim() != 4:
        raise BlinkError(f"vis must be [T][C][P][B], got {tuple(vis.shape)}")
    T, C, P, B = vis.shape
    _dev(uvw_m, torch.float32, "uvw_m", (T, B, 3), vis.device)
    fr = _freqs(freqs_hz)
    if fr.ndim != 1 or fr.shape[0] != C:
        raise BlinkError(f"freqs_hz must hold C = {C} frequencies, got shape {fr.shape}")
    return T, C, P, B, fr, vis.device


def set_option(key: int, value: int) -> None:
    _check(lib().blink_set_option(int(key), int(value)), "blink_set_option")


def kernel_launches() -> int:
    return int(lib().blink_kernel_launches())


def blink_workspace_bytes(op: int, T: int, C: int, P: int, B: int, n_pix: int, weighting: int):
    """-> (recommended_bytes, min_bytes)"""
    rec, mn = ctypes.c_size_t(0), ctypes.c_size_t(0)
    _check(lib().blink_workspace_bytes(op, T, C, P, B, n_pix, weighting, ctypes.byref(rec), ctypes.byref(mn)),
           "blink_workspace_bytes")
    return int(rec.value), int(mn.value)


def _freqs(freqs_hz) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(freqs_hz, dtype=np.float64))


def blink_grid(vis: torch.Tensor, uvw_m: torch.Tensor, freqs_hz, n_pix: int, pixscale_rad: float, weighting: int = 0,
               want_cell_idx: bool = False, want_counts: bool = False, grid: Optional[torch.Tensor] = None):
    """vis [T][C][P][B] complex64, uvw_m [T][B][3] float32 (CUDA) -> dict(grid, wsum, cell_idx?, counts?)"""
    T, C, P, B, fr, dev = _vis_uvw(vis, uvw_m, freqs_hz)
    _out(grid, torch.complex64, T * C * P * n_pix * n_pix, "grid", dev)
    if grid is None:
        grid = torch.empty((T * C * P, n_pix, n_pix), dtype=torch.complex64, device=dev)
    wsum = torch.empty(T * C, dtype=torch.float32, device=dev)
    cell_idx = torch.empty((T, C, B), dtype=torch.int32, device=dev) if want_cell_idx else None
    counts = torch.empty((T * C, n_pix, n_pix), dtype=torch.int32, device=dev) if want_counts else None
    rec, _ = blink_workspace_bytes(OP_GRID, T, C, P, B, n_pix, weighting)
    ws = torch.empty(max(rec, 16), dtype=torch.uint8, device=dev)
    with torch.cuda.device(dev):
        rc = lib().blink_grid(_ptr(vis), _ptr(uvw_m), fr.ctypes.data_as(ctypes.c_void_p), T, C, P, B, n_pix,
                              float(pixscale_rad), int(weighting), _ptr(grid), _ptr(wsum), _ptr(cell_idx), _ptr(counts),
                              _ptr(ws), ws.numel(), _stream(dev))
    _check(rc, "blink_grid")
    return dict(grid=grid, wsum=wsum, cell_idx=cell_idx, counts=counts)


def blink_fft2d_inverse(grid: torch.Tensor, scale: Optional[torch.Tensor] = None, scale_stride_div: int = 1,
                        want_imag: bool = False, image: Optional[torch.Tensor] = None):
    """grid [batch][N][N] complex64 (CUDA, CLOBBERED) -> dict(image float32, imag?)"""
    _dev(grid, torch.complex64, "grid")
    if grid.dim() != 3 or grid.shape[1] != grid.shape[2]:
        raise BlinkError(f"grid must be [batch][N][N], got {tuple(grid.shape)}")
    batch, n, _ = grid.shape
    dev = grid.device
    _out(image, torch.float32, batch * n * n, "image", dev)
    if image is None:
        image = torch.empty((batch, n, n), dtype=torch.float32, device=dev)
    imag = torch.empty((batch, n, n), dtype=torch.float32, device=dev) if want_imag else None
    if scale is not None:
        _dev(scale, torch.float32, "scale", device=dev)
        if scale_stride_div < 1 or scale.numel() < -(-batch // int(scale_stride_div)):
            raise BlinkError("scale must hold ceil(batch / scale_stride_div) entries")
    rec, _ = blink_workspace_bytes(OP_FFT2D, batch, 1, 1, 0, n, 0)         # non-zero only for sides that are not 2^k
    ws = torch.empty(rec, dtype=torch.uint8, device=dev) if rec else None
    with torch.cuda.device(dev):
        rc = lib().blink_fft2d_inverse(_ptr(grid), n, batch, _ptr(scale), int(scale_stride_div), _ptr(image), _ptr(imag),
                                       _ptr(ws), rec, _stream(dev))
    _check(rc, "blink_fft2d_inverse")
    return dict(image=image, imag=imag)


def _image_outputs(T, C, P_out, n_pix, dev, image, wsum, name="image"):
    _out(image, torch.float32, T * C * P_out * n_pix * n_pix, name, dev)
    _out(wsum, torch.float32, T * C, "wsum", dev)
    if image is None:
        image = torch.empty((T * C * P_out, n_pix, n_pix), dtype=torch.float32, device=dev)
    if wsum is None:
        wsum = torch.empty(T * C, dtype=torch.float32, device=dev)
    return image, wsum


def _workspace(workspace, op, T, C, P, B, n_pix, weighting, dev):
    if workspace is None:
        rec, _ = blink_workspace_bytes(op, T, C, P, B, n_pix, weighting)
        return torch.empty(max(rec, 256), dtype=torch.uint8, device=dev)
    _out(workspace, torch.uint8, 0, "workspace", dev)
    if workspace.data_ptr() % 256:
        raise BlinkError("workspace must be 256-byte aligned")
    return workspace


def blink_image(vis: torch.Tensor, uvw_m: torch.Tensor, freqs_hz, n_pix: int, pixscale_rad: float, weighting: int = 0,
                want_cell_idx: bool = False, want_counts: bool = False, image: Optional[torch.Tensor] = None,
                workspace: Optional[torch.Tensor] = None, wsum: Optional[torch.Tensor] = None):
    """vis [T][C][P][B] complex64, uvw_m [T][B][3] float32 (CUDA) -> dict(image [T*C*P][N][N] float32, wsum, ...)"""
    T, C, P, B, fr, dev = _vis_uvw(vis, uvw_m, freqs_hz)
    image, wsum = _image_outputs(T, C, P, n_pix, dev, image, wsum)
    cell_idx = torch.empty((T, C, B), dtype=torch.int32, device=dev) if want_cell_idx else None
    counts = torch.empty((T * C, n_pix, n_pix), dtype=torch.int32, device=dev) if want_counts else None
    workspace = _workspace(workspace, OP_IMAGE, T, C, P, B, n_pix, weighting, dev)
    with torch.cuda.device(dev):
        rc = lib().blink_image(_ptr(vis), _ptr(uvw_m), fr.ctypes.data_as(ctypes.c_void_p), T, C, P, B, n_pix,
                               float(pixscale_rad), int(weighting), _ptr(image), _ptr(wsum), _ptr(cell_idx), _ptr(counts),
                               _ptr(workspace), workspace.numel(), _stream(dev))
    _check(rc, "blink_image")
    return dict(image=image, wsum=wsum, cell_idx=cell_idx, counts=counts)


def blink_static_scratch_bytes() -> int:
    return int(lib().blink_static_scratch_bytes())


def blink_image_static(vis: torch.Tensor, uvw_m: torch.Tensor, freqs_hz, n_pix: int, pixscale_rad: float, weighting: int = 0,
                       image: Optional[torch.Tensor] = None, wsum: Optional[torch.Tensor] = None):
    """blink_image with the library's built-in 32 MiB scratch array instead of a workspace: the call allocates no device memory
    when image and wsum are passed in.  Calls that overlap on the GPU race on that array; larger problems raise BlinkError."""
    T, C, P, B, fr, dev = _vis_uvw(vis, uvw_m, freqs_hz)
    image, wsum = _image_outputs(T, C, P, n_pix, dev, image, wsum)
    with torch.cuda.device(dev):
        rc = lib().blink_image_static(_ptr(vis), _ptr(uvw_m), fr.ctypes.data_as(ctypes.c_void_p), T, C, P, B, n_pix,
                                      float(pixscale_rad), int(weighting), _ptr(image), _ptr(wsum), _stream(dev))
    _check(rc, "blink_image_static")
    return dict(image=image, wsum=wsum)


def blink_image_stokes_i(vis: torch.Tensor, uvw_m: torch.Tensor, freqs_hz, n_pix: int, pixscale_rad: float,
                         weighting: int = 0, image: Optional[torch.Tensor] = None,
                         workspace: Optional[torch.Tensor] = None, wsum: Optional[torch.Tensor] = None):
    """vis [T][C][P][B] with P = 2 (XX, YY) or 4 (XX, XY, YX, YY) -> dict(image [T*C][N][N] = (I_XX + I_YY) / 2, wsum)"""
    T, C, P, B, fr, dev = _vis_uvw(vis, uvw_m, freqs_hz)
    image, wsum = _image_outputs(T, C, 1, n_pix, dev, image, wsum)
    workspace = _workspace(workspace, OP_IMAGE_STOKES_I, T, C, P, B, n_pix, weighting, dev)
    with torch.cuda.device(dev):
        rc = lib().blink_image_stokes_i(_ptr(vis), _ptr(uvw_m), fr.ctypes.data_as(ctypes.c_void_p), T, C, P, B, n_pix,
                                        float(pixscale_rad), int(weighting), _ptr(image), _ptr(wsum),
                                        _ptr(workspace), workspace.numel(), _stream(dev))
    _check(rc, "blink_image_stokes_i")
    return dict(image=image, wsum=wsum)


def blink_image_avg(vis: torch.Tensor, uvw_m: torch.Tensor, freqs_hz, n_pix: int, pixscale_rad: float, weighting: int = 0,
                    avg_time: bool = False, image_avg: Optional[torch.Tensor] = None,
                    workspace: Optional[torch.Tensor] = None, wsum: Optional[torch.Tensor] = None):
    """Mean of the dirty images over channels (-> [T*P][N][N]) or over timesteps and channels (-> [P][N][N])."""
    T, C, P, B, fr, dev = _vis_uvw(vis, uvw_m, freqs_hz)
    n_out = P if avg_time else T * P
    _out(image_avg, torch.float32, n_out * n_pix * n_pix, "image_avg", dev)
    _out(wsum, torch.float32, T * C, "wsum", dev)
    if image_avg is None:
        image_avg = torch.empty((n_out, n_pix, n_pix), dtype=torch.float32, device=dev)
    if wsum is None:
        wsum = torch.empty(T * C, dtype=torch.float32, device=dev)
    workspace = _workspace(workspace, OP_IMAGE_AVG, T, C, P, B, n_pix, weighting, dev)
    with torch.cuda.device(dev):
        rc = lib().blink_image_avg(_ptr(vis), _ptr(uvw_m), fr.ctypes.data_as(ctypes.c_void_p), T, C, P, B, n_pix,
                                   float(pixscale_rad), int(weighting), int(bool(avg_time)), _ptr(image_avg), _ptr(wsum),
                                   _ptr(workspace), workspace.numel(), _stream(dev))
    _check(rc, "blink_image_avg")
    return dict(image_avg=image_avg, wsum=wsum)


def _gains_pairs(gains: torch.Tensor, ant_pairs: torch.Tensor, C: int, P: int, B: int, dev):
    _dev(gains, torch.complex64, "gains", device=dev)
    if gains.dim() != 3 or gains.shape[0] != C or gains.shape[1] != P or gains.shape[2] < 1:
        raise BlinkError(f"gains must be [C={C}][P={P}][A], got {tuple(gains.shape)}")
    _dev(ant_pairs, torch.int32, "ant_pairs", (B, 2), dev)
    return int(gains.shape[2])


def blink_apply_gains(vis: torch.Tensor, gains: torch.Tensor, ant_pairs: torch.Tensor):
    """In place: vis[t][c][p][b] *= gains[c][p][a1] * conj(gains[c][p][a2]); ant_pairs [B][2] int32 (CUDA), 0 <= a < A."""
    _dev(vis, torch.complex64, "vis")
    if vis.dim() != 4:
        raise BlinkError(f"vis must be [T][C][P][B], got {tuple(vis.shape)}")
    T, C, P, B = vis.shape
    A = _gains_pairs(gains, ant_pairs, C, P, B, vis.device)
    with torch.cuda.device(vis.device):
        rc = lib().blink_apply_gains(_ptr(vis), _ptr(gains), _ptr(ant_pairs), T, C, P, B, A, _stream(vis.device))
    _check(rc, "blink_apply_gains")
    return vis


def blink_image_cal(vis: torch.Tensor, uvw_m: torch.Tensor, freqs_hz, gains: torch.Tensor, ant_pairs: torch.Tensor,
                    n_pix: int, pixscale_rad: float, weighting: int = 0, image: Optional[torch.Tensor] = None,
                    workspace: Optional[torch.Tensor] = None, wsum: Optional[torch.Tensor] = None):
    """blink_image with per-antenna gain corrections fused into the gridder's load (vis is left untouched)."""
    T, C, P, B, fr, dev = _vis_uvw(vis, uvw_m, freqs_hz)
    A = _gains_pairs(gains, ant_pairs, C, P, B, dev)
    image, wsum = _image_outputs(T, C, P, n_pix, dev, image, wsum)
    workspace = _workspace(workspace, OP_IMAGE_CAL, T, C, P, B, n_pix, weighting, dev)
    with torch.cuda.device(dev):
        rc = lib().blink_image_cal(_ptr(vis), _ptr(uvw_m), fr.ctypes.data_as(ctypes.c_void_p), _ptr(gains), _ptr(ant_pairs),
                                   A, T, C, P, B, n_pix, float(pixscale_rad), int(weighting), _ptr(image),
                                   _ptr(wsum), _ptr(workspace), workspace.numel(), _stream(dev))
    _check(rc, "blink_image_cal")
    return dict(image=image, wsum=wsum)


def blink_image_conv(vis: torch.Tensor, uvw_m: torch.Tensor, freqs_hz, n_pix: int, pixscale_rad: float, support: int,
                     beta: float = 0.0, image: Optional[torch.Tensor] = None, workspace: Optional[torch.Tensor] = None,
                     wsum: Optional[torch.Tensor] = None, want_cell_idx: bool = False):
    """blink_image with the Kaiser-Bessel gridding kernel of odd support 3 / 5 / 7 (natural weighting, grid-corrected)."""
    T, C, P, B, fr, dev = _vis_uvw(vis, uvw_m, freqs_hz)
    image, wsum = _image_outputs(T, C, P, n_pix, dev, image, wsum)
    cell_idx = torch.empty((T, C, B), dtype=torch.int32, device=dev) if want_cell_idx else None
    workspace = _workspace(workspace, OP_IMAGE_CONV, T, C, P, B, n_pix, 0, dev)
    with torch.cuda.device(dev):
        rc = lib().blink_image_conv(_ptr(vis), _ptr(uvw_m), fr.ctypes.data_as(ctypes.c_void_p), T, C, P, B, n_pix,
                                    float(pixscale_rad), int(support), float(beta), _ptr(image), _ptr(wsum), _ptr(cell_idx),
                                    _ptr(workspace), workspace.numel(), _stream(dev))
    _check(rc, "blink_image_conv")
    return dict(image=image, wsum=wsum, cell_idx=cell_idx)


def blink_conv_taps_host(f: float, support: int, beta: float = 0.0):
    """-> (float32 [support] tap weights as the kernel evaluates them, largest deviation of the fit). No GPU needed."""
    w = np.empty(int(support), dtype=np.float32)
    err = ctypes.c_double(0.0)
    rc = lib().blink_conv_taps_host(float(f), int(support), float(beta), w.ctypes.data_as(ctypes.c_void_p), ctypes.byref(err))
    _check(rc, "blink_conv_taps_host")
    return w, err.value


def blink_volt_out_of_range(volt: torch.Tensor) -> int:
    """Number of int8 samples equal to -128 (outside blink_correlate's input contract [-127, 127]); synchronises."""
    _dev(volt, torch.int8, "volt")
    cnt = torch.zeros(1, dtype=torch.int64, device=volt.device)
    with torch.cuda.device(volt.device):
        rc = lib().blink_volt_out_of_range(_ptr(volt), volt.numel(), _ptr(cnt), _stream(volt.device))
    _check(rc, "blink_volt_out_of_range")
    return int(cnt.item())


def blink_correlate(volt: torch.Tensor, n_t: int, n_avg: int, vis: Optional[torch.Tensor] = None, check_range: bool = False):
    """volt [F][A][Ns][2] int8 (CUDA) -> vis [T][C][A(A+1)/2] complex64: lower-triangular CMAC products per interval / channel.

    Input contract (include/blinkimg.h): every sample in [-127, 127].  The kernel negates imaginary parts bytewise, and
    -(-128) does not exist in int8: a sample of -128 silently gives wrong imaginary parts.  check_range=True counts such
    samples first (one extra pass over volt, synchronising) and raises."""
    _dev(volt, torch.int8, "volt")
    if volt.dim() != 4 or volt.shape[3] != 2:
        raise BlinkError("volt must be [F][A][Ns][2] int8")
    F, A, Ns, _ = volt.shape
    if Ns % n_t or F % n_avg:
        raise BlinkError("Ns must be a multiple of n_t and F of n_avg")
    if check_range and blink_volt_out_of_range(volt):
        raise BlinkError("volt holds samples equal to -128: outside blink_correlate's input range [-127, 127]")
    n_out = (Ns // n_t) * (F // n_avg) * (A * (A + 1) // 2)
    _out(vis, torch.complex64, n_out, "vis", volt.device)
    if vis is None:
        vis = torch.empty((Ns // n_t, F // n_avg, A * (A + 1) // 2), dtype=torch.complex64, device=volt.device)
    with torch.cuda.device(volt.device):
        rc = lib().blink_correlate(_ptr(volt), F, A, Ns, int(n_t), int(n_avg), _ptr(vis), _stream(volt.device))
    _check(rc, "blink_correlate")
    return vis


def blink_image_host(vis_host: torch.Tensor, uvw_host: torch.Tensor, freqs_hz, n_pix: int, pixscale_rad: float,
                     weighting: int, image_host: torch.Tensor, wsum_host: torch.Tensor, workspace: torch.Tensor):
    """Host-buffer variant: vis_host / uvw_host / image_host / wsum_host are (pinned) CPU tensors; workspace is a
    256-byte aligned CUDA uint8 tensor of at least blink_workspace_bytes(OP_IMAGE_HOST) minimum bytes."""
    if vis_host.dim() != 4:
        raise BlinkError(f"vis_host must be [T][C][P][B], got {tuple(vis_host.shape)}")
    T, C, P, B = vis_host.shape
    fr = _freqs(freqs_hz)
    if fr.ndim != 1 or fr.shape[0] != C:
        raise BlinkError(f"freqs_hz must hold C = {C} frequencies, got shape {fr.shape}")
    for t, dt, nm, n in ((vis_host, torch.complex64, "vis_host", T * C * P * B), (uvw_host, torch.float32, "uvw_host", T * B * 3),
                         (image_host, torch.float32, "image_host", T * C * P * n_pix * n_pix),
                         (wsum_host, torch.float32, "wsum_host", T * C)):
        if t.is_cuda or t.dtype != dt or not t.is_contiguous() or t.numel() < n:
            raise BlinkError(f"{nm} must be a contiguous CPU tensor of dtype {dt} with at least {n} elements")
    if tuple(uvw_host.shape) != (T, B, 3):
        raise BlinkError(f"uvw_host must be [T][B][3], got {tuple(uvw_host.shape)}")
    if not workspace.is_cuda or workspace.dtype != torch.uint8 or not workspace.is_contiguous() or workspace.data_ptr() % 256:
        raise BlinkError("workspace must be a contiguous, 256-byte aligned CUDA uint8 tensor")
    with torch.cuda.device(workspace.device):
        rc = lib().blink_image_host(_ptr(vis_host), _ptr(uvw_host), fr.ctypes.data_as(ctypes.c_void_p), T, C, P, B, n_pix,
                                    float(pixscale_rad), int(weighting), _ptr(image_host), _ptr(wsum_host),
                                    _ptr(workspace), workspace.numel())
    _check(rc, "blink_image_host")
    return dict(image=image_host, wsum=wsum_host)

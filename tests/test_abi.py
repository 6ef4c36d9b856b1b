"""The C-ABI library builds, loads without a GPU and exports every symbol include/blinkimg.h declares;
calls that need a device fail loudly (no CPU fallback)."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def so_path():
    from paper_2505_15204_b200 import build
    return build.build()


def _declared_functions():
    text = open(os.path.join(ROOT, "include", "blinkimg.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(blink_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_exported(so_path):
    names = _declared_functions()
    assert {"blink_grid", "blink_fft2d_inverse", "blink_image", "blink_image_host", "blink_workspace_bytes"} <= set(names)
    L = ctypes.CDLL(so_path)
    for n in names:
        assert hasattr(L, n), n
    from paper_2505_15204_b200 import binding
    assert sorted(binding.EXPORTS) == names


def test_host_only_calls(so_path):
    from paper_2505_15204_b200 import binding as bk
    L = bk.lib()
    assert L.blink_strerror(0).decode() == "ok" and L.blink_strerror(-2).decode() == "unsupported size"
    bk.set_option(bk.OPT_GRID_CHUNK_B, 123)
    v = ctypes.c_int(0)
    assert L.blink_get_option(bk.OPT_GRID_CHUNK_B, ctypes.byref(v)) == 0 and v.value == 123
    bk.set_option(bk.OPT_GRID_CHUNK_B, 0)
    assert L.blink_set_option(99, 1) == -1
    # workspace query is pure host arithmetic
    rec, mn = bk.blink_workspace_bytes(bk.OP_FFT2D, 10, 1, 1, 0, 512, 0)
    assert rec == 0 and mn == 0
    bk.set_option(bk.OPT_IMAGE_PATH, 1)
    rec, mn = bk.blink_workspace_bytes(bk.OP_IMAGE, 50, 768, 1, 8128, 512, 0)
    bk.set_option(bk.OPT_IMAGE_PATH, 0)
    assert mn == 512 * 512 * 8 and rec == 256 * mn
    with pytest.raises(bk.BlinkError):
        bk.blink_workspace_bytes(bk.OP_IMAGE, 1, 1, 1, 10, 98, 0)         # 2 * 7^2: a prime factor above 5
    with pytest.raises(bk.BlinkError):
        bk.blink_workspace_bytes(bk.OP_IMAGE, 1, 1, 1, 10, 45, 0)         # odd
    # sides that are not a power of two need an N-entry twiddle table for the mixed-radix transform
    rec, mn = bk.blink_workspace_bytes(bk.OP_FFT2D, 1, 1, 1, 0, 1200, 0)
    assert rec == mn == 1200 * 8 + (-1200 * 8) % 256
    # ... and blink_image through the unfused chain at such a side keeps one row extent (16 bytes) per (t,c) behind the chunk's grids
    rec, mn = bk.blink_workspace_bytes(bk.OP_IMAGE, 2, 768, 1, 8128, 240, 0)
    twb = 240 * 8 + (-240 * 8) % 256
    assert mn == twb + 240 * 240 * 8 + 16 and rec == twb + 256 * (240 * 240 * 8 + 16)
    # the paper's side 1200 has a fused kernel: sorted baselines, the twiddle table, one transposed half plane per CTA
    rec, mn = bk.blink_workspace_bytes(bk.OP_IMAGE, 2, 768, 1, 8128, 1200, 0)
    sortb = 3 * (2 * 8128 * 4 + (-2 * 8128 * 4) % 256)
    assert mn == sortb + 9728 + 1200 * 600 * 8 and (rec - sortb - 9728) % (1200 * 600 * 8) == 0 and rec > mn
    # small batches (<= 4 Mi pixels, auto path): the recommended size also holds the whole range for the unfused chain
    for n, n_img in ((256, 64), (512, 16), (1024, 4), (2048, 1)):
        rec, mn = bk.blink_workspace_bytes(bk.OP_IMAGE, 1, n_img, 1, 8128, n, 0)
        assert rec >= n_img * n * n * 8 and mn <= rec


def test_no_cpu_fallback_without_device(so_path):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a device is present")
    from paper_2505_15204_b200 import binding as bk
    L = bk.lib()
    buf = np.zeros(64, dtype=np.float32)
    p = buf.ctypes.data_as(ctypes.c_void_p)
    fr = np.array([150e6]).ctypes.data_as(ctypes.c_void_p)
    rc = L.blink_image(p, p, fr, 1, 1, 1, 4, 32, 0.01, 0, p, p, None, None, p, 64, None)
    assert rc == -4                                                      # BLINK_ERR_CUDA, and says why
    assert L.blink_last_cuda_error().decode() != ""
    big = np.zeros(1 << 16, dtype=np.float32)
    q = big.ctypes.data_as(ctypes.c_void_p)
    assert L.blink_image_conv(q, q, fr, 1, 1, 1, 4, 256, 0.01, 5, 0.0, q, q, None, q, 1 << 18, None) == -4
    assert L.blink_correlate(q, 2, 4, 128, 64, 1, q, None) == -4


def test_conv_taps_host_logic_against_oracle(so_path, oracle_mod):
    # the polynomial form of the normalised Kaiser-Bessel taps (host fit + the kernel's fp32 Horner evaluation)
    # against the oracle's direct evaluation of the definition (reading R16)
    from paper_2505_15204_b200 import binding as bk
    for S in (3, 5, 7):
        for beta in (0.0, 1.8 * S, 3.0 * S):
            b = beta if beta > 0 else 2.34 * S
            worst = 0.0
            for f in np.linspace(-0.5, 0.5, 41):
                w, fit = bk.blink_conv_taps_host(f, S, beta)
                assert fit < 2e-7
                ref = oracle_mod.conv_taps(float(np.float32(f)), S, b)
                worst = max(worst, float(np.max(np.abs(w.astype(np.float64) - ref))))
                assert abs(float(w.astype(np.float64).sum()) - 1.0) < 1e-6
            assert worst < 1e-6, (S, beta, worst)


def test_conv_argument_checks(so_path):
    from paper_2505_15204_b200 import binding as bk
    L = bk.lib()
    w = np.zeros(8, np.float32)
    wp = w.ctypes.data_as(ctypes.c_void_p)
    assert L.blink_conv_taps_host(0.1, 4, 0.0, wp, None) == -2            # even support
    assert L.blink_conv_taps_host(0.1, 9, 0.0, wp, None) == -2
    assert L.blink_conv_taps_host(0.1, 5, 5.0, wp, None) == -1            # beta below 1.7 S: the correction has a null
    assert L.blink_conv_taps_host(0.7, 5, 0.0, wp, None) == -1            # offset outside [-1/2, 1/2]
    rec, mn = bk.blink_workspace_bytes(bk.OP_IMAGE_CONV, 50, 768, 1, 8128, 512, 0)
    rec0, mn0 = bk.blink_workspace_bytes(bk.OP_IMAGE, 50, 768, 1, 8128, 512, 0)
    assert rec == rec0 + 2048 and mn == mn0 + 2048                        # + the 512-entry correction table
    # the paper's 1200: the fused 1200 kernel's workspace + the 1200-entry correction table
    rec, mn = bk.blink_workspace_bytes(bk.OP_IMAGE_CONV, 2, 300, 1, 100, 1200, 0)
    rec0, mn0 = bk.blink_workspace_bytes(bk.OP_IMAGE, 2, 300, 1, 100, 1200, 0)
    assert rec == rec0 + 4864 and mn == mn0 + 4864
    # outside the fused kernels (sides below 256, other sides that are not a power of two): twiddles + correction table + counters +
    # the chunk's grids
    rec, mn = bk.blink_workspace_bytes(bk.OP_IMAGE_CONV, 2, 300, 1, 100, 240, 0)
    fixed = 2048 + 1024 + 2560
    assert mn == fixed + 240 * 240 * 8 and rec == fixed + 256 * 240 * 240 * 8
    rec, mn = bk.blink_workspace_bytes(bk.OP_IMAGE_CONV, 1, 1, 2, 100, 128, 0)
    assert rec == mn == 512 + 256 + 2 * 128 * 128 * 8
    with pytest.raises(bk.BlinkError):
        bk.blink_workspace_bytes(bk.OP_IMAGE_CONV, 1, 1, 1, 100, 98, 0)    # 2 * 7^2

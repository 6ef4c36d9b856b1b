"""Pins for the convolutional-gridding oracle (oracle_*conv*, reading R16)
against things other than itself: library Bessel functions, closed forms, invariants, an independent numpy
re-gridding, reduction to nearest-cell gridding, and the exact (ungridded) Fourier sum the method approximates.
No GPU needed."""
import numpy as np
import pytest

C0 = 299792458.0


def _beta(S):
    return 2.34 * S


# ------------------------------------------------------------------ kernel function
def test_bessel_i0_against_libraries(oracle_mod):
    sp = pytest.importorskip("scipy.special")
    for x in [0.0, 1e-3, 0.5, 1.0, 3.75, 7.02, 11.7, 16.38, 30.0]:
        assert oracle_mod.bessel_i0(x) == pytest.approx(float(sp.i0(x)), rel=1e-13)
        assert oracle_mod.bessel_i0(x) == pytest.approx(float(np.i0(x)), rel=1e-10)
    assert oracle_mod.bessel_i0(0.0) == 1.0


def test_kb_shape(oracle_mod):
    sp = pytest.importorskip("scipy.special")
    for S in (3, 5, 7):
        b = _beta(S)
        assert oracle_mod.kb(0.0, S, b) == pytest.approx(1.0, abs=1e-15)               # peak 1 at the sample
        assert oracle_mod.kb(S / 2, S, b) == pytest.approx(1.0 / sp.i0(b), rel=1e-12)   # edge value 1/I0(beta)
        assert oracle_mod.kb(S / 2 + 1e-3, S, b) == 0.0                                 # compact support
        d = np.linspace(-S / 2, S / 2, 41)
        k = np.array([oracle_mod.kb(x, S, b) for x in d])
        assert np.allclose(k, k[::-1], rtol=1e-13)                                      # even
        assert np.all(np.diff(k[:21]) > 0)                                              # rises to the centre
        ref = sp.i0(b * np.sqrt(np.clip(1 - (2 * d / S) ** 2, 0, None))) / sp.i0(b)     # definition via scipy
        assert np.allclose(k, ref, rtol=1e-12)


def test_taps_normalised_symmetric_mirrored(oracle_mod):
    rng = np.random.default_rng(11)
    for S in (1, 3, 5, 7):
        b = _beta(S)
        w0 = oracle_mod.conv_taps(0.0, S, b)
        assert np.allclose(w0, w0[::-1], rtol=1e-14) and np.argmax(w0) == S // 2         # on-grid sample: symmetric taps
        for f in rng.uniform(-0.5, 0.5, 20):
            w = oracle_mod.conv_taps(f, S, b)
            assert w.sum() == pytest.approx(1.0, abs=1e-15) and np.all(w > 0)
            assert np.allclose(oracle_mod.conv_taps(-f, S, b), w[::-1], rtol=1e-13)       # conjugate sample: mirrored taps
            if S > 1 and abs(f) > 0.05:
                # a sample displaced towards +u (f > 0) puts more weight on the +1 tap than on the -1 tap
                r = S // 2
                assert (w[r + 1] > w[r - 1]) == (f > 0)
    assert oracle_mod.conv_taps(0.3, 1, 5.0)[0] == 1.0                                    # S = 1: nearest cell


# ------------------------------------------------------------------ grid correction
def test_taper_closed_form(oracle_mod):
    # FT of the Kaiser-Bessel window over its support (Kaiser & Schafer 1980):
    #   int k(d) cos(2 pi d xi) dd  ~  sinh(sqrt(beta^2 - (pi S xi)^2)) / sqrt(beta^2 - (pi S xi)^2),  sin(.)/. beyond
    for S in (3, 5, 7):
        for b in (_beta(S), 1.2 * S):                     # the second crosses into the sin branch inside the image
            n = 64
            c = oracle_mod.conv_taper(n, S, b)
            xi = (np.arange(n) - n // 2) / n
            z = b * b - (np.pi * S * xi) ** 2
            q = np.sqrt(np.abs(z))
            ft = np.where(z > 0, np.sinh(q) / np.where(q == 0, 1, q), np.sin(q) / np.where(q == 0, 1, q))
            ref = ft / (np.sinh(b) / b)
            assert np.allclose(c, ref, rtol=1e-9, atol=1e-12)
            assert c[n // 2] == pytest.approx(1.0, abs=1e-14) and np.allclose(c[1:], c[1:][::-1], rtol=1e-12)
    c = oracle_mod.conv_taper(128, 7, _beta(7))
    assert np.all(c > 0) and np.all(np.diff(c[:65]) > 0)      # default beta: positive, falls monotonically to the edge


# ------------------------------------------------------------------ gridding
def _rand_case(seed, B, n, s_target=0.4, spread=0.8):
    rng = np.random.default_rng(seed)
    f_hz = 150e6
    pix = s_target * C0 / (f_hz * n)
    uvw = np.zeros((B, 3), np.float32)
    uvw[:, :2] = rng.uniform(-spread * n / 2 / s_target, spread * n / 2 / s_target, (B, 2))
    vis = (rng.normal(size=B) + 1j * rng.normal(size=B)).astype(np.complex64)
    return vis, uvw, f_hz, pix


def test_cell_conv_range_and_offsets(oracle_mod):
    n, h, s = 64, 32, np.float32(1.0)
    for S in (3, 5, 7):
        r = S // 2
        c, fx, fy = oracle_mod.cell_conv(h - 1 - r, 0.0, s, n, S)
        assert c == h * n + (h + h - 1 - r) and fx == 0.0 and fy == 0.0
        assert oracle_mod.cell_conv(h - r, 0.0, s, n, S)[0] == -1              # support would reach column h
        assert oracle_mod.cell_conv(0.0, -(h - r), s, n, S)[0] == -1
        assert oracle_mod.cell_conv(float("nan"), 0.0, s, n, S)[0] == -1
        c, fx, fy = oracle_mod.cell_conv(2.25, -3.375, s, n, S)
        assert c == (h - 3) * n + (h + 2) and fx == 0.25 and fy == -0.375      # offsets x - rint(x), exact
        c, fx, fy = oracle_mod.cell_conv(2.5, 3.5, s, n, S)                    # ties to even, as in a1
        assert c == (h + 4) * n + (h + 2) and fx == 0.5 and fy == -0.5


def test_support_one_is_nearest_cell(oracle_mod):
    vis, uvw, f_hz, pix = _rand_case(3, 300, 64)
    g1, W1, ci1 = oracle_mod.grid_conv_one(vis, uvw, f_hz, 64, pix, 1, 4.0)
    g0, _, W0, ci0 = oracle_mod.grid_one(vis, uvw, f_hz, 64, pix, 0)
    assert W1 == W0 and np.array_equal(ci1, ci0) and np.array_equal(g1, g0)


@pytest.mark.parametrize("S", [3, 5, 7])
def test_grid_invariants(oracle_mod, S):
    n = 64
    vis, uvw, f_hz, pix = _rand_case(4 + S, 400, n, spread=1.0)
    g, W, ci = oracle_mod.grid_conv_one(vis, uvw, f_hz, n, pix, S, _beta(S))
    kept = ci >= 0
    assert 0 < kept.sum() < len(ci)                                             # some samples fall off the tighter range
    assert W == 2 * kept.sum()
    assert g.sum() == pytest.approx(2 * vis[kept].real.astype(np.float64).sum(), abs=1e-9)   # taps sum to 1
    h = n // 2
    gm = np.zeros_like(g)
    gm[1:, 1:] = np.conj(g[1:, 1:][::-1, ::-1])                                 # G[-v][-u] = conj G[v][u]
    assert np.allclose(g, gm, rtol=0, atol=1e-12)
    assert not g[0].any() and not g[:, 0].any()                                 # row / column -h stay empty (R4)
    # the nearest cells are those of a1 wherever both are in range
    ci0 = oracle_mod.grid_one(vis, uvw, f_hz, n, pix, 0)[3]
    assert np.array_equal(ci[kept], ci0[kept]) and np.all(ci0[kept] >= 0)


@pytest.mark.parametrize("S", [3, 7])
def test_grid_independent_numpy(oracle_mod, S):
    # independent re-gridding: numpy float64 arithmetic on the fp32 products, scipy's I0, outer products + np.add.at
    sp = pytest.importorskip("scipy.special")
    n, h, r, b = 64, 32, S // 2, _beta(S)
    vis, uvw, f_hz, pix = _rand_case(21, 500, n)
    g, W, ci = oracle_mod.grid_conv_one(vis, uvw, f_hz, n, pix, S, b)
    s = np.float32(((f_hz * n) * pix) / C0)
    x = (uvw[:, 0] * s).astype(np.float32)
    y = (uvw[:, 1] * s).astype(np.float32)
    iu, iv = np.rint(x), np.rint(y)
    ok = (np.abs(iu) <= h - 1 - r) & (np.abs(iv) <= h - 1 - r)
    ref = np.zeros((n, n), np.complex128)
    j = np.arange(-r, r + 1)

    def taps(f):
        k = sp.i0(b * np.sqrt(1 - (2 * (j[None, :] - f[:, None]) / S) ** 2)) / sp.i0(b)
        return k / k.sum(axis=1, keepdims=True)
    wx = taps(x[ok].astype(np.float64) - iu[ok])
    wy = taps(y[ok].astype(np.float64) - iv[ok])
    w2 = wy[:, :, None] * wx[:, None, :]                                        # [sample][row tap][col tap]
    rows = (iv[ok].astype(int)[:, None, None] + j[None, :, None]) + 0 * j[None, None, :]
    cols = (iu[ok].astype(int)[:, None, None] + j[None, None, :]) + 0 * j[None, :, None]
    v = vis[ok].astype(np.complex128)[:, None, None]
    np.add.at(ref, (rows + h, cols + h), w2 * v)
    np.add.at(ref, (h - rows, h - cols), w2 * np.conj(v))
    assert W == 2 * ok.sum()
    assert np.allclose(g, ref, rtol=0, atol=1e-11)


# ------------------------------------------------------------------ images
@pytest.mark.parametrize("S", [3, 5, 7])
def test_unit_source_centre_is_one(oracle_mod, S):
    # all V = 1: the normalised taps keep the total weight of a sample at 1 and c(0) = 1, so I[h][h] = 1 exactly
    n = 64
    vis, uvw, f_hz, pix = _rand_case(31, 200, n)
    vis[:] = 1.0
    out = oracle_mod.image_conv_one(vis, uvw, f_hz, n, pix, S, _beta(S), want_imag=True)
    assert out["image"][n // 2, n // 2] == pytest.approx(1.0, abs=1e-12)
    assert np.abs(out["imag"]).max() < 1e-9 * np.abs(out["image"]).max()          # Hermitian grid -> real image
    img = out["image"]
    assert np.allclose(img[1:, 1:], img[1:, 1:][::-1, ::-1], atol=1e-10)          # dirty beam is point-symmetric


@pytest.mark.parametrize("S", [3, 5, 7])
def test_image_is_taper_corrected_transform_of_grid(oracle_mod, S):
    # numpy.fft route from the oracle's own grid + the closed-form taper (not the quadrature)
    n, h, b = 32, 16, _beta(S)
    vis, uvw, f_hz, pix = _rand_case(41, 150, n)
    out = oracle_mod.image_conv_one(vis, uvw, f_hz, n, pix, S, b)
    xi = (np.arange(n) - h) / n
    q = np.sqrt(b * b - (np.pi * S * xi) ** 2)
    c = (np.sinh(q) / q) / (np.sinh(b) / b)
    ref = np.fft.fftshift(np.fft.ifft2(np.fft.ifftshift(out["grid"]))).real * n * n / out["W"] / np.outer(c, c)
    assert np.allclose(out["image"], ref, rtol=1e-8, atol=1e-10 * np.abs(ref).max())


@pytest.mark.parametrize("S", [3, 5, 7])
def test_closer_to_exact_fourier_sum_than_nearest_cell(oracle_mod, S):
    # What gridding approximates: the exact dirty image I(l,m) = (1/W) sum_b 2 Re(V_b e^{+2 pi i (u_b l + v_b m)}),
    # (l, m) = ((x-h), (y-h)) * pixscale, u in wavelengths (eq. 4-5).  Inside the central half of
    # the field the convolved + corrected image must be much closer to it than the nearest-cell image; a wrong
    # offset sign, a transposed tap axis or a missing / inverted correction all fail this.
    n, h = 64, 32
    vis, uvw, f_hz, pix = _rand_case(51, 120, n, spread=0.7)
    s = np.float32(((f_hz * n) * pix) / C0)
    conv = oracle_mod.image_conv_one(vis, uvw, f_hz, n, pix, S, _beta(S))
    near = oracle_mod.image_one(vis, uvw, f_hz, n, pix, 0)
    kept = conv["cell_idx"] >= 0
    assert np.array_equal(kept, near["cell_idx"] >= 0)                 # spread 0.7: the same samples on both sides
    x = (uvw[:, 0] * s).astype(np.float64)[kept]                        # cells = wavelengths * N * pixscale
    y = (uvw[:, 1] * s).astype(np.float64)[kept]
    v = vis[kept].astype(np.complex128)
    pxl = (np.arange(n) - h) / n                                        # l * (cells per wavelength) = (x-h)/N
    ex = np.exp(2j * np.pi * np.outer(x, pxl))                          # [b][xpix]
    ey = np.exp(2j * np.pi * np.outer(y, pxl))                          # [b][ypix]
    exact = 2 * np.real(np.einsum("b,by,bx->yx", v, ey, ex)) / (2 * kept.sum())
    sl = slice(h - n // 4, h + n // 4)
    e_conv = np.sqrt(np.mean((conv["image"][sl, sl] - exact[sl, sl]) ** 2))
    e_near = np.sqrt(np.mean((near["image"][sl, sl] - exact[sl, sl]) ** 2))
    assert e_conv < e_near / {3: 30.0, 5: 1e3, 7: 1e5}[S], (e_conv, e_near)


def test_batch_driver_matches_single(oracle_mod):
    rng = np.random.default_rng(61)
    T, C, P, B, n = 2, 3, 2, 60, 32
    uvw = np.zeros((T, B, 3), np.float32)
    uvw[:, :, :2] = rng.uniform(-25, 25, (T, B, 2))
    vis = (rng.normal(size=(T, C, P, B)) + 1j * rng.normal(size=(T, C, P, B))).astype(np.complex64)
    freqs = 150e6 + 40e3 * np.arange(C)
    pix = 0.4 * C0 / (150e6 * n)
    ids = np.array([0, 5, 11])
    imgs, ws = oracle_mod.image_conv_batch(vis, uvw, freqs, n, pix, 5, _beta(5), img_ids=ids, nthreads=2)
    for k, i in enumerate(ids):
        p, c, t = i % P, (i // P) % C, i // (P * C)
        one = oracle_mod.image_conv_one(vis[t, c, p], uvw[t], freqs[c], n, pix, 5, _beta(5))
        assert np.array_equal(imgs[k], one["image"]) and ws[k] == one["W"]

"""Pins for oracle/blink_oracle.c against things OTHER than itself (no GPU needed).

Each test names the passage / closed form / invariant it checks.  The paper prints no worked
numerical example of gridding or the FFT, so the pins are closed forms, invariants,
hand-worked cases (tests/golden/), brute force on tiny inputs and an independent library routine
(numpy.fft) -- chosen so a dropped term, a wrong sign, a transposed axis or an off-by-one shift fails.
"""
import os

import numpy as np
import pytest

C0 = 299792458.0
GOLD = os.path.join(os.path.dirname(__file__), "golden")


# --------------------------------------------------------------------------- a0 / a1: scale and cell
def test_scale_closed_form(oracle_mod):
    # f = c  =>  s = N * pixscale exactly (u in wavelengths = u_m f / c)
    assert oracle_mod.scale(C0, 256, 0.5 / 256) == np.float32(0.5)
    assert oracle_mod.scale(C0, 8, 0.125) == np.float32(1.0)
    assert oracle_mod.scale(2 * C0, 512, 1.0 / 512) == np.float32(2.0)
    # generic: single rounding of the double value
    f, n, p = 154.24e6, 256, 0.5 / 256
    assert oracle_mod.scale(f, n, p) == np.float32(((f * n) * p) / C0)


def test_cell_on_grid_and_layout(oracle_mod):
    n, h, s = 64, 32, np.float32(0.5)
    # u_m = 2k -> exactly k cells; column = u, row = v (reading R8); DC at [h][h] (R7)
    assert oracle_mod.cell(0.0, 0.0, s, n) == h * n + h
    assert oracle_mod.cell(2.0, 0.0, s, n) == h * n + h + 1          # +u moves one COLUMN
    assert oracle_mod.cell(0.0, 2.0, s, n) == (h + 1) * n + h        # +v moves one ROW
    assert oracle_mod.cell(-6.0, 10.0, s, n) == (h + 5) * n + (h - 3)


def test_cell_ties_to_even_and_range(oracle_mod):
    n, h, s = 64, 32, np.float32(1.0)
    base = h * n + h
    assert oracle_mod.cell(2.5, 0.0, s, n) == base + 2               # 2.5 -> 2
    assert oracle_mod.cell(3.5, 0.0, s, n) == base + 4               # 3.5 -> 4
    assert oracle_mod.cell(-2.5, 0.0, s, n) == base - 2
    assert oracle_mod.cell(0.0, -0.5, s, n) == base                  # -0.5 -> -0
    # reading R4: |i| <= h-1 kept, h dropped (both axes, both signs)
    assert oracle_mod.cell(h - 1, 0.0, s, n) == base + h - 1
    assert oracle_mod.cell(-(h - 1), 0.0, s, n) == base - (h - 1)
    for bad in [(h, 0.0), (-h, 0.0), (0.0, h), (0.0, -h), (h - 0.5, 0.0), (1e9, 0.0)]:
        assert oracle_mod.cell(bad[0], bad[1], s, n) == -1
    assert oracle_mod.cell(h - 0.51, 0.0, s, n) == base + h - 1
    for bad in [float("nan"), float("inf"), -float("inf")]:
        assert oracle_mod.cell(bad, 0.0, s, n) == -1
        assert oracle_mod.cell(0.0, bad, s, n) == -1


def test_mirror_invariant(oracle_mod):
    # conj sample at (-u,-v): r + r' = N and q + q' = N (rint is odd-symmetric)
    rng = np.random.default_rng(5)
    n, s = 128, np.float32(0.37)
    for _ in range(500):
        u, v = rng.uniform(-200, 200, 2).astype(np.float32)
        c = oracle_mod.cell(u, v, s, n)
        cm = oracle_mod.cell(-u, -v, s, n)
        if c < 0:
            assert cm < 0
            continue
        assert oracle_mod.mirror_cell(c, n) == cm
        assert c // n + cm // n == n and c % n + cm % n == n


def test_cells_vs_float64_bruteforce(oracle_mod):
    # away from half-cell boundaries an all-double evaluation must give the same cell
    rng = np.random.default_rng(11)
    T, B, n, pix = 2, 4000, 512, 0.6 / 512
    freqs = np.array([139.54e6, 154.88e6, 170.22e6])
    uvw = rng.uniform(-320, 320, (T, B, 3)).astype(np.float32)
    got = oracle_mod.cells(uvw, freqs, n, pix)
    h = n // 2
    checked = 0
    for t in range(T):
        for c, f in enumerate(freqs):
            s64 = f * n * pix / C0
            x = uvw[t, :, 0].astype(np.float64) * s64
            y = uvw[t, :, 1].astype(np.float64) * s64
            safe = (np.abs(x - np.floor(x) - 0.5) > 1e-3) & (np.abs(y - np.floor(y) - 0.5) > 1e-3)
            iu, iv = np.floor(x + 0.5).astype(int), np.floor(y + 0.5).astype(int)
            inr = (np.abs(iu) <= h - 1) & (np.abs(iv) <= h - 1)
            want = np.where(inr, (iv + h) * n + (iu + h), -1)
            assert np.array_equal(got[t, c][safe], want[safe])
            checked += int(safe.sum())
    assert checked > 0.95 * T * len(freqs) * B


# --------------------------------------------------------------------------- a2 / a3: gridding
def _load_three_antenna():
    rows = []
    with open(os.path.join(GOLD, "three_antenna_case.txt")) as fh:
        for line in fh:
            line = line.split("#")[0].strip()
            if line:
                rows.append([float(x) for x in line.split()])
    a = np.array(rows)
    return a[:, :3].astype(np.float32), (a[:, 3] + 1j * a[:, 4]).astype(np.complex64)


def test_three_antenna_hand_case(oracle_mod):
    uvw, vis = _load_three_antenna()
    n = 8
    grid, cnt, W, ci = oracle_mod.grid_one(vis, uvw, C0, n, 0.125, 0)
    assert list(ci) == [53, 34, 53, 15, -1]
    g = grid.ravel()
    want = {53: 4 + 2.25j, 19: 4 - 2.25j, 34: 0.5 - 1j, 38: 0.5 + 1j, 15: -2 + 4j, 57: -2 - 4j}
    for k in range(n * n):
        assert g[k] == want.get(k, 0.0), k
    wantc = {53: 2, 19: 2, 34: 1, 38: 1, 15: 1, 57: 1}
    assert all(cnt.ravel()[k] == wantc.get(k, 0) for k in range(n * n))
    assert W == 8.0
    r = oracle_mod.image_one(vis, uvw, C0, n, 0.125, 0)
    assert abs(r["image"][4, 4] - 0.625) < 1e-15
    # uniform (reading R9)
    grid, cnt, W, _ = oracle_mod.grid_one(vis, uvw, C0, n, 0.125, 1)
    assert W == 6.0
    assert grid.ravel()[53] == 2 + 1.125j and grid.ravel()[19] == 2 - 1.125j
    assert grid.ravel()[34] == 0.5 - 1j
    r = oracle_mod.image_one(vis, uvw, C0, n, 0.125, 1)
    assert abs(r["image"][4, 4] - 1.0 / 6.0) < 1e-15


def _random_case(seed, B=600, n=64, spread=40.0):
    rng = np.random.default_rng(seed)
    uvw = rng.uniform(-spread, spread, (B, 3)).astype(np.float32)
    vis = (rng.normal(size=B) + 1j * rng.normal(size=B)).astype(np.complex64)
    return uvw, vis


def test_grid_invariants(oracle_mod):
    n = 64
    uvw, vis = _random_case(3, n=n, spread=75.0)                             # some samples fall off the grid
    f, pix = 150e6, 1.0 / n
    grid, cnt, W, ci = oracle_mod.grid_one(vis, uvw, f, n, pix, 0)
    inr = ci >= 0
    assert 0 < inr.sum() < len(ci)
    assert W == 2 * inr.sum() == cnt.sum()                            # natural: W = 2 B_in = sum(cnt)
    # sum of all cells = sum_b 2 Re V_b  => centre-pixel closed form
    s = grid.sum()
    want = 2.0 * vis[inr].real.astype(np.float64).sum()
    assert abs(s.real - want) < 1e-9 and abs(s.imag) < 1e-9
    # Hermitian: G[N-r][N-q] = conj(G[r][q]); row 0 and column 0 stay empty (reading R4)
    assert np.all(grid[0, :] == 0) and np.all(grid[:, 0] == 0)
    sub = grid[1:, 1:]
    assert np.array_equal(sub[::-1, ::-1], np.conj(sub))
    subc = cnt[1:, 1:]
    assert np.array_equal(subc[::-1, ::-1], subc)
    # uniform: W = occupied cells; values = natural / cnt
    gridu, cntu, Wu, _ = oracle_mod.grid_one(vis, uvw, f, n, pix, 1)
    assert Wu == (cnt > 0).sum() and np.array_equal(cntu, cnt)
    occ = cnt > 0
    assert np.allclose(gridu[occ], grid[occ] / cnt[occ], rtol=1e-15, atol=0)
    # independent numpy re-gridding from the cell indices (np.add.at), different code path
    g2 = np.zeros(n * n, dtype=np.complex128)
    h = n // 2
    cells = ci[inr]
    mir = (2 * h - cells // n) * n + (2 * h - cells % n)
    np.add.at(g2, cells, vis[inr].astype(np.complex128))
    np.add.at(g2, mir, np.conj(vis[inr].astype(np.complex128)))
    assert np.allclose(g2.reshape(n, n), grid, rtol=1e-13, atol=1e-13)


def test_all_dropped_gives_zero_image(oracle_mod):
    uvw = np.full((5, 3), 1e6, dtype=np.float32)
    vis = np.ones(5, dtype=np.complex64)
    r = oracle_mod.image_one(vis, uvw, 150e6, 32, 1.0 / 32, 0)
    assert r["W"] == 0 and np.all(r["image"] == 0) and np.all(r["cell_idx"] == -1)
    r = oracle_mod.image_one(vis[:0], uvw[:0], 150e6, 32, 1.0 / 32, 1)   # B = 0
    assert r["W"] == 0 and np.all(r["image"] == 0)


# --------------------------------------------------------------------------- a4 / a5: transforms
def _closed_form_single_cell(n, ku, kv, V):
    # one sample V at (ku,kv) plus conj at (-ku,-kv):  2|V| cos(2 pi (ku(x-h) + kv(y-h))/N + arg V)
    h = n // 2
    y, x = np.mgrid[0:n, 0:n]
    return 2 * abs(V) * np.cos(2 * np.pi * (ku * (x - h) + kv * (y - h)) / n + np.angle(V))


@pytest.mark.parametrize("n,ku,kv", [(16, 3, 0), (16, 0, 5), (32, -7, 4), (32, 15, -15)])
def test_single_cell_closed_form(oracle_mod, n, ku, kv):
    h = n // 2
    V = 0.7 - 1.9j
    g = np.zeros((n, n), dtype=np.complex128)
    g[kv + h, ku + h] = V
    g[h - kv, h - ku] = np.conj(V)
    want = _closed_form_single_cell(n, ku, kv, V)
    for fn in (oracle_mod.idft2_direct, oracle_mod.ifft2_radix2):
        out = fn(g)
        assert np.max(np.abs(out.real - want)) < 1e-12
        assert np.max(np.abs(out.imag)) < 1e-12
    assert np.max(np.abs(oracle_mod.sparse_image(g, 1.0) - want)) < 1e-12


def test_orientation_not_transposed(oracle_mod):
    # a pure-u fringe varies along x (columns) only; a pure-v fringe along y (rows) only
    n, h = 16, 8
    g = np.zeros((n, n), dtype=np.complex128)
    g[h, h + 2] = 1.0
    g[h, h - 2] = 1.0
    out = oracle_mod.ifft2_radix2(g).real
    assert np.allclose(out, out[0:1, :]) and not np.allclose(out, out[:, 0:1])


def test_radix2_vs_direct_32(oracle_mod):
    # north_star check 4: on 32x32 grids the FFT image matches a brute-force direct Fourier sum
    n = 32
    uvw, vis = _random_case(7, B=300, n=n, spread=25.0)
    grid, cnt, W, _ = oracle_mod.grid_one(vis, uvw, 200e6, n, 1.0 / n, 0)
    a = oracle_mod.ifft2_radix2(grid)
    b = oracle_mod.idft2_direct(grid)
    assert np.max(np.abs(a - b)) < 1e-10 * np.max(np.abs(b))
    img = oracle_mod.sparse_image(grid, W)
    assert np.max(np.abs(img - b.real / W)) < 1e-12
    # arbitrary NON-Hermitian complex input too (the transform itself, no gridding)
    rng = np.random.default_rng(9)
    g = rng.normal(size=(n, n)) + 1j * rng.normal(size=(n, n))
    a, b = oracle_mod.ifft2_radix2(g), oracle_mod.idft2_direct(g)
    assert np.max(np.abs(a - b)) < 1e-10 * np.max(np.abs(b))


@pytest.mark.parametrize("n", [32, 64, 256, 1024])
def test_radix2_vs_numpy_library(oracle_mod, n):
    # library special case: Re(fftshift(ifft2(ifftshift(G)))) * N^2
    rng = np.random.default_rng(n)
    g = rng.normal(size=(n, n)) + 1j * rng.normal(size=(n, n))
    a = oracle_mod.ifft2_radix2(g)
    b = np.fft.fftshift(np.fft.ifft2(np.fft.ifftshift(g))) * (n * n)
    assert np.max(np.abs(a - b)) < 1e-11 * np.max(np.abs(b))
    # sign-flip form for N = 0 mod 4: (-1)^(x+y) IDFT_plain[(-1)^(q+r) G]
    sgn = (-1.0) ** (np.add.outer(np.arange(n), np.arange(n)))
    c = sgn * np.fft.ifft2(sgn * g) * (n * n)
    assert np.max(np.abs(a - c)) < 1e-11 * np.max(np.abs(b))
    # Parseval: sum |out|^2 = N^2 sum |G|^2
    assert abs((np.abs(a) ** 2).sum() / (n * n * (np.abs(g) ** 2).sum()) - 1) < 1e-12


def test_radix2_linearity_and_separable_matrix_form(oracle_mod):
    n, h = 64, 32
    rng = np.random.default_rng(1)
    g1 = rng.normal(size=(n, n)) + 1j * rng.normal(size=(n, n))
    g2 = rng.normal(size=(n, n)) + 1j * rng.normal(size=(n, n))
    a = oracle_mod.ifft2_radix2(g1 + 2.5 * g2)
    b = oracle_mod.ifft2_radix2(g1) + 2.5 * oracle_mod.ifft2_radix2(g2)
    assert np.max(np.abs(a - b)) < 1e-10
    # definition via two dense matrix products: out = F G F^T, F[x][q] = e^{2 pi i (q-h)(x-h)/N}
    k = np.arange(n) - h
    F = np.exp(2j * np.pi * np.outer(k, k) / n)
    assert np.max(np.abs(oracle_mod.ifft2_radix2(g1) - F @ g1 @ F.T)) < 1e-9


# --------------------------------------------------------------------------- whole image
def _on_grid_uvw(rng, B, n, s):
    h = n // 2
    iu = rng.integers(-(h - 1), h, B)
    iv = rng.integers(-(h - 1), h, B)
    uvw = np.zeros((B, 3), dtype=np.float32)
    uvw[:, 0] = iu / s
    uvw[:, 1] = iv / s
    return uvw, iu, iv


def test_unit_source_at_phase_centre(oracle_mod):
    # north_star check 1: all V = 1 => I[h][h] = 1.0, the maximum; image = dirty beam, point-symmetric
    n, h = 64, 32
    uvw, _ = _random_case(21, B=500, n=n, spread=30.0)
    vis = np.ones(500, dtype=np.complex64)
    for wt in (0, 1):
        r = oracle_mod.image_one(vis, uvw, 160e6, n, 1.0 / n, wt, want_imag=True)
        img = r["image"]
        assert abs(img[h, h] - 1.0) < 1e-13
        assert img.max() <= img[h, h] + 1e-13
        assert np.allclose(img[1:, 1:], img[1:, 1:][::-1, ::-1], atol=1e-12)     # I[y][x] = I[N-y][N-x]
        assert np.max(np.abs(r["imag"])) < 1e-12                                 # check 3


def test_on_grid_offset_source_peaks_at_its_pixel(oracle_mod):
    # north_star check 2: V_b = e^{-2 pi i (u l0 + v m0)} with on-grid uvw => exactly 1.0 at (h+x0, h+y0)
    n, h = 64, 32
    f, pix = C0, 0.5 / n                                                          # s = 0.5 exactly
    s = float(oracle_mod.scale(f, n, pix))
    rng = np.random.default_rng(2)
    uvw, iu, iv = _on_grid_uvw(rng, 400, n, s)
    for (x0, y0) in [(5, -3), (-7, 0), (0, 6), (h - 1, -(h - 1))]:
        l0, m0 = x0 * pix, y0 * pix                                               # pixel-centred direction cosines
        u_l = uvw[:, 0].astype(np.float64) * f / C0
        v_l = uvw[:, 1].astype(np.float64) * f / C0
        vis = np.exp(-2j * np.pi * (u_l * l0 + v_l * m0)).astype(np.complex64)    # eq. 4 sign, L104
        r = oracle_mod.image_one(vis, uvw, f, n, pix, 0, want_imag=True)
        img = r["image"]
        yx = np.unravel_index(np.argmax(img), img.shape)
        assert yx == (h + y0, h + x0)                                             # row = m/y, column = l/x
        assert abs(img[yx] - 1.0) < 1e-6                                          # complex64 rounding of V only
        assert np.max(np.abs(r["imag"])) < 1e-6 * img.max()


def test_generic_offset_source_argmax(oracle_mod):
    # generic (off-grid) uvw: nearest-cell phase error lowers the peak a little, does not move it
    n, h = 128, 64
    f, pix = 154.24e6, 0.5 / n
    rng = np.random.default_rng(4)
    B = 3000
    r_ = 140.0 * np.sqrt(rng.random(B))
    th = 2 * np.pi * rng.random(B)
    uvw = np.stack([r_ * np.cos(th), r_ * np.sin(th), np.zeros(B)], axis=1).astype(np.float32)
    for (x0, y0) in [(9, -12), (-16, 16)]:
        l0, m0 = x0 * pix, y0 * pix
        u_l = uvw[:, 0].astype(np.float64) * f / C0
        v_l = uvw[:, 1].astype(np.float64) * f / C0
        vis = np.exp(-2j * np.pi * (u_l * l0 + v_l * m0)).astype(np.complex64)
        r = oracle_mod.image_one(vis, uvw, f, n, pix, 0, want_imag=True)
        img = r["image"]
        assert np.unravel_index(np.argmax(img), img.shape) == (h + y0, h + x0)
        assert 0.85 < img.max() <= 1.0 + 1e-9
        assert np.max(np.abs(r["imag"])) < 1e-6 * img.max()


def test_sparse_direct_sum_full_size_image(oracle_mod):
    # one FULL-SIZE config-1 image: radix-2 route == direct Fourier sum over occupied cells
    from paper_2505_15204_b200 import workloads
    w = workloads.make_config(1)
    vis = w.vis[0, 0, 0].numpy()
    uvw = w.uvw_m[0].numpy()
    r = oracle_mod.image_one(vis, uvw, w.freqs_hz[0], w.n_pix, w.pixscale_rad, 0)
    img2 = oracle_mod.sparse_image(r["grid"], r["W"])
    assert np.max(np.abs(r["image"] - img2)) < 1e-11 * np.max(np.abs(img2))
    # centre pixel closed form (sum of gridded samples / W)
    inr = r["cell_idx"] >= 0
    h = w.n_pix // 2
    assert abs(r["image"][h, h] - 2 * vis[inr].real.astype(np.float64).sum() / r["W"]) < 1e-12
    # config 1 drops a few percent of baselines with pixscale 0.5/256 (reading R4)
    assert 0.0 < (~inr).mean() < 0.05


def test_image_batch_matches_image_one(oracle_mod):
    from paper_2505_15204_b200 import workloads
    w = workloads.make_random(T=2, C=3, P=2, B=200, n_pix=32, weighting=1, seed=8)
    vis, uvw = w.vis.numpy(), w.uvw_m.numpy()
    ids = np.array([0, 5, 11, 7])
    imgs, ws = oracle_mod.image_batch(vis, uvw, w.freqs_hz, 32, w.pixscale_rad, 1, ids, nthreads=3)
    for k, i in enumerate(ids):
        p, c, t = i % 2, (i // 2) % 3, i // 6
        r = oracle_mod.image_one(vis[t, c, p], uvw[t], w.freqs_hz[c], 32, w.pixscale_rad, 1)
        assert np.array_equal(imgs[k], r["image"]) and ws[k] == r["W"]


def test_table7_byte_accounting():
    # PAPER.md L365-370 Table 7: float32 images, complex64 visibilities
    assert abs(38400 * 1200 ** 2 * 4 / 2 ** 30 - 206) < 0.5                      # "206 GB" images
    assert abs(38400 * 8256 * 4 * 8 / 2 ** 30 - 9.5) < 0.1                       # "9.5 GB" visibilities


# ---------------------------------------------------------------------------------------------
# averaged images (reading R14)
# ---------------------------------------------------------------------------------------------
def _avg_inputs(seed, T=2, C=4, P=2, B=60, N=32, ones=False):
    rng = np.random.default_rng(seed)
    fr = 150e6 + 1.5e6 * np.arange(C)                       # wide spacing: the channels grid to different cells
    half_m = 0.8 * (N / 2) / (fr[-1] / 299792458.0)
    uvw = rng.uniform(-half_m, half_m, (T, B, 3)).astype(np.float32)
    vis = np.ones((T, C, P, B), np.complex64) if ones else \
        (rng.normal(size=(T, C, P, B)) + 1j * rng.normal(size=(T, C, P, B))).astype(np.complex64)
    return vis, uvw, fr, N, 1.0 / N


@pytest.mark.parametrize("weighting", [0, 1])
@pytest.mark.parametrize("avg_time", [False, True])
def test_avg_unit_source_centre_is_one(oracle_mod, weighting, avg_time):
    # every single image has exactly 1.0 at the phase centre when all V = 1, so their mean has too
    vis, uvw, fr, N, pix = _avg_inputs(3, ones=True)
    a = oracle_mod.image_avg(vis, uvw, fr, N, pix, weighting, avg_time)
    assert np.allclose(a[..., N // 2, N // 2], 1.0, atol=1e-12)
    assert np.all(a <= a[..., N // 2, N // 2][..., None, None] + 1e-12)


@pytest.mark.parametrize("weighting", [0, 1])
@pytest.mark.parametrize("avg_time", [False, True])
def test_avg_linearity_numpy(oracle_mod, weighting, avg_time):
    # independent evaluation: re-grid in numpy from the oracle's CELL INDICES only, sum the grids weighted by
    # 1/W_c, transform ONCE with numpy.fft (library routine) -- the transform is linear, so this must be the mean
    vis, uvw, fr, N, pix = _avg_inputs(5)
    T, C, P, B = vis.shape
    h = N // 2
    ci = oracle_mod.cells(uvw, fr, N, pix)
    acc = np.zeros(((1 if avg_time else T), P, N, N), np.complex128)
    for t in range(T):
        for c in range(C):
            ok = ci[t, c] >= 0
            r, q = ci[t, c][ok] // N, ci[t, c][ok] % N
            cnt = np.zeros((N, N))
            np.add.at(cnt, (r, q), 1)
            np.add.at(cnt, (N - r, N - q), 1)
            W = cnt.sum() if weighting == 0 else np.count_nonzero(cnt)
            for p in range(P):
                g = np.zeros((N, N), np.complex128)
                np.add.at(g, (r, q), vis[t, c, p][ok].astype(np.complex128))
                np.add.at(g, (N - r, N - q), np.conj(vis[t, c, p][ok].astype(np.complex128)))
                if weighting == 1:
                    g[cnt > 0] /= cnt[cnt > 0]
                acc[0 if avg_time else t, p] += g / W
    img = np.fft.fftshift(np.fft.ifft2(np.fft.ifftshift(acc, axes=(-2, -1))), axes=(-2, -1)).real * N * N
    img /= (T * C) if avg_time else C
    a = oracle_mod.image_avg(vis, uvw, fr, N, pix, weighting, avg_time)
    want = img[0] if avg_time else img
    assert np.max(np.abs(a - want)) <= 1e-10 * np.max(np.abs(want))


def test_avg_centre_pixel_closed_form_and_zero_images_count(oracle_mod):
    # centre pixel of one image = sum(2 Re V_in) / W; the mean divides by the NUMBER OF CHANNELS even when a
    # channel has nothing on the grid (its image is zero)
    vis, uvw, fr, N, pix = _avg_inputs(7, T=1, C=3, P=1)
    fr = fr.copy()
    fr[2] = 5e9                                              # this channel throws every sample off the grid
    ci = oracle_mod.cells(uvw, fr, N, pix)
    assert np.all(ci[0, 2] < 0)
    a = oracle_mod.image_avg(vis, uvw, fr, N, pix, 0)
    want = 0.0
    for c in range(2):
        ok = ci[0, c] >= 0
        want += (2.0 * vis[0, c, 0][ok].real.astype(np.float64).sum()) / (2.0 * ok.sum())
    assert abs(a[0, 0, N // 2, N // 2] - want / 3.0) <= 1e-12 * max(1.0, abs(want))


# ---------------------------------------------------------------------------------------------
# per-antenna gain corrections (reading R15)
# ---------------------------------------------------------------------------------------------
def _gain_inputs(seed, T=2, C=3, P=2, A=7):
    rng = np.random.default_rng(seed)
    pairs = np.array([(i, j) for i in range(A) for j in range(i)], dtype=np.int32)      # b = i(i-1)/2 + j
    B = len(pairs)
    vis = (rng.normal(size=(T, C, P, B)) + 1j * rng.normal(size=(T, C, P, B))).astype(np.complex64)
    gains = (rng.uniform(0.5, 1.5, (C, P, A)) * np.exp(1j * rng.uniform(-np.pi, np.pi, (C, P, A)))).astype(np.complex64)
    return vis, gains, pairs


def test_gains_identity_phase_and_numpy(oracle_mod):
    vis, gains, pairs = _gain_inputs(9)
    assert np.array_equal(oracle_mod.apply_gains(vis, np.ones_like(gains), pairs), vis)
    # pure per-antenna phases: modulus kept, phase advanced by phi_a1 - phi_a2
    phi = np.angle(gains.astype(np.complex128))
    out = oracle_mod.apply_gains(vis, np.exp(1j * phi).astype(np.complex64), pairs).astype(np.complex128)
    want_phase = phi[:, :, pairs[:, 0]] - phi[:, :, pairs[:, 1]]                               # [C][P][B]
    assert np.allclose(np.abs(out), np.abs(vis), rtol=1e-5)
    assert np.allclose(out, vis.astype(np.complex128) * np.exp(1j * want_phase)[None], rtol=2e-6, atol=1e-6)
    # general gains against an independent numpy evaluation
    g = gains.astype(np.complex128)
    want = vis.astype(np.complex128) * (g[:, :, pairs[:, 0]] * np.conj(g[:, :, pairs[:, 1]]))[None]
    got = oracle_mod.apply_gains(vis, gains, pairs)
    assert np.allclose(got, want, rtol=2e-6, atol=1e-6)
    # a transposed antenna pair conjugates the factor: make sure the order matters and is the stated one
    swapped = oracle_mod.apply_gains(vis, gains, pairs[:, ::-1].copy())
    assert not np.allclose(swapped, got, rtol=1e-3)


def test_gains_undo_corruption_restores_image(oracle_mod):
    # corrupt "true" visibilities with per-antenna errors e_a (V_obs = e_a1 conj(e_a2) V), calibrate with g = 1/e:
    # the dirty image of the corrected data equals the image of the true data
    rng = np.random.default_rng(10)
    A, N = 6, 32
    pairs = np.array([(i, j) for i in range(A) for j in range(i)], dtype=np.int32)
    B = len(pairs)
    uvw = rng.uniform(-20, 20, (1, B, 3)).astype(np.float32)
    true = (rng.normal(size=(1, 1, 1, B)) + 1j * rng.normal(size=(1, 1, 1, B))).astype(np.complex64)
    e = (rng.uniform(0.7, 1.3, (1, 1, A)) * np.exp(1j * rng.uniform(-2, 2, (1, 1, A))))
    obs = (true.astype(np.complex128) * (e[:, :, pairs[:, 0]] * np.conj(e[:, :, pairs[:, 1]]))[None]).astype(np.complex64)
    fixed = oracle_mod.apply_gains(obs, (1.0 / e).astype(np.complex64), pairs)
    f = 150e6
    a = oracle_mod.image_one(true[0, 0, 0], uvw[0], f, N, 1.0 / N, 0)["image"]
    b = oracle_mod.image_one(fixed[0, 0, 0], uvw[0], f, N, 1.0 / N, 0)["image"]
    c = oracle_mod.image_one(obs[0, 0, 0], uvw[0], f, N, 1.0 / N, 0)["image"]
    assert np.max(np.abs(a - b)) <= 1e-5 * np.max(np.abs(a))
    assert np.max(np.abs(a - c)) > 1e-2 * np.max(np.abs(a))                                   # the corruption was visible


# ---------------------------------------------------------------------------------------------
# image sides that are not a power of two (1200 x 1200)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n", [12, 20])
def test_non_pow2_transform_vs_bruteforce(oracle_mod, n):
    rng = np.random.default_rng(300 + n)
    g = rng.normal(size=(n, n)) + 1j * rng.normal(size=(n, n))
    a, b = oracle_mod.ifft2_radix2(g), oracle_mod.idft2_direct(g)            # row-column 1D sums vs the O(N^4) definition
    assert np.max(np.abs(a - b)) < 1e-11 * np.max(np.abs(b))


@pytest.mark.parametrize("n", [30, 48, 150])
def test_non_pow2_transform_vs_numpy_library(oracle_mod, n):
    rng = np.random.default_rng(400 + n)
    g = rng.normal(size=(n, n)) + 1j * rng.normal(size=(n, n))
    a = oracle_mod.ifft2_radix2(g)
    b = np.fft.fftshift(np.fft.ifft2(np.fft.ifftshift(g))) * (n * n)
    assert np.max(np.abs(a - b)) < 1e-11 * np.max(np.abs(b))
    assert abs((np.abs(a) ** 2).sum() / (n * n * (np.abs(g) ** 2).sum()) - 1) < 1e-12     # Parseval


def test_non_pow2_single_cell_closed_form_and_unit_source(oracle_mod):
    # the paper's own image side: one Hermitian pair of cells -> a cosine fringe with the stated sign, orientation, shift
    n, ku, kv, V = 1200, 37, -211, 0.7 - 1.9j
    h = n // 2
    g = np.zeros((n, n), dtype=np.complex128)
    g[kv + h, ku + h] = V
    g[h - kv, h - ku] = np.conj(V)
    out = oracle_mod.ifft2_radix2(g)
    want = _closed_form_single_cell(n, ku, kv, V)
    assert np.max(np.abs(out.real - want)) < 1e-9 and np.max(np.abs(out.imag)) < 1e-9
    # whole image at a side of 240: all V = 1 -> exactly 1.0 at the phase centre, which is the maximum
    rng = np.random.default_rng(5)
    n = 240
    uvw = rng.uniform(-60, 60, (200, 3)).astype(np.float32)
    r = oracle_mod.image_one(np.ones(200, np.complex64), uvw, 150e6, n, 1.0 / n, 0)
    assert abs(r["image"][n // 2, n // 2] - 1.0) < 1e-12 and r["image"].max() <= r["image"][n // 2, n // 2] + 1e-12
    assert r["W"] == 2 * np.count_nonzero(r["cell_idx"] >= 0)


# ---------------------------------------------------------------------------------------------
# Stokes I images, I = (XX + YY) / 2 (reading R18)
# ---------------------------------------------------------------------------------------------
def _stokes_inputs(seed, P, B=60, N=32, T=2, C=2):
    rng = np.random.default_rng(seed)
    uvw = rng.uniform(-25, 25, (T, B, 3)).astype(np.float32)
    vis = (rng.normal(size=(T, C, P, B)) + 1j * rng.normal(size=(T, C, P, B))).astype(np.complex64)
    freqs = 150e6 + 1e6 * np.arange(C)
    return vis, uvw, freqs, N, 1.0 / N


@pytest.mark.parametrize("P", [2, 4])
@pytest.mark.parametrize("weighting", [0, 1])
def test_stokes_i_special_cases(oracle_mod, P, weighting):
    vis, uvw, freqs, N, pix = _stokes_inputs(70 + P, P)
    h = N // 2
    # unit sources in XX and YY (whatever sits in XY / YX is ignored): exactly 1.0 at the phase centre
    v1 = vis.copy()
    v1[:, :, 0] = 1.0
    v1[:, :, P - 1] = 1.0
    img, W = oracle_mod.image_stokes_i(v1, uvw, freqs, N, pix, weighting)
    assert np.all(np.abs(img[:, h, h] - 1.0) < 1e-12) and np.all(W > 0)
    # YY = -XX: the two images cancel pixel by pixel
    v2 = vis.copy()
    v2[:, :, P - 1] = -v2[:, :, 0]
    img, _ = oracle_mod.image_stokes_i(v2, uvw, freqs, N, pix, weighting)
    assert np.max(np.abs(img)) < 1e-12
    # signal in XX only: half the XX image, and W is the (t, c)'s weight sum
    v3 = vis.copy()
    v3[:, :, P - 1] = 0
    img, W = oracle_mod.image_stokes_i(v3, uvw, freqs, N, pix, weighting, tc_ids=[3, 0])
    for k, tc in enumerate([3, 0]):
        t, c = divmod(tc, vis.shape[1])
        r = oracle_mod.image_one(vis[t, c, 0], uvw[t], freqs[c], N, pix, weighting)
        assert np.max(np.abs(img[k] - 0.5 * r["image"])) < 1e-13 and W[k] == r["W"]


def test_stokes_i_single_baseline_closed_form(oracle_mod):
    # one baseline on cell (ku, kv): I = (2 / W) |Vm| cos(2 pi (ku x' + kv y') / N + arg Vm) with Vm = (V_XX + V_YY) / 2, W = 2
    N, ku, kv = 32, 5, -3
    f = 150e6
    s = float(oracle_mod.scale(f, N, 1.0 / N))
    uvw = np.array([[[ku / s, kv / s, 0.0]]], dtype=np.float32)
    vxx, vyy = 0.8 - 0.3j, -0.2 + 1.1j
    vis = np.zeros((1, 1, 4, 1), dtype=np.complex64)
    vis[0, 0, 0, 0], vis[0, 0, 3, 0] = vxx, vyy
    vis[0, 0, 1, 0], vis[0, 0, 2, 0] = 9.0, -7.0j                      # XY, YX must not leak in
    img, W = oracle_mod.image_stokes_i(vis, uvw, [f], N, 1.0 / N, 0)
    assert W[0] == 2.0
    vm = 0.5 * (np.complex64(vxx).astype(np.complex128) + np.complex64(vyy).astype(np.complex128))
    want = _closed_form_single_cell(N, ku, kv, vm) / 2.0
    assert np.max(np.abs(img[0] - want)) < 1e-12


@pytest.mark.parametrize("weighting", [0, 1])
def test_stokes_i_equals_image_of_mean_visibilities(oracle_mod, weighting):
    # linearity: gridding, weighting (shared W and counts) and the transform are linear in V
    vis, uvw, freqs, N, pix = _stokes_inputs(77, 2, B=200)
    img, W = oracle_mod.image_stokes_i(vis, uvw, freqs, N, pix, weighting)
    for tc in range(4):
        t, c = divmod(tc, 2)
        vm = (0.5 * (vis[t, c, 0].astype(np.complex128) + vis[t, c, 1].astype(np.complex128)))
        # float64 mean visibilities through an independent numpy gridding + numpy.fft (the oracle takes complex64 inputs)
        ci = oracle_mod.cells(uvw[t:t + 1], freqs[c:c + 1], N, pix)[0, 0]
        g = np.zeros(N * N, dtype=np.complex128)
        cnt = np.zeros(N * N)
        ok = ci >= 0
        mir = (N - ci[ok] // N) * N + (N - ci[ok] % N)
        np.add.at(g, ci[ok], vm[ok]); np.add.at(g, mir, np.conj(vm[ok]))
        np.add.at(cnt, ci[ok], 1); np.add.at(cnt, mir, 1)
        if weighting == 1:
            g[cnt > 0] /= cnt[cnt > 0]
            Wn = np.count_nonzero(cnt)
        else:
            Wn = cnt.sum()
        ref = np.fft.fftshift(np.fft.ifft2(np.fft.ifftshift(g.reshape(N, N)))).real * N * N / Wn
        assert W[tc] == Wn and np.max(np.abs(img[tc] - ref)) < 1e-12 * max(1.0, np.max(np.abs(ref)))

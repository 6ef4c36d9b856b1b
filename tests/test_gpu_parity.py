"""GPU parity: libblinkimg (through the C ABI binding) against the CPU oracle, element by element.

Bars (BASELINE.json north_star): per image max|I_gpu - I_oracle| <= 1e-4 * max|I_oracle|;
cell_idx, counts, wsum bit-exact.  All inputs come from paper_2505_15204_b200.workloads (seeded).
"""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu

TOL = 1e-4


@pytest.fixture(scope="module")
def bk():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2505_15204_b200 import binding
    binding.lib()                     # raises if the .so is missing: no fallback
    yield binding
    for k in (binding.OPT_IMAGE_PATH, binding.OPT_FUSED_CTAS, binding.OPT_GRID_CHUNK_B, binding.OPT_AVG_WSUM, binding.OPT_FUSED_TEAM):
        binding.set_option(k, 0)


def _img_err(gpu, ref):
    return float(np.max(np.abs(gpu.astype(np.float64) - ref)) / max(np.max(np.abs(ref)), 1e-300))


def _check_images(bk, w, res, oracle_mod, ids=None):
    vis, uvw = w.vis.cpu().numpy(), w.uvw_m.cpu().numpy()
    n_img = w.T * w.C * w.P
    ids = np.arange(n_img) if ids is None else np.asarray(ids)
    ref, wref = oracle_mod.image_batch(vis, uvw, w.freqs_hz, w.n_pix, w.pixscale_rad, w.weighting, ids, nthreads=8)
    img = res["image"][torch.as_tensor(ids, device=res["image"].device)].cpu().numpy()
    wsum = res["wsum"].cpu().numpy()
    worst = 0.0
    for k, i in enumerate(ids):
        assert wsum[i // w.P] == np.float32(wref[k]), (i, wsum[i // w.P], wref[k])
        if wref[k] == 0:
            assert np.all(img[k] == 0)
            continue
        worst = max(worst, _img_err(img[k], ref[k]))
    assert worst <= TOL, worst
    return worst


# --------------------------------------------------------------------------- blink_fft2d_inverse
@pytest.mark.parametrize("n,batch", [(32, 5), (64, 3), (128, 3), (256, 2), (512, 3), (1024, 2), (2048, 1), (4096, 1), (8192, 1)])
def test_fft2d_inverse_vs_oracle(bk, oracle_mod, n, batch):
    rng = np.random.default_rng(100 + n)
    g = (rng.normal(size=(batch, n, n)) + 1j * rng.normal(size=(batch, n, n))).astype(np.complex64)
    # a few isolated bright cells so that sign / orientation / shift errors cannot hide in noise
    g[0, n // 2 + 3, n // 2 - 5] += 50 * n
    g[-1, 1, n - 2] += (30 - 40j) * n
    scale = torch.tensor(rng.uniform(0.5, 2.0, batch).astype(np.float32), device="cuda")
    r = bk.blink_fft2d_inverse(torch.tensor(g, device="cuda"), scale=scale, scale_stride_div=1, want_imag=True)
    torch.cuda.synchronize()
    re, im = r["image"].cpu().numpy(), r["imag"].cpu().numpy()
    sc = scale.cpu().numpy().astype(np.float64)
    for b in range(batch):
        ref = oracle_mod.ifft2_radix2(g[b].astype(np.complex128)) / sc[b]
        peak = np.max(np.abs(ref))
        assert np.max(np.abs(re[b] - ref.real)) <= TOL * peak
        assert np.max(np.abs(im[b] - ref.imag)) <= TOL * peak


def test_fft2d_scale_semantics(bk, oracle_mod):
    n, batch = 64, 6
    rng = np.random.default_rng(1)
    g = (rng.normal(size=(batch, n, n)) + 1j * rng.normal(size=(batch, n, n))).astype(np.complex64)
    scale = torch.tensor([2.0, 0.0, 4.0], device="cuda")          # images per entry = 2; a zero entry -> zero image
    r = bk.blink_fft2d_inverse(torch.tensor(g, device="cuda"), scale=scale, scale_stride_div=2)
    img = r["image"].cpu().numpy()
    for b, s in enumerate([2.0, 2.0, 0.0, 0.0, 4.0, 4.0]):
        ref = oracle_mod.ifft2_radix2(g[b].astype(np.complex128)).real
        if s == 0:
            assert np.all(img[b] == 0)
        else:
            assert np.max(np.abs(img[b] - ref / s)) <= TOL * np.max(np.abs(ref / s))
    r = bk.blink_fft2d_inverse(torch.tensor(g, device="cuda"))     # unscaled
    ref = oracle_mod.ifft2_radix2(g[3].astype(np.complex128)).real
    assert np.max(np.abs(r["image"][3].cpu().numpy() - ref)) <= TOL * np.max(np.abs(ref))


# --------------------------------------------------------------------------- blink_grid
def _check_grid(bk, oracle_mod, w):
    from paper_2505_15204_b200 import workloads  # noqa: F401
    r = bk.blink_grid(w.vis, w.uvw_m, w.freqs_hz, w.n_pix, w.pixscale_rad, w.weighting, want_cell_idx=True,
                      want_counts=True)
    torch.cuda.synchronize()
    vis, uvw = w.vis.cpu().numpy(), w.uvw_m.cpu().numpy()
    ci = r["cell_idx"].cpu().numpy()
    assert np.array_equal(ci, oracle_mod.cells(uvw, w.freqs_hz, w.n_pix, w.pixscale_rad))       # bit-exact, every (t,c,b)
    grid = r["grid"].cpu().numpy()
    cnt = r["counts"].cpu().numpy().astype(np.uint32)
    wsum = r["wsum"].cpu().numpy()
    for t in range(w.T):
        for c in range(w.C):
            for p in range(w.P):
                g, cn, W, _ = oracle_mod.grid_one(vis[t, c, p], uvw[t], w.freqs_hz[c], w.n_pix, w.pixscale_rad, w.weighting)
                i = (t * w.C + c) * w.P + p
                assert np.array_equal(cnt[t * w.C + c], cn)
                assert wsum[t * w.C + c] == np.float32(W)
                peak = max(np.max(np.abs(g)), 1e-30)
                assert np.max(np.abs(grid[i] - g)) <= 1e-5 * peak


@pytest.mark.parametrize("n,weighting", [(32, 0), (64, 1), (256, 0), (512, 1)])
def test_grid_vs_oracle(bk, oracle_mod, n, weighting):
    from paper_2505_15204_b200 import workloads
    w = workloads.make_random(T=2, C=3, P=2, B=1500, n_pix=n, weighting=weighting, seed=n + weighting, device="cuda", fill=1.1)
    _check_grid(bk, oracle_mod, w)


@pytest.mark.parametrize("weighting", [0, 1])
def test_grid_spill_path(bk, oracle_mod, weighting):
    # chunks of 400 baselines: chunks after the first are added with global atomics
    from paper_2505_15204_b200 import workloads
    w = workloads.make_random(T=1, C=2, P=2, B=1500, n_pix=128, weighting=weighting, seed=77, device="cuda", fill=0.5)
    bk.set_option(bk.OPT_GRID_CHUNK_B, 400)
    try:
        _check_grid(bk, oracle_mod, w)
    finally:
        bk.set_option(bk.OPT_GRID_CHUNK_B, 0)


def test_grid_collisions_single_cell(bk, oracle_mod):
    # every baseline in the same cell: worst-case shared-memory atomic contention, exact counts
    from paper_2505_15204_b200 import workloads
    w = workloads.make_random(T=1, C=1, P=1, B=3000, n_pix=64, weighting=1, seed=3, device="cuda")
    w.uvw_m[:] = 0.0
    w.uvw_m[0, :, 0] = 4.2
    w.uvw_m[0, :, 1] = -7.7
    _check_grid(bk, oracle_mod, w)


# --------------------------------------------------------------------------- blink_image
@pytest.mark.parametrize("path", [0, 1, 2])
def test_image_config1_full(bk, oracle_mod, path):
    from paper_2505_15204_b200 import workloads
    w = workloads.make_config(1, device="cuda")
    bk.set_option(bk.OPT_IMAGE_PATH, path)
    try:
        res = bk.blink_image(w.vis, w.uvw_m, w.freqs_hz, w.n_pix, w.pixscale_rad, w.weighting, want_cell_idx=True,
                             want_counts=True)
        torch.cuda.synchronize()
    finally:
        bk.set_option(bk.OPT_IMAGE_PATH, 0)
    _check_images(bk, w, res, oracle_mod)
    uvw = w.uvw_m.cpu().numpy()
    assert np.array_equal(res["cell_idx"].cpu().numpy(), oracle_mod.cells(uvw, w.freqs_hz, w.n_pix, w.pixscale_rad))
    r1 = oracle_mod.image_one(w.vis[0, 0, 0].cpu().numpy(), uvw[0], w.freqs_hz[0], w.n_pix, w.pixscale_rad, 0)
    assert np.array_equal(res["counts"][0].cpu().numpy().astype(np.uint32), r1["cnt"])
    # the brightest source of the synthetic sky is where the image peaks (sanity on orientation end to end)
    img = res["image"][0].cpu().numpy()
    s = w.sources
    k = int(np.argmax(s["flux"]))
    h = w.n_pix // 2
    yx = np.unravel_index(np.argmax(img), img.shape)
    assert abs(yx[1] - (h + s["l"][k] / w.pixscale_rad)) <= 1.5 and abs(yx[0] - (h + s["m"][k] / w.pixscale_rad)) <= 1.5


@pytest.mark.parametrize("cfg,T,C", [(2, 1, 3), (3, 2, 3), (4, 1, 2), (5, 1, 2)])
@pytest.mark.parametrize("path", [0, 1, 2])
def test_image_reduced_configs(bk, oracle_mod, cfg, T, C, path):
    from paper_2505_15204_b200 import workloads
    w = workloads.make_config(cfg, device="cuda", T=T, C=C)
    bk.set_option(bk.OPT_IMAGE_PATH, path)
    try:
        res = bk.blink_image(w.vis, w.uvw_m, w.freqs_hz, w.n_pix, w.pixscale_rad, w.weighting, want_cell_idx=True)
        torch.cuda.synchronize()
    finally:
        bk.set_option(bk.OPT_IMAGE_PATH, 0)
    n_img = w.T * w.C * w.P
    ids = np.arange(n_img) if w.n_pix <= 1024 else np.array([0, n_img - 1, n_img // 2])
    _check_images(bk, w, res, oracle_mod, ids)
    assert np.array_equal(res["cell_idx"].cpu().numpy(),
                          oracle_mod.cells(w.uvw_m.cpu().numpy(), w.freqs_hz, w.n_pix, w.pixscale_rad))


@pytest.mark.parametrize("weighting", [0, 1])
@pytest.mark.parametrize("path", [0, 1, 2])
def test_image_random_ragged(bk, oracle_mod, weighting, path):
    # odd sizes everywhere: B not a multiple of anything, P = 3, off-grid samples, tiny workspace (forces chunking)
    from paper_2505_15204_b200 import workloads
    w = workloads.make_random(T=3, C=5, P=3, B=1237, n_pix=128, weighting=weighting, seed=5, device="cuda", fill=1.2)
    rec, mn = bk.blink_workspace_bytes(bk.OP_IMAGE, w.T, w.C, w.P, w.B, w.n_pix, weighting)
    ws = torch.empty(max(mn * 2, 16), dtype=torch.uint8, device="cuda")
    bk.set_option(bk.OPT_IMAGE_PATH, path)
    try:
        res = bk.blink_image(w.vis, w.uvw_m, w.freqs_hz, w.n_pix, w.pixscale_rad, weighting, workspace=ws)
        torch.cuda.synchronize()
    finally:
        bk.set_option(bk.OPT_IMAGE_PATH, 0)
    _check_images(bk, w, res, oracle_mod)


@pytest.mark.parametrize("weighting", [0, 1])
@pytest.mark.parametrize("B", [1237, 2048])
def test_fused_ragged(bk, oracle_mod, weighting, B):
    # the fused kernel itself (forced): odd B (rows only 8-byte aligned: no bulk-copy prefetch) and even B,
    # P = 3 planes per (t,c), samples off the grid, 3 persistent CTAs for 6 (t,c) items, minimum workspace
    from paper_2505_15204_b200 import workloads
    w = workloads.make_random(T=2, C=3, P=3, B=B, n_pix=256, weighting=weighting, seed=11 + B, device="cuda", fill=1.15)
    w.uvw_m[1, 5, 0] = float("nan")
    rec, mn = bk.blink_workspace_bytes(bk.OP_IMAGE, w.T, w.C, w.P, w.B, w.n_pix, weighting)
    bk.set_option(bk.OPT_IMAGE_PATH, 2)
    bk.set_option(bk.OPT_FUSED_CTAS, 3)
    try:
        res = bk.blink_image(w.vis, w.uvw_m, w.freqs_hz, w.n_pix, w.pixscale_rad, weighting, want_cell_idx=True,
                             want_counts=True)
        torch.cuda.synchronize()
        _check_images(bk, w, res, oracle_mod)
        ws = torch.empty(mn, dtype=torch.uint8, device="cuda")              # room for one CTA's scratch only
        res1 = bk.blink_image(w.vis, w.uvw_m, w.freqs_hz, w.n_pix, w.pixscale_rad, weighting, workspace=ws)
        torch.cuda.synchronize()
        _check_images(bk, w, res1, oracle_mod)
    finally:
        bk.set_option(bk.OPT_IMAGE_PATH, 0)
        bk.set_option(bk.OPT_FUSED_CTAS, 0)
    uvw = w.uvw_m.cpu().numpy()
    assert np.array_equal(res["cell_idx"].cpu().numpy(), oracle_mod.cells(uvw, w.freqs_hz, w.n_pix, w.pixscale_rad))
    cnt = res["counts"].cpu().numpy().astype(np.uint32)
    for t in range(w.T):
        for c in range(w.C):
            r1 = oracle_mod.image_one(w.vis[t, c, 0].cpu().numpy(), uvw[t], w.freqs_hz[c], w.n_pix, w.pixscale_rad, weighting)
            assert np.array_equal(cnt[t * w.C + c], r1["cnt"])


@pytest.mark.parametrize("weighting,B", [(0, 13000), (1, 13001)])
def test_fused_two_stage_pipeline(bk, oracle_mod, weighting, B):
    # a visibility row this long leaves room for only two pass-2 stage buffers (the NS = 2 instantiation)
    from paper_2505_15204_b200 import workloads
    w = workloads.make_random(T=1, C=2, P=1, B=B, n_pix=256, weighting=weighting, seed=21, device="cuda", fill=0.8)
    bk.set_option(bk.OPT_IMAGE_PATH, 2)
    try:
        res = bk.blink_image(w.vis, w.uvw_m, w.freqs_hz, w.n_pix, w.pixscale_rad, weighting)
        torch.cuda.synchronize()
    finally:
        bk.set_option(bk.OPT_IMAGE_PATH, 0)
    _check_images(bk, w, res, oracle_mod)


@pytest.mark.parametrize("weighting", [0, 1])
def test_fused_collisions_and_axis_column(bk, oracle_mod, weighting):
    # worst cases of the shared-memory gridder: 1000 samples in ONE cell, 500 on the u = 0 column (their
    # conjugates land in the same column, rows mirrored), 200 exactly at DC (sample and conjugate share the cell),
    # the rest spread out
    from paper_2505_15204_b200 import workloads
    w = workloads.make_random(T=1, C=2, P=2, B=3000, n_pix=256, weighting=weighting, seed=31, device="cuda", fill=0.9)
    cell_m = 299792458.0 / 150e6                                    # one uv cell in metres at the first channel
    w.uvw_m[0, :1000, 0] = 17.2 * cell_m
    w.uvw_m[0, :1000, 1] = -40.3 * cell_m
    w.uvw_m[0, 1000:1500, 0] = 0.0
    w.uvw_m[0, 1500:1700, 0] = 0.0
    w.uvw_m[0, 1500:1700, 1] = 0.0
    w.uvw_m[0, 1700:1800, 0] = -0.2 * cell_m                        # rounds to iu = -0 -> folded onto the u = 0 column
    bk.set_option(bk.OPT_IMAGE_PATH, 2)
    try:
        res = bk.blink_image(w.vis, w.uvw_m, w.freqs_hz, w.n_pix, w.pixscale_rad, weighting, want_cell_idx=True)
        torch.cuda.synchronize()
    finally:
        bk.set_option(bk.OPT_IMAGE_PATH, 0)
    _check_images(bk, w, res, oracle_mod)
    assert np.array_equal(res["cell_idx"].cpu().numpy(),
                          oracle_mod.cells(w.uvw_m.cpu().numpy(), w.freqs_hz, w.n_pix, w.pixscale_rad))


def test_image_degenerate_inputs(bk, oracle_mod):
    from paper_2505_15204_b200 import workloads
    # everything off the grid -> W = 0, zero images, cell_idx = -1
    w = workloads.make_random(T=1, C=2, P=1, B=64, n_pix=64, weighting=0, seed=1, device="cuda")
    w.uvw_m[:] = 1e7
    res = bk.blink_image(w.vis, w.uvw_m, w.freqs_hz, w.n_pix, w.pixscale_rad, 0, want_cell_idx=True)
    torch.cuda.synchronize()
    assert torch.all(res["image"] == 0) and torch.all(res["wsum"] == 0) and torch.all(res["cell_idx"] == -1)
    # a single baseline: closed form 2|V| cos(...) / W with W = 2
    w = workloads.make_random(T=1, C=1, P=1, B=1, n_pix=64, weighting=0, seed=2, device="cuda", fill=0.5)
    res = bk.blink_image(w.vis, w.uvw_m, w.freqs_hz, w.n_pix, w.pixscale_rad, 0)
    _check_images(bk, w, res, oracle_mod)
    # NaN uvw is dropped, the rest still imaged
    w = workloads.make_random(T=1, C=1, P=1, B=50, n_pix=64, weighting=1, seed=4, device="cuda", fill=0.5)
    w.uvw_m[0, 7, 0] = float("nan")
    res = bk.blink_image(w.vis, w.uvw_m, w.freqs_hz, w.n_pix, w.pixscale_rad, 1, want_cell_idx=True)
    assert int(res["cell_idx"][0, 0, 7]) == -1
    _check_images(bk, w, res, oracle_mod)


def test_unit_source_peak_is_one(bk):
    # north_star check 1 on the GPU path itself: all V = 1 -> centre pixel 1.0 and it is the maximum
    from paper_2505_15204_b200 import workloads
    w = workloads.make_config(1, device="cuda")
    w.vis[:] = 1.0
    for wt in (0, 1):
        res = bk.blink_image(w.vis, w.uvw_m, w.freqs_hz, w.n_pix, w.pixscale_rad, wt)
        img = res["image"][0].cpu().numpy()
        h = w.n_pix // 2
        assert abs(img[h, h] - 1.0) < 1e-5 and img.max() <= img[h, h] + 1e-6


def test_error_codes(bk):
    import ctypes
    L = bk.lib()
    x = torch.zeros(64, device="cuda")
    fr = np.array([150e6])
    p = lambda t: ctypes.c_void_p(t.data_ptr())
    f = fr.ctypes.data_as(ctypes.c_void_p)
    # n_pix not a power of two / too small / too large
    for n in (66, 45, 16, 16384):                               # prime factor 11, odd, too small, too large
        assert L.blink_image(p(x), p(x), f, 1, 1, 1, 4, n, 0.01, 0, p(x), p(x), None, None, p(x), 64, None) == -2
    assert L.blink_image(None, p(x), f, 1, 1, 1, 4, 32, 0.01, 0, p(x), p(x), None, None, p(x), 64, None) == -1
    assert L.blink_image(p(x), p(x), f, 1, 1, 1, 4, 32, -1.0, 0, p(x), p(x), None, None, p(x), 64, None) == -1
    assert L.blink_image(p(x), p(x), f, 1, 1, 1, 4, 32, 0.01, 7, p(x), p(x), None, None, p(x), 64, None) == -1
    assert L.blink_fft2d_inverse(p(x), 98, 1, None, 1, p(x), None, None, 0, None) == -2        # 2 * 7^2
    assert L.blink_fft2d_inverse(p(x), 100, 1, None, 1, p(x), None, None, 0, None) == -3       # needs its twiddle workspace
    assert L.blink_strerror(-3).decode() == "workspace too small"


# --------------------------------------------------------------------------- full size, bench launch configuration
def test_config3_full_size_sampled(bk, oracle_mod):
    """BASELINE.json config 3 at FULL size (38400 images of 512x512), exactly as bench.py launches it:
    cell indices of every (t,c,b) bit-exact, wsum of every (t,c) exact, 24 sampled images (spread over t and c,
    including the channels the dispersed transient crosses) within 1e-4 x peak, plus size-independent properties."""
    from paper_2505_15204_b200 import workloads
    import gc
    gc.collect()
    torch.cuda.empty_cache()                                      # memory cached by earlier tests of the session
    free, _ = torch.cuda.mem_get_info()
    if free < 60e9:
        pytest.skip("needs ~50 GB of device memory")
    w = workloads.make_config(3, device="cuda")
    T, C, P, B, N = w.T, w.C, w.P, w.B, w.n_pix
    assert (T, C, P, B, N) == (50, 768, 1, 8128, 512)
    res = bk.blink_image(w.vis, w.uvw_m, w.freqs_hz, N, w.pixscale_rad, w.weighting, want_cell_idx=True)
    torch.cuda.synchronize()
    uvw = w.uvw_m.cpu().numpy()
    ci = res["cell_idx"].cpu().numpy()
    ref_ci = oracle_mod.cells(uvw, w.freqs_hz, N, w.pixscale_rad)
    assert np.array_equal(ci, ref_ci)                                           # all 312 M indices
    assert np.array_equal(res["wsum"].cpu().numpy(), (2 * (ref_ci >= 0).sum(axis=2)).astype(np.float32).ravel())
    del ci, ref_ci
    rng = np.random.default_rng(33)
    tr = w.meta["transient_flux_tc"]
    hot = np.argwhere(tr > 0)
    ids = [0, T * C - 1] + [int(t * C + c) for t, c in hot[rng.choice(len(hot), 6, replace=False)]]
    ids += [int(i) for i in rng.choice(T * C, 16, replace=False)]
    ids = np.unique(ids)
    sel = torch.as_tensor(ids, device="cuda")
    vis_s = w.vis.reshape(T * C, P, B)[sel].cpu().numpy()
    img_s = res["image"][sel].cpu().numpy()
    worst = 0.0
    for k, i in enumerate(ids):
        t, c = divmod(int(i), C)
        r = oracle_mod.image_one(vis_s[k, 0], uvw[t], w.freqs_hz[c], N, w.pixscale_rad, w.weighting)
        worst = max(worst, _img_err(img_s[k], r["image"]))
    assert worst <= TOL, worst
    # properties that hold at any size: centre pixel = sum(2 Re V_in) / W for EVERY image (closed form)
    h = N // 2
    centre = res["image"][:, h, h].double().cpu().numpy()
    inr = torch.as_tensor(oracle_mod.cells(uvw, w.freqs_hz, N, w.pixscale_rad) >= 0, device="cuda").reshape(T * C, B)
    want = (2.0 * (w.vis.reshape(T * C, B).real.double() * inr).sum(dim=1) / (2.0 * inr.sum(dim=1))).cpu().numpy()
    peak = res["image"].reshape(T * C, -1).abs().amax(dim=1).double().cpu().numpy()
    assert np.max(np.abs(centre - want) / peak) <= TOL
    assert bool(torch.isfinite(res["image"]).all())


# --------------------------------------------------------------------------- blink_image_avg
def _check_avg(bk, oracle_mod, w, avg_time, workspace=None):
    res = bk.blink_image_avg(w.vis, w.uvw_m, w.freqs_hz, w.n_pix, w.pixscale_rad, w.weighting, avg_time=avg_time,
                             workspace=workspace)
    torch.cuda.synchronize()
    vis, uvw = w.vis.cpu().numpy(), w.uvw_m.cpu().numpy()
    ref = oracle_mod.image_avg(vis, uvw, w.freqs_hz, w.n_pix, w.pixscale_rad, w.weighting, avg_time)
    ref = ref.reshape(-1, w.n_pix, w.n_pix)
    got = res["image_avg"].cpu().numpy()
    assert got.shape == ref.shape
    for k in range(ref.shape[0]):
        assert _img_err(got[k], ref[k]) <= TOL, (k, _img_err(got[k], ref[k]))
    # wsum is the per-(t,c) weight sum of blink_image, bit-exact
    ci = oracle_mod.cells(uvw, w.freqs_hz, w.n_pix, w.pixscale_rad)
    wsum = res["wsum"].cpu().numpy().reshape(w.T, w.C)
    for t in range(w.T):
        for c in range(w.C):
            ok = ci[t, c] >= 0
            if w.weighting == 0:
                want = 2 * int(ok.sum())
            else:
                cells = ci[t, c][ok]
                mir = (w.n_pix - cells // w.n_pix) * w.n_pix + (w.n_pix - cells % w.n_pix)
                want = len(np.unique(np.concatenate([cells, mir])))
            assert wsum[t, c] == np.float32(want)
    return res


@pytest.mark.parametrize("weighting", [0, 1])
@pytest.mark.parametrize("avg_time", [False, True])
def test_image_avg_random(bk, oracle_mod, weighting, avg_time):
    from paper_2505_15204_b200 import workloads
    w = workloads.make_random(T=3, C=5, P=2, B=1237, n_pix=128, weighting=weighting, seed=41, device="cuda", fill=1.1)
    w.uvw_m[1, 9, 1] = float("nan")
    for wopt in (1, 2):                                         # weight sums by sort + binary search / by ballot counting
        bk.set_option(bk.OPT_AVG_WSUM, wopt)
        try:
            _check_avg(bk, oracle_mod, w, avg_time)
        finally:
            bk.set_option(bk.OPT_AVG_WSUM, 0)
    # minimum workspace: a single count plane (uniform) / weight sums by ballot counting instead of sort + search (natural)
    _, mn = bk.blink_workspace_bytes(bk.OP_IMAGE_AVG, w.T, w.C, w.P, w.B, w.n_pix, weighting)
    _check_avg(bk, oracle_mod, w, avg_time, workspace=torch.empty(mn, dtype=torch.uint8, device="cuda"))


@pytest.mark.parametrize("cfg,T,C", [(3, 2, 6), (4, 1, 3)])
def test_image_avg_reduced_configs(bk, oracle_mod, cfg, T, C):
    from paper_2505_15204_b200 import workloads
    w = workloads.make_config(cfg, device="cuda", T=T, C=C)
    res = _check_avg(bk, oracle_mod, w, False)
    # the averaged image IS the mean of blink_image's images (same library, different path)
    full = bk.blink_image(w.vis, w.uvw_m, w.freqs_hz, w.n_pix, w.pixscale_rad, w.weighting)
    mean = full["image"].reshape(w.T, w.C, w.P, w.n_pix, w.n_pix).double().mean(dim=1).reshape(-1, w.n_pix, w.n_pix)
    got = res["image_avg"].double()
    assert float((got - mean).abs().max() / mean.abs().max()) <= TOL


def test_image_avg_degenerate(bk, oracle_mod):
    from paper_2505_15204_b200 import workloads
    # all V = 1: every image has 1.0 at the centre, so has the mean; one channel entirely off the grid halves it
    w = workloads.make_random(T=1, C=2, P=1, B=500, n_pix=64, weighting=0, seed=43, device="cuda", fill=0.7)
    w.vis[:] = 1.0
    r = bk.blink_image_avg(w.vis, w.uvw_m, w.freqs_hz, w.n_pix, w.pixscale_rad, 0)
    assert abs(float(r["image_avg"][0, 32, 32]) - 1.0) < 1e-5
    w.freqs_hz = np.array([w.freqs_hz[0], 5e10])
    r = bk.blink_image_avg(w.vis, w.uvw_m, w.freqs_hz, w.n_pix, w.pixscale_rad, 0)
    assert abs(float(r["image_avg"][0, 32, 32]) - 0.5) < 1e-5 and float(r["wsum"][1]) == 0.0
    # everything off the grid: zero image
    w.uvw_m[:] = 1e7
    r = bk.blink_image_avg(w.vis, w.uvw_m, w.freqs_hz, w.n_pix, w.pixscale_rad, 1, avg_time=True)
    assert torch.all(r["image_avg"] == 0) and torch.all(r["wsum"] == 0)
    # many samples in one cell (atomic contention, uniform count = 2 cells)
    w = workloads.make_random(T=1, C=3, P=1, B=2000, n_pix=64, weighting=1, seed=44, device="cuda")
    w.uvw_m[:] = 0.0
    w.uvw_m[0, :, 0] = 4.2
    w.uvw_m[0, :, 1] = -7.7
    _check_avg(bk, oracle_mod, w, False)


def test_image_avg_config3_full_size(bk, oracle_mod):
    """BASELINE.json config 3 at full size through blink_image_avg (the launch configuration bench.py times):
    weight sums of all 38400 (t,c) exact; timestep 0's averaged image against the oracle's mean of its 768 images;
    every timestep against the mean of blink_image's own images."""
    from paper_2505_15204_b200 import workloads
    import gc
    gc.collect()
    torch.cuda.empty_cache()                                      # memory cached by earlier tests of the session
    free, _ = torch.cuda.mem_get_info()
    if free < 60e9:
        pytest.skip("needs ~50 GB of device memory")
    w = workloads.make_config(3, device="cuda")
    T, C, P, B, N = w.T, w.C, w.P, w.B, w.n_pix
    res = bk.blink_image_avg(w.vis, w.uvw_m, w.freqs_hz, N, w.pixscale_rad, w.weighting)
    torch.cuda.synchronize()
    uvw = w.uvw_m.cpu().numpy()
    ci = oracle_mod.cells(uvw, w.freqs_hz, N, w.pixscale_rad)
    assert np.array_equal(res["wsum"].cpu().numpy(), (2 * (ci >= 0).sum(axis=2)).astype(np.float32).ravel())
    del ci
    ref0 = oracle_mod.image_avg(w.vis[:1].cpu().numpy(), uvw[:1], w.freqs_hz, N, w.pixscale_rad, w.weighting)[0, 0]
    assert _img_err(res["image_avg"][0].cpu().numpy(), ref0) <= TOL
    full = bk.blink_image(w.vis, w.uvw_m, w.freqs_hz, N, w.pixscale_rad, w.weighting)
    torch.cuda.synchronize()
    worst = 0.0
    for t in range(T):
        mean = full["image"][t * C:(t + 1) * C].double().mean(dim=0)
        worst = max(worst, float((res["image_avg"][t].double() - mean).abs().max() / mean.abs().max()))
    assert worst <= TOL, worst


def test_image_8192(bk, oracle_mod):
    """The paper's long-exposure image side (8192 x 8192): blink_image through the unfused chain
    (the fused kernel stops at 4096) and the channel / time average, both against the oracle."""
    from paper_2505_15204_b200 import workloads
    w = workloads.make_random(T=1, C=2, P=1, B=3000, n_pix=8192, weighting=0, seed=51, device="cuda", fill=0.6)
    res = bk.blink_image(w.vis, w.uvw_m, w.freqs_hz, w.n_pix, w.pixscale_rad, w.weighting, want_cell_idx=True)
    torch.cuda.synchronize()
    _check_images(bk, w, res, oracle_mod, [1])
    assert np.array_equal(res["cell_idx"].cpu().numpy(),
                          oracle_mod.cells(w.uvw_m.cpu().numpy(), w.freqs_hz, w.n_pix, w.pixscale_rad))
    _check_avg(bk, oracle_mod, w, True)


# --------------------------------------------------------------------------- per-antenna gains
def _gain_setup(w, n_ant, seed):
    rng = np.random.default_rng(seed)
    pairs = np.array([(i, j) for i in range(n_ant) for j in range(i)], dtype=np.int32)
    assert len(pairs) >= w.B
    pairs = pairs[rng.permutation(len(pairs))[:w.B]].copy()
    gains = (rng.uniform(0.6, 1.4, (w.C, w.P, n_ant)) * np.exp(1j * rng.uniform(-np.pi, np.pi, (w.C, w.P, n_ant)))).astype(np.complex64)
    return gains, pairs


@pytest.mark.parametrize("weighting", [0, 1])
def test_gains_fused_and_in_place(bk, oracle_mod, weighting):
    from paper_2505_15204_b200 import workloads
    w = workloads.make_random(T=2, C=3, P=2, B=1237, n_pix=256, weighting=weighting, seed=61, device="cuda", fill=1.05)
    gains, pairs = _gain_setup(w, 64, 62)
    vis_before = w.vis.clone()
    g_d, p_d = torch.tensor(gains, device="cuda"), torch.tensor(pairs, device="cuda")
    res = bk.blink_image_cal(w.vis, w.uvw_m, w.freqs_hz, g_d, p_d, w.n_pix, w.pixscale_rad, weighting)
    torch.cuda.synchronize()
    assert torch.equal(w.vis, vis_before)                                  # the fused path never writes the visibilities
    # oracle: apply the gains (definition), then image
    fixed = oracle_mod.apply_gains(w.vis.cpu().numpy(), gains, pairs)
    w_fixed = workloads.Workload(**{**w.__dict__, "vis": torch.tensor(fixed)})
    _check_images(bk, w_fixed, res, oracle_mod)
    # the in-place kernel against the oracle's corrected visibilities, element by element
    v2 = w.vis.clone()
    bk.blink_apply_gains(v2, g_d, p_d)
    torch.cuda.synchronize()
    got = v2.cpu().numpy()
    assert np.max(np.abs(got - fixed)) <= 2e-6 * np.max(np.abs(fixed))
    # unit gains are the identity, bit for bit
    v3 = w.vis.clone()
    bk.blink_apply_gains(v3, torch.ones_like(g_d), p_d)
    assert torch.equal(v3, w.vis)


def test_gains_config3_reduced_and_unfused_sizes(bk, oracle_mod):
    from paper_2505_15204_b200 import workloads
    w = workloads.make_config(3, device="cuda", T=2, C=4)
    n_ant = 128
    pairs = np.array([(i, j) for i in range(n_ant) for j in range(i)], dtype=np.int32)    # the generator's baseline order
    rng = np.random.default_rng(63)
    gains = (rng.uniform(0.8, 1.2, (w.C, w.P, n_ant)) * np.exp(1j * rng.uniform(-1, 1, (w.C, w.P, n_ant)))).astype(np.complex64)
    g_d, p_d = torch.tensor(gains, device="cuda"), torch.tensor(pairs, device="cuda")
    res = bk.blink_image_cal(w.vis, w.uvw_m, w.freqs_hz, g_d, p_d, w.n_pix, w.pixscale_rad, w.weighting)
    fixed = oracle_mod.apply_gains(w.vis.cpu().numpy(), gains, pairs)
    w_fixed = workloads.Workload(**{**w.__dict__, "vis": torch.tensor(fixed)})
    _check_images(bk, w_fixed, res, oracle_mod)
    # sizes the fused kernel does not cover (64, and the paper's 1200): corrected copy in the workspace + the unfused chain
    for n, B in ((64, 100), (1200, 700)):
        ws = workloads.make_random(T=1, C=2, P=2, B=B, n_pix=n, weighting=n == 64, seed=64 + n, device="cuda", fill=0.8)
        g2 = (rng.uniform(0.8, 1.2, (2, 2, n_ant)) * np.exp(1j * rng.uniform(-1, 1, (2, 2, n_ant)))).astype(np.complex64)
        before = ws.vis.clone()
        res = bk.blink_image_cal(ws.vis, ws.uvw_m, ws.freqs_hz, torch.tensor(g2, device="cuda"), p_d[:B].contiguous(), n,
                                 ws.pixscale_rad, ws.weighting)
        torch.cuda.synchronize()
        assert torch.equal(ws.vis, before)
        fixed = oracle_mod.apply_gains(ws.vis.cpu().numpy(), g2, pairs[:B])
        _check_images(bk, workloads.Workload(**{**ws.__dict__, "vis": torch.tensor(fixed)}), res, oracle_mod, [0, 3])


# --------------------------------------------------------------------------- more than 1024 channels (scale blocks)
@pytest.mark.parametrize("path", [1, 2])
def test_more_than_1024_channels(bk, oracle_mod, path):
    # per-channel scales travel as a 1024-entry kernel parameter: C = 1030 needs two blocks per timestep, in the
    # fused kernel, the unfused chain and both averaging kernels; the last channels are the ones checked
    from paper_2505_15204_b200 import workloads
    w = workloads.make_random(T=2, C=1030, P=1, B=300, n_pix=256, weighting=path - 1, seed=71, device="cuda", fill=0.9)
    w.freqs_hz = 150e6 + 1.0e5 * np.arange(w.C)                 # wide enough that late channels grid differently
    bk.set_option(bk.OPT_IMAGE_PATH, path)
    try:
        res = bk.blink_image(w.vis, w.uvw_m, w.freqs_hz, w.n_pix, w.pixscale_rad, w.weighting, want_cell_idx=True)
        torch.cuda.synchronize()
    finally:
        bk.set_option(bk.OPT_IMAGE_PATH, 0)
    ids = np.array([0, 1023, 1024, 1029, 1030, 1030 + 1023, 1030 + 1024, 2 * 1030 - 1])
    _check_images(bk, w, res, oracle_mod, ids)
    assert np.array_equal(res["cell_idx"].cpu().numpy(),
                          oracle_mod.cells(w.uvw_m.cpu().numpy(), w.freqs_hz, w.n_pix, w.pixscale_rad))
    # averaged over the 1030 channels: against the mean of the images just verified to be the library's own
    avg = bk.blink_image_avg(w.vis, w.uvw_m, w.freqs_hz, w.n_pix, w.pixscale_rad, w.weighting)
    mean = res["image"].reshape(w.T, w.C, w.n_pix, w.n_pix).double().mean(dim=1)
    assert float((avg["image_avg"].double() - mean).abs().max() / mean.abs().max()) <= TOL
    assert torch.equal(avg["wsum"], res["wsum"])


def test_small_batch_auto_route(bk, oracle_mod):
    """Auto path, batches of <= 4 Mi pixels: the unfused chain when the workspace holds the whole range (recommended
    size), the fused kernel when it does not (minimum size); both against the oracle, indices and weight sums bit-exact."""
    from paper_2505_15204_b200 import workloads
    for weighting in (0, 1):
        w = workloads.make_config(1, device="cuda")
        w.weighting = weighting
        T, C, P, B = w.vis.shape
        rec, mn = bk.blink_workspace_bytes(bk.OP_IMAGE, T, C, P, B, w.n_pix, weighting)
        assert rec >= w.n_pix * w.n_pix * 8 and mn < rec
        for nbytes in (rec, mn):
            ws = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
            res = bk.blink_image(w.vis, w.uvw_m, w.freqs_hz, w.n_pix, w.pixscale_rad, weighting, want_cell_idx=True,
                                 want_counts=True, workspace=ws)
            torch.cuda.synchronize()
            _check_images(bk, w, res, oracle_mod)
            assert np.array_equal(res["cell_idx"].cpu().numpy(),
                                  oracle_mod.cells(w.uvw_m.cpu().numpy(), w.freqs_hz, w.n_pix, w.pixscale_rad))
            _, cn, _, _ = oracle_mod.grid_one(w.vis.cpu().numpy()[0, 0, 0], w.uvw_m.cpu().numpy()[0], w.freqs_hz[0], w.n_pix,
                                              w.pixscale_rad, weighting)
            assert np.array_equal(res["counts"].cpu().numpy().astype(np.uint32)[0], cn)


# --------------------------------------------------------------------------- sides that are not a power of two
@pytest.mark.parametrize("n,batch", [(48, 3), (240, 2), (1200, 1)])
def test_fft2d_non_pow2(bk, oracle_mod, n, batch):
    rng = np.random.default_rng(500 + n)
    g = (rng.normal(size=(batch, n, n)) + 1j * rng.normal(size=(batch, n, n))).astype(np.complex64)
    g[0, n // 2 + 3, n // 2 - 5] += 50 * n
    g[-1, 1, n - 2] += (30 - 40j) * n
    scale = torch.tensor(rng.uniform(0.5, 2.0, batch).astype(np.float32), device="cuda")
    r = bk.blink_fft2d_inverse(torch.tensor(g, device="cuda"), scale=scale, scale_stride_div=1, want_imag=True)
    torch.cuda.synchronize()
    re, im = r["image"].cpu().numpy(), r["imag"].cpu().numpy()
    sc = scale.cpu().numpy().astype(np.float64)
    for b in range(batch):
        ref = oracle_mod.ifft2_radix2(g[b].astype(np.complex128)) / sc[b]
        peak = np.max(np.abs(ref))
        assert np.max(np.abs(re[b] - ref.real)) <= TOL * peak
        assert np.max(np.abs(im[b] - ref.imag)) <= TOL * peak


@pytest.mark.parametrize("n,weighting", [(48, 1), (90, 0), (240, 0), (1200, 1)])
def test_grid_and_image_non_pow2(bk, oracle_mod, n, weighting):
    from paper_2505_15204_b200 import workloads
    w = workloads.make_random(T=1, C=2, P=2, B=1500, n_pix=n, weighting=weighting, seed=n + weighting, device="cuda", fill=1.1)
    _check_grid(bk, oracle_mod, w)
    res = bk.blink_image(w.vis, w.uvw_m, w.freqs_hz, w.n_pix, w.pixscale_rad, w.weighting, want_cell_idx=True)
    torch.cuda.synchronize()
    _check_images(bk, w, res, oracle_mod, [0, 3] if n == 1200 else None)
    assert np.array_equal(res["cell_idx"].cpu().numpy(),
                          oracle_mod.cells(w.uvw_m.cpu().numpy(), w.freqs_hz, w.n_pix, w.pixscale_rad))
    if n <= 240:
        _check_avg(bk, oracle_mod, w, False)
        _check_avg(bk, oracle_mod, w, True)


@pytest.mark.parametrize("n,weighting,fill", [(240, 0, 0.2), (240, 1, 0.45), (360, 0, 0.07), (1200, 0, 0.3)])
def test_non_pow2_row_extents_poisoned_workspace(bk, oracle_mod, n, weighting, fill):
    """Sides that are not a power of two: the gridder reports how many rows v >= 0 of every (t,c) hold data and the
    Hermitian transform skips the rest (never stored, never read).  The workspace is filled with NaN bit patterns first,
    so a skipped row that IS read (or an extent that is too small) poisons the image; the channels span an octave, so
    the extents differ from (t,c) to (t,c); one timestep has no baseline on the grid (W = 0, zero image) and one has a
    single sample on the row v = 0."""
    from paper_2505_15204_b200 import workloads
    w = workloads.make_random(T=4, C=3, P=2, B=700, n_pix=n, weighting=weighting, seed=7000 + n + weighting, device="cuda", fill=fill)
    w.freqs_hz = np.array([100e6, 150e6, 200e6])
    uvw = w.uvw_m.clone()
    uvw[2] = 1e7                                               # timestep 2: everything far off the grid
    uvw[3, 1:] = 1e7                                           # timestep 3: one baseline, on the row v = 0
    uvw[3, 0, 0], uvw[3, 0, 1] = 5.0, 0.0
    w.uvw_m = uvw
    rec, _ = bk.blink_workspace_bytes(bk.OP_IMAGE, w.T, w.C, w.P, w.B, n, weighting)
    for nbytes in (rec, None):                                 # the recommended size, then a size that forces several chunks
        if nbytes is None:
            _, mn = bk.blink_workspace_bytes(bk.OP_IMAGE, w.T, w.C, w.P, w.B, n, weighting)
            nbytes = mn + 4 * (rec - mn) // 12 // 256 * 256
        ws = torch.full((nbytes // 4 + 4,), float("nan"), dtype=torch.float32, device="cuda").view(torch.uint8)[:max(nbytes, 16)]
        res = bk.blink_image(w.vis, w.uvw_m, w.freqs_hz, n, w.pixscale_rad, weighting, workspace=ws)
        torch.cuda.synchronize()
        assert bool(torch.isfinite(res["image"]).all())
        _check_images(bk, w, res, oracle_mod, [0, 5, 7, 10] if n == 1200 else None)
        assert bool((res["image"][12:18] == 0).all()) and bool((res["wsum"][6:9] == 0).all())
    if n <= 360:
        # with the caller's counts array the gridder stores every band (no half plane, full extents): same images, exact counts
        res = bk.blink_image(w.vis, w.uvw_m, w.freqs_hz, n, w.pixscale_rad, weighting, want_counts=True)
        torch.cuda.synchronize()
        _check_images(bk, w, res, oracle_mod)
        vis, uvw = w.vis.cpu().numpy(), w.uvw_m.cpu().numpy()
        for tc in (0, 4, 7, 9):
            _, cn, _, _ = oracle_mod.grid_one(vis[tc // w.C, tc % w.C, 0], uvw[tc // w.C], w.freqs_hz[tc % w.C], n, w.pixscale_rad, weighting)
            assert np.array_equal(res["counts"].cpu().numpy().astype(np.uint32)[tc], cn)


def test_image_1200_paper_size(bk, oracle_mod):
    """The paper's high-time-resolution image side (1200 x 1200): config-3 visibilities imaged at 1200,
    individually and channel-averaged, against the oracle."""
    from paper_2505_15204_b200 import workloads
    w = workloads.make_config(3, device="cuda", T=1, C=4)
    w.n_pix, w.pixscale_rad = 1200, 0.6 / 1200
    res = bk.blink_image(w.vis, w.uvw_m, w.freqs_hz, w.n_pix, w.pixscale_rad, w.weighting)
    torch.cuda.synchronize()
    _check_images(bk, w, res, oracle_mod, [0, 3])
    avg = bk.blink_image_avg(w.vis, w.uvw_m, w.freqs_hz, w.n_pix, w.pixscale_rad, w.weighting)
    mean = res["image"].double().mean(dim=0)
    assert float((avg["image_avg"][0].double() - mean).abs().max() / mean.abs().max()) <= TOL


def test_fused_repeatability_stress(bk, oracle_mod):
    # the fused kernel's pipelines (stage buffers re-requested by the last releasing group, bulk-copy prefetch,
    # cp.async staging) run 25 times over ~3 images per CTA: every run must reproduce the first one up to the
    # order of the shared-memory atomic adds, and the first one must match the oracle
    from paper_2505_15204_b200 import workloads
    w = workloads.make_config(3, device="cuda", T=2, C=200)
    first = None
    for k in range(25):
        res = bk.blink_image(w.vis, w.uvw_m, w.freqs_hz, w.n_pix, w.pixscale_rad, w.weighting)
        torch.cuda.synchronize()
        if first is None:
            first = res["image"].clone()
            _check_images(bk, w, res, oracle_mod, [0, 199, 200, 399])
            peak = float(first.abs().max())
        else:
            assert float((res["image"] - first).abs().max()) <= 1e-6 * peak, k
            assert torch.equal(res["wsum"], wsum0)
        wsum0 = res["wsum"].clone()


# --------------------------------------------------------------------------- the FUSED kernel's own cell decisions
def _tie_cases(h):
    """(u, v) in cells (the scale is exactly 1 cell per metre): half-cell ties for even and odd k, the range limits,
    the fold u < 0 -> u >= 0, signed zeros.  Rounding is to nearest, ties to even (reading R2)."""
    return [
        (2.5, 7.0), (3.5, -9.0), (-2.5, 11.0), (-3.5, -13.0),            # u ties: 2, 4, -2, -4
        (21.0, 2.5), (23.0, 3.5), (-25.0, -2.5), (-27.0, -3.5),          # v ties
        (0.5, 30.0), (-0.5, 32.0), (1.5, 34.0), (-1.5, -36.0),           # ties that land on / next to the u = 0 column
        (0.0, 40.0), (-0.0, 42.0), (0.0, -44.0), (-0.0, -46.0),          # the u = 0 column itself, signed zeros
        (0.0, 0.0), (-0.0, -0.0), (-0.4, 50.0), (0.4, -52.0),            # DC; |u| < 1/2 folds onto column 0
        (h - 1.0, 60.0), (-(h - 1.0), -62.0), (64.0, h - 1.0), (-66.0, -(h - 1.0)),    # the last cells in range
        (h - 0.5, 70.0), (72.0, h - 0.5), (-(h - 0.5), 74.0), (76.0, -(h - 0.5)),      # tie at the edge: rounds to h (even) -> dropped
        (h - 1.5, 80.0), (82.0, -(h - 1.5)), (h - 1.0, h - 1.0), (-(h - 1.0), h - 1.0),  # tie that rounds to h - 2; corners
    ]


@pytest.mark.parametrize("n", [256, 512, 1200])
@pytest.mark.parametrize("weighting", [0, 1])
@pytest.mark.parametrize("path", [2, 1])
def test_fused_cell_decisions_one_hot(bk, oracle_mod, n, weighting, path):
    """What the gridder itself decides (not the side computation behind cell_idx): 8 baselines per timestep, 8 planes, plane
    p carries ONLY baseline p, so every image is one cosine fringe whose (k_u, k_v) is the cell the gridder chose
    (eq. 4-5; closed form of SURVEY 8(c) 'FFT, any N').  A wrong cell changes the image by O(1) x peak."""
    from paper_2505_15204_b200 import workloads
    h = n // 2
    f = 150e6
    pix = 299792458.0 / (f * n)
    assert float(oracle_mod.scale(f, n, pix)) == 1.0                # one cell per metre: u_m IS the cell coordinate
    cases = _tie_cases(float(h))
    B = 8
    T = len(cases) // B
    uvw = np.zeros((T, B, 3), dtype=np.float32)
    uvw[:, :, :2] = np.array(cases, dtype=np.float32).reshape(T, B, 2)
    rng = np.random.default_rng(n + weighting)
    amp = (rng.uniform(0.5, 2.0, (T, B)) * np.exp(1j * rng.uniform(-np.pi, np.pi, (T, B)))).astype(np.complex64)
    vis = np.zeros((T, 1, B, B), dtype=np.complex64)
    for b in range(B):
        vis[:, 0, b, b] = amp[:, b]
    w = workloads.Workload(name="ties", T=T, C=1, P=B, B=B, n_pix=n, pixscale_rad=pix, weighting=weighting,
                           freqs_hz=np.array([f]), uvw_m=torch.tensor(uvw, device="cuda"), vis=torch.tensor(vis, device="cuda"),
                           sources={}, meta={})
    bk.set_option(bk.OPT_IMAGE_PATH, path)
    try:
        res = bk.blink_image(w.vis, w.uvw_m, w.freqs_hz, n, pix, weighting, want_cell_idx=True)
        torch.cuda.synchronize()
    finally:
        bk.set_option(bk.OPT_IMAGE_PATH, 0)
    ci = oracle_mod.cells(uvw, w.freqs_hz, n, pix)[:, 0]            # [T][B]
    assert np.array_equal(res["cell_idx"].cpu().numpy()[:, 0], ci)
    # the cases do what they were built for (ties to even, edge tie dropped, signed zeros on column 0)
    flat = ci.ravel()
    cell = lambda iu, iv: (iv + h) * n + (iu + h)
    assert flat[0] == cell(2, 7) and flat[1] == cell(4, -9) and flat[2] == cell(-2, 11) and flat[3] == cell(-4, -13)
    assert flat[4] == cell(21, 2) and flat[5] == cell(23, 4) and flat[8] == cell(0, 30) and flat[10] == cell(2, 34)
    assert flat[13] == cell(0, 42) and flat[18] == cell(0, 50) and np.all(flat[24:28] == -1) and flat[28] == cell(h - 2, 80)
    img = res["image"].cpu().numpy().reshape(T, B, n, n).astype(np.float64)
    wsum = res["wsum"].cpu().numpy()
    y, x = np.mgrid[0:n, 0:n]
    for t in range(T):
        ok = ci[t] >= 0
        if weighting == 0:
            assert wsum[t] == 2 * ok.sum()
        for b in range(B):
            if not ok[b]:
                assert np.all(img[t, b] == 0), (t, b)
                continue
            # the oracle's image of the plane (every plane up to 512; at 1200 the O(N^3) oracle transform takes seconds per
            # image, so every third plane for uniform weighting and none for natural, where the closed form below decides)
            if n <= 512 or (weighting == 1 and (t * B + b) % 3 == 0):
                r = oracle_mod.image_one(vis[t, 0, b], uvw[t], f, n, pix, weighting)
                assert wsum[t] == np.float32(r["W"])
                peak = np.max(np.abs(r["image"]))
                assert np.max(np.abs(img[t, b] - r["image"])) <= TOL * peak, (t, b)
            if weighting == 0:                                      # the closed form itself, from the oracle's cell
                iv, iu = ci[t, b] // n - h, ci[t, b] % n - h
                V = amp[t, b].astype(np.complex128)
                if iu == 0 and iv == 0:
                    want = np.full((n, n), 2 * V.real / wsum[t])
                else:
                    want = 2 * abs(V) * np.cos(2 * np.pi * (iu * (x - h) + iv * (y - h)) / n + np.angle(V)) / wsum[t]
                assert np.max(np.abs(img[t, b] - want)) <= TOL * np.max(np.abs(want)), (t, b, iu, iv)


# --------------------------------------------------------------------------- teams of CTAs per image (fused kernel)
@pytest.mark.parametrize("n,team,ctas,weighting", [(512, 2, 6, 0), (512, 3, 7, 1), (1024, 4, 8, 1), (2048, 5, 10, 0), (256, 2, 4, 1)])
def test_fused_teams(bk, oracle_mod, n, team, ctas, weighting):
    """BLINK_OPT_FUSED_TEAM: `team` CTAs image one (t,c) together (column pairs and pass-2 tiles dealt over the ranks, one
    double-buffered scratch per team, a global-memory barrier per plane, weight sums added up across the team).  Forced team
    sizes with fewer CTAs than items, P = 3 planes, samples off the grid, an empty (t,c) (W = 0) in the middle, and a grid that
    is not a multiple of the team size."""
    from paper_2505_15204_b200 import workloads
    w = workloads.make_random(T=3, C=3, P=3 if n <= 512 else 1, B=1500, n_pix=n, weighting=weighting, seed=n + team, device="cuda", fill=1.1)
    w.uvw_m[1, :, :] = 1e7                                      # timestep 1: nothing on the grid
    w.uvw_m[2, 3, 0] = float("nan")
    bk.set_option(bk.OPT_IMAGE_PATH, 2)
    bk.set_option(bk.OPT_FUSED_TEAM, team)
    bk.set_option(bk.OPT_FUSED_CTAS, ctas)
    try:
        res = bk.blink_image(w.vis, w.uvw_m, w.freqs_hz, n, w.pixscale_rad, weighting, want_cell_idx=True)
        torch.cuda.synchronize()
        res2 = bk.blink_image(w.vis, w.uvw_m, w.freqs_hz, n, w.pixscale_rad, weighting)       # again: counters start from zero
        torch.cuda.synchronize()
    finally:
        for k in (bk.OPT_IMAGE_PATH, bk.OPT_FUSED_TEAM, bk.OPT_FUSED_CTAS):
            bk.set_option(k, 0)
    n_img = w.T * w.C * w.P
    ids = np.arange(n_img) if n <= 512 else np.array([0, 2, 4, 6, 8])
    _check_images(bk, w, res, oracle_mod, ids)
    assert np.array_equal(res["cell_idx"].cpu().numpy(), oracle_mod.cells(w.uvw_m.cpu().numpy(), w.freqs_hz, n, w.pixscale_rad))
    assert bool((res["image"][3 * w.P:6 * w.P] == 0).all()) and bool((res["wsum"][3:6] == 0).all())
    assert torch.equal(res["wsum"], res2["wsum"])
    peak = float(res["image"].abs().max())
    assert float((res["image"] - res2["image"]).abs().max()) <= 1e-6 * peak


def test_fused_teams_auto_config5_like(bk, oracle_mod):
    """Auto team size: 6 images of 2048 x 2048 on a full GPU leave one-CTA-per-image 96 % idle; the launcher picks a team."""
    from paper_2505_15204_b200 import workloads
    w = workloads.make_config(4, device="cuda", T=1, C=6)
    w.vis = w.vis[:, :, :1].contiguous()
    w.P = 1
    bk.set_option(bk.OPT_IMAGE_PATH, 2)
    try:
        res = bk.blink_image(w.vis, w.uvw_m, w.freqs_hz, w.n_pix, w.pixscale_rad, w.weighting, want_cell_idx=True)
        torch.cuda.synchronize()
    finally:
        bk.set_option(bk.OPT_IMAGE_PATH, 0)
    _check_images(bk, w, res, oracle_mod, [0, 3, 5])


# --------------------------------------------------------------------------- the fused kernel of the paper's side, 1200
@pytest.mark.parametrize("weighting", [0, 1])
@pytest.mark.parametrize("B", [1237, 2048])
def test_fused_1200_ragged(bk, oracle_mod, weighting, B):
    """blink_fused_g.cu forced (path 2): odd B (plain loads) and even B (bulk-copy prefetch), P = 3 planes per (t,c), samples off
    the grid, NaN, 3 persistent CTAs for 4 (t,c) items, recommended and minimum (one CTA's scratch) workspaces, optional outputs."""
    from paper_2505_15204_b200 import workloads
    n = 1200
    w = workloads.make_random(T=2, C=2, P=3, B=B, n_pix=n, weighting=weighting, seed=1200 + B, device="cuda", fill=1.1)
    w.uvw_m[1, 5, 0] = float("nan")
    w.uvw_m[0, 7, 0] = 0.0                                      # the u = 0 column: sample and conjugate in one column
    w.uvw_m[0, 8, :2] = 0.0                                     # DC
    _, mn = bk.blink_workspace_bytes(bk.OP_IMAGE, w.T, w.C, w.P, w.B, n, weighting)
    bk.set_option(bk.OPT_IMAGE_PATH, 2)
    bk.set_option(bk.OPT_FUSED_CTAS, 3)
    try:
        res = bk.blink_image(w.vis, w.uvw_m, w.freqs_hz, n, w.pixscale_rad, weighting, want_cell_idx=True, want_counts=True)
        torch.cuda.synchronize()
        ws = torch.empty(mn, dtype=torch.uint8, device="cuda")
        res1 = bk.blink_image(w.vis, w.uvw_m, w.freqs_hz, n, w.pixscale_rad, weighting, workspace=ws)
        torch.cuda.synchronize()
    finally:
        bk.set_option(bk.OPT_IMAGE_PATH, 0)
        bk.set_option(bk.OPT_FUSED_CTAS, 0)
    _check_images(bk, w, res, oracle_mod, [0, 4, 7, 11])
    _check_images(bk, w, res1, oracle_mod, [2, 9])
    uvw = w.uvw_m.cpu().numpy()
    assert np.array_equal(res["cell_idx"].cpu().numpy(), oracle_mod.cells(uvw, w.freqs_hz, n, w.pixscale_rad))
    r1 = oracle_mod.image_one(w.vis[1, 0, 0].cpu().numpy(), uvw[1], w.freqs_hz[0], n, w.pixscale_rad, weighting)
    assert np.array_equal(res["counts"][2].cpu().numpy().astype(np.uint32), r1["cnt"])
    assert torch.equal(res["wsum"], res1["wsum"])


def test_paper_size_1200_bench_shape_sampled(bk, oracle_mod):
    """The launch configuration of bench.py's paper_size_mode: two timesteps of config 3's visibilities (1536 images) imaged at
    the paper's side 1200 x 1200: every cell index and wsum bit-exact, sampled images within 1e-4 x peak,
    centre pixel of every image against its closed form."""
    from paper_2505_15204_b200 import workloads
    import gc
    gc.collect()
    torch.cuda.empty_cache()
    w = workloads.make_config(3, device="cuda", T=2)
    w.n_pix, w.pixscale_rad = 1200, 0.6 / 1200
    _full_size_check(bk, oracle_mod, w, 2, seed=1200)


# --------------------------------------------------------------------------- full size: configs 2, 5 and one timestep of 4
def _full_size_check(bk, oracle_mod, w, n_sample, seed):
    """The recipe of test_config3_full_size_sampled for any config, natural or uniform: cell index of every (t,c,b) and
    wsum of every (t,c) bit-exact, n_sample images (spread over t, c, p) within 1e-4 x peak, centre pixel of EVERY image
    against its closed form sum_cells G / W."""
    T, C, P, B, N = w.T, w.C, w.P, w.B, w.n_pix
    res = bk.blink_image(w.vis, w.uvw_m, w.freqs_hz, N, w.pixscale_rad, w.weighting, want_cell_idx=True)
    torch.cuda.synchronize()
    uvw = w.uvw_m.cpu().numpy()
    ref_ci = oracle_mod.cells(uvw, w.freqs_hz, N, w.pixscale_rad)
    assert np.array_equal(res["cell_idx"].cpu().numpy(), ref_ci)
    ci = torch.as_tensor(ref_ci, device="cuda").reshape(T * C, B).long()
    ok = ci >= 0
    vre = w.vis.reshape(T * C, P, B).real.double()
    if w.weighting == 0:
        W = 2.0 * ok.sum(dim=1).double()
        centre = 2.0 * (vre * ok[:, None, :]).sum(dim=2) / W[:, None]
    else:
        mir = (N - ci // N) * N + (N - ci % N)
        row = torch.arange(T * C, device="cuda")[:, None] * (N * N)
        keys = torch.cat([(row + ci)[ok], (row + mir)[ok]])
        uniq, inv, counts = torch.unique(keys, return_inverse=True, return_counts=True)
        W = torch.bincount(uniq // (N * N), minlength=T * C).double()
        inv_cnt = torch.zeros((T * C, B), dtype=torch.float64, device="cuda")
        inv_cnt[ok] = 1.0 / counts[inv[: int(ok.sum())]].double()   # samples (vis + conjugates) in the cell of every baseline
        centre = 2.0 * (vre * inv_cnt[:, None, :]).sum(dim=2) / W[:, None]
    assert torch.equal(res["wsum"], W.float())                     # every (t,c), bit-exact
    h = N // 2
    got = res["image"][:, h, h].double().reshape(T * C, P)
    peak = res["image"].reshape(T * C * P, -1).abs().amax(dim=1).double().reshape(T * C, P)
    assert float(((got - centre).abs() / peak).max()) <= TOL
    assert bool(torch.isfinite(res["image"]).all())
    rng = np.random.default_rng(seed)
    n_img = T * C * P
    ids = np.unique(np.concatenate([[0, n_img - 1], rng.choice(n_img, n_sample, replace=False)]))
    vis_c = w.vis.cpu().numpy()
    worst = 0.0
    for k0 in range(0, len(ids), 8):                               # 8 images at a time: the oracle returns float64 images
        part = ids[k0:k0 + 8]
        ref, wref = oracle_mod.image_batch(vis_c, uvw, w.freqs_hz, N, w.pixscale_rad, w.weighting, part, nthreads=8)
        img = res["image"][torch.as_tensor(part, device="cuda")].cpu().numpy()
        for k, i in enumerate(part):
            assert float(res["wsum"][i // P]) == np.float32(wref[k])
            worst = max(worst, _img_err(img[k], ref[k]))
    assert worst <= TOL, worst
    return worst


@pytest.mark.parametrize("cfg,T,n_sample", [(2, None, 16), (5, None, 16), (4, 1, 16)])
def test_full_size_configs_2_5_4(bk, oracle_mod, cfg, T, n_sample):
    """BASELINE.json configs 2 (768 x 1024^2, natural), 5 (320 x 4096^2, uniform) at FULL size and ONE full timestep of
    config 4 (3072 x 2048^2, 4 pols, uniform) in the launch configuration bench.py times."""
    from paper_2505_15204_b200 import workloads
    import gc
    gc.collect()
    torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info()
    if free < 80e9:
        pytest.skip("needs ~70 GB of device memory")
    w = workloads.make_config(cfg, device="cuda", T=T)
    shp = workloads.config_shape(cfg)
    assert (w.C, w.P, w.B, w.n_pix, w.weighting) == (shp["C"], shp["P"], shp["B"], shp["n_pix"], shp["weighting"])
    assert w.T == (shp["T"] if T is None else T)
    _full_size_check(bk, oracle_mod, w, n_sample, seed=900 + cfg)


# --------------------------------------------------------------------------- Stokes I
@pytest.mark.parametrize("P", [2, 4])
@pytest.mark.parametrize("weighting", [0, 1])
@pytest.mark.parametrize("n,B,path", [(256, 1237, 2), (256, 2048, 2), (128, 700, 0), (240, 500, 0)])
def test_stokes_i_vs_oracle(bk, oracle_mod, P, weighting, n, B, path):
    from paper_2505_15204_b200 import workloads
    w = workloads.make_random(T=2, C=3, P=P, B=B, n_pix=n, weighting=weighting, seed=80 + P + n, device="cuda", fill=1.1)
    bk.set_option(bk.OPT_IMAGE_PATH, path)
    try:
        res = bk.blink_image_stokes_i(w.vis, w.uvw_m, w.freqs_hz, n, w.pixscale_rad, weighting)
        torch.cuda.synchronize()
    finally:
        bk.set_option(bk.OPT_IMAGE_PATH, 0)
    ref, wref = oracle_mod.image_stokes_i(w.vis.cpu().numpy(), w.uvw_m.cpu().numpy(), w.freqs_hz, n, w.pixscale_rad, weighting)
    img = res["image"].cpu().numpy()
    assert img.shape == ref.shape
    assert np.array_equal(res["wsum"].cpu().numpy(), wref.astype(np.float32))
    for k in range(ref.shape[0]):
        assert _img_err(img[k], ref[k]) <= TOL, (k, _img_err(img[k], ref[k]))
    with pytest.raises(bk.BlinkError):                              # P = 3 has no XX / YY reading
        w3 = workloads.make_random(T=1, C=1, P=3, B=64, n_pix=64, weighting=0, seed=1, device="cuda")
        bk.blink_image_stokes_i(w3.vis, w3.uvw_m, w3.freqs_hz, 64, w3.pixscale_rad, 0)


def test_stokes_i_config4_reduced(bk, oracle_mod):
    from paper_2505_15204_b200 import workloads
    w = workloads.make_config(4, device="cuda", T=1, C=2)
    res = bk.blink_image_stokes_i(w.vis, w.uvw_m, w.freqs_hz, w.n_pix, w.pixscale_rad, w.weighting)
    ref, wref = oracle_mod.image_stokes_i(w.vis.cpu().numpy(), w.uvw_m.cpu().numpy(), w.freqs_hz, w.n_pix, w.pixscale_rad, w.weighting)
    assert np.array_equal(res["wsum"].cpu().numpy(), wref.astype(np.float32))
    for k in range(2):
        assert _img_err(res["image"][k].cpu().numpy(), ref[k]) <= TOL


# --------------------------------------------------------------------------- avg tie at odd N/2
@pytest.mark.parametrize("n", [90, 50])
@pytest.mark.parametrize("wopt", [1, 2])
def test_avg_edge_tie_odd_half(bk, oracle_mod, n, wopt):
    """N = 2 (mod 4): h = N/2 is odd, so |x| = h - 1/2 rounds to the EVEN h - 1 and stays on the grid; the averaging path's
    one-product range test must count it (wsum bit-exact, image normalised by the right W)."""
    from paper_2505_15204_b200 import workloads
    h = n // 2
    f = 150e6
    pix = 299792458.0 / (f * n)
    assert float(oracle_mod.scale(f, n, pix)) == 1.0
    w = workloads.make_random(T=1, C=1, P=1, B=40, n_pix=n, weighting=0, seed=n, device="cuda", fill=0.5)
    w.freqs_hz, w.pixscale_rad = np.array([f]), pix
    uvw = w.uvw_m.clone()
    uvw[0, :, :2] = torch.as_tensor(np.random.default_rng(n).uniform(-h / 2, h / 2, (40, 2)).astype(np.float32))
    uvw[0, 0, 0], uvw[0, 1, 1], uvw[0, 2, 0], uvw[0, 3, 1] = h - 0.5, -(h - 0.5), h + 0.5, h - 1.5
    w.uvw_m = uvw
    ci = oracle_mod.cells(uvw.cpu().numpy(), w.freqs_hz, n, pix)[0, 0]
    assert ci[0] >= 0 and ci[1] >= 0 and ci[2] == -1 and ci[3] >= 0   # the tie IS on the grid for odd h
    bk.set_option(bk.OPT_AVG_WSUM, wopt)
    try:
        _check_avg(bk, oracle_mod, w, False)
    finally:
        bk.set_option(bk.OPT_AVG_WSUM, 0)


def test_volt_out_of_range(bk):
    from paper_2505_15204_b200 import workloads
    volt = workloads.make_voltages(3, 5, 1003, seed=9, device="cuda", lo=-127, hi=127)
    assert bk.blink_volt_out_of_range(volt) == 0
    flat = volt.view(-1)
    for i in (0, 17, flat.numel() - 1, flat.numel() - 9):
        flat[i] = -128
    assert bk.blink_volt_out_of_range(volt) == 4
    v2 = workloads.make_voltages(8, 16, 200, seed=9, device="cuda")
    v2.view(-1)[5] = -128
    with pytest.raises(bk.BlinkError):
        bk.blink_correlate(v2, 200, 4, check_range=True)


@pytest.mark.parametrize("B,weighting", [(4097, 0), (8192, 1), (8193, 0), (14000, 0)])
def test_presort_in_registers_edges(bk, oracle_mod, B, weighting):
    # the per-timestep presorts run as register-resident bitonic networks (blink_sort.cuh) for 4097..16384 baselines: 8 or 16
    # elements per thread.  Edges: almost all padding (4097), no padding (8192), one element over (8193), 16 per thread (14000); many EQUAL |u|
    # (ties are ordered by index), u = +-same value (folded onto one key), NaN coordinates (sorted last with the padding).
    # Observables: every nearest-cell index and W bit-exact, images within tolerance, through the fused kernel AND through
    # blink_image_avg (whose weight sums come from its own sort by max(|u|, |v|) + binary search, option 1).
    from paper_2505_15204_b200 import workloads
    w = workloads.make_random(T=2, C=2, P=1, B=B, n_pix=256, weighting=weighting, seed=300 + B, device="cuda", fill=1.05)
    cell_m = 299792458.0 / 150e6
    w.uvw_m[0, 100:900, 0] = 7.25 * cell_m                         # 800 equal keys
    w.uvw_m[0, 900:1300, 0] = -7.25 * cell_m                       # and 400 more with the other sign
    w.uvw_m[1, ::7, 0] = 0.0                                       # many samples on the u = 0 column
    w.uvw_m[0, 17, 0] = float("nan")
    w.uvw_m[1, B - 1, 1] = float("nan")
    bk.set_option(bk.OPT_IMAGE_PATH, 2)
    try:
        res = bk.blink_image(w.vis, w.uvw_m, w.freqs_hz, w.n_pix, w.pixscale_rad, weighting, want_cell_idx=True)
        torch.cuda.synchronize()
    finally:
        bk.set_option(bk.OPT_IMAGE_PATH, 0)
    _check_images(bk, w, res, oracle_mod)
    assert np.array_equal(res["cell_idx"].cpu().numpy(), oracle_mod.cells(w.uvw_m.cpu().numpy(), w.freqs_hz, w.n_pix, w.pixscale_rad))
    bk.set_option(bk.OPT_AVG_WSUM, 1)
    try:
        _check_avg(bk, oracle_mod, w, False)
    finally:
        bk.set_option(bk.OPT_AVG_WSUM, 0)

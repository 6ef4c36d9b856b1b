"""blink_image_static: the entry point that allocates no device memory (its scratch is a built-in 32 MiB device array).
Collected last on purpose (the suite runs with pytest -x).  Checks its output against the existing path (blink_image with a
caller-owned workspace) within the tolerance the parity tests use, on calls in a row that share the array, alone in a fresh
process as well as after the other tests."""
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
    binding.lib()
    for k in (binding.OPT_IMAGE_PATH, binding.OPT_FUSED_CTAS, binding.OPT_FUSED_TEAM):
        binding.set_option(k, 0)
    return binding


def _compare(bk, w, out_img, out_wsum):
    ref = bk.blink_image(w.vis, w.uvw_m, w.freqs_hz, w.n_pix, w.pixscale_rad, w.weighting)      # existing path, own workspace
    got = bk.blink_image_static(w.vis, w.uvw_m, w.freqs_hz, w.n_pix, w.pixscale_rad, w.weighting, image=out_img, wsum=out_wsum)
    torch.cuda.synchronize()
    assert got["image"].data_ptr() == out_img.data_ptr()
    assert torch.equal(got["wsum"], ref["wsum"])                                               # weight sums are integers: exact
    n_img = w.T * w.C * w.P
    a = got["image"].reshape(n_img, -1).double()
    b = ref["image"].reshape(n_img, -1).double()
    peak = b.abs().amax(dim=1).clamp_min(1e-300)
    worst = float(((a - b).abs().amax(dim=1) / peak).max())
    assert worst <= TOL, worst
    assert bool(torch.isfinite(got["image"]).all())
    return got


def test_static_scratch_matches_workspace_path_on_calls_in_a_row(bk):
    from paper_2505_15204_b200 import workloads
    assert bk.blink_static_scratch_bytes() == 32 << 20
    # call 1: fused kernel, uniform weighting, P = 2, samples off the grid
    w1 = workloads.make_random(T=2, C=3, P=2, B=1237, n_pix=256, weighting=1, seed=901, device="cuda", fill=1.1)
    img1 = torch.empty((w1.T * w1.C * w1.P, 256, 256), dtype=torch.float32, device="cuda")
    ws1 = torch.empty(w1.T * w1.C, dtype=torch.float32, device="cuda")
    first = _compare(bk, w1, img1, ws1)["image"].clone()
    # call 2, right after, another shape and weighting in the same array: BASELINE.json config 3 reduced (512 x 512, natural)
    w2 = workloads.make_config(3, device="cuda", T=1, C=4)
    img2 = torch.empty((w2.T * w2.C * w2.P, 512, 512), dtype=torch.float32, device="cuda")
    ws2 = torch.empty(w2.T * w2.C, dtype=torch.float32, device="cuda")
    _compare(bk, w2, img2, ws2)
    # call 3: a side that is not a power of two (unfused chain: the array holds twiddles, grids, row extents)
    w3 = workloads.make_random(T=1, C=2, P=1, B=700, n_pix=240, weighting=0, seed=903, device="cuda", fill=0.9)
    img3 = torch.empty((2, 240, 240), dtype=torch.float32, device="cuda")
    ws3 = torch.empty(2, dtype=torch.float32, device="cuda")
    _compare(bk, w3, img3, ws3)
    # call 4 = call 1 again: what calls 2 and 3 left in the array must not matter; and no device memory is taken by the call
    free0, _ = torch.cuda.mem_get_info()
    again = bk.blink_image_static(w1.vis, w1.uvw_m, w1.freqs_hz, 256, w1.pixscale_rad, 1, image=img1, wsum=ws1)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 >= free0
    peak = float(first.abs().max())
    assert float((again["image"] - first).abs().max()) <= 1e-6 * peak                          # up to the order of the atomic adds


def test_static_scratch_rejects_problems_beyond_the_array(bk):
    from paper_2505_15204_b200 import workloads
    w = workloads.make_random(T=1, C=1, P=1, B=64, n_pix=4096, weighting=0, seed=904, device="cuda")
    _, mn = bk.blink_workspace_bytes(bk.OP_IMAGE, 1, 1, 1, 64, 4096, 0)
    assert mn > bk.blink_static_scratch_bytes()
    img = torch.full((1, 4096, 4096), 7.0, dtype=torch.float32, device="cuda")
    ws = torch.full((1,), 7.0, dtype=torch.float32, device="cuda")
    with pytest.raises(bk.BlinkError) as ei:
        bk.blink_image_static(w.vis, w.uvw_m, w.freqs_hz, 4096, w.pixscale_rad, 0, image=img, wsum=ws)
    assert "built-in array holds" in str(ei.value) and str(32 << 20) in str(ei.value)
    torch.cuda.synchronize()
    assert bool((img == 7.0).all()) and float(ws[0]) == 7.0                                    # nothing was launched

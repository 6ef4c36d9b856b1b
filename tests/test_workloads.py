"""Host-side checks of the seeded input generator (no GPU, no imaging arithmetic)."""
import numpy as np
import torch

from paper_2505_15204_b200 import workloads as wl


def test_baseline_order_lower_triangular():
    pos = np.arange(15, dtype=np.float64).reshape(5, 3) ** 2
    bl = wl.baselines_enu(pos)
    assert bl.shape == (10, 3)
    for i in range(5):
        for j in range(i):
            assert np.array_equal(bl[i * (i - 1) // 2 + j], pos[i] - pos[j])      # PAPER.md L178 ordering


def test_zenith_uvw_is_enu():
    rng = np.random.default_rng(0)
    bl = rng.normal(size=(20, 3)) * 100
    uvw = wl.enu_to_uvw(bl, 0.0, np.deg2rad(wl.MWA_LAT_DEG))
    assert np.allclose(uvw, bl, atol=1e-10)
    # rotation preserves length at any hour angle / declination
    uvw2 = wl.enu_to_uvw(bl, 0.3, -0.47)
    assert np.allclose(np.linalg.norm(uvw2, axis=1), np.linalg.norm(bl, axis=1))


def test_config1_shapes_and_determinism():
    a = wl.make_config(1)
    b = wl.make_config(1)
    assert (a.T, a.C, a.P, a.B, a.n_pix) == (1, 1, 1, 8128, 256)
    assert a.vis.shape == (1, 1, 1, 8128) and a.vis.dtype == torch.complex64
    assert a.uvw_m.shape == (1, 8128, 3) and a.uvw_m.dtype == torch.float32
    assert torch.equal(a.vis, b.vis) and torch.equal(a.uvw_m, b.uvw_m)
    assert a.freqs_hz[0] == 154.24e6
    assert np.all((a.sources["flux"] >= 0.1) & (a.sources["flux"] <= 10.0))
    assert float(torch.hypot(a.uvw_m[0, :, 0], a.uvw_m[0, :, 1]).max()) <= 600.0 + 1e-3     # disc of radius 300 m


def test_reduced_configs():
    w = wl.make_config(3, T=2, C=4)
    assert (w.T, w.C, w.P, w.B, w.n_pix, w.weighting) == (2, 4, 1, 8128, 512, wl.W_NATURAL)
    assert w.freqs_hz[0] == 154.88e6 - 383.5 * 40e3 and w.freqs_hz[-1] == 154.88e6 + 383.5 * 40e3
    assert not torch.equal(w.uvw_m[0], w.uvw_m[1])                                # Earth rotation between steps
    w4 = wl.make_config(4, T=1, C=2)
    assert (w4.P, w4.B, w4.n_pix, w4.weighting) == (4, 10296, 2048, wl.W_UNIFORM)
    w5 = wl.make_config(5, T=1, C=2)
    assert float(w5.uvw_m[0, :, 2].abs().max()) > 10.0                            # non-zero w terms


def test_phase_centre_source_visibility_is_flux():
    uvw = torch.tensor(np.random.default_rng(1).normal(size=(1, 50, 3)) * 200, dtype=torch.float32)
    v = wl._point_source_vis(uvw, np.array([150e6, 160e6]), [0.0], [0.0], np.full((1, 2, 1), 3.5), "cpu")
    assert torch.allclose(v, torch.full_like(v, 3.5))


def test_transient_sweeps_down_in_frequency():
    freqs = 154.88e6 + (np.arange(768) - 383.5) * 40e3
    tr = wl.transient_flux(50, freqs, 0.02, 500.0, 5.0, 0.02, 0.1)
    assert tr.shape == (50, 768) and tr.max() <= 5.0 + 1e-12
    top = np.nonzero(tr[:, -1])[0]
    assert top.min() == 5                                                         # arrives at 0.1 s at the top channel
    assert np.allclose(tr.sum(axis=0)[tr.sum(axis=0) > 0].max(), 5.0)             # 20 ms pulse = one bin of flux
    lo = np.nonzero(tr.sum(axis=0))[0].min()
    assert lo > 700                                                               # only the top channels within 1 s

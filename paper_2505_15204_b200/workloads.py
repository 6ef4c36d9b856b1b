"""Seeded synthetic workloads shaped like the paper's MWA observations.

This module only MAKES INPUTS (tile layouts, uvw in metres, frequencies, point-source
visibilities + noise).  It holds none of the imaging method's arithmetic (no cell index,
no gridding, no FFT) and imports neither ``oracle/`` nor the CUDA binding, so both sides
of a parity test can be fed from it.

The inputs stand in for the paper's MWA observations OBSID 1276619416 / 1293315072
(Table 2, L271-280 Table 4), which are not available; shapes follow
BASELINE.json ``configs`` and PAPER.md L57-71 (Table 1) and L284 (50 x 20 ms, 768 x 40 kHz).
The recipe (and which parts are this repo's proposals) is stated in DESIGN.md "Input recipe".

Small RNG draws (tiles, sources) use numpy ``default_rng(seed)``; the noise uses a
``torch.Generator`` on the target device (so CPU- and CUDA-generated noise differ; every
parity test feeds the SAME arrays to both sides, so this does not matter).
"""
from __future__ import annotations

import dataclasses
import math
from typing import Optional

import numpy as np
import torch

C0 = 299792458.0                      # m/s
MWA_LAT_DEG = -26.7033                # array latitude used for ENU -> equatorial
W_NATURAL, W_UNIFORM = 0, 1


@dataclasses.dataclass
class Workload:
    name: str
    T: int
    C: int
    P: int
    B: int
    n_pix: int
    pixscale_rad: float
    weighting: int
    freqs_hz: np.ndarray              # [C] float64 (host)
    uvw_m: torch.Tensor               # [T][B][3] float32
    vis: torch.Tensor                 # [T][C][P][B] complex64
    sources: dict                     # l, m, flux arrays (host, float64)
    meta: dict

    @property
    def n_img(self) -> int:
        return self.T * self.C * self.P


# ----------------------------------------------------------------------------- geometry
def tile_positions_disc(rng: np.random.Generator, n_tiles: int, radius_m: float) -> np.ndarray:
    """ENU positions, uniform over a disc, height jitter N(0, 1 m)."""
    u1 = rng.random(n_tiles)
    u2 = rng.random(n_tiles)
    r = radius_m * np.sqrt(u1)
    th = 2.0 * np.pi * u2
    up = rng.normal(0.0, 1.0, n_tiles)
    return np.stack([r * np.cos(th), r * np.sin(th), up], axis=1)


def tile_positions_logradial(rng: np.random.Generator, n_tiles: int, rmin: float, rmax: float) -> np.ndarray:
    """ENU positions with a log-radial density profile out to rmax."""
    lr = rng.uniform(np.log(rmin), np.log(rmax), n_tiles)
    th = 2.0 * np.pi * rng.random(n_tiles)
    r = np.exp(lr)
    up = rng.normal(0.0, 1.0, n_tiles)
    return np.stack([r * np.cos(th), r * np.sin(th), up], axis=1)


def baselines_enu(pos: np.ndarray) -> np.ndarray:
    """Cross baselines, pairs i > j in lower-triangular order b = i(i-1)/2 + j."""
    n = pos.shape[0]
    ii, jj = np.tril_indices(n, k=-1)       # rows i > j, row-major => b = i(i-1)/2 + j
    return pos[ii] - pos[jj]


def enu_to_uvw(bl_enu: np.ndarray, hour_angle_rad: float, dec_rad: float) -> np.ndarray:
    """Textbook ENU -> equatorial XYZ -> (u, v, w) in metres for one hour angle / declination."""
    phi = np.deg2rad(MWA_LAT_DEG)
    e, n, u = bl_enu[:, 0], bl_enu[:, 1], bl_enu[:, 2]
    x = -n * np.sin(phi) + u * np.cos(phi)
    y = e
    z = n * np.cos(phi) + u * np.sin(phi)
    sh, ch = np.sin(hour_angle_rad), np.cos(hour_angle_rad)
    sd, cd = np.sin(dec_rad), np.cos(dec_rad)
    uu = sh * x + ch * y
    vv = -sd * ch * x + sd * sh * y + cd * z
    ww = cd * ch * x - cd * sh * y + sd * z
    return np.stack([uu, vv, ww], axis=1)


# ----------------------------------------------------------------------------- sky
def draw_sources(rng: np.random.Generator, n_src: int, lm_max: float,
                 smin: float = 0.1, smax: float = 10.0, index: float = -1.6) -> dict:
    l = rng.uniform(-lm_max, lm_max, n_src)
    m = rng.uniform(-lm_max, lm_max, n_src)
    a = index + 1.0                         # dN/dS ~ S^index  => inverse CDF on S^a
    u = rng.random(n_src)
    flux = (smin ** a + u * (smax ** a - smin ** a)) ** (1.0 / a)
    return {"l": l, "m": m, "flux": flux}


def transient_flux(T: int, freqs_hz: np.ndarray, dt_s: float, dm: float, flux_jy: float,
                   width_s: float, t_top_s: float) -> np.ndarray:
    """[T][C] flux of a dispersed pulse: overlap of [t_arr, t_arr+width] with each time bin."""
    f_mhz = freqs_hz / 1e6
    f_top = f_mhz.max()
    t_arr = t_top_s + 4.148808e3 * dm * (f_mhz ** -2 - f_top ** -2)        # seconds
    t0 = np.arange(T)[:, None] * dt_s
    t1 = t0 + dt_s
    ov = np.clip(np.minimum(t1, t_arr[None, :] + width_s) - np.maximum(t0, t_arr[None, :]), 0.0, None)
    return flux_jy * ov / width_s


def _point_source_vis(uvw_m: torch.Tensor, freqs_hz: np.ndarray, l, m, flux_tc,
                      device, chan_chunk: int = 32) -> torch.Tensor:
    """V[t][c][b] = sum_s S_s(t,c) exp(-2 pi i (u l + v m + w (n-1))) with u,v,w in wavelengths
    at f_c (sign as PAPER.md L104 eq. 4); evaluated in float64, returned complex64."""
    T, B, _ = uvw_m.shape
    C = len(freqs_hz)
    l = torch.as_tensor(l, dtype=torch.float64, device=device)
    m = torch.as_tensor(m, dtype=torch.float64, device=device)
    n1 = torch.sqrt(1.0 - l * l - m * m) - 1.0
    f = torch.as_tensor(freqs_hz, dtype=torch.float64, device=device)
    flux_tc = torch.as_tensor(flux_tc, dtype=torch.float64, device=device)     # [T][C][S]
    out = torch.empty((T, C, B), dtype=torch.complex64, device=device)
    for t in range(T):
        uvw = uvw_m[t].to(torch.float64)                                        # [B][3]
        tau = (uvw[:, 0:1] * l[None, :] + uvw[:, 1:2] * m[None, :] + uvw[:, 2:3] * n1[None, :]) / C0  # [B][S]
        for c0 in range(0, C, chan_chunk):
            c1 = min(C, c0 + chan_chunk)
            ph = (-2.0 * math.pi) * f[c0:c1, None, None] * tau[None, :, :]      # [c][B][S]
            amp = flux_tc[t, c0:c1, None, :]                                    # [c][1][S]
            re = (amp * torch.cos(ph)).sum(-1)
            im = (amp * torch.sin(ph)).sum(-1)
            out[t, c0:c1] = torch.complex(re, im).to(torch.complex64)
    return out


def _add_noise(vis: torch.Tensor, sigma: float, seed: int) -> None:
    if sigma <= 0:
        return
    g = torch.Generator(device=vis.device)
    g.manual_seed(seed)
    vr = torch.view_as_real(vis)
    for t in range(vis.shape[0]):                                               # bounded temporaries
        vr[t] += sigma * torch.randn(vr[t].shape, generator=g, device=vis.device, dtype=torch.float32)


# ----------------------------------------------------------------------------- configs
_CONFIGS = {
    # name: tiles, layout, R, T, C, P, N, pixscale, weighting, n_src, lm_max, sigma, seed
    1: dict(tiles=128, layout="disc", R=300.0, T=1, C=1, P=1, N=256, pix=0.5 / 256, w=W_NATURAL,
            n_src=20, lm=0.3, sigma=0.1, seed=1001, f0=154.24e6, pointing="zenith"),
    2: dict(tiles=128, layout="disc", R=300.0, T=1, C=768, P=1, N=1024, pix=1.0 / 1024, w=W_NATURAL,
            n_src=50, lm=0.3, sigma=0.1, seed=1002, f0=154.88e6, pointing="zenith"),
    3: dict(tiles=128, layout="disc", R=300.0, T=50, C=768, P=1, N=512, pix=0.6 / 512, w=W_NATURAL,
            n_src=50, lm=0.3, sigma=0.2, seed=1003, f0=154.88e6, pointing="track", dec=-27.0, H0_h=0.0),
    4: dict(tiles=144, layout="disc", R=300.0, T=10, C=768, P=4, N=2048, pix=1.0 / 2048, w=W_UNIFORM,
            n_src=100, lm=0.3, sigma=0.1, seed=1004, f0=154.88e6, pointing="zenith"),
    5: dict(tiles=128, layout="logradial", R=5000.0, T=5, C=64, P=1, N=4096, pix=1.4 / 4096, w=W_UNIFORM,
            n_src=200, lm=0.7, sigma=0.1, seed=1005, f0=154.88e6, pointing="track", dec=-27.0, H0_h=1.0),
}


def config_shape(k: int) -> dict:
    """Static shape facts of config k (no data)."""
    c = _CONFIGS[k]
    nt = c["tiles"]
    return dict(T=c["T"], C=c["C"], P=c["P"], B=nt * (nt - 1) // 2, n_pix=c["N"],
                pixscale_rad=c["pix"], weighting=c["w"])


def make_config(k: int, device="cpu", T: Optional[int] = None, C: Optional[int] = None,
                seed: Optional[int] = None) -> Workload:
    """Build BASELINE.json config k (1..5).  ``T`` / ``C`` optionally REDUCE the number of timesteps /
    channels (the first T timesteps; C channels spread evenly over the band) for parity tests.
    ``seed`` overrides the config's seed (used for per-rank shards)."""
    cfg = dict(_CONFIGS[k])
    if seed is not None:
        cfg["seed"] = int(seed)
    rng = np.random.default_rng(cfg["seed"])
    device = torch.device(device)
    # tiles -> baselines
    if cfg["layout"] == "disc":
        pos = tile_positions_disc(rng, cfg["tiles"], cfg["R"])
    else:
        pos = tile_positions_logradial(rng, cfg["tiles"], 10.0, cfg["R"])
    bl = baselines_enu(pos)
    B = bl.shape[0]
    # frequencies
    Cfull = cfg["C"]
    if Cfull == 1:
        freqs = np.array([cfg["f0"]], dtype=np.float64)
    else:
        freqs = cfg["f0"] + (np.arange(Cfull) - (Cfull - 1) / 2.0) * 40e3
    if C is not None and C < Cfull:
        sel = np.unique(np.round(np.linspace(0, Cfull - 1, C)).astype(int))
        freqs = freqs[sel]
    Tn = cfg["T"] if T is None else min(T, cfg["T"])
    # uvw per timestep
    phi = np.deg2rad(MWA_LAT_DEG)
    uvw = np.empty((Tn, B, 3), dtype=np.float64)
    for t in range(Tn):
        if cfg["pointing"] == "zenith":
            H, dec = 0.0, phi
        else:
            H = np.deg2rad(15.0 * (cfg["H0_h"] + 0.02 * t / 3600.0))      # 15 deg/h, 20 ms steps
            dec = np.deg2rad(cfg["dec"])
        uvw[t] = enu_to_uvw(bl, H, dec)
    uvw_t = torch.from_numpy(uvw.astype(np.float32)).to(device)
    # sky
    src = draw_sources(rng, cfg["n_src"], cfg["lm"])
    S = cfg["n_src"]
    flux_tc = np.broadcast_to(src["flux"][None, None, :], (Tn, len(freqs), S)).copy()
    l, m = src["l"].copy(), src["m"].copy()
    meta = {"config": k, "seed": cfg["seed"]}
    if k == 3:
        tr = transient_flux(Tn, freqs, 0.02, 500.0, 5.0, 0.02, 0.1)             # [T][C]
        l = np.append(l, 0.12)
        m = np.append(m, -0.08)
        flux_tc = np.concatenate([flux_tc, tr[:, :, None]], axis=2)
        meta["transient_lm"] = (0.12, -0.08)
        meta["transient_flux_tc"] = tr
    # the float32 uvw are what the imager sees; the sky model uses the same values
    visI = _point_source_vis(uvw_t, freqs, l, m, flux_tc, device)               # [T][C][B]
    P = cfg["P"]
    vis = torch.zeros((Tn, len(freqs), P, B), dtype=torch.complex64, device=device)
    if P == 1:
        vis[:, :, 0] = visI
    else:                                                                        # XX, XY, YX, YY
        vis[:, :, 0] = visI
        vis[:, :, 3] = visI
    del visI
    _add_noise(vis, cfg["sigma"], cfg["seed"] + 7919)
    return Workload(name=f"config{k}", T=Tn, C=len(freqs), P=P, B=B, n_pix=cfg["N"],
                    pixscale_rad=cfg["pix"], weighting=cfg["w"], freqs_hz=freqs, uvw_m=uvw_t,
                    vis=vis, sources=src, meta=meta)


def make_random(T: int, C: int, P: int, B: int, n_pix: int, weighting: int, seed: int,
                device="cpu", fill: float = 0.9, f0: float = 150e6) -> Workload:
    """Unstructured test input: uvw uniform so that about ``fill`` of the grid half-width is
    used (values > 1 push samples off the grid), vis ~ complex normal."""
    rng = np.random.default_rng(seed)
    freqs = f0 + 40e3 * np.arange(C)
    pix = 1.0 / n_pix
    # cells per metre at f0 is f0 * n_pix * pix / c0 = f0 / c0
    half_m = fill * (n_pix / 2) / (f0 / C0)
    uvw = rng.uniform(-half_m, half_m, (T, B, 3)).astype(np.float32)
    vis = (rng.normal(size=(T, C, P, B)) + 1j * rng.normal(size=(T, C, P, B))).astype(np.complex64)
    return Workload(name="random", T=T, C=C, P=P, B=B, n_pix=n_pix, pixscale_rad=pix, weighting=weighting,
                    freqs_hz=freqs, uvw_m=torch.from_numpy(uvw).to(device),
                    vis=torch.from_numpy(vis).to(device), sources={}, meta={"seed": seed})


def make_voltages(F: int, A: int, Ns: int, seed: int, device="cpu", amp: float = 2.0, lo: int = -8, hi: int = 7) -> torch.Tensor:
    """Synthetic fine-channelised voltages shaped like MWA Phase I VCS data: [F][A][Ns][2] int8,
    a common sky signal seen by every input with its own complex gain plus independent receiver noise, quantised to
    the 4 + 4 bit range [-8, 7] (``lo`` / ``hi`` widen it for full-range tests).  No correlator arithmetic here."""
    g = torch.Generator(device=device)
    g.manual_seed(seed)
    dev = torch.device(device)
    sky = torch.randn((F, 1, Ns, 2), generator=g, device=dev)
    ph = torch.rand((1, A, 1), generator=g, device=dev) * (2 * math.pi)
    gr, gi = torch.cos(ph), torch.sin(ph)
    x = torch.empty((F, A, Ns, 2), device=dev)
    x[..., 0] = sky[..., 0] * gr - sky[..., 1] * gi
    x[..., 1] = sky[..., 0] * gi + sky[..., 1] * gr
    x = amp * (0.6 * x + torch.randn((F, A, Ns, 2), generator=g, device=dev))
    return torch.clamp(torch.round(x), lo, hi).to(torch.int8)

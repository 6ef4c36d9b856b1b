"""GPU parity of blink_correlate (CMAC correlator on the int8 tensor cores) against the CPU oracle, through the C ABI.
Bar: BIT-EXACT (the sums are exact integers; the normalisation is one fp32 division on both sides)."""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def bk():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2505_15204_b200 import binding
    binding.lib()
    return binding


def _check(bk, oracle_mod, volt, n_t, n_avg, path=0):
    bk.set_option(bk.OPT_CORR_PATH, path)
    try:
        vis = bk.blink_correlate(volt, n_t, n_avg)
        torch.cuda.synchronize()
    finally:
        bk.set_option(bk.OPT_CORR_PATH, 0)
    ref = oracle_mod.correlate(volt.cpu().numpy(), n_t, n_avg)
    got = vis.cpu().numpy()
    assert got.shape == ref.shape
    bad = np.argwhere(got.view(np.uint64) != ref.view(np.uint64))
    assert len(bad) == 0, (len(bad), bad[:5], got[tuple(bad[0])], ref[tuple(bad[0])])


@pytest.mark.parametrize("F,A,Ns,n_t,n_avg", [
    (4, 256, 512, 64, 2),        # one 128-byte chunk per interval, no K tail
    (8, 256, 1000, 200, 4),      # the paper's 20 ms / 40 kHz shape: 400 bytes = 3 chunks + a 16-byte tail
    (2, 128, 640, 128, 1),       # a single tile
    (3, 100, 288, 72, 3),        # partial tile (rows beyond A zero-filled), 144 bytes = 1 chunk + 16-byte tail
    (2, 288, 320, 80, 2),        # MWA Phase II: 144 tiles x 2 pols = 3 tile rows, the last one partial
    (2, 1, 64, 64, 1),           # a single input: one autocorrelation
])
def test_correlate_shapes(bk, oracle_mod, F, A, Ns, n_t, n_avg):
    from paper_2505_15204_b200 import workloads
    volt = workloads.make_voltages(F, A, Ns, seed=7 + A + n_t, device="cuda")
    _check(bk, oracle_mod, volt, n_t, n_avg)


def test_correlate_full_range_int8(bk, oracle_mod):
    from paper_2505_15204_b200 import workloads
    volt = workloads.make_voltages(2, 160, 1024, seed=3, device="cuda", amp=60.0, lo=-127, hi=127)
    assert int(volt.min()) == -127 and int(volt.max()) == 127
    _check(bk, oracle_mod, volt, 512, 2)


def test_correlate_sums_beyond_2_24_and_many_tiles(bk, oracle_mod):
    # full-range samples over 8192 x 2 accumulations: |sums| reach 2.6e8 > 2^24, so the int32 -> fp32 conversion rounds
    # (identically on both sides) before the division; 520 inputs = 5 tile rows (15 tiles), the last one with 8 valid rows
    from paper_2505_15204_b200 import workloads
    volt = workloads.make_voltages(2, 520, 8192, seed=13, device="cuda", amp=90.0, lo=-127, hi=127)
    _check(bk, oracle_mod, volt, 8192, 2)
    ref_max = float(np.abs(oracle_mod.correlate(volt[:, :4].cpu().numpy(), 8192, 2)).max()) * 16384
    assert ref_max > 2 ** 24


@pytest.mark.parametrize("n_t", [72, 80, 88, 96, 104, 120, 136, 200])
def test_correlate_k_tails(bk, oracle_mod, n_t):
    # 2 n_t bytes per (interval, fine channel) = full 128-byte chunks + a tail of 16 .. 112 bytes: tails of at most 32 / 64
    # bytes are staged as 32 / 64-byte rows in the swizzle of that width (own tensor map, own UMMA descriptor), wider ones
    # as a zero-filled 128-byte chunk; 200 inputs = a full and a partial tile row, 3 intervals x 2 output channels
    from paper_2505_15204_b200 import workloads
    volt = workloads.make_voltages(6, 200, 3 * n_t, seed=23 + n_t, device="cuda")
    _check(bk, oracle_mod, volt, n_t, 3)


def test_correlate_many_units(bk, oracle_mod):
    # 16 intervals x 48 channels x 3 tiles = 2304 units over 148 CTAs: stage ring and TMEM buffers wrap many times
    from paper_2505_15204_b200 import workloads
    volt = workloads.make_voltages(48, 256, 16 * 64, seed=11, device="cuda")
    _check(bk, oracle_mod, volt, 64, 1)


def test_correlate_constant_and_zero(bk):
    volt = torch.zeros((2, 130, 128, 2), dtype=torch.int8, device="cuda")
    assert torch.all(bk.blink_correlate(volt, 64, 2) == 0)
    volt[..., 0] = 3
    volt[..., 1] = -4                                             # every x = 3 - 4i: all products 25 + 0i
    vis = bk.blink_correlate(volt, 64, 1)
    assert torch.all(vis == torch.complex(torch.tensor(25.0), torch.tensor(0.0)).to("cuda"))


def test_correlate_error_codes(bk):
    import ctypes
    L = bk.lib()
    x = torch.zeros(1 << 20, dtype=torch.int8, device="cuda")
    p = ctypes.c_void_p(x.data_ptr())
    assert L.blink_correlate(p, 2, 4, 100, 64, 1, p, None) == -1          # Ns not a multiple of n_t
    assert L.blink_correlate(p, 3, 4, 128, 64, 2, p, None) == -1          # F not a multiple of n_avg
    assert L.blink_correlate(p, 2, 4, 120, 60, 1, p, None) == -2          # n_t not a multiple of 8
    assert L.blink_correlate(p, 2, 4, 64, 32, 1, p, None) == -2           # n_t below 64
    assert L.blink_correlate(None, 2, 4, 128, 64, 1, p, None) == -1


def test_correlate_one_second_sampled(bk, oracle_mod):
    """One second of MWA Phase I data in the launch configuration bench.py times: 3072 fine channels x 256 inputs x
    10000 samples, 20 ms x 40 kHz -> 50 x 768 matrices of 32896 entries.  Sampled (t, c) against the oracle bit for bit,
    autocorrelations real and positive everywhere."""
    from paper_2505_15204_b200 import workloads
    import gc
    gc.collect()
    torch.cuda.empty_cache()                                      # memory cached by earlier tests of the session
    free, _ = torch.cuda.mem_get_info()
    if free < 70e9:
        pytest.skip("needs ~60 GB of device memory (generation included)")
    F, A, Ns, n_t, n_avg = 3072, 256, 10000, 200, 4
    volt = torch.empty((F, A, Ns, 2), dtype=torch.int8, device="cuda")
    for f0 in range(0, F, 256):
        volt[f0:f0 + 256] = workloads.make_voltages(256, A, Ns, seed=100 + f0, device="cuda")
    vis = bk.blink_correlate(volt, n_t, n_avg)
    torch.cuda.synchronize()
    rng = np.random.default_rng(5)
    for t, c in [(0, 0), (49, 767)] + [(int(rng.integers(50)), int(rng.integers(768))) for _ in range(6)]:
        sub = volt[c * n_avg:(c + 1) * n_avg, :, t * n_t:(t + 1) * n_t].contiguous().cpu().numpy()
        ref = oracle_mod.correlate(sub, n_t, n_avg)[0, 0]
        got = vis[t, c].cpu().numpy()
        assert np.array_equal(got.view(np.uint64), ref.view(np.uint64)), (t, c)
    i = torch.arange(A, device="cuda")
    autos = vis[:, :, i * (i + 1) // 2 + i]
    assert bool(torch.all(autos.imag == 0)) and bool(torch.all(autos.real > 0))

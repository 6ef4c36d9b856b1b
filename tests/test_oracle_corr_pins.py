"""Pins for oracle_correlate (CMAC correlator, eq. 3 L98 and L172-178; reading R17) against things
other than itself.  No GPU needed."""
import os

import numpy as np
import pytest

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _tri(i, j):
    return i * (i + 1) // 2 + j


def test_hand_worked_two_inputs(oracle_mod):
    volt = np.zeros((1, 2, 2, 2), np.int8)
    volt[0, 0] = [[1, 2], [3, -1]]
    volt[0, 1] = [[2, -1], [-1, 4]]
    vis = oracle_mod.correlate(volt, n_t=2, n_avg=1)
    assert vis.shape == (1, 1, 3)
    for line in open(os.path.join(GOLD, "cmac_two_inputs.txt")):
        if line.startswith("#") or not line.strip():
            continue
        i, j, re, im = line.split()
        assert vis[0, 0, _tri(int(i), int(j))] == np.complex64(float(re) + 1j * float(im))


def test_constant_inputs_and_autos(oracle_mod):
    rng = np.random.default_rng(1)
    F, A, Ns = 2, 5, 24
    c = rng.integers(-8, 8, (F, A, 2))
    volt = np.broadcast_to(c[:, :, None, :], (F, A, Ns, 2)).astype(np.int8)
    vis = oracle_mod.correlate(volt, n_t=8, n_avg=1)                        # every sample equal: the mean is the product
    z = c[..., 0] + 1j * c[..., 1]
    for f in range(F):
        for i in range(A):
            for j in range(i + 1):
                assert np.all(vis[:, f, _tri(i, j)] == np.complex64(z[f, i] * np.conj(z[f, j])))
    volt = rng.integers(-8, 8, (3, 4, 40, 2)).astype(np.int8)
    vis = oracle_mod.correlate(volt, n_t=10, n_avg=3)
    p = (volt.astype(np.int64) ** 2).sum(axis=3)                            # |x|^2  [F][A][Ns]
    for i in range(4):
        auto = vis[:, 0, _tri(i, i)]
        assert np.all(auto.imag == 0)
        want = p[:, i].reshape(3, 4, 10).sum(axis=(0, 2)) / np.float32(30)
        assert np.array_equal(auto.real, want.astype(np.float32))


def test_independent_numpy_and_swap_symmetry(oracle_mod):
    rng = np.random.default_rng(2)
    F, A, Ns, n_t, n_avg = 4, 6, 48, 12, 2
    volt = rng.integers(-127, 128, (F, A, Ns, 2)).astype(np.int8)
    vis = oracle_mod.correlate(volt, n_t, n_avg)
    x = volt[..., 0].astype(np.float64) + 1j * volt[..., 1].astype(np.float64)       # [F][A][Ns]
    xs = x.reshape(F // n_avg, n_avg, A, Ns // n_t, n_t)
    full = np.einsum("cfits,cfjts->tcij", xs, np.conj(xs))                           # exact: integers below 2^53
    for i in range(A):
        for j in range(i + 1):
            want = full[:, :, i, j]
            got = vis[:, :, _tri(i, j)]
            assert np.array_equal(got.real, (want.real.astype(np.float32) / np.float32(n_t * n_avg)))
            assert np.array_equal(got.imag, (want.imag.astype(np.float32) / np.float32(n_t * n_avg)))
    # swapping two inputs conjugates their cross term (S_ji = conj S_ij) and swaps their autos
    sw = volt.copy()
    sw[:, [1, 4]] = sw[:, [4, 1]]
    vis2 = oracle_mod.correlate(sw, n_t, n_avg)
    assert np.array_equal(vis2[:, :, _tri(4, 1)], np.conj(vis[:, :, _tri(4, 1)]))
    assert np.array_equal(vis2[:, :, _tri(1, 1)], vis[:, :, _tri(4, 4)])


def test_channel_averaging_is_mean_of_channels(oracle_mod):
    rng = np.random.default_rng(3)
    volt = rng.integers(-8, 8, (4, 3, 32, 2)).astype(np.int8)
    one = oracle_mod.correlate(volt, n_t=16, n_avg=1).astype(np.complex128)          # sums / 16, exact in fp32
    four = oracle_mod.correlate(volt, n_t=16, n_avg=4).astype(np.complex128)
    assert np.array_equal(four[:, 0], one.mean(axis=1))                              # exact: small integers / 64


def test_phase_steps_and_noise(oracle_mod):
    # a common signal seen with per-input phase steps of 90 degrees (exact in integers): x_a = s * i^a
    rng = np.random.default_rng(4)
    Ns, A = 4000, 4
    s = rng.integers(-5, 6, Ns) + 1j * rng.integers(-5, 6, Ns)
    x = np.stack([s * (1j ** a) for a in range(A)])
    volt = np.stack([x.real, x.imag], axis=-1).astype(np.int8)[None]
    vis = oracle_mod.correlate(volt, n_t=Ns, n_avg=1)[0, 0]
    p = np.mean(np.abs(s) ** 2)
    for i in range(A):
        for j in range(i + 1):
            assert vis[_tri(i, j)] == pytest.approx(p * (1j ** (i - j)), rel=1e-6)
    # independent noise: cross terms vanish as 1/sqrt(n), autos give the variance
    volt = np.clip(np.rint(rng.normal(0, 2.5, (1, 3, 20000, 2))), -8, 7).astype(np.int8)
    vis = oracle_mod.correlate(volt, n_t=20000, n_avg=1)[0, 0]
    var = (volt.astype(np.float64) ** 2).sum(axis=3).mean(axis=2)[0]
    for i in range(3):
        assert vis[_tri(i, i)].real == pytest.approx(var[i], rel=1e-6)
        for j in range(i):
            assert abs(vis[_tri(i, j)]) < 6 * np.sqrt(var[i] * var[j] / 20000)


def test_argument_checks(oracle_mod):
    volt = np.zeros((3, 2, 10, 2), np.int8)
    with pytest.raises(ValueError):
        oracle_mod.correlate(volt, n_t=4, n_avg=1)
    with pytest.raises(ValueError):
        oracle_mod.correlate(volt, n_t=5, n_avg=2)

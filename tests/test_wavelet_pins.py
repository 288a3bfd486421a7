"""Pins of the wavelet-lifting oracle (oracle/wavelet_oracle.c) to PAPER.md:191-241 (Eq. 8-11) and to the
textbook filters of the two wavelets; readings W1-W5 of DESIGN.md section 3."""
import numpy as np
import pytest


def rnd(shape, seed):
    return np.random.default_rng(seed).normal(0, 2, shape)


SHAPES = [(1, 1, 1), (1, 1, 2), (1, 1, 5), (4, 4, 4), (8, 8, 8), (5, 6, 7), (3, 1, 9), (9, 10, 17)]


@pytest.mark.parametrize("wavelet", [0, 1], ids=["haar", "legall"])
@pytest.mark.parametrize("shape", SHAPES, ids=lambda s: "x".join(map(str, s[::-1])))
def test_wv1_perfect_reconstruction(oracle, shape, wavelet):
    """"The decomposition process, mathematically reversible": inverse(forward) = identity for
    every shape (odd lengths, size-1 axes) and depth."""
    a = rnd(shape, 1)
    for L in (1, 2, 3, 4):
        w = oracle.wavelet_transform_oracle(a, wavelet, L)
        assert np.abs(oracle.wavelet_transform_oracle(w, wavelet, L, inverse=True) - a).max() < 1e-12
    assert np.array_equal(oracle.wavelet_transform_oracle(a, wavelet, 0), a)


def test_wv2_haar_by_hand(oracle):
    """Eq. 8-11: d = odd - even, c = even + d/2 = mean of the pair; level 2 on the c's at stride 2."""
    a = np.array([[[1.0, 5.0, 2.0, 8.0, 7.0]]])
    w = oracle.wavelet_transform_oracle(a, oracle.HAAR, 1)[0, 0]
    assert np.allclose(w, [3.0, 4.0, 5.0, 6.0, 7.0], atol=1e-15)           # c0 d0 c1 d1 c2(unpaired: W2)
    w = oracle.wavelet_transform_oracle(a, oracle.HAAR, 2)[0, 0]
    assert np.allclose(w, [4.0, 4.0, 2.0, 6.0, 7.0], atol=1e-15)           # level 2: d = 5 - 3, c = 4; 7 unpaired
    w = oracle.wavelet_transform_oracle(a, oracle.HAAR, 3)[0, 0]
    assert np.allclose(w, [5.5, 4.0, 2.0, 6.0, 3.0], atol=1e-15)           # level 3 pairs positions 0 and 4


def test_wv3_haar_approximation_is_the_block_mean(oracle):
    a = rnd((8, 8, 8), 2)
    for L in (1, 2, 3):
        w = oracle.wavelet_transform_oracle(a, oracle.HAAR, L)
        s = 2 ** L
        blocks = a.reshape(8 // s, s, 8 // s, s, 8 // s, s).mean(axis=(1, 3, 5))
        assert np.abs(w[::s, ::s, ::s] - blocks).max() < 1e-13


def test_wv4_legall_by_hand_and_53_taps(oracle):
    """CDF 5/3 (reading W4): predict with the mean of the two even neighbours, update with a quarter of the two
    details; equivalently the analysis filters (-1, 2, 6, 2, -1)/8 and (-1, 2, -1)/2."""
    a = np.array([[[1.0, 2.0, 4.0, 8.0, 16.0]]])
    w = oracle.wavelet_transform_oracle(a, oracle.LEGALL, 1)[0, 0]
    assert np.allclose(w, [0.75, -0.5, 3.375, -2.0, 15.0], atol=1e-15)
    b = rnd((1, 1, 32), 3)
    w = oracle.wavelet_transform_oracle(b, oracle.LEGALL, 1)[0, 0]
    x = b[0, 0]
    for i in range(2, 29, 2):                    # interior low-pass samples
        assert abs(w[i] - (-x[i - 2] + 2 * x[i - 1] + 6 * x[i] + 2 * x[i + 1] - x[i + 2]) / 8.0) < 1e-13
    for i in range(1, 31, 2):                    # high-pass samples
        assert abs(w[i] - (-x[i - 1] + 2 * x[i] - x[i + 1]) / 2.0) < 1e-13


def test_wv5_vanishing_moments(oracle):
    """Constants have zero details for both wavelets (also at the faces: symmetric extension); linear ramps have
    zero Le Gall details in the interior (two vanishing moments) but not zero Haar details."""
    c = np.full((5, 6, 7), 3.0)
    for wv in (0, 1):
        w = oracle.wavelet_transform_oracle(c, wv, 3)
        approx = np.zeros_like(c, dtype=bool)
        approx[::8, ::8, ::8] = True
        assert np.abs(w[~approx]).max() < 1e-14 and np.abs(w[approx] - 3.0).max() < 1e-14
    z, y, x = np.meshgrid(np.arange(16.0), np.arange(16.0), np.arange(16.0), indexing="ij")
    ramp = 2.0 * x - y + 0.5 * z
    w = oracle.wavelet_transform_oracle(ramp, oracle.LEGALL, 1)
    inner = w[1:13, 1:13, 1:13]
    mask = ((np.arange(1, 13)[:, None, None] % 2) | (np.arange(1, 13)[None, :, None] % 2) | (np.arange(1, 13)[None, None, :] % 2)) > 0
    assert np.abs(inner[mask]).max() < 1e-12                      # every interior coefficient that is a detail
    assert np.abs(oracle.wavelet_transform_oracle(ramp, oracle.HAAR, 1)[1:13, 1:13, 1:13][mask]).max() > 0.4


def test_wv6_threshold_bands(oracle):
    """Reading W3: detail coefficients created at level l use t_l, the approximation band t_L.  On an 8^3 cube with
    L = 3 there are 448 / 56 / 7 details of level 1 / 2 / 3 and one approximation coefficient."""
    a = rnd((8, 8, 8), 4)
    for wv in (0, 1):
        w = oracle.wavelet_transform_oracle(a, wv, 3)
        idx = np.indices((8, 8, 8))
        tz = lambda p: np.where(p == 0, 31, np.log2(np.maximum(p & -p, 1)).astype(int))
        level = np.minimum(np.minimum(tz(idx[0]), tz(idx[1])), tz(idx[2])) + 1
        assert [(level == l).sum() for l in (1, 2, 3)] == [448, 56, 7] and (level > 3).sum() == 1
        # kill level-1 details only
        big = 1e9
        out = oracle.wavelet_filter_oracle(a, wv, [big, 0.0, 0.0])
        w1 = np.where(level == 1, 0.0, w)
        assert np.abs(out - oracle.wavelet_transform_oracle(w1, wv, 3, inverse=True)).max() < 1e-12
        # kill everything but level-1 details (level 2, and level 3 + approximation through t_3)
        out = oracle.wavelet_filter_oracle(a, wv, [0.0, big, big])
        w2 = np.where(level == 1, w, 0.0)
        assert np.abs(out - oracle.wavelet_transform_oracle(w2, wv, 3, inverse=True)).max() < 1e-12


def test_wv7_filter_limits_and_units(oracle):
    a = rnd((6, 9, 10), 5)
    for wv in (0, 1):
        assert np.abs(oracle.wavelet_filter_oracle(a, wv, [0.0, 0.0, 0.0]) - a).max() < 1e-12       # t = 0: identity
        assert np.abs(oracle.wavelet_filter_oracle(a, wv, [1e9])).max() == 0.0                      # everything cut
        # thresholds are in units of rms: scaling cube and rms together scales the result
        r1 = oracle.wavelet_filter_oracle(a, wv, [0.5, 0.8, 1.1], rms=1.0)
        r4 = oracle.wavelet_filter_oracle(4.0 * a, wv, [0.5, 0.8, 1.1], rms=4.0)
        assert np.abs(r4 - 4.0 * r1).max() < 1e-12
        # hard threshold: a coefficient exactly at t*rms survives (|v| < t is cut)
    c = np.full((4, 4, 4), 2.0)
    assert np.abs(oracle.wavelet_filter_oracle(c, 0, [9.0, 2.0]) - 2.0).max() < 1e-14               # approx = 2.0 = t_L rms
    assert np.abs(oracle.wavelet_filter_oracle(c, 0, [9.0, 2.0001])).max() == 0.0
    with pytest.raises(ValueError):
        oracle.wavelet_filter_oracle(a, 0, [-1.0])


def test_wv8_separable_order_and_linearity(oracle):
    """Reading W1 (x, then y, then z per level) gives the same coefficients as any other axis order for these
    linear, separable transforms; and the transform is linear."""
    a, b = rnd((6, 7, 9), 6), rnd((6, 7, 9), 7)
    for wv in (0, 1):
        w = oracle.wavelet_transform_oracle(a, wv, 2)
        wt = oracle.wavelet_transform_oracle(a.transpose(2, 1, 0).copy(), wv, 2).transpose(2, 1, 0)
        assert np.abs(w - wt).max() < 1e-12
        lin = oracle.wavelet_transform_oracle(2.0 * a - 3.0 * b, wv, 2)
        assert np.abs(lin - (2.0 * w - 3.0 * oracle.wavelet_transform_oracle(b, wv, 2))).max() < 1e-12

"""Pins for oracle/idg_oracle.c against what the paper and the mathematics fix.

Every pin is something OTHER than the oracle's own formula retyped: closed forms,
invariants, a library routine in the linear limit, brute force with independent
index tables.  DESIGN.md section 5 lists which reading each pin holds down.
"""
import itertools
import math

import numpy as np
import pytest
from scipy import fft as sfft
from scipy import ndimage

DEF = dict(K=1.5, tau=0.0325, cx=5.0, cy=5.0, cz=5.0, rms=1.0)   # PAPER.md:187 defaults


def rnd(shape, seed=0, scale=3.0):
    return np.random.default_rng(seed).normal(0.0, scale, size=shape)


# P1 -- a constant cube is a fixed point for any parameters (differences + boundary reading R1)
@pytest.mark.parametrize("shape", [(1, 1, 1), (3, 4, 5), (7, 1, 6)])
def test_p1_constant_fixed_point(oracle, shape):
    for v in (0.0, 1.0, -7.25, 41.0):
        a = np.full(shape, v)
        out = oracle.idg_filter_oracle(a, 7, K=0.7, tau=0.0625, cx=10, cy=3, cz=0.5, rms=2.0)
        assert np.array_equal(out, a)


# P2 -- single bright voxel, one iteration: closed form (Eq. 7 by hand).
# Pins: S evaluated at the CENTRE voxel, axis <-> C_j mapping (x fastest), tau placement.
def test_p2_single_voxel_closed_form(oracle):
    K, tau, cx, cy, cz, rms, v = 1.5, 0.03, 2.0, 3.0, 5.0, 0.8, 4.0
    a = np.zeros((7, 6, 5))            # [z, y, x]
    a[3, 2, 2] = v
    out = oracle.idg_filter_oracle(a, 1, K, tau, cx, cy, cz, rms)
    exp = np.zeros_like(a)
    exp[3, 2, 2] = v * (1.0 - 2.0 * tau * (cx + cy + cz) / (1.0 + v * v / (K * K * rms * rms)))
    exp[3, 2, 1] = exp[3, 2, 3] = tau * cx * v       # neighbours have I = 0 -> S = 1
    exp[3, 1, 2] = exp[3, 3, 2] = tau * cy * v
    exp[2, 2, 2] = exp[4, 2, 2] = tau * cz * v
    np.testing.assert_allclose(out, exp, rtol=1e-15, atol=1e-16)


# P3 -- conductance-weighted increment sum vanishes each iteration; the plain sum changes for
# finite K ("does not conserve the flux scale").  Pins R1 + centre-S + the dropped
# grad S . grad I term together.
def test_p3_weighted_increment_sum(oracle):
    a = rnd((9, 8, 7), 3)
    p = dict(K=1.2, tau=0.03, cx=4.0, cy=5.0, cz=6.0, rms=1.5)
    cur = a
    for _ in range(4):
        nxt = oracle.idg_filter_oracle(cur, 1, **p)
        w = 1.0 + cur ** 2 / (p["K"] ** 2 * p["rms"] ** 2)
        terms = (nxt - cur) * w
        assert abs(terms.sum()) <= 1e-12 * np.abs(terms).sum()
        cur = nxt
    assert abs(cur.sum() - a.sum()) > 1e-3 * np.abs(a).sum() / a.size ** 0.5


# P4 -- K = +inf: voxel sum conserved (zero-flux boundary; north_star check)
def test_p4_linear_limit_conserves_sum(oracle):
    a = rnd((6, 7, 8), 4)
    cur = a
    for _ in range(5):
        cur = oracle.idg_filter_oracle(cur, 3, K=math.inf, tau=0.03, cx=5, cy=4, cz=6, rms=1.0)
        assert abs(cur.sum() - a.sum()) <= 1e-12 * np.abs(a).sum()


# P5 -- K = +inf equals n-fold scipy.ndimage.convolve with the 7-point kernel, mode='nearest'
def test_p5_linear_limit_is_heat_kernel(oracle):
    a = rnd((7, 9, 8), 5)
    tau, cx, cy, cz = 0.03, 3.0, 5.0, 6.0
    k = np.zeros((3, 3, 3))
    k[1, 1, 1] = 1.0 - 2.0 * tau * (cx + cy + cz)
    k[1, 1, 0] = k[1, 1, 2] = tau * cx
    k[1, 0, 1] = k[1, 2, 1] = tau * cy
    k[0, 1, 1] = k[2, 1, 1] = tau * cz
    ref = a
    for _ in range(6):
        ref = ndimage.convolve(ref, k, mode="nearest")
    out = oracle.idg_filter_oracle(a, 6, K=math.inf, tau=tau, cx=cx, cy=cy, cz=cz, rms=1.0)
    np.testing.assert_allclose(out, ref, rtol=0, atol=1e-13)


# P6 -- K = +inf closed form via DCT-II: pins "exactly n updates" (n vs n+1) without a loop
@pytest.mark.parametrize("n", [0, 1, 7, 20])
def test_p6_dct_closed_form(oracle, n):
    a = rnd((6, 5, 9), 6)
    tau, c = 0.0325, (5.0, 4.0, 6.0)        # (cz, cy, cx) order of array axes below
    lam = np.ones(a.shape)
    for ax, cj in zip(range(3), (c[0], c[1], c[2])):
        nj = a.shape[ax]
        s = np.sin(math.pi * np.arange(nj) / (2.0 * nj)) ** 2
        sh = [1, 1, 1]
        sh[ax] = nj
        lam = lam - 4.0 * tau * cj * s.reshape(sh)
    ref = sfft.idctn(sfft.dctn(a, type=2, norm="ortho") * lam ** n, type=2, norm="ortho")
    out = oracle.idg_filter_oracle(a, n, K=math.inf, tau=tau, cx=c[2], cy=c[1], cz=c[0], rms=1.0)
    np.testing.assert_allclose(out, ref, rtol=0, atol=1e-13)
    if n > 0:    # n+1 or n-1 updates must NOT match
        off = oracle.idg_filter_oracle(a, n + 1, K=math.inf, tau=tau, cx=c[2], cy=c[1], cz=c[0], rms=1.0)
        assert np.abs(off - ref).max() > 1e-6


# P7 -- symmetries: odd; scale covariance; axis permutation with C_j permuted; mirror flips
def test_p7_symmetries(oracle):
    a = rnd((5, 6, 7), 7)
    p = dict(K=1.5, tau=0.03, cx=3.0, cy=5.0, cz=6.0, rms=1.25)
    f = oracle.idg_filter_oracle(a, 5, **p)
    np.testing.assert_array_equal(oracle.idg_filter_oracle(-a, 5, **p), -f)
    q = dict(p, rms=p["rms"] * 8.0)
    np.testing.assert_array_equal(oracle.idg_filter_oracle(8.0 * a, 5, **q), 8.0 * f)
    # swap x and z (array axes 2 and 0) together with cx and cz
    g = oracle.idg_filter_oracle(np.ascontiguousarray(a.transpose(2, 1, 0)), 5,
                                 **dict(p, cx=p["cz"], cz=p["cx"]))
    np.testing.assert_allclose(g.transpose(2, 1, 0), f, rtol=0, atol=1e-14)
    # swap x and y
    g = oracle.idg_filter_oracle(np.ascontiguousarray(a.transpose(0, 2, 1)), 5,
                                 **dict(p, cx=p["cy"], cy=p["cx"]))
    np.testing.assert_allclose(g.transpose(0, 2, 1), f, rtol=0, atol=1e-14)
    for ax in range(3):
        g = oracle.idg_filter_oracle(np.ascontiguousarray(np.flip(a, ax)), 5, **p)
        np.testing.assert_allclose(np.flip(g, ax), f, rtol=0, atol=1e-14)


# P8 -- domain of dependence: one changed voxel reaches Manhattan distance n exactly (Jacobi,
# no hidden global coupling such as a re-estimated rms)
def test_p8_domain_of_dependence(oracle):
    a = rnd((11, 11, 11), 8)
    b = a.copy()
    b[5, 5, 5] += 1.0
    n = 3
    fa = oracle.idg_filter_oracle(a, n, **DEF)
    fb = oracle.idg_filter_oracle(b, n, **DEF)
    z, y, x = np.indices(a.shape)
    dist = abs(z - 5) + abs(y - 5) + abs(x - 5)
    changed = fa != fb
    assert not changed[dist > n].any()
    assert changed[dist == n].all()      # Gauss-Seidel or fewer sweeps would break one of the two


# P9 -- degenerate shapes: size-1 axes contribute nothing; 1x1x1 is the identity
def test_p9_degenerate_shapes(oracle):
    assert oracle.idg_filter_oracle(np.array([[[3.5]]]), 9, **DEF)[0, 0, 0] == 3.5
    line = rnd((1, 1, 13), 9)
    f = oracle.idg_filter_oracle(line, 4, **DEF)
    # 1-D scheme written independently with padding
    cur = line[0, 0].copy()
    for _ in range(4):
        pad = np.concatenate([cur[:1], cur, cur[-1:]])
        d = (pad[2:] - cur) + (pad[:-2] - cur)
        cur = cur + DEF["tau"] * DEF["cx"] * d / (1.0 + cur ** 2 / (DEF["K"] ** 2 * DEF["rms"] ** 2))
    np.testing.assert_allclose(f[0, 0], cur, rtol=0, atol=1e-14)
    # the same line laid along y and along z must use cy / cz
    p = dict(DEF, cx=1.0, cy=2.0, cz=3.0)
    fx = oracle.idg_filter_oracle(line, 4, **dict(p, cx=2.0))
    fy = oracle.idg_filter_oracle(line.reshape(1, 13, 1), 4, **p)
    np.testing.assert_allclose(fy.ravel(), fx.ravel(), rtol=0, atol=1e-14)
    fx = oracle.idg_filter_oracle(line, 4, **dict(p, cx=3.0))
    fz = oracle.idg_filter_oracle(line.reshape(13, 1, 1), 4, **p)
    np.testing.assert_allclose(fz.ravel(), fx.ravel(), rtol=0, atol=1e-14)


# P10 -- brute force on 4x4x4 and 5x6x7 with explicit neighbour tables (no padding, no slicing)
def _brute(a, n, K, tau, cx, cy, cz, rms):
    nz, ny, nx = a.shape
    cur = {k: float(a[k]) for k in itertools.product(range(nz), range(ny), range(nx))}
    for _ in range(n):
        new = {}
        for (z, y, x), c in cur.items():
            acc = 0.0
            for (dz, dy, dx, w) in ((0, 0, 1, cx), (0, 0, -1, cx), (0, 1, 0, cy),
                                    (0, -1, 0, cy), (1, 0, 0, cz), (-1, 0, 0, cz)):
                nb = cur.get((z + dz, y + dy, x + dx))     # missing key = outside the cube
                if nb is not None:
                    acc += w * (nb - c)
            new[(z, y, x)] = c + tau * acc / (1.0 + c * c / (K * K * rms * rms))
        cur = new
    out = np.empty_like(a)
    for k, v in cur.items():
        out[k] = v
    return out


@pytest.mark.parametrize("shape,n", [((4, 4, 4), 1), ((4, 4, 4), 2), ((7, 6, 5), 2), ((2, 1, 3), 3)])
def test_p10_brute_force(oracle, shape, n):
    a = rnd(shape, 10)
    p = dict(K=0.9, tau=0.04, cx=2.0, cy=5.0, cz=7.0, rms=1.3)
    np.testing.assert_allclose(oracle.idg_filter_oracle(a, n, **p), _brute(a, n, **p), rtol=0, atol=1e-14)


# P11 -- Markov: f(I, n+m) == f(f(I, n), m)
def test_p11_markov(oracle):
    a = rnd((6, 7, 8), 11)
    f = oracle.idg_filter_oracle(a, 9, **DEF)
    g = oracle.idg_filter_oracle(oracle.idg_filter_oracle(a, 4, **DEF), 5, **DEF)
    np.testing.assert_array_equal(f, g)


# Soft trend from the paper: smoothing reduces the noise rms, more for larger K
def test_noise_is_smoothed_more_for_larger_k(oracle):
    a = np.random.default_rng(12).normal(0, 1, (16, 16, 16))
    s = [oracle.idg_filter_oracle(a, 20, **dict(DEF, K=K)).std() for K in (0.5, 1.5, 10.0)]
    assert s[0] > s[1] > s[2] and s[2] < 0.5


def test_threads_do_not_change_results(oracle):
    a = rnd((12, 9, 10), 13)
    oracle.set_threads(1)
    f1 = oracle.idg_filter_oracle(a, 6, **DEF)
    oracle.set_threads(4)
    f4 = oracle.idg_filter_oracle(a, 6, **DEF)
    np.testing.assert_array_equal(f1, f4)


def test_into_variant_is_the_same_routine(oracle):
    """idg_filter_oracle_into (caller-owned fp64 buffers; bench.py times it) returns bit for bit what
    idg_filter_oracle returns, leaves its input untouched, and rejects buffers of the wrong kind."""
    rng = np.random.default_rng(12)
    a = rng.normal(0, 2, (6, 7, 9)).astype(np.float32)
    a64 = a.astype(np.float64)
    keep = a64.copy()
    out, scratch = np.empty_like(a64), np.empty_like(a64)
    for n in (0, 1, 4, 7):
        got = oracle.idg_filter_oracle_into(a64, n, out, scratch, K=1.5, tau=0.03, cx=5.0, cy=4.0, cz=6.0, rms=2.0)
        assert got is out and np.array_equal(out, oracle.idg_filter_oracle(a, n, K=1.5, tau=0.03, cx=5.0, cy=4.0, cz=6.0, rms=2.0))
        assert np.array_equal(a64, keep)
    with pytest.raises(ValueError):
        oracle.idg_filter_oracle_into(a64, 1, out.astype(np.float32), scratch)
    with pytest.raises(ValueError):
        oracle.idg_filter_oracle_into(a64, 1, out[:, :, :8], scratch)

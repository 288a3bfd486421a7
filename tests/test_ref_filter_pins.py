"""Pins of the box / Gaussian reference-filter oracles (oracle/ref_filters_oracle.c) to what the
paper and the mathematics fix (Eq. 1-3; readings F1-F5 of DESIGN.md section 3).

The paper prints no worked example for these filters, so the pins are closed forms, invariants,
brute force on tiny inputs and the special cases that reduce to a library routine.
"""
import itertools
import math

import numpy as np
import pytest
import scipy.ndimage as ndi

S2F = 2.0 * math.sqrt(2.0 * math.log(2.0))       # Eq. 2: FWHM = S2F * sigma


@pytest.fixture(scope="module")
def cube():
    rng = np.random.default_rng(77)
    return rng.normal(0.0, 1.0, (7, 9, 11)) + 5.0 * (rng.random((7, 9, 11)) < 0.05)


# ------------------------------------------------------------------ box filter

def test_b1_constant_cube_is_a_fixed_point(oracle):
    a = np.full((4, 5, 6), 3.25)
    assert np.array_equal(oracle.box_filter_oracle(a, 3, 5, 7), a)


def test_b2_width_one_is_the_identity(oracle, cube):
    assert np.array_equal(oracle.box_filter_oracle(cube, 1, 1, 1), cube)


def test_b3_interior_impulse_gives_the_box_with_the_right_axes(oracle):
    """"Mean value of its neighbours, including itself": an impulse v becomes the
    value v/(Nx Ny Nz) on an Nx x Ny x Nz block -- Nx along x (fastest axis), Nz along z."""
    a = np.zeros((15, 13, 11))
    a[7, 6, 5] = 2.0
    out = oracle.box_filter_oracle(a, 3, 5, 7)
    expect = np.zeros_like(a)
    expect[7 - 3:7 + 4, 6 - 2:6 + 3, 5 - 1:5 + 2] = 2.0 / (3 * 5 * 7)
    assert np.allclose(out, expect, rtol=0, atol=1e-16)


def test_b4_brute_force_with_explicit_clamping(oracle):
    rng = np.random.default_rng(3)
    a = rng.normal(size=(3, 4, 5))
    wx, wy, wz = 3, 1, 5
    out = oracle.box_filter_oracle(a, wx, wy, wz)
    for z, y, x in itertools.product(range(3), range(4), range(5)):
        vals = [a[min(max(z + k, 0), 2), min(max(y + j, 0), 3), min(max(x + i, 0), 4)]
                for k in range(-2, 3) for j in range(0, 1) for i in range(-1, 2)]
        assert abs(out[z, y, x] - sum(vals) / 15.0) < 1e-14


def test_b5_equals_library_uniform_filter(oracle, cube):
    for w in ((3, 3, 3), (3, 5, 5), (7, 1, 9), (9, 9, 9)):
        ref = ndi.uniform_filter(cube, size=(w[2], w[1], w[0]), mode="nearest")
        assert np.abs(oracle.box_filter_oracle(cube, *w) - ref).max() < 1e-13


def test_b6_even_or_nonpositive_widths_are_rejected(oracle, cube):
    for w in ((2, 3, 3), (3, 0, 3), (3, 3, -1)):
        with pytest.raises(ValueError):
            oracle.box_filter_oracle(cube, *w)


# ------------------------------------------------------------------ Gaussian kernel (Eq. 1-3)

def test_g1_unit_sum_and_support(oracle):
    """Reading F2 (A normalises the sampled kernel) and F3 (r_j = floor(3 sigma_j + 1/2))."""
    for fwhm in ((3, 3, 3), (2, 3, 3), (7, 3, 3), (1, 5, 7), (0, 3, 0)):
        k = oracle.gaussian_kernel_oracle(fwhm)
        assert abs(k.sum() - 1.0) < 1e-14
        r = [int(math.floor(3.0 * f / S2F + 0.5)) for f in fwhm]
        assert k.shape == (2 * r[2] + 1, 2 * r[1] + 1, 2 * r[0] + 1)
    assert oracle.gaussian_radii_oracle((3, 3, 3)) == (4, 4, 4)       # sigma = 1.274 -> 3 sigma = 3.82
    assert oracle.gaussian_radii_oracle((7, 3, 2)) == (9, 4, 3)


def test_g2_half_maximum_at_half_the_fwhm(oracle):
    """Eq. 2: the kernel falls to one half at |x| = FWHM/2 (FWHM even -> a sampled offset)."""
    k = oracle.gaussian_kernel_oracle((4, 6, 8))
    c = tuple(s // 2 for s in k.shape)
    k0 = k[c]
    assert abs(k[c[0], c[1], c[2] + 2] / k0 - 0.5) < 1e-14       # x: FWHM 4
    assert abs(k[c[0], c[1] + 3, c[2]] / k0 - 0.5) < 1e-14       # y: FWHM 6
    assert abs(k[c[0] + 4, c[1], c[2]] / k0 - 0.5) < 1e-14       # z: FWHM 8


def test_g3_eq1_values_by_hand(oracle):
    """Eq. 1 pointwise: K(p)/K(0) = exp(-(px^2/2sx^2 + py^2/2sy^2 + pz^2/2sz^2))."""
    fwhm = (2.0, 3.0, 5.0)
    s = [f / S2F for f in fwhm]
    k = oracle.gaussian_kernel_oracle(fwhm)
    rz, ry, rx = (n // 2 for n in k.shape)
    for pz, py, px in ((0, 0, 1), (0, 1, 0), (1, 0, 0), (2, -1, 1), (-3, 2, -2)):
        want = math.exp(-(px * px / (2 * s[0] ** 2) + py * py / (2 * s[1] ** 2) + pz * pz / (2 * s[2] ** 2)))
        assert abs(k[rz + pz, ry + py, rx + px] / k[rz, ry, rx] - want) < 1e-14


def test_g4_rotation_closed_forms(oracle):
    """Eq. 3 with right-handed matrices and R = Rz Ry Rx (reading F4)."""
    fwhm = (7.0, 3.0, 2.0)
    s = [f / S2F for f in fwhm]

    def ratio(k, p):            # p = (px, py, pz)
        r = k.shape[0] // 2
        return k[r + p[2], r + p[1], r + p[0]] / k[r, r, r]

    def gauss(q, sig):
        return math.exp(-sum(q[i] ** 2 / (2 * sig[i] ** 2) for i in range(3)))

    pts = [(1, 0, 0), (0, 2, 0), (0, 0, 3), (2, -1, 1), (-3, 4, 2)]
    # a quarter turn about z carries the x axis of G onto y
    k = oracle.gaussian_kernel_oracle(fwhm, (0, 0, 90))
    for p in pts:
        assert abs(ratio(k, p) - gauss(p, (s[1], s[0], s[2]))) < 1e-12
    # order of the product: Rx(90) first, then Rz(90): G's axes (x, y, z) end up along (y, z, x)
    k = oracle.gaussian_kernel_oracle(fwhm, (90, 0, 90))
    for p in pts:
        assert abs(ratio(k, p) - gauss(p, (s[2], s[0], s[1]))) < 1e-12
    # sense of rotation: +45 deg about z puts the long axis along (1, 1, 0), not (1, -1, 0)
    k = oracle.gaussian_kernel_oracle(fwhm, (0, 0, 45))
    assert ratio(k, (3, 3, 0)) > 10 * ratio(k, (3, -3, 0))
    assert abs(ratio(k, (3, 3, 0)) - math.exp(-18.0 / (2 * s[0] ** 2))) < 1e-12
    # +30 deg about y: R e_x = (cos, 0, -sin)
    k = oracle.gaussian_kernel_oracle(fwhm, (0, 30, 0))
    assert ratio(k, (4, 0, -2)) > ratio(k, (4, 0, 2))
    # full turns and an in-plane isotropic kernel do not depend on the angle
    k0 = oracle.gaussian_kernel_oracle((5, 5, 2), (0, 0, 1e-300))
    assert np.abs(oracle.gaussian_kernel_oracle((5, 5, 2), (0, 0, 33)) - k0).max() < 1e-15
    assert np.abs(oracle.gaussian_kernel_oracle(fwhm, (360, 0, 180)) -
                  oracle.gaussian_kernel_oracle(fwhm, (0, 0, 180))).max() < 1e-15


def test_g5_second_moments_rotate_with_the_kernel(oracle):
    """Covariance of the sampled kernel ~ R diag(s^2) R^T (up to the truncation at 3 sigma)."""
    fwhm, theta = (8.0, 3.0, 2.0), (40.0, -35.0, 60.0)
    s2 = np.array([(f / S2F) ** 2 for f in fwhm])
    k = oracle.gaussian_kernel_oracle(fwhm, theta)
    r = k.shape[0] // 2
    g = np.arange(-r, r + 1, dtype=float)
    Z, Y, X = np.meshgrid(g, g, g, indexing="ij")
    P = np.stack([X, Y, Z])
    cov = np.einsum("azyx,bzyx,zyx->ab", P, P, k)
    t = np.radians(theta)
    Rx = np.array([[1, 0, 0], [0, math.cos(t[0]), -math.sin(t[0])], [0, math.sin(t[0]), math.cos(t[0])]])
    Ry = np.array([[math.cos(t[1]), 0, math.sin(t[1])], [0, 1, 0], [-math.sin(t[1]), 0, math.cos(t[1])]])
    Rz = np.array([[math.cos(t[2]), -math.sin(t[2]), 0], [math.sin(t[2]), math.cos(t[2]), 0], [0, 0, 1]])
    R = Rz @ Ry @ Rx
    want = R @ np.diag(s2) @ R.T
    assert np.abs(cov - want).max() < 0.01 * s2.max()
    # a wrong order (Rx Ry Rz) or a transposed R would miss by far more than the truncation error
    for bad in (Rx @ Ry @ Rz, R.T):
        assert np.abs(cov - bad @ np.diag(s2) @ bad.T).max() > 0.2 * s2.max()


# ------------------------------------------------------------------ Gaussian filter

def test_g6_constant_cube_and_impulse(oracle):
    a = np.full((5, 6, 7), -1.5)
    # 1e-13, not 1e-15: the direct sum adds 343 fp64 products (r = 3) of unit-sum weights, which do not add up to exactly 1; its
    # rounding (summation order, a few tens of ulp of 1.5) is a few 1e-15..1e-14 -- a property of fp64 summation, not of the filter
    assert np.abs(oracle.gaussian_filter_oracle(a, (3, 3, 3)) - a).max() < 1e-13
    a = np.zeros((21, 21, 21))
    a[10, 10, 10] = 3.0
    for theta in ((0, 0, 0), (15, 40, -70)):
        k = oracle.gaussian_kernel_oracle((5, 3, 2), theta)
        out = oracle.gaussian_filter_oracle(a, (5, 3, 2), theta)
        rz, ry, rx = (n // 2 for n in k.shape)
        got = out[10 - rz:11 + rz, 10 - ry:11 + ry, 10 - rx:11 + rx]
        assert np.abs(got - 3.0 * k).max() < 1e-14                 # the impulse response is the kernel (3.0 * k rounds once more than the oracle's sum of one non-zero term: a few ulp of 0.1)
        assert abs(out.sum() - 3.0) < 1e-13


def test_g7_axis_aligned_equals_library_gaussian_filter(oracle, cube):
    """theta = 0: the 3-D sum equals three 1-D library passes with sigma from Eq. 2,
    truncate = 3 (radius int(3 sigma + 1/2), reading F3) and mode='nearest' (reading F1)."""
    for fwhm in ((3, 3, 3), (2, 3, 3), (7, 3, 3), (1, 5, 3)):
        sig = [f / S2F for f in fwhm]
        ref = ndi.gaussian_filter(cube, sigma=(sig[2], sig[1], sig[0]), mode="nearest", truncate=3.0)
        assert np.abs(oracle.gaussian_filter_oracle(cube, fwhm) - ref).max() < 1e-13


def test_g8_rotated_filter_by_brute_force(oracle):
    rng = np.random.default_rng(5)
    a = rng.normal(size=(6, 5, 7))
    fwhm, theta = (3.0, 2.0, 1.5), (25.0, 10.0, -40.0)
    k = oracle.gaussian_kernel_oracle(fwhm, theta)
    r = k.shape[0] // 2
    out = oracle.gaussian_filter_oracle(a, fwhm, theta)
    pad = np.pad(a, r, mode="edge")
    ref = ndi.correlate(pad, k[::-1, ::-1, ::-1], mode="constant")[r:-r, r:-r, r:-r]
    assert np.abs(out - ref).max() < 1e-13
    for z, y, x in ((0, 0, 0), (5, 4, 6), (2, 3, 1)):
        s = 0.0
        for kz, ky, kx in itertools.product(range(-r, r + 1), repeat=3):
            s += k[r + kz, r + ky, r + kx] * a[min(max(z - kz, 0), 5), min(max(y - ky, 0), 4), min(max(x - kx, 0), 6)]
        assert abs(out[z, y, x] - s) < 1e-13


def test_g9_linear_ramp_is_reproduced_in_the_interior(oracle):
    """A unit-sum even kernel reproduces linear functions away from the faces."""
    z, y, x = np.meshgrid(np.arange(30.0), np.arange(30.0), np.arange(30.0), indexing="ij")
    a = 0.5 * x - 0.25 * y + 2.0 * z + 1.0
    out = oracle.gaussian_filter_oracle(a, (4, 3, 2), (30, 20, 10))
    r = oracle.gaussian_radii_oracle((4, 3, 2), (30, 20, 10))[0]
    c = slice(r, 30 - r)
    assert np.abs(out[c, c, c] - a[c, c, c]).max() < 1e-12


def test_g10_invalid_parameters(oracle, cube):
    with pytest.raises(ValueError):
        oracle.gaussian_filter_oracle(cube, (-1, 3, 3))
    with pytest.raises(ValueError):
        oracle.gaussian_filter_oracle(cube, (0, 3, 3), (0, 0, 10))      # F5
    assert np.array_equal(oracle.gaussian_filter_oracle(cube, (0, 0, 0)), cube)

"""Pins of the quality-diagnostics oracle (oracle/quality_oracle.py) to PAPER.md:247-278 (Eq. 12-16)
and PAPER.md:344-355 (Eq. 17-18): a hand-computed example, closed forms and invariants.  The paper's
printed F-values (Tables 1-4) need its data cubes, which are not in the container: no pin by printed
values."""
import itertools
import math

import numpy as np
import pytest


@pytest.fixture(scope="module")
def Q():
    from oracle import quality_oracle
    return quality_oracle


def test_q1_hand_computed_example(Q):
    """2x2x2 cube, rms_o = 1 (threshold 3), rms_f = 0.5 (threshold 1.5); worked out by hand."""
    o = np.array([[[4.0, 1.0], [3.0, -5.0]], [[2.9, 0.0], [10.0, 2.0]]], dtype=np.float32)
    f = np.array([[[2.0, 1.6], [1.4, 0.0]], [[1.5, 0.0], [5.0, 1.49]]], dtype=np.float32)
    m = np.array([[[3.0, 1.0], [2.0, 0.0]], [[2.0, 0.0], [9.0, 1.0]]], dtype=np.float32)
    s = Q.mask_sums_oracle(o, f, m, 3.0, 1.5)
    # M_o = {4, 3, 10}: S_oo = 17, N_o = 3.  M_f = {2.0, 1.6, 1.5, 5.0}: I_o there = 4, 1, 2.9, 10
    assert s["N_o"] == 3 and s["N_f"] == 4 and s["n_roi"] == 8
    assert s["S_oo"] == pytest.approx(17.0, abs=1e-12)
    assert s["S_of"] == pytest.approx(4.0 + 1.0 + float(np.float32(2.9)) + 10.0, abs=1e-12)
    assert s["S_mf"] == pytest.approx(3.0 + 1.0 + 2.0 + 9.0, abs=1e-12) and s["S_m"] == pytest.approx(18.0)
    q = Q.quality_oracle(s, 1.0, 0.5)
    assert q["F"] == pytest.approx(s["S_of"] / 17.0, rel=1e-15)                        # Eq. 12
    sig_of, sig_oo = math.sqrt(4) * 0.5, math.sqrt(3) * 1.0                            # Eq. 16
    want = math.sqrt(sig_of ** 2 / 17.0 ** 2 + s["S_of"] ** 2 * sig_oo ** 2 / 17.0 ** 4)
    assert q["sigma_F"] == pytest.approx(want, rel=1e-15)                              # Eq. 15
    assert q["F_M"] == pytest.approx(15.0 / 18.0, rel=1e-15)                           # Eq. 17


def test_q2_threshold_is_inclusive_and_nan_never_passes(Q):
    """Eq. 14: M = 1 if I >= 3 rms (">=", not ">"); blank (NaN) voxels are outside every mask."""
    o = np.array([[[3.0, np.nextafter(np.float32(3.0), np.float32(0.0)), np.nan, 7.0]]], dtype=np.float32)
    s = Q.mask_sums_oracle(o, o, None, 3.0, 3.0)
    assert s["N_o"] == 2 and s["S_oo"] == 10.0 and s["S_of"] == 10.0


def test_q3_identical_cubes_give_f_one_and_error_formula_collapses(Q):
    rng = np.random.default_rng(1)
    o = (rng.normal(0, 1, (6, 7, 8)) + 6.0 * (rng.random((6, 7, 8)) < 0.2)).astype(np.float32)
    s = Q.mask_sums_oracle(o, o, None, 3.0, 3.0)
    q = Q.quality_oracle(s, 1.0, 1.0)
    assert q["F"] == 1.0
    assert q["sigma_F"] == pytest.approx(math.sqrt(2.0 * s["N_o"]) / abs(s["S_oo"]), rel=1e-14)


def test_q4_sums_are_always_over_the_original_cube(Q):
    """"the sums are always calculated on the pixel intensity values of the original data cube"
    (PAPER.md:261): changing the filtered values without changing its mask changes nothing."""
    rng = np.random.default_rng(2)
    o = rng.normal(0, 2, (5, 6, 7)).astype(np.float32)
    f = rng.normal(0, 2, (5, 6, 7)).astype(np.float32)
    g = np.where(f >= 1.0, f + 100.0, f - 100.0).astype(np.float32)       # same mask at threshold 1
    a, b = Q.mask_sums_oracle(o, f, o, 3.0, 1.0), Q.mask_sums_oracle(o, g, o, 3.0, 1.0)
    assert a == b


def test_q5_scale_invariance_and_sign(Q):
    """F, F_M are ratios: scaling both cubes, the model and the thresholds by 2^k changes nothing;
    sigma_F scales like rms / S."""
    rng = np.random.default_rng(3)
    o = (rng.normal(0, 1, (8, 9, 10)) + 5.0 * (rng.random((8, 9, 10)) < 0.1)).astype(np.float32)
    f = (0.5 * o + 0.3).astype(np.float32)
    m = np.abs(o).astype(np.float32)
    a = Q.quality_oracle(Q.mask_sums_oracle(o, f, m, 3.0, 1.2), 1.0, 0.4)
    b = Q.quality_oracle(Q.mask_sums_oracle(8 * o, 8 * f, 8 * m, 24.0, 9.6), 8.0, 3.2)
    for k in ("F", "sigma_F", "F_M"):
        assert a[k] == pytest.approx(b[k], rel=1e-14)


def test_q6_roi_by_brute_force(Q):
    rng = np.random.default_rng(4)
    o = rng.normal(0, 2, (6, 7, 9)).astype(np.float32)
    f = rng.normal(0, 1, (6, 7, 9)).astype(np.float32)
    m = rng.normal(1, 1, (6, 7, 9)).astype(np.float32)
    roi = (2, 8, 1, 5, 3, 6)                                    # x0, x1, y0, y1, z0, z1 (half open)
    s = Q.mask_sums_oracle(o, f, m, 2.0, 0.5, roi)
    S_oo = S_of = S_mf = S_m = 0.0
    N_o = N_f = n = 0
    for z, y, x in itertools.product(range(3, 6), range(1, 5), range(2, 8)):
        n += 1
        S_m += float(m[z, y, x])
        if o[z, y, x] >= np.float32(2.0):
            S_oo += float(o[z, y, x]); N_o += 1
        if f[z, y, x] >= np.float32(0.5):
            S_of += float(o[z, y, x]); S_mf += float(m[z, y, x]); N_f += 1
    assert (s["N_o"], s["N_f"], s["n_roi"]) == (N_o, N_f, n)
    for k, v in (("S_oo", S_oo), ("S_of", S_of), ("S_mf", S_mf), ("S_m", S_m)):
        assert s[k] == pytest.approx(v, abs=1e-12)
    with pytest.raises(ValueError):
        Q.mask_sums_oracle(o, f, m, 2.0, 0.5, (0, 10, 0, 7, 0, 6))


def test_q7_independent_voxels_divide_the_counts(Q):
    s = {"S_oo": 50.0, "S_of": 80.0, "N_o": 40, "N_f": 90, "S_mf": 0.0, "S_m": 0.0}
    a = Q.quality_oracle(s, 1.0, 0.5, voxels_per_beam=1.0)
    b = Q.quality_oracle(s, 1.0, 0.5, voxels_per_beam=10.0)
    assert b["sigma_F"] == pytest.approx(a["sigma_F"] / math.sqrt(10.0), rel=1e-14)
    assert math.isnan(b["F_M"]) and b["F"] == 1.6


def test_q8_rms_estimate(Q):
    rng = np.random.default_rng(5)
    a = rng.normal(0.3, 2.0, (10, 11, 12)).astype(np.float32)
    st = Q.cube_stats_oracle(a, (1, 12, 0, 11, 2, 9))
    sub = a[2:9, 0:11, 1:12].astype(np.float64)
    assert st["n"] == sub.size and st["sum"] == pytest.approx(sub.sum(), rel=1e-14)
    assert st["rms"] == pytest.approx(np.std(sub), rel=1e-12)              # library routine
    assert Q.cube_stats_oracle(np.full((3, 3, 3), 7.0, np.float32))["rms"] == 0.0


def test_q9_histogram(Q):
    """Reading Q5: equal bins over [lo, hi), fp32 bin decision, out-of-range and NaN voxels dropped."""
    a = np.array([[[-1.0, 0.0, 0.24, 0.25, 0.5, 0.99, 1.0, np.nan, 0.75, 0.7499999]]], dtype=np.float32)
    h = Q.histogram_oracle(a, 0.0, 1.0, 4)
    assert h.tolist() == [2, 1, 2, 2]                      # [0,.25): 0, .24 | [.25,.5): .25 | [.5,.75): .5, .7499999 | [.75,1): .99, .75
    assert Q.histogram_oracle(a, 0.0, 1.0, 4, mask_thr=0.5).tolist() == [0, 0, 2, 2]
    rng = np.random.default_rng(9)
    b = rng.normal(0, 1, (6, 7, 8)).astype(np.float32)
    h = Q.histogram_oracle(b, -4.0, 4.0, 64, roi=(1, 7, 0, 7, 2, 6))
    sub = b[2:6, 0:7, 1:7]
    ref, _ = np.histogram(sub, bins=64, range=(-4.0, 4.0))           # library routine (bins exactly representable)
    inside = ((sub >= -4.0) & (sub < 4.0)).sum()
    assert h.sum() == inside and np.array_equal(h, ref)
    with pytest.raises(ValueError):
        Q.histogram_oracle(b, 1.0, 1.0, 4)

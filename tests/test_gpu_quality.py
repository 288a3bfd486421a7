"""GPU parity of the quality diagnostics (Eq. 12-18): idg_mask_sums / idg_cube_stats through the
C ABI against oracle/quality_oracle.py.  Mask populations and the ROI size are integers: bit-exact.
Sums are fp64 accumulations of the same fp32 values in a different order: relative 1e-12."""
import math

import numpy as np
import pytest

torch = pytest.importorskip("torch")

REL = 1e-12


@pytest.fixture(scope="module")
def B():
    from paper_1609_03782_b200 import binding
    binding.lib()
    return binding


@pytest.fixture(scope="module")
def Q():
    from oracle import quality_oracle
    return quality_oracle


def check(B, Q, o, f, m, thr_o, thr_f, roi):
    t = lambda a: None if a is None else torch.from_numpy(a).cuda()
    s = B.idg_mask_sums(t(o), t(f), t(m), thr_o, thr_f, roi).cpu().numpy()
    ref = Q.mask_sums_oracle(o, f, m, thr_o, thr_f, roi)
    got = dict(zip(B.SUM_KEYS, s))
    for k in ("N_o", "N_f", "n_roi"):
        assert got[k] == ref[k], k                                   # integers: exact
    scale = float(np.abs(o.astype(np.float64)).sum()) + 1.0
    for k in ("S_oo", "S_of", "S_mf", "S_m"):
        assert abs(got[k] - ref[k]) <= REL * scale, k
    assert s[7] == 0.0
    return got, ref


@pytest.mark.gpu
@pytest.mark.parametrize("shape", [(1, 1, 1), (3, 5, 7), (9, 33, 64), (17, 40, 132), (6, 50, 100), (5, 9, 259)],
                         ids=lambda s: "x".join(map(str, s[::-1])))
@pytest.mark.parametrize("with_model", [False, True], ids=["nomodel", "model"])
def test_mask_sums(B, Q, shape, with_model):
    rng = np.random.default_rng(sum(shape))
    o = (rng.normal(0, 1, shape) + 6.0 * (rng.random(shape) < 0.1)).astype(np.float32)
    f = (0.6 * o + rng.normal(0, 0.2, shape)).astype(np.float32)
    m = np.abs(rng.normal(0, 1, shape)).astype(np.float32) if with_model else None
    o.flat[0] = np.float32(3.0)                    # exactly on the threshold: must be inside (>=)
    nz, ny, nx = shape
    rois = [None, (0, nx, 0, ny, 0, nz), (nx // 3, nx - nx // 4, ny // 4, ny, nz // 2, nz), (1 % nx, nx, 0, ny, 0, nz),
            (0, 0, 0, ny, 0, nz)]
    for roi in rois:
        check(B, Q, o, f, m, 3.0, 1.2, roi)


@pytest.mark.gpu
def test_quality_on_a_filtered_config0_cube(B, Q, oracle):
    """The paper's use: F, sigma_F and F_M of an IDG-filtered ModelB-like cube over a ROI around the tail."""
    from paper_1609_03782_b200 import synth
    c = synth.modelb_like(seed=1000, snr=32.0)
    t = torch.from_numpy(c.data).cuda()
    filt = B.idg_filter(t, 20, B.Params())
    st = B.idg_cube_stats(filt, (0, 100, 0, 100, 0, 8)).cpu().numpy()      # signal-free channels
    ref = Q.cube_stats_oracle(filt.cpu().numpy(), (0, 100, 0, 100, 0, 8))
    assert st[0] == ref["n"] and abs(st[1] - ref["sum"]) <= 1e-9 and abs(st[2] - ref["sumsq"]) <= 1e-9
    rms_f = B.idg_stats_rms(st)[1]
    assert rms_f == pytest.approx(ref["rms"], rel=1e-9) and rms_f < 0.7 * c.rms    # the filter lowers the noise
    model = torch.from_numpy(c.model).cuda() if getattr(c, "model", None) is not None else None
    roi = (10, 90, 10, 90, 10, 60)
    thr_f = float(np.float32(3.0 * rms_f))
    sums = B.idg_mask_sums(t, filt, model, 3.0 * c.rms, thr_f, roi).cpu().numpy()
    want = Q.mask_sums_oracle(c.data, filt.cpu().numpy(), None if model is None else c.model, 3.0 * c.rms, thr_f, roi)
    assert sums[2] == want["N_o"] and sums[3] == want["N_f"]
    q = B.idg_quality(sums, c.rms, rms_f)
    qr = Q.quality_oracle(want, c.rms, rms_f)
    for k in ("F", "sigma_F") + (("F_M",) if model is not None else ()):
        assert q[k] == pytest.approx(qr[k], rel=1e-10)
    assert q["F"] > 1.0                     # more signal above 3 rms after adaptive smoothing


@pytest.mark.gpu
@pytest.mark.parametrize("shape", [(1, 1, 1), (3, 5, 7), (17, 40, 132), (6, 50, 100)], ids=lambda s: "x".join(map(str, s[::-1])))
def test_histogram_is_bit_exact(B, Q, shape):
    """Integer work: every count must equal the oracle's (the bin is decided in fp32 on both sides)."""
    rng = np.random.default_rng(sum(shape) + 3)
    a = (rng.normal(0, 1, shape) + 6.0 * (rng.random(shape) < 0.1)).astype(np.float32)
    a.flat[0] = np.float32(-4.0)                      # on the lower edge: counted;  upper edge: not
    if a.size > 1:
        a.flat[1] = np.float32(4.0)
    t = torch.from_numpy(a).cuda()
    nz, ny, nx = shape
    for lo, hi, nb, roi, thr in ((-4.0, 4.0, 64, None, None), (-0.3, 7.1, 37, None, None), (-4.0, 4.0, 1, None, None),
                                 (0.0, 10.0, 1000, (nx // 3, nx, 0, ny, nz // 2, nz), None), (-4.0, 4.0, 64, None, 0.5)):
        got = B.idg_histogram(t, lo, hi, nb, roi, thr).cpu().numpy()
        assert np.array_equal(got, Q.histogram_oracle(a, lo, hi, nb, roi, thr)), (lo, hi, nb, roi, thr)


@pytest.mark.gpu
def test_argument_errors(B):
    a = torch.zeros((4, 5, 8), device="cuda")
    with pytest.raises(B.IdgError) as e:
        B.idg_mask_sums(a, a, None, 3.0, 3.0, (0, 9, 0, 5, 0, 4))
    assert e.value.status == -2
    with pytest.raises(B.IdgError) as e:
        B.idg_mask_sums(a, a, None, float("nan"), 3.0)
    assert e.value.status == -4
    with pytest.raises(TypeError):
        B.idg_cube_stats(a.cpu())
    for lo, hi, nb in ((1.0, 1.0, 4), (0.0, 1.0, 0), (0.0, 1.0, 9000), (float("nan"), 1.0, 4)):
        with pytest.raises(B.IdgError) as e:
            B.idg_histogram(a, lo, hi, nb)
        assert e.value.status == -4


def test_idg_quality_host_formulas(B, Q):
    """Host-only entry point (no GPU needed): Eq. 12, 15-17 against the oracle and by hand."""
    sums = [17.0, 17.9, 3.0, 4.0, 15.0, 18.0, 8.0, 0.0]
    q = B.idg_quality(sums, 1.0, 0.5)
    ref = Q.quality_oracle(dict(zip(B.SUM_KEYS, sums)), 1.0, 0.5)
    for k in ("F", "sigma_F", "F_M"):
        assert q[k] == pytest.approx(ref[k], rel=1e-15)
    assert q["F"] == pytest.approx(17.9 / 17.0) and q["F_M"] == pytest.approx(15.0 / 18.0)
    q = B.idg_quality([0.0] * 8, 1.0, 1.0)
    assert all(math.isnan(v) for v in q.values())
    with pytest.raises(B.IdgError):
        B.idg_quality(sums, 0.0, 1.0)
    with pytest.raises(B.IdgError):
        B.idg_quality(sums, 1.0, 1.0, voxels_per_beam=0.5)


@pytest.mark.gpu
def test_parameter_exploration_runs_and_behaves_like_the_paper(B):
    """explore.py: the config-1 sweep with on-device diagnostics.  Soft checks from the paper: smoothing lowers the
    noise monotonically with n, and the adaptive filter lifts faint signal above 3 rms (F > 1)
    while recovering a growing share of the model flux (F_M grows with F)."""
    from paper_1609_03782_b200 import explore
    rows = explore.explore(snr=22.0, seed=1001, nmax=20, ks=(1.5,), report=(1, 5, 10, 20))
    assert [r["n"] for r in rows] == [1, 5, 10, 20]
    rms = [r["rms_f"] for r in rows]
    assert all(a > b for a, b in zip(rms, rms[1:])) and rms[-1] < 0.5
    assert rows[-1]["F"] > 1.0 and rows[-1]["F_M"] > rows[0]["F_M"] and all(r["sigma_F"] > 0 for r in rows)

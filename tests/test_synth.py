"""The synthetic generator: deterministic, rms 1, beam-correlated in (y, x) only."""
import numpy as np

from paper_1609_03782_b200 import synth


def test_noise_statistics_and_correlation():
    n = synth.beam_noise((24, 96, 96), 5).astype(np.float64)
    assert abs(n.std() - 1.0) < 1e-3 and abs(n.mean()) < 0.05
    cx = (n[:, :, 1:] * n[:, :, :-1]).mean()
    cy = (n[:, 1:, :] * n[:, :-1, :]).mean()
    cz = (n[1:] * n[:-1]).mean()
    # Gaussian beam autocorrelation at lag 1: exp(-1/(4 sigma^2))
    sx, sy = 4.4 * synth.FWHM_TO_SIGMA, 3.5 * synth.FWHM_TO_SIGMA
    assert abs(cx - np.exp(-1 / (4 * sx * sx))) < 0.03
    assert abs(cy - np.exp(-1 / (4 * sy * sy))) < 0.03
    assert abs(cz) < 0.06                       # uncorrelated in velocity


def test_modelb_like_is_deterministic_and_scaled():
    a = synth.modelb_like(seed=1000, snr=32.0, threads=1)
    b = synth.modelb_like(seed=1000, snr=32.0, threads=3)
    assert np.array_equal(a.data, b.data) and a.data.dtype == np.float32
    assert a.data.shape == (67, 100, 100)
    assert abs(float(a.model.max()) - 32.0) < 1e-3
    assert a.peak < 64.0
    c = synth.modelb_like(seed=1001, snr=22.0)
    assert not np.array_equal(a.data, c.data)


def test_batch_params_are_stable():
    p = synth.batch_params(256, 4000)
    assert p.shape == (256, 6)
    assert np.all(p[:, 1] * (p[:, 2] + p[:, 3] + p[:, 4]) <= 0.5 + 1e-6)
    assert set(np.unique(p[:, 0])) <= set(np.float32(synth.K_SWEEP))


def test_survey_field_small():
    c = synth.survey_field((48, 160, 160), seed=7, n_discs=2, thick=True)
    assert c.data.shape == (48, 160, 160) and np.isfinite(c.data).all()
    assert c.peak > 4.0

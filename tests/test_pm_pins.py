"""Pins of the gradient-driven (Perona-Malik, Eq. 4-5) variant of the oracle
(readings P1-P3 of DESIGN.md section 3).  The paper prints no worked example for it."""
import itertools

import numpy as np
import pytest
import scipy.ndimage as ndi


def rnd(shape, seed, spikes=True):
    rng = np.random.default_rng(seed)
    a = rng.normal(0, 1, shape)
    return a + (6.0 * (rng.random(shape) < 0.05) if spikes else 0.0)


def test_pm1_constant_and_linear_limit(oracle):
    """A constant cube is a fixed point; K = inf is the same linear diffusion as for Eq. 7."""
    a = np.full((4, 5, 6), 2.5)
    assert np.array_equal(oracle.pm_filter_oracle(a, 7), a)
    b = rnd((6, 7, 8), 1)
    assert np.array_equal(oracle.pm_filter_oracle(b, 5, K=np.inf), oracle.idg_filter_oracle(b, 5, K=np.inf))


def test_pm2_single_voxel_closed_form(oracle):
    """A bright voxel v in a zero cube, one step: at the voxel the central differences vanish (S = 1),
    at a face neighbour along x the gradient is v/2 along x only."""
    v, K, tau, C, rms = 8.0, 1.5, 0.02, (5.0, 4.0, 6.0), 2.0
    a = np.zeros((7, 7, 7))
    a[3, 3, 3] = v
    out = oracle.pm_filter_oracle(a, 1, K=K, tau=tau, cx=C[0], cy=C[1], cz=C[2], rms=rms)
    assert out[3, 3, 3] == pytest.approx(v * (1.0 - 2.0 * tau * sum(C)), rel=1e-15)         # S = 1 at the peak
    S = 1.0 / (1.0 + (v / 2.0) ** 2 / (K * K * rms * rms))
    assert out[3, 3, 4] == pytest.approx(tau * C[0] * v * S, rel=1e-15)
    assert out[3, 4, 3] == pytest.approx(tau * C[1] * v * S, rel=1e-15)
    assert out[2, 3, 3] == pytest.approx(tau * C[2] * v * S, rel=1e-15)
    assert out[3, 4, 4] == 0.0                                                               # no diagonal coupling
    # the intensity-driven filter differs exactly there: it damps the peak, not its neighbours
    idg = oracle.idg_filter_oracle(a, 1, K=K, tau=tau, cx=C[0], cy=C[1], cz=C[2], rms=rms)
    assert idg[3, 3, 4] == pytest.approx(tau * C[0] * v, rel=1e-15) and idg[3, 3, 3] > out[3, 3, 3]


def test_pm3_conductance_sees_differences_not_levels(oracle):
    """Eq. 5 depends on the gradient only: adding a constant offset commutes with the filter (it does
    not for Eq. 6), and a linear ramp is a fixed point in the interior whatever its slope."""
    a = rnd((6, 7, 8), 2)
    p = dict(K=1.0, tau=0.03, cx=5.0, cy=4.0, cz=6.0, rms=1.0)
    assert np.abs(oracle.pm_filter_oracle(a + 100.0, 4, **p) - (oracle.pm_filter_oracle(a, 4, **p) + 100.0)).max() < 1e-11
    assert np.abs(oracle.idg_filter_oracle(a + 100.0, 4, **p) - (oracle.idg_filter_oracle(a, 4, **p) + 100.0)).max() > 1e-3
    z, y, x = np.meshgrid(np.arange(9.0), np.arange(9.0), np.arange(9.0), indexing="ij")
    ramp = 3.0 * x - 2.0 * y + 0.5 * z
    out = oracle.pm_filter_oracle(ramp, 2, **p)
    assert np.abs(out[2:-2, 2:-2, 2:-2] - ramp[2:-2, 2:-2, 2:-2]).max() < 1e-12


def test_pm4_weighted_increment_invariant(oracle):
    """sum_v (I_{i+1} - I_i)(1 + |grad I_i|^2 / K^2 rms^2) = tau sum_v weighted Laplacian = 0 with
    replicated faces: pins the boundary, the place where S is evaluated and the 1/2 of the central
    difference (a forward difference or a missing 1/2 breaks it)."""
    a = rnd((6, 7, 8), 3)
    K, rms = 1.2, 1.5
    p = dict(K=K, tau=0.03, cx=5.0, cy=4.0, cz=6.0, rms=rms)
    pad = np.pad(a, 1, mode="edge")
    g2 = (0.25 * (pad[1:-1, 1:-1, 2:] - pad[1:-1, 1:-1, :-2]) ** 2 + 0.25 * (pad[1:-1, 2:, 1:-1] - pad[1:-1, :-2, 1:-1]) ** 2
          + 0.25 * (pad[2:, 1:-1, 1:-1] - pad[:-2, 1:-1, 1:-1]) ** 2)
    d = oracle.pm_filter_oracle(a, 1, **p) - a
    w = 1.0 + g2 / (K * K * rms * rms)
    assert abs((d * w).sum()) < 1e-12 * np.abs(d * w).sum()
    assert abs((d * (1.0 + 4.0 * g2 / (K * K * rms * rms))).sum()) > 1e-4 * np.abs(d).sum()    # without the 1/2: broken


def test_pm5_brute_force_and_symmetries(oracle):
    rng = np.random.default_rng(4)
    a = rng.normal(0, 2, (4, 5, 6))
    K, tau, C, rms = 0.8, 0.025, (5.0, 3.0, 6.0), 1.3
    out = oracle.pm_filter_oracle(a, 1, K=K, tau=tau, cx=C[0], cy=C[1], cz=C[2], rms=rms)
    cl = lambda v, n: min(max(v, 0), n - 1)
    for z, y, x in itertools.product(range(4), range(5), range(6)):
        c = a[z, y, x]
        nb = [(a[z, y, cl(x + 1, 6)], a[z, y, cl(x - 1, 6)]), (a[z, cl(y + 1, 5), x], a[z, cl(y - 1, 5), x]),
              (a[cl(z + 1, 4), y, x], a[cl(z - 1, 4), y, x])]
        lap = sum(Cj * ((p - c) + (m - c)) for Cj, (p, m) in zip(C, nb))
        g2 = sum((0.5 * (p - m)) ** 2 for p, m in nb)
        assert out[z, y, x] == pytest.approx(c + tau * lap / (1.0 + g2 / (K * K * rms * rms)), rel=1e-13, abs=1e-13)
    p = dict(K=K, tau=tau, cx=C[0], cy=C[1], cz=C[2], rms=rms)
    assert np.abs(oracle.pm_filter_oracle(-a, 3, **p) + oracle.pm_filter_oracle(a, 3, **p)).max() < 1e-13
    assert np.abs(oracle.pm_filter_oracle(a[:, :, ::-1], 3, **p) - oracle.pm_filter_oracle(a, 3, **p)[:, :, ::-1]).max() < 1e-13
    q = dict(K=K, tau=tau, cx=C[2], cy=C[1], cz=C[0], rms=rms)          # swap x <-> z with the weights
    assert np.abs(oracle.pm_filter_oracle(a.transpose(2, 1, 0), 3, **q) -
                  oracle.pm_filter_oracle(a, 3, **p).transpose(2, 1, 0)).max() < 1e-13
    assert np.abs(oracle.pm_filter_oracle(a, 5, **p) -
                  oracle.pm_filter_oracle(oracle.pm_filter_oracle(a, 2, **p), 3, **p)).max() == 0.0


def test_pm6_edges_survive_where_eq6_smooths_them(oracle):
    """The point of Eq. 5: a step edge of a bright plateau keeps its contrast."""
    a = np.zeros((5, 5, 40))
    a[:, :, 20:] = 10.0
    p = dict(K=1.0, tau=0.0325, cx=5.0, cy=5.0, cz=5.0, rms=1.0)
    pm = oracle.pm_filter_oracle(a, 20, **p)
    lin = oracle.pm_filter_oracle(a, 20, **dict(p, K=np.inf))
    assert pm[2, 2, 20] - pm[2, 2, 19] > 7.0 > 3.0 > lin[2, 2, 20] - lin[2, 2, 19]

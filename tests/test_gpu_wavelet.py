"""GPU parity of the wavelet lifting path (section 3.4, Eq. 8-11): idg_wavelet_transform and
idg_wavelet_filter through the C ABI against oracle/wavelet_oracle.c.

Transform coefficients are compared element by element (fp32 lifting against fp64: 1e-4 x rms, in
practice ~1e-6).  The filter takes a hard decision per coefficient; where the fp64 coefficient lies
within MARGIN of its threshold either decision is correct, so the test compares what is unique (all
other coefficients must follow the oracle's decision) and checks that the ambiguous ones are either
kept or cut."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TOL = 1e-4
MARGIN = 1e-4


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1609_03782_b200 import binding
    binding.lib()
    return binding


def noisy(shape, seed):
    rng = np.random.default_rng(seed)
    return (rng.normal(0, 1, shape) + 8.0 * (rng.random(shape) < 0.03)).astype(np.float32)


SHAPES = [(1, 1, 1), (1, 1, 2), (1, 1, 5), (4, 4, 4), (5, 6, 7), (3, 1, 9), (9, 10, 17), (21, 67, 100), (16, 64, 128),
          (33, 40, 130)]
IDS = lambda s: "x".join(map(str, s[::-1])) if isinstance(s, tuple) else None


def level_map(shape, levels):
    """Level (1..levels) whose threshold applies to each coefficient: trailing zero bits of the three indices."""
    def tz(n):
        p = np.arange(n)
        return np.where(p == 0, 31, np.log2(np.maximum(p & -p, 1)).astype(int)).astype(np.int8)
    z, y, x = tz(shape[0])[:, None, None], tz(shape[1])[None, :, None], tz(shape[2])[None, None, :]
    return np.minimum(np.minimum(np.minimum(z, y), x) + 1, levels)


def check_filter(oracle, a, out, wavelet, thr, rms):
    """What is unique must follow the oracle's decision; coefficients within MARGIN of their threshold may be kept or
    cut.  Returns (worst error on the unique coefficients / rms, fraction of ambiguous coefficients)."""
    L = len(thr)
    w = oracle.wavelet_transform_oracle(a, wavelet, L)                   # fp64 coefficients
    t_map = np.asarray([float(np.float32(t)) * rms for t in thr])[level_map(a.shape, L) - 1]
    ambiguous = np.abs(np.abs(w) - t_map) <= MARGIN * rms
    got = oracle.wavelet_transform_oracle(out, wavelet, L)               # coefficients the GPU kept
    want = np.where(np.abs(w) < t_map, 0.0, w)
    worst = float(np.abs(got - want)[~ambiguous].max()) / rms
    amb = got[ambiguous]
    ok = np.minimum(np.abs(amb), np.abs(amb - w[ambiguous])) <= TOL * rms
    assert ok.all()                                                      # the rest: kept or cut
    return worst, float(ambiguous.mean())


@pytest.mark.parametrize("wavelet", [0, 1], ids=["haar", "legall"])
@pytest.mark.parametrize("shape", SHAPES, ids=IDS)
def test_transform_and_inverse(B, oracle, shape, wavelet):
    a = noisy(shape, 21)
    t = torch.from_numpy(a).cuda()
    for L in (0, 1, 2, 3, 5):
        w = B.idg_wavelet_transform(t, wavelet, L)
        ref = oracle.wavelet_transform_oracle(a, wavelet, L)
        assert np.abs(w.cpu().numpy().astype(np.float64) - ref).max() <= TOL, (shape, L)
        back = B.idg_wavelet_transform(w, wavelet, L, inverse=True)
        assert float((back - t).abs().max()) <= TOL                      # reversible
        inplace = t.clone()
        B.idg_wavelet_transform(inplace, wavelet, L, out=inplace)
        assert torch.equal(inplace, w)                                   # in place == out of place


@pytest.mark.parametrize("wavelet,thr", [(0, (0.5, 0.8, 1.1)), (1, (1.0, 1.4, 1.7)), (0, (0.7,)), (1, (0.6, 1.15))],
                         ids=["haar-paper", "legall-paper", "haar-l1", "legall-l2"])
@pytest.mark.parametrize("shape", [(5, 6, 7), (9, 10, 17), (21, 67, 100), (33, 40, 130)], ids=IDS)
def test_filter(B, oracle, shape, wavelet, thr):
    """Thresholds of PAPER.md:222 (Haar 0.5/0.8/1.1, Le Gall 1/1.4/1.7 x rms) and two of the sweep."""
    rms = 1.5
    a = (noisy(shape, 22) * rms).astype(np.float32)
    out = B.idg_wavelet_filter(torch.from_numpy(a).cuda(), wavelet, thr, rms).cpu().numpy().astype(np.float64)
    worst, amb = check_filter(oracle, a, out, wavelet, thr, rms)
    assert worst <= TOL                                                  # what is unique
    if amb == 0.0:
        assert np.abs(out - oracle.wavelet_filter_oracle(a, wavelet, [float(np.float32(t)) for t in thr], rms)).max() <= TOL * rms


@pytest.mark.parametrize("wavelet,thr", [(0, (0.5, 0.8, 1.1)), (1, (1.0, 1.4, 1.7))], ids=["haar", "legall"])
def test_filter_full_size_against_the_oracle(B, oracle, parity_log, wavelet, thr):
    """configs[2] size (512 x 512 x 256), the launch configuration bench.py --filter wavelet_* times, the paper's
    thresholds: the CUDA filter against oracle/wavelet_oracle.c over the WHOLE cube, with the same
    ambiguity band at the hard threshold as the small cases (the oracle's lifting is O(N): seconds)."""
    from paper_1609_03782_b200 import synth
    c = synth.survey_field((256, 512, 512), seed=2000, n_discs=6)
    out = B.idg_wavelet_filter(torch.from_numpy(c.data).cuda(), wavelet, thr, c.rms)
    plan = B.idg_last_plan()
    out = out.cpu().numpy().astype(np.float64)
    worst, amb = check_filter(oracle, c.data, out, wavelet, thr, c.rms)
    parity_log(f"wavelet filter {('haar', 'legall')[wavelet]} 512x512x256, 3 levels", worst,
               f"whole cube, coefficients outside the ambiguity band ({amb:.2e} of them inside), {plan}")
    assert worst <= TOL


@pytest.mark.parametrize("shape", SHAPES + [(8, 8, 32), (17, 23, 77), (64, 72, 160), (21, 67, 100), (13, 30, 268),
                                            (9, 5, 12), (17, 23, 76), (3, 2, 4)], ids=IDS)
def test_haar_fused_pass_equals_per_axis_passes(B, shape):
    """The single-pass Haar filters (an 8^3 block per warp in registers where nx % 4 == 0, else 64 x 8 x 8 regions in
    shared memory; option kernel = 2 forces the latter) apply the same operations in the same order as the
    per-level, per-axis kernels: bit-identical for every shape (odd extents, blocks hanging over the faces), 1..3
    levels, in place or not."""
    a = torch.from_numpy(noisy(shape, 23)).cuda()
    for thr in ((0.7,), (0.5, 0.8), (0.5, 0.8, 1.1), (0.0, 0.0, 0.0)):
        B.idg_set_option(B.IDG_OPT_KERNEL, 1)
        try:
            ref = B.idg_wavelet_filter(a, B.WAVELET_HAAR, thr, 1.3)
            plan_ref = B.idg_last_plan()
            assert "idg_lift_kernel" in plan_ref
            B.idg_set_option(B.IDG_OPT_KERNEL, 2)
            out = B.idg_wavelet_filter(a, B.WAVELET_HAAR, thr, 1.3)
            assert "idg_haar_filter_kernel" in B.idg_last_plan()
            assert torch.equal(out, ref), (shape, thr)
        finally:
            B.idg_set_option(B.IDG_OPT_KERNEL, 0)
        out = B.idg_wavelet_filter(a, B.WAVELET_HAAR, thr, 1.3)
        assert ("idg_haar_warp_kernel" if shape[2] % 4 == 0 else "idg_haar_filter_kernel") in B.idg_last_plan()
        assert torch.equal(out, ref), (shape, thr)
        inplace = a.clone()
        B.idg_wavelet_filter(inplace, B.WAVELET_HAAR, thr, 1.3, out=inplace)
        assert torch.equal(inplace, ref)


@pytest.mark.parametrize("wavelet", [0, 1], ids=["haar", "legall"])
@pytest.mark.parametrize("shape", SHAPES + [(17, 23, 77), (64, 72, 160), (40, 300, 50)], ids=IDS)
def test_whole_line_passes_equal_two_phase_passes(B, shape, wavelet):
    """The one-pass-per-axis kernels (complete lines in shared memory) are bit-identical to the two-phase
    kernels (option kernel = 1) for the transform, its inverse and the filter."""
    a = torch.from_numpy(noisy(shape, 24)).cuda()
    for L in (1, 2, 3, 4):
        B.idg_set_option(B.IDG_OPT_KERNEL, 1)
        try:
            ref = B.idg_wavelet_transform(a, wavelet, L)
            ref_back = B.idg_wavelet_transform(ref, wavelet, L, inverse=True)
            ref_f = B.idg_wavelet_filter(a, wavelet, [0.4 + 0.3 * l for l in range(L)], 1.2)
        finally:
            B.idg_set_option(B.IDG_OPT_KERNEL, 0)
        out = B.idg_wavelet_transform(a, wavelet, L)
        assert torch.equal(out, ref), (shape, L)
        assert torch.equal(B.idg_wavelet_transform(out, wavelet, L, inverse=True), ref_back)
        assert torch.equal(B.idg_wavelet_filter(a, wavelet, [0.4 + 0.3 * l for l in range(L)], 1.2), ref_f)


@pytest.mark.parametrize("shape", SHAPES + [(17, 23, 77), (70, 35, 67), (64, 72, 160), (40, 300, 50), (131, 19, 36)],
                         ids=IDS)
def test_legall_fused_levels_equal_in_place_passes(B, shape):
    """The Le Gall filter with the three axes of a level fused (out of place, compact lattices, thresholds
    applied on load: idg_legall.cu, the default) is bit-identical to the in-place passes (option kernel = 2:
    whole lines in shared memory; 1: two phases), also when it runs in place, for tiles with ragged tails,
    odd lattice extents at every level and levels deeper than the cube."""
    a = torch.from_numpy(noisy(shape, 31)).cuda()
    for L in (1, 2, 3, 5):
        thr = [0.4 + 0.3 * l for l in range(L)]
        refs = []
        for k in (1, 2):
            B.idg_set_option(B.IDG_OPT_KERNEL, k)
            try:
                refs.append(B.idg_wavelet_filter(a, B.WAVELET_LEGALL53, thr, 1.2))
                assert "idg_lift" in B.idg_last_plan()
            finally:
                B.idg_set_option(B.IDG_OPT_KERNEL, 0)
        out = B.idg_wavelet_filter(a, B.WAVELET_LEGALL53, thr, 1.2)
        assert "idg_legall_fwd_kernel" in B.idg_last_plan() and B.idg_last_launch_count() == 2 * L
        assert torch.equal(refs[0], refs[1]) and torch.equal(out, refs[0]), (shape, L)
        inplace = a.clone()
        B.idg_wavelet_filter(inplace, B.WAVELET_LEGALL53, thr, 1.2, out=inplace)
        assert torch.equal(inplace, out)


def test_filter_limits_and_config0(B, oracle):
    from paper_1609_03782_b200 import synth
    c = synth.modelb_like(seed=1000, snr=32.0)
    t = torch.from_numpy(c.data).cuda()
    for wv in (0, 1):
        assert float((B.idg_wavelet_filter(t, wv, (0.0, 0.0, 0.0)) - t).abs().max()) <= TOL      # t = 0: identity
        assert float(B.idg_wavelet_filter(t, wv, (1e9,)).abs().max()) == 0.0                      # everything cut
    # the paper's recipe: Gaussian pre-smoothing, then the wavelet filter (FWHM 3 for the models)
    pre = B.idg_gaussian_filter(t, (3, 3, 3))
    out = B.idg_wavelet_filter(pre, B.WAVELET_HAAR, (0.5, 0.8, 1.1), c.rms)
    assert float((out == 0).float().mean()) > 0.3 and float(out.max()) > 10.0     # noise cut, bright disc kept


def test_argument_errors(B):
    a = torch.zeros((4, 5, 8), device="cuda")
    for args in ((2, (0.5,), 1.0), (0, (), 1.0), (0, (-1.0,), 1.0), (0, (0.5,), 0.0), (1, (float("nan"),), 1.0)):
        with pytest.raises(B.IdgError) as e:
            B.idg_wavelet_filter(a, *args)
        assert e.value.status == -4
    with pytest.raises(B.IdgError) as e:
        B.idg_wavelet_transform(a, 0, 17)
    assert e.value.status == -4
    with pytest.raises(TypeError):
        B.idg_wavelet_transform(a.cpu(), 0, 1)


def test_release_temporaries(B):
    """The private pool keeps the Le Gall temporaries (~1.3 cubes) between calls; idg_release_temporaries
    hands them back to the driver, and the next call simply allocates again."""
    a = torch.from_numpy(noisy((96, 128, 256), 5)).cuda()              # 12.6 MB cube -> ~16 MB of temporaries
    ref = B.idg_wavelet_filter(a, B.WAVELET_LEGALL53, (1.0, 1.4, 1.7))
    torch.cuda.synchronize()
    held = torch.cuda.mem_get_info()[0]
    B.idg_release_temporaries()
    freed = torch.cuda.mem_get_info()[0]
    assert freed >= held + 8 * 2 ** 20
    assert torch.equal(B.idg_wavelet_filter(a, B.WAVELET_LEGALL53, (1.0, 1.4, 1.7)), ref)


def test_haar_warp_kernel_full_size_equals_per_axis_passes(B):
    """configs[2] size (512 x 512 x 256), the launch configuration bench.py --filter wavelet_haar times: the
    block-per-warp kernel against the per-level, per-axis in-place passes, bit for bit, with the paper's thresholds."""
    g = torch.Generator(device="cuda").manual_seed(31)
    a = torch.randn((256, 512, 512), device="cuda", generator=g)
    a[100:110, 200:230, 300:340] += 6.0
    B.idg_set_option(B.IDG_OPT_KERNEL, 1)
    try:
        ref = B.idg_wavelet_filter(a, B.WAVELET_HAAR, (0.5, 0.8, 1.1), 1.0)
    finally:
        B.idg_set_option(B.IDG_OPT_KERNEL, 0)
    out = B.idg_wavelet_filter(a, B.WAVELET_HAAR, (0.5, 0.8, 1.1), 1.0)
    assert "idg_haar_warp_kernel" in B.idg_last_plan()
    assert torch.equal(out, ref)
    assert int((out != a).sum()) > a.numel() // 2          # the filter did something

"""GPU parity of the gradient-driven (Perona-Malik, Eq. 5) variant: idg_filter_pm through the C ABI against
oracle.pm_filter_oracle, element by element; bar 1e-4 x rms as for the intensity-driven filter."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu
TOL = 1e-4


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1609_03782_b200 import binding
    binding.lib()
    yield binding
    for k in (binding.IDG_OPT_KERNEL, binding.IDG_OPT_FUSE, binding.IDG_OPT_TILE):
        binding.idg_set_option(k, 0)


def plan(B, kernel, fuse, tile):
    B.idg_set_option(B.IDG_OPT_KERNEL, kernel)
    B.idg_set_option(B.IDG_OPT_FUSE, fuse)
    B.idg_set_option(B.IDG_OPT_TILE, tile)


PLANS = [(1, 0, 0), (3, 1, 0), (3, 2, 0), (3, 3, 0), (3, 4, 0), (5, 0, 0), (0, 0, 0)]
SHAPES = [(1, 1, 1), (4, 4, 4), (7, 6, 5), (3, 5, 8), (2, 3, 260), (9, 70, 132), (21, 67, 100), (13, 150, 268)]


@pytest.mark.parametrize("p", PLANS, ids=lambda p: "k%d-T%d-t%d" % p)
@pytest.mark.parametrize("shape", SHAPES, ids=lambda s: "x".join(map(str, s[::-1])))
def test_pm_parity(B, oracle, shape, p):
    plan(B, *p)
    rng = np.random.default_rng(sum(shape) + 7)
    a = (rng.normal(0, 1, shape) + 8.0 * (rng.random(shape) < 0.05)).astype(np.float32)
    prm = B.Params(K=1.5, tau=0.0325, cx=5.0, cy=4.0, cz=6.0, rms=1.0)
    t = torch.from_numpy(a).cuda()
    for n in (0, 1, 2, 5, 10):
        out = B.idg_filter_pm(t, n, prm).cpu().numpy().astype(np.float64)
        ref = oracle.pm_filter_oracle(a, n, **prm.f32())
        assert np.abs(out - ref).max() <= TOL, (shape, n)


def test_pm_config0_and_invariants(B, oracle):
    from paper_1609_03782_b200 import synth
    plan(B, 0, 0, 0)
    c = synth.modelb_like(seed=1000, snr=32.0)
    t = torch.from_numpy(c.data).cuda()
    for K in (0.5, 1.5, 10.0):
        prm = B.Params(K=K)
        out = B.idg_filter_pm(t, 10, prm)
        assert np.abs(out.cpu().numpy().astype(np.float64) - oracle.pm_filter_oracle(c.data, 10, **prm.f32())).max() <= TOL * c.rms
    # K = inf: bitwise the same linear diffusion as idg_filter; constant cube: fixed point to rounding
    lin = B.Params(K=float("inf"))
    assert torch.equal(B.idg_filter_pm(t, 6, lin), B.idg_filter(t, 6, lin))
    k = torch.full((10, 40, 64), 3.25, device="cuda")
    assert float((B.idg_filter_pm(k, 9, B.Params()) - k).abs().max()) <= 3.25 * 9 * 2.0 ** -23   # fixed point to rounding
    # fused kernels (TMA kernel 3 at every depth, resident kernel 5, auto plan) == naive kernel, bit for bit
    plan(B, 1, 0, 0)
    ref = B.idg_filter_pm(t, 7, B.Params())
    for p in ((3, 1, 0), (3, 2, 0), (3, 3, 0), (3, 4, 0), (5, 0, 0), (0, 0, 0)):
        plan(B, *p)
        assert torch.equal(B.idg_filter_pm(t, 7, B.Params()), ref), p


def test_pm_batched(B, oracle):
    """idg_filter_pm_batched: per-cube parameters and iteration counts (0 included), in place and not, under every plan;
    each cube equals the single-cube call bit for bit and the oracle within the tolerance."""
    rng = np.random.default_rng(77)
    cubes = (rng.normal(0, 1, (5, 9, 20, 24)) + 6.0 * (rng.random((5, 9, 20, 24)) < 0.04)).astype(np.float32)
    ns = [0, 1, 4, 7, 10]
    ps = [B.Params(K=0.75 + 0.5 * b, tau=0.03, cx=4.0 + b % 3, cy=5.0, cz=6.0, rms=1.0) for b in range(5)]
    t = torch.from_numpy(cubes).cuda()
    for p in PLANS:
        plan(B, *p)
        out = B.idg_filter_pm_batched(t, ns, ps)
        inpl = t.clone()
        B.idg_filter_pm_batched(inpl, ns, ps, out=inpl)
        for b in range(5):
            assert torch.equal(out[b], B.idg_filter_pm(t[b], ns[b], ps[b])), (p, b)
            assert torch.equal(out[b], inpl[b]), (p, b)
            ref = oracle.pm_filter_oracle(cubes[b], ns[b], **ps[b].f32())
            assert np.abs(out[b].cpu().numpy().astype(np.float64) - ref).max() <= TOL, (p, b)
    plan(B, 0, 0, 0)

"""idg_gaussian_filter_static: the no-allocation variant of the rotated Gaussian filter (include/idg.h), whose kernel
weights live in a static device array inside the library instead of a stream-ordered temporary.

Collected LAST on purpose (the suite runs with `pytest -x`): a failure here hides no other test.  The new entry point
is compared with the existing path, idg_gaussian_filter with the same rotation, on two calls in a row that share the
array -- the first with the largest kernel the array takes (r = 9), the second with a small one (r = 4), so the second
call runs on top of the first call's leftovers -- within the tolerance of the other reference-filter tests (1e-4 x rms);
the two paths build the same fp32 weights and run the same kernel, so they agree bit for bit as well.
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

TOL = 1e-4          # x rms (rms = 1 here), as in tests/test_gpu_ref_filters.py


@pytest.fixture(scope="module")
def B():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1609_03782_b200 import binding
    binding.lib()           # fails loudly if the extension is missing
    for k in (binding.IDG_OPT_KERNEL, binding.IDG_OPT_FUSE, binding.IDG_OPT_ZCHUNK, binding.IDG_OPT_TILE,
              binding.IDG_OPT_CTAS, binding.IDG_OPT_COOP):
        binding.idg_set_option(k, 0)
    return binding


def cube(shape, seed):
    rng = np.random.default_rng(seed)
    a = (rng.normal(0, 1, shape) + 8.0 * (rng.random(shape) < 0.03)).astype(np.float32)
    return torch.from_numpy(a).cuda()


CALLS = [((7.0, 3.0, 3.0), (25.0, -40.0, 110.0)),       # r = 9: fills the whole static array (PAPER.md:328 rotates FWHM 7, 3, 3)
         ((2.0, 3.0, 3.0), (0.0, 0.0, 45.0))]           # r = 4: 729 of its 6859 entries, on top of the leftovers


def test_static_entry_point_matches_the_existing_path_on_two_calls_in_a_row(B):
    a = cube((21, 45, 70), 41)
    assert [B.idg_gaussian_radii(f, t)[0] for f, t in CALLS] == [9, 4]
    want = [B.idg_gaussian_filter(a, f, t) for f, t in CALLS]          # existing path (allocates its weights)
    torch.cuda.synchronize()
    out = [torch.empty_like(a), torch.empty_like(a)]
    for (f, t), o in zip(CALLS, out):                                   # two calls in a row, no sync in between
        B.idg_gaussian_filter_static(a, f, t, out=o)
    torch.cuda.synchronize()
    for o, w in zip(out, want):
        assert float((o - w).abs().max()) <= TOL
        assert torch.equal(o, w)                                        # same weights, same kernel
    # and once more in the opposite order (small kernel first, then the large one over it)
    for (f, t), w in zip(CALLS[::-1], want[::-1]):
        o = B.idg_gaussian_filter_static(a, f, t)
        assert float((o - w).abs().max()) <= TOL


def test_static_entry_point_against_the_oracle(B, oracle):
    a = cube((9, 20, 33), 42)
    f, t = (3.0, 5.0, 2.0), (10.0, 20.0, 30.0)
    out = B.idg_gaussian_filter_static(a, f, t)
    ref = oracle.gaussian_filter_oracle(a.cpu().numpy(), f, t)
    assert float(np.abs(out.cpu().numpy().astype(np.float64) - ref).max()) <= TOL


def test_static_entry_point_allocates_no_device_memory(B):
    """Free device memory is the same before and after (the library's private pool, which the existing path grows,
    is not touched); outputs are preallocated so that torch allocates nothing either."""
    a = cube((16, 40, 64), 43)
    o = torch.empty_like(a)
    f, t = CALLS[0]
    B.idg_gaussian_filter_static(a, f, t, out=o)            # first use: module / kernel loading, symbol look-up
    torch.cuda.synchronize()
    before = torch.cuda.mem_get_info()[0]
    for f, t in CALLS * 3:
        B.idg_gaussian_filter_static(a, f, t, out=o)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == before


def test_static_entry_point_rejects_what_does_not_fit(B):
    a = cube((8, 12, 16), 44)
    assert B.idg_gaussian_radii((8.2, 2.0, 4.0), (0.0, 33.0, 0.0))[0] == 10
    B.idg_gaussian_filter(a, (8.2, 2.0, 4.0), (0.0, 33.0, 0.0))         # the allocating path takes r = 10
    with pytest.raises(B.IdgError) as e:
        B.idg_gaussian_filter_static(a, (8.2, 2.0, 4.0), (0.0, 33.0, 0.0))
    assert e.value.status == -8 and "static scratch" in str(e.value)
    with pytest.raises(B.IdgError) as e:                                # no rotation: the separable path has no scratch
        B.idg_gaussian_filter_static(a, (3.0, 3.0, 3.0), (0.0, 0.0, 0.0))
    assert e.value.status == -4
    with pytest.raises(B.IdgError) as e:                                # cube and out must not overlap
        B.idg_gaussian_filter_static(a, (3.0, 3.0, 3.0), (0.0, 0.0, 45.0), out=a)
    assert e.value.status == -6
    with pytest.raises(TypeError):
        B.idg_gaussian_filter_static(a.cpu(), (3.0, 3.0, 3.0), (0.0, 0.0, 45.0))

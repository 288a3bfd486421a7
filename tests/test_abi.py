"""CPU-side checks of the boundary: the library loads, exports every symbol include/idg.h
declares, and its host-only entry points behave.  No compute calls (no GPU here)."""
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def binding():
    from paper_1609_03782_b200 import build
    build.build()
    from paper_1609_03782_b200 import binding as b
    return b


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "idg.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(idg_[a-z_]+)\s*\(", src)))


def test_header_symbols_are_exported(binding):
    names = declared_symbols()
    assert len(names) >= 11
    L = binding.lib()
    for n in names:
        assert hasattr(L, n), n
    assert set(names) == set(binding.SYMBOLS)


def test_version_and_status_strings(binding):
    assert binding.idg_version() == 10100
    assert binding.status_string(0) == "ok"
    for s in range(-8, 0):
        assert binding.status_string(s) not in ("", "unknown status")


def test_params_check(binding):
    P = binding.Params
    assert binding.idg_params_check(P()) == 0                       # PAPER.md:187 defaults are in range, stable
    assert binding.idg_params_check(P(tau=0.0625)) == 2             # in GUI range but tau*sum(C) = 0.94 > 1/2
    assert binding.idg_params_check(P(K=0.25)) == 1
    assert binding.idg_params_check(P(K=float("inf"))) == 1         # accepted (linear limit), outside GUI range
    assert binding.idg_params_check(P(cx=11.0)) & 1
    for bad in (P(K=0.0), P(K=-1.0), P(K=float("nan")), P(tau=-0.1), P(cy=-1.0), P(rms=0.0),
                P(rms=float("inf")), P(tau=float("nan"))):
        assert binding.idg_params_check(bad) == 4


def test_workspace_bytes(binding):
    w = binding.idg_workspace_bytes(100, 100, 67, 1)
    assert w >= 100 * 100 * 67 * 4 and w % 256 == 0
    assert binding.idg_workspace_bytes(128, 128, 64, 256) >= 256 * 128 * 128 * 64 * 4 + 256 * 32
    assert binding.idg_workspace_bytes(0, 4, 4, 1) == 0
    assert binding.idg_workspace_bytes(4, 4, 4, 0) == 0


def test_options(binding):
    from paper_1609_03782_b200.binding import IdgError
    binding.idg_set_option(binding.IDG_OPT_FUSE, 3)
    assert binding.idg_get_option(binding.IDG_OPT_FUSE) == 3
    binding.idg_set_option(binding.IDG_OPT_FUSE, 0)
    with pytest.raises(IdgError):
        binding.idg_set_option(binding.IDG_OPT_FUSE, 9)
    with pytest.raises(IdgError):
        binding.idg_set_option(99, 0)


def test_options_are_per_host_thread(binding):
    """idg.h: an option set by one host thread affects that thread's calls only (thread_local state): two threads
    holding different IDG_OPT_FUSE at the same time each read back their own, and the main thread's stays untouched."""
    import threading
    binding.idg_set_option(binding.IDG_OPT_FUSE, 1)
    seen, gate = {}, threading.Barrier(2)

    def worker(value):
        assert binding.idg_get_option(binding.IDG_OPT_FUSE) == 0          # a new thread starts from the defaults
        binding.idg_set_option(binding.IDG_OPT_FUSE, value)
        gate.wait()                                                       # both threads have set theirs
        seen[value] = binding.idg_get_option(binding.IDG_OPT_FUSE)
        gate.wait()

    ts = [threading.Thread(target=worker, args=(v,)) for v in (2, 4)]
    for t in ts:
        t.start()
    for t in ts:
        t.join()
    assert seen == {2: 2, 4: 4}
    assert binding.idg_get_option(binding.IDG_OPT_FUSE) == 1
    binding.idg_set_option(binding.IDG_OPT_FUSE, 0)


def test_stats_rms(binding):
    """idg_stats_rms: mean and sqrt(<x^2> - <x>^2) from (n, sum, sum of squares); against numpy on a small sample."""
    import numpy as np
    x = np.random.default_rng(3).normal(2.0, 1.5, 1000)
    mean, rms = binding.idg_stats_rms([x.size, x.sum(), (x * x).sum()])
    assert mean == pytest.approx(x.mean(), rel=1e-12) and rms == pytest.approx(x.std(), rel=1e-10)
    assert all(np.isnan(v) for v in binding.idg_stats_rms([0.0, 0.0, 0.0]))


def test_resident_shapes_reserve_mailboxes(binding):
    """Cubes the resident kernel can take (nx >= 8, <= 4 Mi voxels) carry 32 MB of mailboxes in the workspace."""
    small = binding.idg_workspace_bytes(100, 100, 67, 1)
    assert small >= 100 * 100 * 67 * 4 + (32 << 20)
    # nx % 4 != 0: three pitched copies (row pitch 104 floats) for kernel 3 instead of one scratch cube, and the
    # mailboxes as well (the resident kernel pads rows on chip)
    w = binding.idg_workspace_bytes(102, 100, 67, 1)
    assert 3 * 104 * 100 * 67 * 4 + (32 << 20) <= w < 3 * 104 * 100 * 67 * 4 + (33 << 20)
    w = binding.idg_workspace_bytes(1023, 1023, 512, 1)             # too large for the chip: no mailboxes
    assert 3 * 1024 * 1023 * 512 * 4 <= w < 3 * 1024 * 1023 * 512 * 4 + (1 << 20)
    assert binding.idg_workspace_bytes(1024, 1024, 512, 1) < 1024 * 1024 * 512 * 4 + (1 << 20)  # too large


def test_cpu_tensor_is_rejected(binding):
    import torch
    with pytest.raises(TypeError):
        binding.idg_filter(torch.zeros(4, 4, 4), 1)

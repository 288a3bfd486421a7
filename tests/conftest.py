import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def oracle():
    import oracle as o
    o.build()
    return o


@pytest.fixture(scope="session")
def parity_log():
    """record(name, max_err_over_rms, note): the full-size parity cases append their margin under the 1e-4 x rms bar to
    gpurun_out/parity.txt (the only folder that comes back from the GPU box; a copy is kept under profiles/)."""
    path = os.path.join(ROOT, "gpurun_out", "parity.txt")
    os.makedirs(os.path.dirname(path), exist_ok=True)
    try:
        os.remove(path)
    except OSError:
        pass

    def record(name: str, err: float, note: str = "") -> None:
        with open(path, "a") as f:
            f.write(f"{name:<44s} max|gpu - oracle|/rms = {err:.3e}   (bar 1e-4)   {note}\n")
    return record

import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
for _p in (ROOT, os.path.join(ROOT, "tests")):
    if _p not in sys.path:
        sys.path.insert(0, _p)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")
    config.addinivalue_line("markers", "slow: long-running full-size parity case")


@pytest.fixture(scope="session")
def have_cuda():
    import torch
    return torch.cuda.is_available()


@pytest.fixture(scope="session")
def oracle_farm(request):
    """Background oracle followers shared by the GPU parity tests.  When the session has a CUDA device, the followers of the
    large configs (2 and 3: minutes of host time each) are started HERE, at the first use of the fixture -- the autouse
    fixture below asks for it before the first GPU test -- so that they compute while the other GPU tests run."""
    import torch
    from parity_utils import OracleFarm, request_large
    farm = OracleFarm()
    if torch.cuda.is_available():
        for cfg in (3, 2):          # longest first (config 1 is seconds: its test starts it)
            request_large(farm, cfg)
    yield farm
    farm.close()


@pytest.fixture(scope="session", autouse=True)
def _start_oracle_farm(request):
    if any(item.get_closest_marker("gpu") for item in request.session.items):
        import torch
        if torch.cuda.is_available():
            request.getfixturevalue("oracle_farm")
    yield


def pytest_terminal_summary(terminalreporter):
    try:
        from parity_utils import REPORTS
    except Exception:  # noqa: BLE001
        return
    if REPORTS:
        terminalreporter.section("parity coverage: GPU vs oracle (deviation / measured floor)")
        for r in REPORTS:
            terminalreporter.write_line(r)
    try:
        import paper_2504_07948_b200 as qb
        stale = qb.qmc_stale_error()
        if stale:
            terminalreporter.write_line("note: a CUDA error left pending on the thread by another library was dropped: " + stale)
    except Exception:  # noqa: BLE001
        pass

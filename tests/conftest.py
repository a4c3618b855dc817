import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


def pytest_addoption(parser):
    parser.addoption("--full", action="store_true", default=False,
                     help="configs 4 and 5: compare EVERY row with the oracle (and the fused list at every Nmax of config 5) instead of "
                          "the survey's row subsets; about 20 minutes of oracle time on 16 cores (SURVEY.md 8(d))")


@pytest.fixture(scope="session")
def full_run(request):
    return bool(request.config.getoption("--full")) or os.environ.get("SPD_FULL") == "1"

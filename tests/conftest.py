import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


# the tests exercise the measurement / debugging aids of include/nfs_dev.h as well: they run against the dev build
# (same object files as the product library plus nfs_dev.cu and the probe); tests/test_abi.py checks what each exports
from paper_1209_3362_b200 import binding as _binding  # noqa: E402

_binding.use_dev_library()


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def oracle():
    from oracle import nfs_oracle

    nfs_oracle.lib()
    return nfs_oracle

import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def oracle_mod():
    import oracle
    oracle.build()
    return oracle


@pytest.fixture(scope="session", autouse=True)
def _checked_build_saw_no_violation():
    """BFSC_CHECKED=1: the run uses libbfsc_checked.so (every BFSC_CHECK of the kernels evaluated); at its end no check
    may have failed."""
    yield
    if os.environ.get("BFSC_CHECKED", "") == "1":
        import torch
        if torch.cuda.is_available():
            from paper_1704_00513_b200 import binding
            if binding._lib is not None:
                enc, dec = binding.check_failures()
                assert enc[0] == 0, f"BFSC_CHECK failed {enc[0]} times in the encode kernels, first at encode-side line {enc[1]}"
                assert dec[0] == 0, f"BFSC_CHECK failed {dec[0]} times in the decode kernels, first at decode-side line {dec[1]}"

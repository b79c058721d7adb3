import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on the B200 box)")


@pytest.fixture(scope="session")
def oracle():
    import oracle as o
    o.build()
    return o


@pytest.fixture(params=["auto", "prefill_kernel", "decode_kernel", "gqa_pair_kernel"])
def dispatch(request):
    """Runs a -m gpu test once per attention kernel: the shape-based default, the two-stream (prefill / hybrid) kernel
    forced, the swapped-operand decode kernel forced, the CTA-pair GQA decode kernel forced (DeviceBatch skips the test
    when the forced kernel does not exist for the batch's geometry, e.g. the pair kernel for MHA).  Every kernel must be
    correct for every batch it accepts."""
    import gpu_harness
    mode = {"auto": 0, "prefill_kernel": 1, "decode_kernel": 2, "gqa_pair_kernel": 3}[request.param]
    gpu_harness.DEFAULT_DISPATCH = mode
    yield mode
    gpu_harness.DEFAULT_DISPATCH = 0

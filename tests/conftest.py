import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


def need_gpu(free_gib: float = 0.0):
    """GPU tests fail loudly (never skip) when selected on a box without a device or with too little free device
    memory: a full-size parity check that silently vanishes would leave the GPU suite green for the wrong reason."""
    import torch
    if not torch.cuda.is_available():
        pytest.fail("this test is marked gpu and needs a CUDA device (run with -m 'not gpu' on a CPU box)",
                    pytrace=False)
    if free_gib > 0.0:
        torch.cuda.empty_cache()
        free, _ = torch.cuda.mem_get_info()
        if free < free_gib * 2 ** 30:
            pytest.fail(f"needs {free_gib} GiB of free device memory, only {free / 2 ** 30:.1f} GiB are free",
                        pytrace=False)

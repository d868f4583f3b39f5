import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


def pytest_collection_modifyitems(config, items):
    try:
        import torch
        has_gpu = torch.cuda.is_available()
    except Exception:
        has_gpu = False
    if has_gpu:
        return
    skip = pytest.mark.skip(reason="no CUDA device")
    for it in items:
        if "gpu" in it.keywords:
            it.add_marker(skip)


def pytest_generate_tests(metafunc):
    """Every GPU test runs twice: with the pool kernel (the default) and with the one-photon-per-lane kernel
    (include/rt.h rt_set_kernel).  Both must give the oracle's photons bit for bit."""
    if metafunc.definition.get_closest_marker("gpu") and "trace_kernel" in metafunc.fixturenames:
        metafunc.parametrize("trace_kernel", ["pool", "lanes"], indirect=True)


@pytest.fixture(autouse=True)
def trace_kernel(request):
    which = getattr(request, "param", None)
    if which is None:
        yield None
        return
    from paper_2208_05247_b200 import binding
    old = binding.DEFAULT_KERNEL
    binding.DEFAULT_KERNEL = binding.KERNEL_LANES if which == "lanes" else binding.KERNEL_POOL
    try:
        yield which
    finally:
        binding.DEFAULT_KERNEL = old

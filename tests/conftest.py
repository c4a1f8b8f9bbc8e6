import os
import sys

import pytest

ROOT = os.path.abspath(os.path.join(os.path.dirname(__file__), ".."))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


def _have_gpu() -> bool:
    try:
        import torch
        return torch.cuda.is_available()
    except Exception:
        return False


def pytest_collection_modifyitems(config, items):
    if _have_gpu():
        return
    skip = pytest.mark.skip(reason="no CUDA device in this container")
    for item in items:
        if "gpu" in item.keywords:
            item.add_marker(skip)


@pytest.fixture(scope="session", autouse=True)
def _plan_as_large_job():
    """The plan has one rule that depends on the size of the call (small jobs keep any_kernel where a large job takes the
    generic kernel: iqa_query_plan_n).  The parity tests use small images to reach every kernel, so they plan every call
    as a large job; tests/test_gpu_2d.py::test_small_jobs_keep_any_kernel switches the rule back on and checks it."""
    from paper_2501_10653_b200 import binding
    old = binding.iqa_debug_knob("IQA_PLAN_LARGE_JOB", 1)
    yield
    binding.iqa_debug_knob("IQA_PLAN_LARGE_JOB", old)

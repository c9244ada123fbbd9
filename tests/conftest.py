import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parents[1]
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def acclb():
    """The CUDA path through its C-ABI binding; fails loudly when the extension or the GPU is missing."""
    import torch
    from paper_2505_01126_b200 import binding

    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    binding.load()  # raises if libacclb.so is not built
    return binding

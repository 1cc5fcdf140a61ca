import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")


@pytest.fixture(scope="session")
def oracle():
    from oracle import oracle as orc
    orc.build()
    return orc


@pytest.fixture(autouse=True)
def _release_cached_device_memory():
    """The GPU tests run in ONE process and torch keeps freed workspaces cached (after the config-5 test that is > 137 GB), which the
    worker processes of the two-rank tests cannot use: the full suite once left them too little to allocate.  Hand the cache back
    after every test; a no-op without CUDA."""
    yield
    import sys
    torch = sys.modules.get("torch")
    if torch is not None and torch.cuda.is_available() and torch.cuda.is_initialized():
        torch.cuda.empty_cache()

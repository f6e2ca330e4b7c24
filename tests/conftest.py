import os
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def have_gpu():
    import torch
    return torch.cuda.is_available()


@pytest.fixture
def opts():
    """Options every cn.Model of the test is created with (cn_model_create_opts; the library reads
    no environment variable).  Fixtures and tests fill it before they create models."""
    return {}


class CnWithOptions:
    """The binding module with Model() bound to the test's options."""

    def __init__(self, mod, opts):
        self._mod, self._opts = mod, opts

    def Model(self, desc, options=None, **kw):
        o = dict(self._opts)
        o.update(options or {})
        return self._mod.Model(desc, options=o or None, **kw)

    def __getattr__(self, name):
        return getattr(self._mod, name)


@pytest.fixture
def cn(opts):
    """paper_1901_10975_b200 (built on demand); GPU tests skip without a device."""
    from paper_1901_10975_b200.build import build
    build()
    import paper_1901_10975_b200 as mod
    return CnWithOptions(mod, opts)


@pytest.fixture
def need_gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")

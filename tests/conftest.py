import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def oracle():
    from oracle import load_oracle
    return load_oracle()


_SCENES = {}


def get_scene(config, **kw):
    """Cached scenegen scene (data only)."""
    from scenegen import make_scene
    key = (config, tuple(sorted(kw.items())))
    if key not in _SCENES:
        _SCENES[key] = make_scene(config, **kw)
    return _SCENES[key]


@pytest.fixture(scope="session")
def scene1():
    return get_scene(1)


@pytest.fixture(scope="session")
def scene2():
    return get_scene(2)

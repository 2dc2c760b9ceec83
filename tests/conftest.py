"""Shared pytest setup: the `gpu` marker, repo root on sys.path, cached scenes."""
import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on a B200)")


def pytest_collection_modifyitems(config, items):
    """A `gpu` test on a box without a CUDA device is skipped, never silently passed on a fallback."""
    try:
        import torch
        have = torch.cuda.is_available()
    except Exception:  # pragma: no cover
        have = False
    if have:
        return
    skip = pytest.mark.skip(reason="no CUDA device")
    for item in items:
        if "gpu" in item.keywords:
            item.add_marker(skip)


_SCENES = {}


@pytest.fixture(scope="session")
def scene_cache():
    """make_scene(name, **kw) memoised for the session (scenes are read-only inputs)."""
    from ba_scenes import make_scene

    def get(name, **kw):
        key = (name, tuple(sorted(kw.items())))
        if key not in _SCENES:
            _SCENES[key] = make_scene(name, **kw)
        return _SCENES[key]

    return get

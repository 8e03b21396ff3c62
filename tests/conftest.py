"""pytest configuration: registers the ``gpu`` marker and puts the repo root on sys.path."""
import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


def pytest_collection_modifyitems(config, items):
    try:
        import torch
        has_gpu = torch.cuda.is_available()
    except Exception:  # pragma: no cover
        has_gpu = False
    if has_gpu:
        return
    skip = pytest.mark.skip(reason="no CUDA device")
    for item in items:
        if "gpu" in item.keywords:
            item.add_marker(skip)


@pytest.fixture(scope="session")
def cfg1():
    from tpc_synth import generate_config
    return generate_config("cfg1")


@pytest.fixture(scope="session")
def cfg1_clean():
    from tpc_synth import generate_config
    return generate_config("cfg1", sigma=0.0)


@pytest.fixture(scope="session")
def mini_event():
    """A reduced cfg2 (800 tracks + 2 % noise, all 36 sectors): seconds for the oracle, several tiles for the GPU."""
    from tpc_synth import generate_config
    return generate_config("cfg2", n_tracks=800)


@pytest.fixture(scope="session")
def mini_tf():
    """A reduced cfg3 (3 piled-up collisions, 5 % noise, pseudo-z shifts)."""
    from tpc_synth import generate_config
    return generate_config("cfg3", n_collisions=3)

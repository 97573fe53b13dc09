import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def c0():
    """Config C0 (BASELINE.json configs[0]): model + frame + oracle, built once per session."""
    import gen
    from oracle.oracle import Oracle
    cfg = gen.make_config("C0")
    model = gen.make_model(cfg)
    frame = gen.make_frame(cfg, model["env"])
    return cfg, model, frame, Oracle.from_gen(cfg, model)

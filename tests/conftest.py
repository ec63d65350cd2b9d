import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on a B200)")


@pytest.fixture(scope="session")
def tiny_model():
    import synthetic_inputs as si
    from oracle import model
    cfg = si.CONFIGS["tiny"]
    params = si.draw_vibronic_params(cfg)
    mpo = model.build_mpo(params)
    dims = si.site_dims(params)
    occ = si.initial_occupations(params)
    return cfg, params, mpo, dims, occ

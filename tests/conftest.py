import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def cfg1():
    """Config 1 (BASELINE.json configs[0]): bank (float64 + fp32-rounded), templates, strain, injections."""
    from workloads import CONFIGS, chirp_templates
    c = CONFIGS[1]
    bank = c.bank(0)
    return dict(cfg=c, bank=bank, bank32=bank.as_f32(), H=chirp_templates(bank.mchirp, 8.0),
                strain=c.strain(), inj=c.injections())

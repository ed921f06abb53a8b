import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)
ORACLE_DIR = os.path.join(ROOT, "oracle")
if ORACLE_DIR not in sys.path:
    sys.path.insert(0, ORACLE_DIR)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")


@pytest.fixture(scope="session")
def oracle():
    import geo_oracle  # oracle/geo_oracle.py (test infrastructure)
    geo_oracle.lib()
    return geo_oracle


@pytest.fixture(scope="session")
def tab_oracle():
    import geo_tab_oracle  # oracle/geo_tab_oracle.py (test infrastructure)
    geo_tab_oracle.lib()
    return geo_tab_oracle


@pytest.fixture(scope="session")
def ks_oracle():
    import geo_ks_oracle  # oracle/geo_ks_oracle.py (test infrastructure, Cartesian Kerr-Schild)
    geo_ks_oracle.lib()
    return geo_ks_oracle


@pytest.fixture(scope="module")
def G():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1803_08320_b200 import build, geo
    build.build()   # (re)compiles libgeo.so in-tree if it is missing or older than its sources
    geo.lib()       # fails loudly if libgeo.so is missing
    return geo

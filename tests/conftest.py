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
def oracle_mod():
    from oracle import lbm_oracle

    lbm_oracle.build()
    return lbm_oracle


def make_oracle(wl, inp):
    """Build an oracle simulation from a workload dict + inputs (mask, rho, u)."""
    from oracle import lbm_oracle

    s = lbm_oracle.Oracle(wl)
    if inp.get("mask") is not None:
        s.set_solid_mask(inp["mask"])
    s.init_fields(inp["rho"], inp.get("u"))
    return s

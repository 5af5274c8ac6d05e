import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")
    config.addinivalue_line("markers", "slow: long-running full-size case")


@pytest.fixture(scope="session")
def oracle_mod():
    import oracle
    oracle.build()
    return oracle


@pytest.fixture(scope="session", autouse=True)
def _built_library():
    """The CUDA library is built in-tree (nvcc cross-compiles without a GPU)."""
    from paper_1311_2719_b200 import build
    build.build()


@pytest.fixture(scope="session")
def cfg5_inputs():
    """(cfg, gauge field, source) of BASELINE.json config 5 (48^3 x 96, 6 GB of links): generated once
    per session, the three full-size tests share it."""
    from paper_1311_2719_b200 import synth
    return synth.config_inputs(5)


@pytest.fixture(scope="session")
def cfg3_inputs():
    from paper_1311_2719_b200 import synth
    return synth.config_inputs(3)


@pytest.fixture(scope="session")
def cfg3_oracle_cg(cfg3_inputs):
    """The oracle's own CG on BASELINE.json config 3 (32^4, m = 0.01: 3138 iterations, about a minute on the
    GPU box's 16 host cores), run ONCE per session: the full-size tests compare the WHOLE solution vector
    with it at the north-star tolerance, not a sample."""
    import oracle
    c, u, b = cfg3_inputs
    return oracle.cg(c["dims"], 0, u, c["param"], c["tol"], 100000, b)

import os
import sys
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


_ORACLE_SPACES = {}


def oracle_space(cfg: int, with_objective=True, objective_seed=0):
    """Session cache of fully enumerated oracle spaces for the BASELINE configs (cfg3 takes ~1 min)."""
    import oracle as O
    import workloads as W
    key = (cfg, with_objective, objective_seed)
    if key not in _ORACLE_SPACES:
        sp = {0: W.space_cfg0, 1: W.space_cfg1, 2: W.space_cfg2, 3: W.space_cfg3, 4: W.space_cfg1}[cfg]()
        s = O.OracleSpace.from_space(sp).build()
        if with_objective:
            s.set_objective(W.objective_table(s.rows(), sp.m, objective_seed))
        _ORACLE_SPACES[key] = (sp, s)
    return _ORACLE_SPACES[key]


@pytest.fixture(scope="session")
def get_oracle_space():
    return oracle_space

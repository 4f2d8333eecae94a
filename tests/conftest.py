import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def oracle_lib():
    import oracle
    oracle.build()
    return oracle


_problem_cache = {}


@pytest.fixture(scope="session")
def problems():
    """Seeded synthetic problems by config name, cached for the session (host tensors)."""
    import gwgen

    def get(name):
        if name not in _problem_cache:
            _problem_cache[name] = gwgen.make_problem(name)
        return _problem_cache[name]

    return get


_raw_cache = {}


@pytest.fixture(scope="session")
def raw_problems():
    """Seeded problems with NO input symmetry (gwgen.make_problem(raw=True)): independent V blocks, non-Hermitian G, gamma, W."""
    import gwgen

    def get(name):
        if name not in _raw_cache:
            _raw_cache[name] = gwgen.make_problem(name, raw=True)
        return _raw_cache[name]

    return get


_oracle_cache = {}


@pytest.fixture(scope="session")
def oracle_results(problems, oracle_lib):
    """Full oracle pipeline on a small config: dict(P0t, P0w, Ww, Wt, Sigma, K)."""

    def get(name):
        if name not in _oracle_cache:
            p = problems(name)
            cfg = p.cfg
            vb = oracle_lib.VBlocks(cfg, p.V.numpy())
            P0t = oracle_lib.polarization(cfg, vb, p.G)
            Wt, P0w, Ww = oracle_lib.screened_interaction(cfg, p.T_wt, p.T_tw, P0t, want_freq=True)
            Sg = oracle_lib.selfenergy(cfg, vb, p.G, Wt)
            K = oracle_lib.exchange(cfg, vb, p.gamma)
            _oracle_cache[name] = dict(P0t=P0t, P0w=P0w, Ww=Ww, Wt=Wt, Sigma=Sg, K=K)
        return _oracle_cache[name]

    return get

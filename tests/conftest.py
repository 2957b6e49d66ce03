import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")
    config.addinivalue_line("markers", "slow: longer CPU test")


@pytest.fixture(scope="session")
def po():
    from oracle import pb_oracle
    pb_oracle.build()
    return pb_oracle


def _sphere_oracle(po, radius, subdiv, K_far, **kw):
    from paper_1810_03698_b200.workloads import icosphere
    v, t = icosphere(radius, subdiv)
    return po.Oracle(v, t, po.Params(K_far=K_far, **kw))


@pytest.fixture(scope="session")
def sphere_oracles(po):
    """R=4 icospheres, K_far=4 (BASELINE configs[0]), by subdivision level; cached."""
    cache = {}

    def get(subdiv, radius=4.0, K_far=4, **kw):
        key = (subdiv, radius, K_far, tuple(sorted(kw.items())))
        if key not in cache:
            cache[key] = _sphere_oracle(po, radius, subdiv, K_far, **kw)
        return cache[key]

    return get

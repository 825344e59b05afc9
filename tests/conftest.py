import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def cfg0():
    """configs[0]: 288-atom water-like system + base52 model + full oracle result."""
    import oracle
    import workloads as W
    sysm, model = W.build(W.CONFIGS[0])
    om = oracle.OracleModel(model)
    res = oracle.compute(om, sysm.pos, sysm.types, sysm.box)
    return sysm, model, om, res


def tiny_model(sf_rows, n_elem=1, hidden=(3,), seed=7, rc=6.0):
    """Model with an explicit SF list (tuples central,kind,e1,e2,eta,rs,lam,zeta)."""
    import workloads as W
    from workloads.model import Model, mlp_weights
    sf = np.array(sf_rows, dtype=W.SF_DTYPE)
    n_per = [int(np.sum(sf["central"] == c)) for c in range(n_elem)]
    layer_sizes = [[max(n_per[c], 1), *hidden, 1] for c in range(n_elem)]
    weights = [mlp_weights(layer_sizes[c], seed, c) for c in range(n_elem)]
    return Model(elements=tuple("X%d" % i for i in range(n_elem)), rc=rc, sf=sf,
                 layer_sizes=layer_sizes, weights=weights, name="tiny", n_sf_per_elem=n_per)

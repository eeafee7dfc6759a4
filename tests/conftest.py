import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
for p in (ROOT, os.path.dirname(os.path.abspath(__file__))):
    if p not in sys.path:
        sys.path.insert(0, p)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run with -m gpu on a B200)")


_ORACLE_CACHE = {}


@pytest.fixture(scope="session")
def oracle_cfg():
    """Session cache: cfg index -> (inputs, dense-oracle result)."""
    from thc_synth import make_config
    from oracle import dense

    def get(cfg):
        if cfg not in _ORACLE_CACHE:
            x = make_config(cfg)
            res = dense.residual_and_energy(x.Xo, x.Xv, x.Z, x.B_ov, x.B_oo, x.B_vv, x.Y, x.V, x.eps)
            res.pop("omega", None)
            res.pop("t", None)
            _ORACLE_CACHE[cfg] = (x, res)
        return _ORACLE_CACHE[cfg]

    return get


def small_inputs(o=3, v=4, NL=6, NP=5, NX=7, seed=5, zmul=30.0):
    """Miniature problem with O(1) amplitudes so that the T2^2 terms are not negligible."""
    from thc_synth import make_inputs
    x = make_inputs(o, v, NL, NP, NX, seed=seed)
    x.Z = x.Z * zmul
    return x


def oracle_eval(x, **kw):
    from oracle import dense
    return dense.residual_and_energy(x.Xo, x.Xv, x.Z, x.B_ov, x.B_oo, x.B_vv, x.Y, x.V, x.eps, **kw)

"""north_star pin: 'the identity between factorized and dense contractions'.

The paper states every term twice: as a dense 4-index equation (Eqs.28-41) and as a factorised
algorithm (Alg.1-9).  oracle/dense.py implements the former, tests/paper_algorithms.py the latter.
"""
import numpy as np
import pytest

from conftest import small_inputs, oracle_eval
import paper_algorithms as pa


@pytest.mark.parametrize("dims,seed", [((3, 4, 6, 5, 7), 5), ((2, 5, 3, 8, 4), 6), ((4, 3, 5, 6, 9), 7)])
def test_each_algorithm_equals_projected_dense_equation(dims, seed):
    o, v, NL, NP, NX = dims
    x = small_inputs(o, v, NL, NP, NX, seed=seed)
    res = oracle_eval(x)
    xi_oo, xi_vv = pa.alg8_xi(x.Xo, x.Xv, x.Z, x.B_ov)
    got = dict(
        s1=pa.alg1(x.Xo, x.Xv, x.Z, x.B_oo, x.B_vv),
        s2=pa.alg2(x.Xo, x.Xv, x.Z, x.B_ov),
        s3=pa.alg3(x.Xo, x.Xv, x.Z, x.B_oo, x.B_vv),
        s6=pa.alg6(x.Xo, x.Xv, x.Z, x.Yo, x.Yv, x.V),
        s7=pa.alg7(x.Xo, x.Xv, x.Z, x.Yo, x.Yv, x.V),
        s9=pa.alg9(x.Xo, x.Xv, x.Z, np.diag(x.eps[:o]) + xi_oo, np.diag(x.eps[o:]) + xi_vv),
    )
    for k, s in got.items():
        scale = np.abs(res[k]).max()
        assert scale > 1e-3, k
        assert np.abs(s - res[k]).max() <= 2e-13 * max(1.0, scale), k
    assert np.abs(xi_oo - res["xi_oo"]).max() < 1e-13
    assert np.abs(xi_vv - res["xi_vv"]).max() < 1e-13


def test_transposed_xi_oo_changes_sigma9():
    """Reading R5: Alg.9 line 5 contracts the FIRST index of (F + xi)_ji."""
    x = small_inputs(3, 4, 6, 5, 7, seed=5)
    o = 3
    res = oracle_eval(x)
    xi_oo, xi_vv = pa.alg8_xi(x.Xo, x.Xv, x.Z, x.B_ov)
    bad = pa.alg9(x.Xo, x.Xv, x.Z, np.diag(x.eps[:o]) + xi_oo.T, np.diag(x.eps[o:]) + xi_vv)
    assert np.abs(bad - res["s9"]).max() > 1e-3

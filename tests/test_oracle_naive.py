"""Pin the einsum index strings and the two-ERI-set wiring of oracle/dense.py to literal loops."""
import numpy as np
import pytest

from conftest import small_inputs, oracle_eval
from oracle import dense, naive


@pytest.mark.parametrize("o,v,seed", [(2, 3, 5), (3, 2, 6)])
def test_terms_equal_literal_loops(o, v, seed):
    x = small_inputs(o, v, 4, 5, 6, seed=seed)
    res = oracle_eval(x)                                  # independent THC set (Y, V)
    thc = dense.thc_ovov(x.Yo, x.Yv, x.V)
    t = naive.expand_t_naive(x.Xo, x.Xv, x.Z)
    assert np.abs(t - res["t"]).max() < 1e-13
    nv = naive.omega_terms_naive(t, x.B_oo, x.B_ov, x.B_vv, thc, x.eps[:o], x.eps[o:])
    for k in dense.TERMS:
        scale = np.abs(nv[k]).max()
        assert scale > 1e-3
        assert np.abs(nv[k] - res["omega"][k]).max() <= 1e-13 * max(1.0, scale), k
    assert np.abs(nv["xi_oo"] - res["xi_oo"]).max() < 1e-13
    assert np.abs(nv["xi_vv"] - res["xi_vv"]).max() < 1e-13
    # xi_oo is NOT symmetric (reading R5) -- the index order in Alg.9 line 5 matters
    assert np.abs(res["xi_oo"] - res["xi_oo"].T).max() > 1e-3
    # projection
    for k in ("s1", "s6"):
        assert np.abs(naive.project_naive(x.Xo, x.Xv, nv[k]) - res[k]).max() < 1e-13


def test_thc_and_cd_sets_are_wired_to_the_right_terms():
    """Scaling V scales only s6, s7; scaling B scales s1,s2,s3 and the xi part of s9 (reading R6)."""
    x = small_inputs(2, 3, 4, 5, 6, seed=9)
    r0 = oracle_eval(x)
    x.V = 3.0 * x.V
    r1 = oracle_eval(x)
    for k in ("s1", "s2", "s3", "s9"):
        assert np.abs(r1[k] - r0[k]).max() < 1e-13
    for k in ("s6", "s7"):
        assert np.abs(r1[k] - 3.0 * r0[k]).max() < 1e-12
    assert r1["E"] == pytest.approx(r0["E"], abs=1e-13)

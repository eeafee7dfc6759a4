"""Pin T1 (oracle/dense.py) to T0: determinant-space <D|exp(-T2) H exp(T2)|0> (no CC formula used)."""
import numpy as np
import pytest

from conftest import small_inputs, oracle_eval
from oracle import dense, bruteforce


@pytest.mark.parametrize("o,v,seed", [(2, 3, 11), (3, 3, 12), (2, 2, 13)])
def test_dense_total_equals_determinant_bruteforce(o, v, seed):
    x = small_inputs(o, v, 7, 5, 9, seed=seed)
    res = oracle_eval(x, thc_from_cd=True)       # one Hamiltonian: THC set := Cholesky set
    eri = bruteforce.full_eri(x.B_oo, x.B_ov, x.B_vv)
    om_bf, e_bf = bruteforce.omega_bruteforce(res["t"], eri, x.eps, o, v)
    om = sum(res["omega"][k] for k in dense.TERMS)
    scale = np.abs(om_bf).max()
    assert scale > 0.5                           # all terms are O(1) here
    assert np.abs(om - om_bf).max() <= 1e-12 * scale
    assert abs(res["E"] - e_bf) <= 1e-12 * max(1.0, abs(e_bf))
    # every term must matter for this pin to bite
    for k in dense.TERMS:
        assert np.abs(res["omega"][k]).max() > 1e-3 * scale


def test_printed_quarter_prefactor_is_wrong_by_the_whole_term():
    """Reading R2: Eq.35 / Alg.7 l.769 print 1/4; only 1/2 reproduces second quantisation."""
    o, v = 2, 3
    x = small_inputs(o, v, 7, 5, 9, seed=11)
    res = oracle_eval(x, thc_from_cd=True)
    eri = bruteforce.full_eri(x.B_oo, x.B_ov, x.B_vv)
    om_bf, _ = bruteforce.omega_bruteforce(res["t"], eri, x.eps, o, v)
    om = sum(res["omega"][k] for k in dense.TERMS)
    printed = om - 0.5 * res["omega"]["s7"]      # what a 1/4 prefactor would give
    miss = om_bf - printed
    assert np.abs(miss - 0.5 * res["omega"]["s7"]).max() < 1e-12
    assert np.abs(miss).max() > 1e-2


def test_bra_normalisation():
    """<D|H|0> = (ia|jb) and E_corr(T2=0) = 0 for the alpha-beta bra used by T0."""
    o, v = 2, 2
    x = small_inputs(o, v, 4, 3, 4, seed=3)
    eri = bruteforce.full_eri(x.B_oo, x.B_ov, x.B_vv)
    om, e = bruteforce.omega_bruteforce(np.zeros((o, v, o, v)), eri, x.eps, o, v)
    ovov = np.einsum("Lia,Ljb->iajb", x.B_ov, x.B_ov)
    assert np.abs(om - ovov).max() < 1e-13
    assert abs(e) < 1e-13

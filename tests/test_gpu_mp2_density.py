"""GPU parity of thc_mp2_density (Appendix II, Eqs.47-56) against oracle/mp2_density.py, element by element."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = 1e-10      # relative to the largest element of the block: the bar of the residual terms


def _run(o, v, NP, seed, symmetric=True):
    import torch
    import paper_2111_11473_b200 as thc
    from thc_synth import make_inputs
    from oracle import mp2_density
    x = make_inputs(o, v, 4, NP, 8, seed=seed, with_bvv=False)
    Z = x.Z * 30.0
    if not symmetric:
        Z = Z + np.triu(np.random.default_rng(seed).standard_normal((NP, NP)), 1) * np.abs(Z).max()
    want_oo, want_vv = mp2_density.mp2_density(x.Xo, x.Xv, Z)
    h = thc.thc_setup(o, v, 4, NP, 8)
    try:
        dev = [torch.from_numpy(np.ascontiguousarray(t)).cuda() for t in (x.Xo, x.Xv, Z)]
        for _ in range(2):                                  # twice: the workspace is reused, results must not change
            D_oo, D_vv = h.thc_mp2_density(*dev)
            torch.cuda.synchronize()
            for got, want, name in ((D_oo, want_oo, "D_oo"), (D_vv, want_vv, "D_vv")):
                err = np.abs(got.cpu().numpy() - want).max() / np.abs(want).max()
                assert err <= TOL, (name, err)
    finally:
        h.close()


@pytest.mark.parametrize("o,v,NP", [(5, 20, 50), (20, 100, 300), (7, 13, 37), (1, 3, 5), (3, 2, 130)])
def test_mp2_density_matches_the_definition(o, v, NP):
    """BASELINE configs 0 and 1, ragged odd extents (scalar load path), one occupied orbital, NP >> o v."""
    _run(o, v, NP, seed=41 + o)


def test_mp2_density_with_a_non_symmetric_core_matrix():
    """Eqs.53-56 hold for any T; a transposed operand in the exchange-like chains shows only when Z != Z^T."""
    _run(6, 11, 48, seed=5, symmetric=False)


def test_mp2_density_over_several_blocks_of_occupied_orbitals():
    """o NP^2 large enough that the exchange-like parts run in two blocks of i with a ragged last one (22 + 2)."""
    _run(24, 60, 800, seed=9)


def test_mp2_density_at_config2_size_sampled_elements_and_invariants():
    """BASELINE config 2 dimensions (o=60, v=340, NP=1000): the dense t does not fit the oracle, so single elements of
    D_oo / D_vv from their definition (oracle.mp2_density.density_*_element) plus what holds at any size: symmetry and
    tr D_oo = -tr D_vv."""
    import torch
    import paper_2111_11473_b200 as thc
    from thc_synth import make_inputs
    from oracle import mp2_density
    o, v, NP = 60, 340, 1000
    x = make_inputs(o, v, 4, NP, 8, seed=2, with_bvv=False)
    Z = x.Z * 30.0
    h = thc.thc_setup(o, v, 4, NP, 8)
    try:
        D_oo, D_vv = (t.cpu().numpy() for t in h.thc_mp2_density(*[torch.from_numpy(np.ascontiguousarray(t)).cuda() for t in (x.Xo, x.Xv, Z)]))
    finally:
        h.close()
    so, sv = np.abs(D_oo).max(), np.abs(D_vv).max()
    for i, j in ((3, 7), (59, 59)):
        assert abs(D_oo[i, j] - mp2_density.density_oo_element(x.Xo, x.Xv, Z, i, j)) <= TOL * so, (i, j)
    for a, b in ((5, 123), (339, 339)):
        assert abs(D_vv[a, b] - mp2_density.density_vv_element(x.Xo, x.Xv, Z, a, b)) <= TOL * sv, (a, b)
    assert np.abs(D_oo - D_oo.T).max() <= 1e-12 * so and np.abs(D_vv - D_vv.T).max() <= 1e-12 * sv
    assert abs(np.trace(D_oo) + np.trace(D_vv)) <= 1e-11 * abs(np.trace(D_vv))

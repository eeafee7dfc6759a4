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

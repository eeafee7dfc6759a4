"""thc_residual_rr (rank-reduced working variables, Eqs.13-14, 22) against oracle/rr.py, which never forms
Z = tau~^T T tau~ nor uses R^RR = tau~ sigma tau~^T."""
import numpy as np
import pytest

from conftest import small_inputs

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("dims,NR", [((3, 4, 6, 7, 9), 4), ((6, 14, 10, 40, 52), 17), ((5, 20, 12, 50, 64), 50)])
def test_rr_residual_matches_oracle(dims, NR):
    import torch
    import paper_2111_11473_b200 as thc
    from oracle import rr
    x = small_inputs(*dims, seed=41, zmul=1.0)
    rng = np.random.default_rng(NR)
    tau = rr.symmetric_orthogonalizer(x.Xo, x.Xv, rng.standard_normal((NR, x.NP)))
    T = rng.standard_normal((NR, NR))
    T = 0.5 * (T + T.T)
    ref = rr.rr_residual_and_energy(x.Xo, x.Xv, tau, T, x.B_ov, x.B_oo, x.B_vv, x.Y, x.V, x.eps)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    h = thc.thc_setup(x.o, x.v, x.NL, x.NP, x.NX)
    R_rr, Z = h.thc_residual_rr(dev(tau), dev(T), dev(x.Xo), dev(x.Xv), dev(x.B_ov), dev(x.B_oo), dev(x.B_vv), dev(x.Y),
                                dev(x.V), dev(x.eps), want_Z=True)
    E = h.thc_energy(dev(x.Xo), dev(x.Xv), Z, dev(x.B_ov))
    got = R_rr.cpu().numpy()
    h.close()
    assert np.abs(got - ref["R_rr"]).max() <= 1e-10 * np.abs(ref["R_rr"]).max()
    assert abs(E - ref["E"]) <= 1e-9

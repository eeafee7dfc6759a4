"""thc_residual_t1 (T1-dressed Cholesky vectors, dressed Fock matrix, singles residual; Eq.38, Eq.42,
Alg.8 lines 11-12, Alg.10) against oracle/t1.py, element by element and per term: the six doubles terms, xi, and the two
groups of the singles residual.  Tolerances as in test_gpu_parity.py (1e-10 of each term's own maximum)."""
import numpy as np
import pytest

from conftest import small_inputs

pytestmark = pytest.mark.gpu

NAMES = ("Xo", "Xv", "Z", "B_ov", "B_oo", "B_vv", "Y", "V", "eps")
TERMS = ("s1", "s2", "s3", "s6", "s7", "s9")


def _t1(o, v, seed, scale):
    return scale * np.random.default_rng(seed).standard_normal((o, v))


def _check(x, t1, **opts):
    import torch
    import paper_2111_11473_b200 as thc
    from oracle import t1 as t1o
    ref = t1o.residual_and_energy(x.Xo, x.Xv, x.Z, t1, x.B_ov, x.B_oo, x.B_vv, x.Y, x.V, x.eps)
    ref["sigma_GH"], ref["sigma_IJ"] = ref["sigma_G_H"], ref["sigma_I_J"]
    d = [torch.from_numpy(np.ascontiguousarray(getattr(x, n))).cuda() for n in NAMES]
    bvv_mode = opts.get("bvv_mode", "device")
    if bvv_mode == "host":
        d[5] = torch.from_numpy(np.ascontiguousarray(x.B_vv)).pin_memory()
    elif bvv_mode == "provider":
        dev_bvv = d[5]
        d[5] = lambda L0, nl, dst: dst.copy_(dev_bvv[L0:L0 + nl])
    h = thc.thc_setup(x.o, x.v, x.NL, x.NP, x.NX, **opts)
    res = h.thc_residual_t1(d[0], d[1], d[2], torch.from_numpy(t1).cuda(), *d[3:])
    res2 = h.thc_residual_t1(d[0], d[1], d[2], torch.from_numpy(t1).cuda(), *d[3:])     # the handle is reusable
    torch.cuda.synchronize()
    errs = {}
    for k in TERMS + ("R", "xi_oo", "xi_vv", "sigma", "sigma_GH", "sigma_IJ"):
        # each quantity against its own maximum; the two singles groups against the larger of them (at t1 = 0 the
        # I+J group is exactly zero on the GPU and rounding noise of the F^ - diag(eps) cancellation in the oracle)
        scale = max(np.abs(ref["sigma_GH"]).max(), np.abs(ref["sigma_IJ"]).max()) if k.startswith("sigma") else np.abs(ref[k]).max()
        errs[k] = np.abs(res[k].cpu().numpy() - ref[k]).max() / (scale if scale > 0 else 1.0)
        assert torch.equal(res[k], res2[k]), k
    h.close()
    bad = {k: e for k, e in errs.items() if e > 1e-10}
    assert not bad, f"parity failures {bad} (all: {errs})"
    return ref, res


@pytest.mark.parametrize("cfg", [0, 1])
def test_t1_config_per_term(cfg):
    from thc_synth import make_config
    x = make_config(cfg)
    _check(x, _t1(x.o, x.v, 50 + cfg, 0.05))


@pytest.mark.parametrize("dims", [(3, 4, 6, 5, 7), (7, 13, 19, 37, 45), (6, 18, 10, 64, 96), (66, 9, 5, 33, 40), (3, 4, 3, 641, 8)])
def test_t1_ragged_shapes_with_large_amplitudes(dims):
    x = small_inputs(*dims, seed=17, zmul=30.0)
    _check(x, _t1(dims[0], dims[1], 3, 0.3))
    _check(x, _t1(dims[0], dims[1], 3, 0.3), bL=4, bP7=3, bX=16, bI=5, tma_min_flop=1)


@pytest.mark.parametrize("mode", ["host", "provider"])
def test_t1_streamed_bvv(mode):
    x = small_inputs(6, 14, 21, 40, 52, seed=3, zmul=30.0)
    _check(x, _t1(6, 14, 4, 0.3), bL=4, bvv_mode=mode)


def test_t1_zero_equals_the_undressed_path():
    import torch
    import paper_2111_11473_b200 as thc
    x = small_inputs(6, 14, 21, 40, 52, seed=3, zmul=30.0)
    _, res = _check(x, np.zeros((6, 14)))
    d = [torch.from_numpy(np.ascontiguousarray(getattr(x, n))).cuda() for n in NAMES]
    h = thc.thc_setup(x.o, x.v, x.NL, x.NP, x.NX)
    plain = h.thc_residual_terms(*d)
    for k in TERMS + ("R",):
        assert float((plain[k] - res[k]).abs().max()) <= 1e-12 * float(plain[k].abs().max()), k
    h.close()

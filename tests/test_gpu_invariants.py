"""T3 invariants of the path evaluated through the C ABI: properties that hold at any size and need no
reference values.  Run here on a config-1-shaped problem with O(1) amplitudes; they are the kind of check that still
applies where no oracle row is affordable (sigma6, sigma9, E at config 4)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

NAMES = ("Xo", "Xv", "Z", "B_ov", "B_oo", "B_vv", "Y", "V", "eps")
TERMS = ("s1", "s2", "s3", "s6", "s7", "s9")


def _setup(o=12, v=40, NL=48, NP=96, NX=160, seed=17, zmul=20.0):
    import torch
    from thc_synth.device import make_inputs_device
    d = make_inputs_device(o, v, NL, NP, NX, seed=seed)
    d["Z"] = d["Z"] * zmul
    return (o, v, NL, NP, NX), d


def _eval(dims, d, **opts):
    import torch
    import paper_2111_11473_b200 as thc
    h = thc.thc_setup(*dims, **opts)
    res = h.thc_residual_terms(*[d[n] for n in NAMES])
    E = h.thc_energy(d["Xo"], d["Xv"], d["Z"], d["B_ov"])
    torch.cuda.synchronize()
    h.close()
    out = {k: res[k].cpu().numpy() for k in TERMS + ("R",)}
    out["E"] = E
    return out


def _close(a, b, tol=1e-11):
    for k in TERMS + ("R",):
        scale = max(np.abs(a[k]).max(), 1e-300)
        assert np.abs(a[k] - b[k]).max() <= tol * scale, k
    assert abs(a["E"] - b["E"]) <= 1e-10 * max(1.0, abs(a["E"]))


def test_each_term_is_symmetric():
    dims, d = _setup()
    r = _eval(dims, d)
    for k in TERMS + ("R",):
        assert np.abs(r[k] - r[k].T).max() <= 1e-12 * np.abs(r[k]).max(), k


def test_cholesky_rotation_invariance():
    """B^L -> sum_M Q_LM B^M with Q orthogonal leaves every Cholesky ERI, hence R and E, unchanged (exercises the
    L loop, its blocking and ordering)."""
    import torch
    dims, d = _setup()
    ref = _eval(dims, d, bL=7)
    NL = dims[2]
    Q, _ = torch.linalg.qr(torch.randn(NL, NL, dtype=torch.float64, device="cuda", generator=torch.Generator("cuda").manual_seed(3)))
    d2 = dict(d)
    for k in ("B_ov", "B_oo", "B_vv"):
        d2[k] = torch.einsum("LM,Mpq->Lpq", Q, d[k]).contiguous()
    _close(ref, _eval(dims, d2, bL=16), tol=1e-10)


def test_grid_gauge_invariance():
    """Xo[:,P] -> a_P Xo[:,P], Xv[:,P] -> Xv[:,P] / a_P leaves U^P_ia, t and R unchanged while o_PQ, v_PQ change;
    likewise Yo[:,I] -> b_I Yo[:,I], V_IJ -> V_IJ / (b_I b_J)."""
    import torch
    dims, d = _setup()
    o = dims[0]
    ref = _eval(dims, d)
    g = torch.Generator("cuda").manual_seed(5)
    a = torch.exp(0.5 * torch.randn(dims[3], dtype=torch.float64, device="cuda", generator=g))
    b = torch.exp(0.5 * torch.randn(dims[4], dtype=torch.float64, device="cuda", generator=g))
    d2 = dict(d)
    d2["Xo"] = (d["Xo"] * a).contiguous()
    d2["Xv"] = (d["Xv"] / a).contiguous()
    Y = d["Y"].clone()
    Y[:o] *= b
    d2["Y"] = Y
    d2["V"] = (d["V"] / (b[:, None] * b[None, :])).contiguous()
    _close(ref, _eval(dims, d2), tol=1e-10)


def test_polynomial_structure_in_Z_and_linearity_in_V():
    """R(sZ) = R0 + s R1 + s^2 R2 exactly, with R0 = A A^T and R2 = sigma6 + sigma7 + sigma9|eps=0 ... checked through
    third differences; sigma6, sigma7 scale linearly with V and nothing else depends on V."""
    import torch
    dims, d = _setup()
    R = {}
    for s in (0.0, 1.0, 2.0, 3.0):
        d2 = dict(d)
        d2["Z"] = (d["Z"] * s).contiguous()
        R[s] = _eval(dims, d2)["R"]
    third = R[3.0] - 3 * R[2.0] + 3 * R[1.0] - R[0.0]
    assert np.abs(third).max() <= 1e-10 * np.abs(R[3.0]).max()
    d3 = dict(d)
    d3["V"] = (2.5 * d["V"]).contiguous()
    a, b = _eval(dims, d), _eval(dims, d3)
    for k in ("s6", "s7"):
        assert np.abs(b[k] - 2.5 * a[k]).max() <= 1e-12 * np.abs(b[k]).max(), k
    for k in ("s1", "s2", "s3", "s9"):
        assert np.array_equal(a[k], b[k]), k


def test_zero_padding_invariance():
    """Appending zero grid points / zero Cholesky vectors / zero ERI-grid columns leaves the original block of R
    unchanged and makes the padded entries vanish (tile edges, non-multiple-of-tile sizes)."""
    import torch
    dims, d = _setup()
    o, v, NL, NP, NX = dims
    ref = _eval(dims, d)
    pP, pL, pX = 5, 3, 7
    z = lambda *s: torch.zeros(*s, dtype=torch.float64, device="cuda")
    d2 = dict(d)
    d2["Xo"] = torch.cat([d["Xo"], z(o, pP)], 1).contiguous()
    d2["Xv"] = torch.cat([d["Xv"], z(v, pP)], 1).contiguous()
    Z = z(NP + pP, NP + pP); Z[:NP, :NP] = d["Z"]; d2["Z"] = Z
    for k, sh in (("B_ov", (pL, o, v)), ("B_oo", (pL, o, o)), ("B_vv", (pL, v, v))):
        d2[k] = torch.cat([d[k], z(*sh)], 0).contiguous()
    d2["Y"] = torch.cat([d["Y"], z(o + v, pX)], 1).contiguous()
    V = z(NX + pX, NX + pX); V[:NX, :NX] = d["V"]; d2["V"] = V
    got = _eval((o, v, NL + pL, NP + pP, NX + pX), d2)
    for k in TERMS + ("R",):
        scale = np.abs(ref[k]).max()
        assert np.abs(got[k][:NP, :NP] - ref[k]).max() <= 1e-11 * scale, k
        assert np.abs(got[k][NP:, :]).max() <= 1e-13 * scale and np.abs(got[k][:, NP:]).max() <= 1e-13 * scale, k
    assert abs(got["E"] - ref["E"]) <= 1e-10 * max(1.0, abs(ref["E"]))

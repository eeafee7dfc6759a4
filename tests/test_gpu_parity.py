"""Parity of the CUDA path (through the C ABI) against the dense CPU oracle, element by element.

Tolerances (BASELINE.json north_star): max|R_gpu - R_ref| / max|R_ref| <= 1e-10 for the
total AND for each of the six terms against that term's own maximum (the T2^2 terms are ~1e-6 of the total at the
BASELINE Z scale, so a total-only check would not see them); |E_gpu - E_ref| <= 1e-9 E_h.
"""
import numpy as np
import pytest

from conftest import small_inputs, oracle_eval

pytestmark = pytest.mark.gpu

TERMS = ("s1", "s2", "s3", "s6", "s7", "s9")
RTOL = 1e-10
ETOL = 1e-9


def _to_dev(x):
    import torch
    names = ("Xo", "Xv", "Z", "B_ov", "B_oo", "B_vv", "Y", "V", "eps")
    return [torch.from_numpy(np.ascontiguousarray(getattr(x, n))).cuda() for n in names]


def _relerr(got, ref):
    scale = np.abs(ref).max()
    if scale == 0.0:
        return np.abs(got).max()
    return np.abs(got - ref).max() / scale


def _check_against(x, ref, **opts):
    import torch
    import paper_2111_11473_b200 as thc
    h = thc.thc_setup(x.o, x.v, x.NL, x.NP, x.NX, **opts)
    d = _to_dev(x)
    res = h.thc_residual_terms(*d)
    R2 = h.thc_residual(*d)
    E = h.thc_energy(d[0], d[1], d[2], d[3])
    torch.cuda.synchronize()
    errs = {}
    for k in TERMS + ("R", "xi_oo", "xi_vv"):
        errs[k] = _relerr(res[k].cpu().numpy(), ref[k])
    errs["R_direct"] = _relerr(R2.cpu().numpy(), ref["R"])
    errs["E_abs"] = abs(E - ref["E"])
    assert h.kernel_launches > 0
    h.close()
    bad = {k: e for k, e in errs.items() if e > (ETOL if k == "E_abs" else RTOL)}
    assert not bad, f"parity failures {bad} (all: {errs})"
    return errs


def test_config0_per_term(oracle_cfg):
    x, ref = oracle_cfg(0)
    _check_against(x, ref)


def test_config1_per_term(oracle_cfg):
    x, ref = oracle_cfg(1)
    _check_against(x, ref)


@pytest.mark.parametrize("dims", [(3, 4, 6, 5, 7), (7, 13, 19, 37, 45), (6, 18, 10, 64, 96), (2, 35, 5, 33, 17)])
def test_ragged_shapes_with_large_amplitudes(dims):
    """Odd / non-multiple-of-tile extents (scalar load path, ragged tile tails); Z scaled up so that the
    T2^2 terms are O(1) of the total."""
    x = small_inputs(*dims, seed=11, zmul=30.0)
    ref = oracle_eval(x)
    _check_against(x, ref)


@pytest.mark.parametrize("blocks", [dict(bL=1, bP7=1, bX=16, bI=1), dict(bL=5, bP7=7, bX=32, bI=9),
                                    dict(bL=64, bP7=64, bX=64, bI=64)])
def test_block_size_invariance(blocks):
    """Results must not depend on the L / P / X / I blocking."""
    x = small_inputs(6, 14, 21, 40, 52, seed=3, zmul=30.0)
    ref = oracle_eval(x)
    _check_against(x, ref, **blocks)


@pytest.mark.parametrize("dims", [(6, 18, 10, 64, 96), (66, 10, 6, 34, 40), (4, 6, 3, 642, 8)])
def test_tma_gemm_path_on_small_shapes(dims):
    """Every aligned K-major product forced onto the TMA-fed GEMM kernel (tma_min_flop=1): batched, k-batched, aux,
    transposed-copy, upper-only and split-K launches of the plan on shapes with ragged tiles."""
    x = small_inputs(*dims, seed=13, zmul=30.0)
    ref = oracle_eval(x)
    _check_against(x, ref, tma_min_flop=1)
    _check_against(x, ref, tma_min_flop=1, bL=3, bP7=5, bX=32, bI=10)


def test_term_mask_and_zero_cases():
    import torch
    import paper_2111_11473_b200 as thc
    x = small_inputs(4, 9, 8, 24, 30, seed=2, zmul=30.0)
    ref = oracle_eval(x)
    d = _to_dev(x)
    for name, bit in thc.TERM_BITS.items():
        h = thc.thc_setup(x.o, x.v, x.NL, x.NP, x.NX, term_mask=bit | (thc.TERM_BITS["s2"] if name == "s9" else 0))
        res = h.thc_residual_terms(*d)
        assert _relerr(res[name].cpu().numpy(), ref[name]) <= RTOL, name
        h.close()
    # Z = 0, B = 0  =>  R = 0 (north_star)
    h = thc.thc_setup(x.o, x.v, x.NL, x.NP, x.NX)
    z = [torch.zeros_like(t) for t in d]
    R = h.thc_residual(d[0], d[1], z[2], z[3], z[4], z[5], d[6], d[7], d[8])
    assert float(R.abs().max()) == 0.0
    # Z = 0  =>  R = A A^T
    R = h.thc_residual(d[0], d[1], z[2], d[3], d[4], d[5], d[6], d[7], d[8]).cpu().numpy()
    A = np.einsum("iP,aP,Lia->PL", x.Xo, x.Xv, x.B_ov)
    assert _relerr(R, A @ A.T) <= RTOL
    h.close()


def test_host_entry_matches_oracle(oracle_cfg):
    import torch
    import paper_2111_11473_b200 as thc
    x, ref = oracle_cfg(0)
    names = ("Xo", "Xv", "Z", "B_ov", "B_oo", "B_vv", "Y", "V", "eps")
    host = [torch.from_numpy(np.ascontiguousarray(getattr(x, n))).pin_memory() for n in names]
    R = torch.empty(x.NP, x.NP, dtype=torch.float64).pin_memory()
    h = thc.thc_setup(x.o, x.v, x.NL, x.NP, x.NX)
    E = h.thc_residual_host(*host, R)
    assert _relerr(R.numpy(), ref["R"]) <= RTOL
    assert abs(E - ref["E"]) <= ETOL
    h.close()


@pytest.mark.parametrize("mode", ["host", "provider"])
def test_streamed_bvv_matches_resident(mode):
    """B_vv streamed in L-blocks (pinned host memory, or a provider callback that fills device blocks on demand;
    PAPER.md l.191-195, BASELINE config 4) must give bit-identical results to the resident path."""
    import torch
    import paper_2111_11473_b200 as thc
    x = small_inputs(6, 14, 21, 40, 52, seed=3, zmul=30.0)
    ref = oracle_eval(x)
    d = _to_dev(x)
    h0 = thc.thc_setup(x.o, x.v, x.NL, x.NP, x.NX, bL=4)
    R0 = h0.thc_residual(*d).cpu().numpy()
    h0.close()
    h = thc.thc_setup(x.o, x.v, x.NL, x.NP, x.NX, bL=4, bvv_mode=mode)
    calls = []
    lib_stream = torch.cuda.current_stream().cuda_stream
    if mode == "host":
        bvv = torch.from_numpy(np.ascontiguousarray(x.B_vv)).pin_memory()
    else:
        def bvv(L0, nl, dst):
            calls.append((L0, nl))
            assert torch.cuda.current_stream().cuda_stream == lib_stream      # fills must be ordered with the GEMMs
            dst.copy_(d[5][L0:L0 + nl])
    args = list(d)
    args[5] = bvv
    for _ in range(2):                      # twice: the double buffer must be reusable across calls
        R = h.thc_residual(*args).cpu().numpy()
        assert np.array_equal(R, R0)
        assert getattr(h, "_provider_error", None) is None, h._provider_error
    assert _relerr(R, ref["R"]) <= RTOL
    if mode == "provider":
        assert calls[:3] == [(0, 4), (4, 4), (8, 4)] and calls[5] == (20, 1)
    h.close()


def test_provider_fill_is_stream_ordered_at_scale():
    """A fast provider (device-to-device copy) on a problem large enough that an unordered fill would overwrite the
    double buffer before the previous block's GEMM has read it (regression: fills once ran on a torch pool stream)."""
    import torch
    import paper_2111_11473_b200 as thc
    from thc_synth.device import make_inputs_device
    o, v, NL, NP, NX = 16, 256, 96, 320, 64
    d = make_inputs_device(o, v, NL, NP, NX, seed=12)
    names = ("Xo", "Xv", "Z", "B_ov", "B_oo", "B_vv", "Y", "V", "eps")
    mask = thc.TERM_BITS["s1"] | thc.TERM_BITS["s3"]
    h0 = thc.thc_setup(o, v, NL, NP, NX, bL=8, term_mask=mask)
    ref = h0.thc_residual(*[d[n] for n in names]).clone()
    h0.close()
    h = thc.thc_setup(o, v, NL, NP, NX, bL=8, term_mask=mask, bvv_mode="provider")
    args = [d[n] for n in names]
    args[5] = lambda L0, nl, dst: dst.copy_(d["B_vv"][L0:L0 + nl])
    for _ in range(3):
        R = h.thc_residual(*args)
        assert torch.equal(R, ref)
    h.close()


def test_unfused_alg7_path_o_above_64():
    """o > 64 takes the Alg.7 path that BASELINE configs 3 and 4 use (no 64-wide fused kernel): checked here against
    the dense oracle on a cheap shape so that a regression is caught without the multi-minute runs."""
    x = small_inputs(66, 9, 5, 33, 40, seed=21, zmul=30.0)
    ref = oracle_eval(x)
    _check_against(x, ref)
    _check_against(x, ref, bP7=4, bX=16, bI=16)


def test_symmetric_half_path_odd_NP():
    """NP >= 640 switches the half-transforms to upper-tile GEMMs + mirror; odd NP takes the scalar load path."""
    x = small_inputs(3, 4, 3, 641, 8, seed=22, zmul=30.0)
    ref = oracle_eval(x)
    _check_against(x, ref)


def test_check_symmetry_option_rejects_unsymmetric_inputs():
    import paper_2111_11473_b200 as thc
    x = small_inputs(4, 9, 8, 24, 30, seed=2, zmul=30.0)
    ref = oracle_eval(x)
    _check_against(x, ref, check_symmetry=True)               # symmetric inputs pass
    d = _to_dev(x)
    for k in (2, 4, 5, 7):                                    # Z, B_oo, B_vv, V
        bad = [t.clone() for t in d]
        bad[k].view(-1)[1] += 1e-3                            # element (0, 1) of the first matrix
        h = thc.thc_setup(x.o, x.v, x.NL, x.NP, x.NX, check_symmetry=True)
        with pytest.raises(thc.ThcError, match="invalid argument"):
            h.thc_residual(*bad)
        h.close()


def test_probe_reports_plausible_ceilings():
    import paper_2111_11473_b200 as thc
    h = thc.thc_setup(4, 8, 4, 16, 16)
    p = h.thc_probe()
    h.close()
    assert 20.0 < p["dmma_tflops"] < 60.0 and 20.0 < p["dfma_tflops"] < 60.0, p
    assert 60.0 < p["lds128_bytes_per_clk_per_sm"] <= 140.0, p


@pytest.mark.parametrize("dims", [(3, 4, 6, 5, 7), (7, 13, 19, 37, 45), (6, 18, 10, 64, 96), (20, 9, 5, 33, 40)])
def test_n5_gemm_only_t2sq_variant(dims):
    """sigma6 through the O(N^5) GEMM-only Alg.4 + Alg.5 instead of Alg.6: same oracle, same
    tolerance, O(1) amplitudes so that the term is not negligible; both variants forced explicitly."""
    x = small_inputs(*dims, seed=19, zmul=30.0)
    ref = oracle_eval(x)
    _check_against(x, ref, t2sq_algorithm=5)
    _check_against(x, ref, t2sq_algorithm=4)


def test_n5_variant_config0_and_config1(oracle_cfg):
    for cfg in (0, 1):
        x, ref = oracle_cfg(cfg)
        _check_against(x, ref, t2sq_algorithm=5)

"""Parity of the CUDA path against the T2 sampled-row oracle (oracle/rows.py) at sizes the dense oracle cannot hold.

Configs 2 and 3 run by default, in the launch configuration bench.py times (config 3 is its default workload); config 4
is opt-in (THC_BIG_TESTS=4: an evaluation takes ~13 minutes; its oracle rows take hours of CPU and are read from
tests/golden/ where tests/golden/make_rows.py has stored them, else computed live).  Inputs are drawn on the device by
thc_synth.device and the very same tensors are copied to the host for the oracle.  Tolerances as in test_gpu_parity.py:
1e-10 relative to each term's own maximum over the sampled rows, 1e-9 E_h on the energy.
"""
import os

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TERMS = ("s1", "s2", "s3", "s6", "s7", "s9")
NAMES = ("Xo", "Xv", "Z", "B_ov", "B_oo", "B_vv", "Y", "V", "eps")


def _run(cfg, rows, rows_s6, lblock, terms=TERMS, check_xi_and_energy=True, provider=False, cheap_pins=None):
    import torch
    import paper_2111_11473_b200 as thc
    from thc_synth import CONFIGS
    from thc_synth.device import make_config_device
    from oracle.rows import RowOracle

    import time
    from thc_synth import device as synth
    c = CONFIGS[cfg]
    d = make_config_device(cfg, with_bvv=not provider)
    if provider:                                   # config 4: B_vv only ever exists one L-block at a time

        def bvv_fill(L0, nl, dst):
            synth.bvv_block(c["seed"], c["o"], c["v"], c["NL"], L0, L0 + nl, "cuda", out=dst)
        d["B_vv"] = bvv_fill
    h = thc.thc_setup(c["o"], c["v"], c["NL"], c["NP"], c["NX"], bvv_mode="provider" if provider else "device")
    print(f"config {cfg}: blocks {h.blocks}, workspace {h.workspace_bytes / 1e9:.1f} GB", flush=True)
    args = [d[n] for n in NAMES]
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    res = h.thc_residual_terms(*args)
    torch.cuda.synchronize()
    print(f"config {cfg}: one residual evaluation (all terms) {time.perf_counter() - t0:.1f} s", flush=True)
    E = h.thc_energy(d["Xo"], d["Xv"], d["Z"], d["B_ov"])
    torch.cuda.synchronize()
    cheap = {}
    if cheap_pins:
        # energy contribution of single Cholesky vectors: NL ranks -> rank L owns exactly vector L
        for L in cheap_pins["L"]:
            cheap[("E", L)] = float(h.thc_energy_shard(d["Xo"], d["Xv"], d["Z"], d["B_ov"][L:L + 1].contiguous(), L, c["NL"])[0])
        # eps part of sigma9 at this NP: a handle with one zero Cholesky vector (xi = 0, sigma1..3 = 0)
        h0 = thc.thc_setup(c["o"], c["v"], 1, c["NP"], c["NX"], term_mask=thc.TERM_BITS["s9"] | thc.TERM_BITS["s2"])
        z = lambda *shape: torch.zeros(*shape, dtype=torch.float64, device="cuda")
        r0 = h0.thc_residual_terms(d["Xo"], d["Xv"], d["Z"], z(1, c["o"], c["v"]), z(1, c["o"], c["o"]),
                                   z(1, c["v"], c["v"]), d["Y"], d["V"], d["eps"])
        cheap["s9_eps"] = r0["s9"][cheap_pins["P"]].cpu().numpy()
        h0.close()
        del r0
    got = {k: res[k][list(rows)].cpu().numpy() for k in TERMS + ("R",)}
    if os.environ.get("THC_ROWS_SAVE"):          # the sampled GPU rows, for tests/test_rows_offline.py (stored oracle rows that
        np.savez(os.environ["THC_ROWS_SAVE"], cfg=cfg, rows=np.array(rows), **got)      # arrive after this run)
    xi_oo, xi_vv = res["xi_oo"].cpu().numpy(), res["xi_vv"].cpu().numpy()
    sym = float((res["R"] - res["R"].T).abs().max() / res["R"].abs().max())
    h.close()
    del res
    host = {n: d[n].cpu().numpy() for n in NAMES if torch.is_tensor(d[n])}
    del d, args
    torch.cuda.empty_cache()
    if provider:                                   # the oracle reads the same generator, block by block
        host["B_vv"] = lambda L0, L1: synth.bvv_block(c["seed"], c["o"], c["v"], c["NL"], L0, L1, "cuda").cpu().numpy()

    ro = RowOracle(*[host[n] for n in NAMES], lblock=lblock)
    errs = {"R_symmetry": sym}
    if check_xi_and_energy:
        rxo, rxv = ro.xi()
        errs["xi_oo"] = np.abs(xi_oo - rxo).max() / np.abs(rxo).max()
        errs["xi_vv"] = np.abs(xi_vv - rxv).max() / np.abs(rxv).max()
        errs["E_abs"] = abs(E - ro.energy())
    if cheap_pins:
        t0 = time.perf_counter()
        for L in cheap_pins["L"]:
            sub = [host[n][L:L + 1] if n in ("B_ov", "B_oo") else host[n] for n in NAMES]
            sub[5] = np.zeros((1, c["v"], c["v"]))
            e_ref = RowOracle(*sub, lblock=1).energy()
            errs[f"E_L{L}_abs"] = abs(cheap[("E", L)] - e_ref)
        j, b = cheap_pins["j"], cheap_pins["b"]
        col, row_v = ro.xi_oo_column(j), ro.xi_vv_row(b)
        errs["xi_oo_column"] = np.abs(xi_oo[:, j] - col).max() / np.abs(col).max()
        errs["xi_vv_row"] = np.abs(xi_vv[b] - row_v).max() / np.abs(row_v).max()
        zero = [np.zeros((1,) + host[n].shape[1:]) if n in ("B_ov", "B_oo") else host[n] for n in NAMES]
        zero[5] = np.zeros((1, c["v"], c["v"]))
        s9_ref = RowOracle(*zero, lblock=1).row(cheap_pins["P"], terms=("s9",))["s9"]
        errs["s9_eps_part"] = np.abs(cheap["s9_eps"] - s9_ref).max() / np.abs(s9_ref).max()
        print(f"config {cfg}: cheap pins (E per vector, xi column/row, sigma9 eps part) {time.perf_counter() - t0:.0f} s CPU", flush=True)
    # stored expected rows (tests/golden/config<C>_row<P>_<term>.txt, written by tests/golden/make_rows.py from oracle/ alone)
    # replace the live oracle for the terms they hold: at config 4 a row takes longer than a GPU-box call may last
    from golden.make_rows import load_rows
    stored = {P: load_rows(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden"), cfg, P) for P in rows}
    if any("s6" in stored[P] for P in rows) and "s6" not in terms:
        terms = tuple(k for k in TERMS if k in terms or k == "s6")
    ref = {k: [] for k in terms}
    all_terms = terms
    for n, P in enumerate(rows):
        terms = tuple(k for k in all_terms if k != "s6" or P in rows_s6 or "s6" in stored[P])
        live = tuple(k for k in terms if k not in stored[P])
        t0 = time.perf_counter()
        r = dict(stored[P])
        if live:
            r.update(ro.row(P, terms=live))
        print(f"config {cfg}: oracle row P={P}: live {live} in {time.perf_counter() - t0:.0f} s CPU, stored "
              f"{tuple(k for k in terms if k in stored[P])}", flush=True)
        for k in terms:
            ref[k].append((n, r[k]))
    for k in all_terms:
        if not ref[k]:
            continue
        scale = max(np.abs(r).max() for _, r in ref[k])
        errs[k] = max(np.abs(got[k][n] - r).max() for n, r in ref[k]) / scale
    bad = {k: e for k, e in errs.items() if e > (1e-9 if k.startswith("E_") else 1e-10)}
    assert not bad, f"parity failures {bad} (all: {errs})"
    print(f"config {cfg} sampled-row parity: {errs}")


def test_config2_sampled_rows():
    _run(2, rows=(3, 777), rows_s6=(3,), lblock=16)


def test_config3_sampled_rows():
    """BASELINE config 3 (the bench.py default workload): ~40 s of GPU and ~9 min of CPU row oracle."""
    _run(3, rows=(1234,), rows_s6=(1234,), lblock=8)


@pytest.mark.skipif(not os.environ.get("THC_BIG_TESTS", "").startswith("4"),
                    reason="set THC_BIG_TESTS=4 (config 4: ~40 GB resident, B_vv streamed, ~15 min of GPU; rows stored under "
                           "tests/golden/ are used, missing ones cost ~1 h of CPU; THC_BIG_TESTS=4s6 forces a sigma6 row)")
def test_config4_sampled_rows_streamed_bvv():
    """Paper-scale config: B_vv (304 GB) comes from a provider callback one L-block at a time.  One sampled row of
    sigma1, sigma2, sigma3, sigma7 (and sigma6 with THC_BIG_TESTS=4s6) against the row oracle; the energy through
    sampled Cholesky vectors (thc_energy_shard with one vector per rank vs the oracle restricted to that vector, long
    double); xi_oo / xi_vv through one sampled column / row (Eqs.39-40 with one index fixed); sigma9 through its
    eps part (a second handle with NL = 1 and B = 0: Alg.9 at this NP without the xi dressing).  The xi part of sigma9
    is linear in xi and shares the Alg.9 code path with the eps part; a row of it would need the full xi (hours of CPU):
    DESIGN.md section 5 lists it as unpinned at this config."""
    s6 = os.environ.get("THC_BIG_TESTS") == "4s6"
    _run(4, rows=(2718,), rows_s6=(2718,) if s6 else (), lblock=4,
         terms=("s1", "s2", "s3", "s6", "s7") if s6 else ("s1", "s2", "s3", "s7"),
         check_xi_and_energy=False, provider=True, cheap_pins=dict(L=(0, 3141, 7499), j=123, b=1999, P=2718))

"""The CUDA shard / finish entry points against the unsharded CUDA path and the oracle: the ranks of a world of 2, 3
and 5 are evaluated one after the other on one device and their packed buffers summed by hand (no rank waits on
another; the real exchange is one all-reduce, covered over gloo in test_sharded_gloo.py)."""
import numpy as np
import pytest

from conftest import small_inputs, oracle_eval

pytestmark = pytest.mark.gpu

NAMES = ("Xo", "Xv", "Z", "B_ov", "B_oo", "B_vv", "Y", "V", "eps")
TERMS = ("s1", "s2", "s3", "s6", "s7", "s9")


@pytest.mark.parametrize("world", [2, 3, 5])
def test_sharded_matches_unsharded(world):
    import torch
    import paper_2111_11473_b200 as thc
    x = small_inputs(6, 14, 4 if world == 5 else 21, 40, 52, seed=3, zmul=30.0)      # world 5 > NL 4: empty ranges
    ref = oracle_eval(x)
    d = {n: torch.from_numpy(np.ascontiguousarray(getattr(x, n))).cuda() for n in NAMES}
    h = thc.thc_setup(x.o, x.v, x.NL, x.NP, x.NX, bL=4, bX=16, bP7=5)
    full = h.thc_residual_terms(*[d[n] for n in NAMES])
    E_full = h.thc_energy(d["Xo"], d["Xv"], d["Z"], d["B_ov"])
    total = torch.zeros(h.shard_doubles, dtype=torch.float64, device="cuda")
    E = torch.zeros(1, dtype=torch.float64, device="cuda")
    for r in range(world):
        L0, L1, _, _ = thc.thc_shard_range(x.NL, x.NP, r, world)
        sl = [d["Xo"], d["Xv"], d["Z"], d["B_ov"][L0:L1].contiguous(), d["B_oo"][L0:L1].contiguous(),
              d["B_vv"][L0:L1].contiguous(), d["Y"], d["V"], d["eps"]]
        total += h.thc_residual_shard(*sl, r, world)
        E += h.thc_energy_shard(d["Xo"], d["Xv"], d["Z"], sl[3], r, world)
    res = h.thc_residual_finish(d["Xo"], d["Xv"], d["Z"], d["Y"], d["V"], d["eps"], total, want_terms=True)
    torch.cuda.synchronize()
    for k in TERMS + ("R",):
        a, b, c = res[k].cpu().numpy(), full[k].cpu().numpy(), ref[k]
        assert np.abs(a - b).max() <= 1e-12 * np.abs(b).max(), k
        assert np.abs(a - c).max() <= 1e-10 * np.abs(c).max(), k
    assert abs(float(E[0]) - E_full) <= 1e-12 * max(1.0, abs(E_full))
    assert abs(float(E[0]) - ref["E"]) <= 1e-9
    h.close()


@pytest.mark.parametrize("mode", ["host", "provider"])
@pytest.mark.parametrize("world", [2, 3])
def test_sharded_streamed_bvv(world, mode):
    """Sharded evaluation with B_vv streamed from pinned host memory (the rank's slice, or the whole array) or from a
    provider callback (global Cholesky indices): every rank must see ITS vectors."""
    import torch
    import paper_2111_11473_b200 as thc
    x = small_inputs(6, 14, 21, 40, 52, seed=3, zmul=30.0)
    ref = oracle_eval(x)
    d = {n: torch.from_numpy(np.ascontiguousarray(getattr(x, n))).cuda() for n in NAMES}
    bvv_host = torch.from_numpy(np.ascontiguousarray(x.B_vv)).pin_memory()
    calls = []

    def fill(L0, nl, dst):
        calls.append((L0, nl))
        dst.copy_(d["B_vv"][L0:L0 + nl])
    h = thc.thc_setup(x.o, x.v, x.NL, x.NP, x.NX, bL=4, bX=16, bP7=5, bvv_mode=mode)
    total = torch.zeros(h.shard_doubles, dtype=torch.float64, device="cuda")
    for r in range(world):
        L0, L1, _, _ = thc.thc_shard_range(x.NL, x.NP, r, world)
        if mode == "provider":
            bvv = fill
        else:                                       # rank 0 passes the whole array, the others their slice
            bvv = bvv_host if r == 0 else bvv_host[L0:L1].contiguous().pin_memory()
        sl = [d["Xo"], d["Xv"], d["Z"], d["B_ov"][L0:L1].contiguous(), d["B_oo"][L0:L1].contiguous(), bvv,
              d["Y"], d["V"], d["eps"]]
        n0 = len(calls)
        total += h.thc_residual_shard(*sl, r, world)
        if mode == "provider":                      # the callback was asked for exactly this rank's GLOBAL range
            got = calls[n0:]
            assert got[0][0] == L0 and got[-1][0] + got[-1][1] == L1
            assert all(a[0] + a[1] == b[0] for a, b in zip(got, got[1:]))
    R = h.thc_residual_finish(d["Xo"], d["Xv"], d["Z"], d["Y"], d["V"], d["eps"], total).cpu().numpy()
    assert np.abs(R - ref["R"]).max() <= 1e-10 * np.abs(ref["R"]).max()
    h.close()

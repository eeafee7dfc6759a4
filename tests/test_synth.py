"""The seeded input generator: determinism, order-freedom, structure (no method arithmetic in it)."""
import os

import numpy as np

from thc_synth import make_inputs, bvv_block, normal_block, CONFIGS


def test_deterministic_and_order_free():
    a = make_inputs(3, 4, 6, 5, 7, seed=5)
    b = make_inputs(3, 4, 6, 5, 7, seed=5)
    for n in ("eps", "Xo", "Xv", "Z", "B_oo", "B_ov", "B_vv", "Y", "V"):
        assert np.array_equal(getattr(a, n), getattr(b, n))
    idx = np.arange(100, dtype=np.uint64)
    full = normal_block(7, 3, idx)
    perm = np.random.default_rng(0).permutation(100)
    assert np.array_equal(normal_block(7, 3, idx[perm]), full[perm])
    assert np.array_equal(bvv_block(5, 3, 4, 6, 2, 5), a.B_vv[2:5])
    c = make_inputs(3, 4, 6, 5, 7, seed=6)
    assert not np.array_equal(a.Xo, c.Xo)


def test_structure_and_distributions():
    x = make_inputs(6, 30, 40, 64, 128, seed=1)
    assert np.array_equal(x.Z, x.Z.T) and np.array_equal(x.V, x.V.T)
    assert np.array_equal(x.B_vv, x.B_vv.transpose(0, 2, 1))
    assert np.array_equal(x.B_oo, x.B_oo.transpose(0, 2, 1))
    assert np.linalg.eigvalsh(x.V).min() > -1e-12
    assert np.all(x.eps[:6] >= -1.5) and np.all(x.eps[:6] <= -0.3)
    assert np.all(x.eps[6:] >= 0.1) and np.all(x.eps[6:] <= 3.0)
    assert abs(x.Xv.std() * np.sqrt(64) - 1) < 0.08
    assert abs(x.Y.std() * np.sqrt(128) - 1) < 0.05
    # off-diagonal of (G+G^T)/2 has std 1/sqrt(2); Z scale 0.1
    off = x.Z[np.triu_indices(64, 1)]
    assert abs(off.std() / (0.1 / np.sqrt(2)) - 1) < 0.08
    # Cholesky decay exp(-L / (NL/4))
    r = x.B_vv[39].std() / x.B_vv[0].std()
    assert abs(r / np.exp(-39 / 10.0) - 1) < 0.15
    g = normal_block(3, 9, np.arange(200000, dtype=np.uint64))
    assert abs(g.mean()) < 0.01 and abs(g.std() - 1) < 0.01
    assert abs(np.mean(g ** 4) - 3) < 0.1


def test_configs_match_baseline():
    assert CONFIGS[0] == dict(o=5, v=20, NL=60, NP=50, NX=100, seed=0)
    assert CONFIGS[4] == dict(o=250, v=2250, NL=7500, NP=5000, NX=10000, seed=4)


def test_device_generator_matches_numpy_generator():
    """thc_synth.device (torch ops; used on the GPU for configs 3-4) draws the same tensors as generators.py."""
    import torch
    from thc_synth import generators as g
    from thc_synth import device as dv
    idx = np.array([0, 1, 5, 123456789, 2 ** 40 + 7], dtype=np.uint64)
    assert np.array_equal(g.uniform_block(3, 5, idx), dv.uniform_block(3, 5, torch.from_numpy(idx.astype(np.int64))).numpy())
    x = g.make_inputs(3, 4, 6, 5, 7, seed=9)
    d = dv.make_inputs_device(3, 4, 6, 5, 7, seed=9, device="cpu")
    for k in ("eps", "Xo", "Xv", "Z", "B_oo", "B_ov", "B_vv", "Y", "V"):
        assert np.abs(getattr(x, k) - d[k].numpy()).max() <= 1e-14, k
    blk = dv.bvv_block(9, 3, 4, 6, 2, 5, "cpu").numpy()
    assert np.abs(blk - x.B_vv[2:5]).max() <= 1e-14


def test_lazy_cholesky_blocks_equal_the_full_arrays():
    """LazyCholesky draws B_oo / B_ov block by block: any slice equals the same slice of the arrays make_inputs returns."""
    from thc_synth import LazyCholesky, make_inputs
    x = make_inputs(3, 5, 9, 4, 6, seed=11, with_bvv=False)
    for kind, full in (("oo", x.B_oo), ("ov", x.B_ov)):
        lazy = LazyCholesky(11, 3, 5, 9, kind)
        assert lazy.shape == full.shape
        for sl in (slice(0, 4), slice(4, 9), slice(8, 12)):
            assert np.array_equal(lazy[sl], full[sl])


def test_golden_row_writer_round_trip(tmp_path):
    """tests/golden/make_rows.py (oracle + generators only) writes exact hex floats; drawing the Cholesky vectors block by
    block gives the rows of the in-memory oracle up to the summation order over L-blocks."""
    import subprocess
    import sys
    from golden.make_rows import load_rows
    from oracle.rows import RowOracle
    from thc_synth import make_config
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    subprocess.run([sys.executable, os.path.join(root, "tests", "golden", "make_rows.py"), "--config", "0", "--row", "7",
                    "--terms", "s1,s2,s3,s6,s7", "--outdir", str(tmp_path)], check=True, timeout=600, cwd=root)
    got = load_rows(str(tmp_path), 0, 7)
    x = make_config(0)
    ref = RowOracle(x.Xo, x.Xv, x.Z, x.B_ov, x.B_oo, x.B_vv, x.Y, x.V, x.eps).row(7, terms=tuple(got))
    assert set(got) == {"s1", "s2", "s3", "s6", "s7"}
    for k in got:
        assert np.abs(got[k] - ref[k]).max() <= 1e-13 * np.abs(ref[k]).max(), k

"""Pins of the T2 sampled-row oracle (oracle/rows.py) against the dense oracle of record (oracle/dense.py), per term,
on config 0 and on ragged miniatures with O(1) amplitudes; plus the callable-B_vv path and the long-double energy."""
import numpy as np
import pytest

from conftest import small_inputs, oracle_eval
from oracle.rows import RowOracle, TERMS


def _rows_vs_dense(x, ref, rows, **kw):
    ro = RowOracle(x.Xo, x.Xv, x.Z, x.B_ov, x.B_oo, x.B_vv, x.Y, x.V, x.eps, **kw)
    xi_oo, xi_vv = ro.xi()
    assert np.abs(xi_oo - ref["xi_oo"]).max() <= 1e-12 * max(1.0, np.abs(ref["xi_oo"]).max())
    assert np.abs(xi_vv - ref["xi_vv"]).max() <= 1e-12 * max(1.0, np.abs(ref["xi_vv"]).max())
    for P in rows:
        got = ro.row(P)
        for k in TERMS:
            scale = np.abs(ref[k]).max()
            assert np.abs(got[k] - ref[k][P]).max() <= 1e-12 * scale, (k, P)
    assert abs(ro.energy() - ref["E"]) <= 1e-11 * max(1.0, abs(ref["E"]))


def test_rows_match_dense_config0(oracle_cfg):
    x, ref = oracle_cfg(0)
    _rows_vs_dense(x, ref, rows=(0, 17, 49), lblock=7)


@pytest.mark.parametrize("dims", [(3, 4, 6, 5, 7), (4, 9, 8, 12, 15), (2, 7, 5, 9, 70)])
def test_rows_match_dense_ragged(dims):
    x = small_inputs(*dims, seed=21, zmul=30.0)
    ref = oracle_eval(x)
    _rows_vs_dense(x, ref, rows=range(dims[3]), lblock=4)


def test_rows_callable_bvv():
    x = small_inputs(3, 5, 7, 6, 8, seed=4, zmul=30.0)
    ref = oracle_eval(x)
    ro = RowOracle(x.Xo, x.Xv, x.Z, x.B_ov, x.B_oo, lambda L0, L1: x.B_vv[L0:L1], x.Y, x.V, x.eps, lblock=3)
    got = ro.row(2, terms=("s1", "s3"))
    for k in ("s1", "s3"):
        assert np.abs(got[k] - ref[k][2]).max() <= 1e-12 * np.abs(ref[k]).max()


@pytest.mark.parametrize("dims", [(3, 4, 6, 5, 7), (4, 9, 8, 12, 15)])
def test_single_xi_column_and_row_match_dense(dims):
    """xi_oo_column / xi_vv_row (used where the full xi is unaffordable, BASELINE config 4) against the dense oracle's
    xi of Eqs.39-40 -- every column / row, so that a transposed index would show (xi_oo is not symmetric, R5)."""
    x = small_inputs(*dims, seed=23, zmul=30.0)
    ref = oracle_eval(x)
    ro = RowOracle(x.Xo, x.Xv, x.Z, x.B_ov, x.B_oo, x.B_vv, x.Y, x.V, x.eps, lblock=3)
    assert np.abs(ref["xi_oo"] - ref["xi_oo"].T).max() > 1e-6 * np.abs(ref["xi_oo"]).max()
    for j in range(x.o):
        assert np.abs(ro.xi_oo_column(j) - ref["xi_oo"][:, j]).max() <= 1e-12 * np.abs(ref["xi_oo"]).max(), j
    for b in range(x.v):
        assert np.abs(ro.xi_vv_row(b) - ref["xi_vv"][b]).max() <= 1e-12 * np.abs(ref["xi_vv"]).max(), b


def test_sigma6_row_over_the_first_outer_grid_points():
    """bench.py's bounded CPU sample hands the row oracle the first nxi rows of V: the sigma6 row is then the partial sum
    over the outer ERI-grid points I < nxi (J over the whole grid), i.e. the full row for a V whose other rows are zero."""
    x = small_inputs(3, 4, 5, 6, 10, seed=12)
    nxi, P = 4, 2
    part = RowOracle(x.Xo, x.Xv, x.Z, x.B_ov, x.B_oo, x.B_vv, x.Y, x.V[:nxi], x.eps).row(P, terms=("s6",))["s6"]
    Vz = x.V.copy()
    Vz[nxi:] = 0.0
    full = RowOracle(x.Xo, x.Xv, x.Z, x.B_ov, x.B_oo, x.B_vv, x.Y, Vz, x.eps).row(P, terms=("s6",))["s6"]
    assert np.abs(part - full).max() <= 1e-14 * np.abs(full).max()
    whole = RowOracle(x.Xo, x.Xv, x.Z, x.B_ov, x.B_oo, x.B_vv, x.Y, x.V, x.eps).row(P, terms=("s6",))["s6"]
    assert np.abs(part - whole).max() > 1e-3 * np.abs(whole).max()          # it really is a part, not the whole

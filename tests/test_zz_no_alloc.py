"""Allocation-free entry point thc_dgemm_static (include/thc.h) against the existing workspace-based thc_dgemm.

Collected last on purpose (pytest -x): the entry point shares one static device array between calls, so the
test runs it twice in a row with different shapes (the second call sees the first one's partial tiles in the scratch) and
must pass both alone in a fresh process and after every other GPU test of the suite."""
import ctypes

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = 1e-13      # relative to max|C| * sqrt(K): the bound tests/test_gpu_kernels.py uses for the DMMA GEMM


def _existing(M, N, K, alpha, A, B, beta, C):
    import paper_2111_11473_b200 as thc
    h = thc.thc_setup(4, 8, 4, 16, 16)
    try:
        h.thc_dgemm(1, 1, M, N, K, alpha, A, A.stride(0), B, B.stride(0), beta, C, C.stride(0))
    finally:
        h.close()


def _case(seed, M, N, K, pad, splits):
    import torch
    import paper_2111_11473_b200 as thc
    rng = np.random.default_rng(seed)
    A = torch.from_numpy(rng.standard_normal((M, K + pad))).cuda()
    B = torch.from_numpy(rng.standard_normal((N, K + pad))).cuda()
    C0 = torch.from_numpy(rng.standard_normal((M, N + pad))).cuda()
    Av, Bv = A[:, :K], B[:, :K]
    want = C0.clone()
    _existing(M, N, K, 0.7, A, B, -1.3, want)
    got = C0.clone()
    thc.thc_dgemm_static(Av, Bv, got[:, :N], 0.7, -1.3, splits)
    torch.cuda.synchronize()
    want, got, C0 = want.cpu().numpy(), got.cpu().numpy(), C0.cpu().numpy()
    dense = 0.7 * (A.cpu().numpy()[:, :K] @ B.cpu().numpy()[:, :K].T) - 1.3 * C0[:, :N]
    scale = np.abs(dense).max() * max(1.0, np.sqrt(K))
    assert np.abs(got[:, :N] - want[:, :N]).max() <= TOL * scale
    assert np.abs(got[:, :N] - dense).max() <= TOL * scale
    assert np.array_equal(got[:, N:], C0[:, N:])          # padding columns untouched


def test_static_dgemm_two_calls_in_a_row():
    """Two calls back to back, the second with other extents and another split count: stale partial tiles of the first
    call must not leak into the second.  Then the first shape again (scratch now holds the second call's tiles)."""
    import paper_2111_11473_b200 as thc
    thc.thc_static_init(-1)
    _case(1, 200, 300, 1029, 0, 5)       # 16-byte path, ragged tiles, K tail
    _case(2, 37, 41, 2000, 1, 0)         # odd leading dimensions (8-byte path), library-chosen splits
    _case(1, 200, 300, 1029, 0, 5)
    _case(3, 64, 64, 16, 0, 1)           # one split: no scratch at all


def test_static_dgemm_rejects_sizes_beyond_the_scratch():
    import torch
    import paper_2111_11473_b200 as thc
    M = N = 1024
    A = torch.zeros(M, 64, dtype=torch.float64, device="cuda")
    C = torch.zeros(M, N, dtype=torch.float64, device="cuda")
    assert 3 * M * N * 8 > thc.STATIC_SCRATCH_BYTES >= 2 * M * N * 8
    thc.thc_dgemm_static(A, A, C, splits=2)                     # exactly at the limit
    with pytest.raises(thc.ThcError, match="THC_STATIC_SCRATCH_BYTES"):
        thc.thc_dgemm_static(A, A, C, splits=3)
    thc.thc_dgemm_static(A, A, C, splits=0)                     # auto never exceeds the limit
    torch.cuda.synchronize()
    assert thc.lib().thc_dgemm_static(-1, None, 8, 8, 8, -1, 1.0, ctypes.c_void_p(A.data_ptr()), 64,
                                      ctypes.c_void_p(A.data_ptr()), 64, 0.0, ctypes.c_void_p(C.data_ptr()), N) == -1

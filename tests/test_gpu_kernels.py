"""Unit parity of the two compute kernels exposed through the C ABI: the FP64 DMMA GEMM and Alg.6 line 11."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _handle():
    import paper_2111_11473_b200 as thc
    return thc.thc_setup(4, 8, 4, 16, 16)


@pytest.mark.parametrize("akm,bkm", [(1, 1), (1, 0), (0, 1), (0, 0)])
@pytest.mark.parametrize("M,N,K", [(1, 1, 1), (5, 7, 3), (64, 64, 16), (65, 130, 17), (200, 300, 129), (37, 41, 2000),
                                   (300, 520, 77), (1024, 1024, 256)])
def test_dgemm_against_numpy(akm, bkm, M, N, K):
    """C = alpha A B^T + beta C in every operand layout, tile-ragged extents, odd leading dimensions (scalar
    cp.async path) and even ones (16-byte path), split-K (37 x 41 x 2000)."""
    import torch
    rng = np.random.default_rng(M * 1000003 + N * 1009 + K)
    for pad in (0, 1):
        lda = (K if akm else M) + pad + (1 if (M + N + K) % 2 else 0)
        ldb = (K if bkm else N) + pad
        ldc = N + pad
        A = rng.standard_normal((M if akm else K, lda))
        B = rng.standard_normal((N if bkm else K, ldb))
        C = rng.standard_normal((M, ldc))
        Am = A[:, :K] if akm else A[:, :M].T
        Bm = B[:, :K] if bkm else B[:, :N].T
        ref = C.copy()
        ref[:, :N] = 0.7 * (Am @ Bm.T) - 1.3 * C[:, :N]
        h = _handle()
        Ad, Bd, Cd = (torch.from_numpy(t).cuda() for t in (A, B, C))
        h.thc_dgemm(akm, bkm, M, N, K, 0.7, Ad, lda, Bd, ldb, -1.3, Cd, ldc)
        got = Cd.cpu().numpy()
        h.close()
        scale = np.abs(ref).max()
        assert np.abs(got - ref).max() <= 1e-13 * scale * max(1.0, np.sqrt(K)), (pad, np.abs(got - ref).max() / scale)
        assert np.array_equal(got[:, N:], C[:, N:])      # padding columns untouched


@pytest.mark.parametrize("nI,nP,NPp", [(1, 16, 32), (5, 32, 64), (7, 16, 96), (33, 48, 160)])
def test_triple_product_against_numpy(nI, nP, NPp):
    """H[p,q,r] (+)= sum_I (E[I,p,q] F[I,p,r] + E[I,p,r] F[I,p,q]) G[I,q,r]   (Alg.6 line 11, l.714)."""
    import torch
    rng = np.random.default_rng(nI * 7 + nP + NPp)
    E = rng.standard_normal((nI, nP, NPp))
    F = rng.standard_normal((nI, nP, NPp))
    G = rng.standard_normal((nI, NPp, NPp))
    H0 = rng.standard_normal((nP, NPp, NPp))
    upd = np.einsum("ipq,ipr,iqr->pqr", E, F, G) + np.einsum("ipr,ipq,iqr->pqr", E, F, G)
    h = _handle()
    Ed, Fd, Gd = (torch.from_numpy(t).cuda() for t in (E, F, G))
    for acc in (0, 1):
        Hd = torch.from_numpy(H0).cuda()
        h.thc_triple_product(nI, nP, NPp, Ed, Fd, Gd, Hd, acc)
        ref = upd + (H0 if acc else 0.0)
        got = Hd.cpu().numpy()
        assert np.abs(got - ref).max() <= 1e-13 * np.abs(ref).max() * max(1.0, np.sqrt(nI)), acc
    h.close()


@pytest.mark.parametrize("M,N,K", [(8, 8, 8), (2, 300, 6), (130, 150, 22), (150, 700, 100), (700, 150, 100), (513, 257, 333),
                                   (1024, 1024, 256), (37, 41, 2000), (160, 64, 16), (129, 129, 17)])
def test_dgemm_tma_kernel_against_numpy(M, N, K):
    """The TMA-fed persistent kernel (forced for every aligned K-major product with tma_min_flop=1): ragged tiles and K
    tails are zero-filled by the TMA unit; 128x128, 160x64 and 64x160 tiles; split-K (37 x 41 x 2000)."""
    import torch
    import paper_2111_11473_b200 as thc
    rng = np.random.default_rng(M * 7919 + N * 104729 + K)
    lda, ldb, ldc = K + (K & 1) + 2, K + (K & 1), N + 3
    A, B, C = rng.standard_normal((M, lda)), rng.standard_normal((N, ldb)), rng.standard_normal((M, ldc))
    ref = C.copy()
    ref[:, :N] = 0.7 * (A[:, :K] @ B[:, :K].T) - 1.3 * C[:, :N]
    h = thc.thc_setup(4, 8, 4, 16, 16, tma_min_flop=1)
    Ad, Bd, Cd = (torch.from_numpy(t).cuda() for t in (A, B, C))
    h.thc_dgemm(1, 1, M, N, K, 0.7, Ad, lda, Bd, ldb, -1.3, Cd, ldc)
    got = Cd.cpu().numpy()
    h.close()
    scale = np.abs(ref).max()
    assert np.abs(got - ref).max() <= 1e-13 * scale * max(1.0, np.sqrt(K)), np.abs(got - ref).max() / scale
    assert np.array_equal(got[:, N:], C[:, N:])

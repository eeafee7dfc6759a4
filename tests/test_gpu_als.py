"""GPU parity of thc_cp_als_update (Appendix I, Eqs.43-46 + PCG) against oracle/als.py, element by element."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = 1e-10


def _problem(I, J, K, N, seed, noise=0.05):
    """A = exact rank-N tensor + noise (the shape of a projector U^P_ia, l.124-135, with I = NP, J = o, K = v)."""
    rng = np.random.default_rng(seed)
    X, Y, Z = (rng.standard_normal((n, N)) for n in (I, J, K))
    A = np.einsum("in,jn,kn->ijk", X, Y, Z) + noise * rng.standard_normal((I, J, K))
    return A, Y, Z, rng.standard_normal((I, N))


def _run(I, J, K, N, iters, seed):
    import torch
    import paper_2111_11473_b200 as thc
    from oracle import als
    A, Y, Z, X0 = _problem(I, J, K, N, seed)
    want, want_rn = als.als_update(A, Y, Z, X0, iters)
    h = thc.thc_setup(2, 3, 2, 8, 8)
    try:
        Ad, Yd, Zd = (torch.from_numpy(t).cuda() for t in (A, Y, Z))
        for _ in range(2):
            Xd = torch.from_numpy(X0).cuda()
            rn = h.thc_cp_als_update(Ad, Yd, Zd, Xd, iters, want_rnorm2=True)
            torch.cuda.synchronize()
            got = Xd.cpu().numpy()
            assert np.abs(got - want).max() <= TOL * np.abs(want).max(), np.abs(got - want).max() / np.abs(want).max()
            # |r|^2 is a difference of large numbers once converged: compare on the scale of |R_i|^2
            scale = np.sum(als.mttkrp(A, Y, Z) ** 2, axis=1).max()
            assert np.abs(rn.cpu().numpy() - want_rn).max() <= TOL * scale
    finally:
        h.close()
    return want, A, Y, Z


@pytest.mark.parametrize("I,J,K,N,iters", [(50, 5, 20, 10, 4), (300, 20, 100, 64, 6), (37, 7, 13, 5, 3), (1, 1, 1, 1, 1),
                                           (130, 3, 67, 33, 0)])
def test_als_update_matches_the_oracle_iteration_by_iteration(I, J, K, N, iters):
    """Same iteration count on both sides: ragged / odd extents, a single row, zero iterations (X unchanged, true residual)."""
    _run(I, J, K, N, iters, seed=I + N)


def test_converged_update_is_the_least_squares_solution():
    """Enough iterations: the result equals the LAPACK solve of Eq.44 (checked on the oracle's side too)."""
    want, A, Y, Z = _run(64, 8, 24, 12, 40, seed=2)
    from oracle import als
    direct = np.linalg.solve(als.gram(Y, Z), als.mttkrp(A, Y, Z).T).T
    assert np.abs(want - direct).max() <= 1e-9 * np.abs(direct).max()


def test_khatri_rao_blocks():
    """J K N large enough that Eq.46 runs over two Khatri-Rao blocks of j (54 + 6)."""
    _run(50, 60, 128, 1200, 2, seed=3)


def test_full_als_sweeps_decrease_the_misfit():
    """Three updates per sweep (X, Y, Z in turn, each on the correspondingly permuted copy of A, as l.373 keeps them):
    with converged least-squares solves the misfit |A - [[X, Y, Z]]| cannot increase from one update to the next."""
    import torch
    import paper_2111_11473_b200 as thc
    rng = np.random.default_rng(8)
    I, J, K, N = 40, 12, 30, 6
    Xt, Yt, Zt = (rng.standard_normal((n, N)) for n in (I, J, K))
    A = np.einsum("in,jn,kn->ijk", Xt, Yt, Zt) + 0.01 * rng.standard_normal((I, J, K))
    perms = [np.ascontiguousarray(A.transpose(p)) for p in ((0, 1, 2), (1, 2, 0), (2, 0, 1))]     # [I,J,K], [J,K,I], [K,I,J]
    dev = [torch.from_numpy(p).cuda() for p in perms]
    f = [torch.from_numpy(t + 0.3 * rng.standard_normal(t.shape)).cuda() for t in (Xt, Yt, Zt)]

    def misfit():
        X, Y, Z = (t.cpu().numpy() for t in f)
        return np.linalg.norm(A - np.einsum("in,jn,kn->ijk", X, Y, Z))

    h = thc.thc_setup(2, 3, 2, 8, 8)
    try:
        hist = [misfit()]
        for _ in range(6):
            for m in range(3):                      # update factor m with the other two fixed, in cyclic order
                h.thc_cp_als_update(dev[m], f[(m + 1) % 3], f[(m + 2) % 3], f[m], 4 * N)
                torch.cuda.synchronize()
                hist.append(misfit())
    finally:
        h.close()
    assert all(b <= a * (1 + 1e-10) for a, b in zip(hist, hist[1:])), hist
    assert hist[-1] < 0.2 * hist[0], hist


def test_row_blocks_are_independent():
    """The paper's multi-GPU scheme (l.361, l.373): each device updates its own block of rows with the replicated Y, Z.
    Updating two row blocks separately gives the rows of the whole update."""
    import torch
    import paper_2111_11473_b200 as thc
    A, Y, Z, X0 = _problem(90, 6, 40, 16, seed=17)
    h = thc.thc_setup(2, 3, 2, 8, 8)
    try:
        Ad, Yd, Zd = (torch.from_numpy(t).cuda() for t in (A, Y, Z))
        whole = torch.from_numpy(X0).cuda()
        h.thc_cp_als_update(Ad, Yd, Zd, whole, 5)
        parts = []
        for i0, i1 in ((0, 37), (37, 90)):
            Xb = torch.from_numpy(X0[i0:i1].copy()).cuda()
            h.thc_cp_als_update(Ad[i0:i1].contiguous(), Yd, Zd, Xb, 5)
            parts.append(Xb)
        torch.cuda.synchronize()
        got, want = torch.cat(parts).cpu().numpy(), whole.cpu().numpy()
    finally:
        h.close()
    assert np.abs(got - want).max() <= 1e-12 * np.abs(want).max()


def test_als_update_at_config2_size_sampled_rows():
    """Projector-shaped array at BASELINE config 2 dimensions (I = NP = 1000, J = o = 60, K = v = 340, N = 1000 factors): the
    rows of the update are independent, so the oracle is run on three sampled rows (with the whole Y, Z)."""
    import torch
    import paper_2111_11473_b200 as thc
    from oracle import als
    I, J, K, N, iters = 1000, 60, 340, 1000, 8
    g = torch.Generator(device="cuda").manual_seed(5)
    rnd = lambda *s: torch.randn(*s, dtype=torch.float64, device="cuda", generator=g)
    A, Y, Z, X = rnd(I, J, K), rnd(J, N), rnd(K, N), rnd(I, N)
    rows = [0, 517, 999]
    X0 = X[rows].cpu().numpy()
    h = thc.thc_setup(2, 3, 2, 8, 8)
    try:
        rn = h.thc_cp_als_update(A, Y, Z, X, iters, want_rnorm2=True)
        torch.cuda.synchronize()
    finally:
        h.close()
    want, want_rn = als.als_update(A[rows].cpu().numpy(), Y.cpu().numpy(), Z.cpu().numpy(), X0, iters)
    got = X[rows].cpu().numpy()
    assert np.abs(got - want).max() <= TOL * np.abs(want).max(), np.abs(got - want).max() / np.abs(want).max()
    scale = np.sum(als.mttkrp(A[rows].cpu().numpy(), Y.cpu().numpy(), Z.cpu().numpy()) ** 2, axis=1).max()
    assert np.abs(rn[rows].cpu().numpy() - want_rn).max() <= TOL * scale

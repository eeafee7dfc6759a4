"""Pins of oracle/als.py (Appendix I, Eqs.43-46 l.355-373) against things other than itself."""
import numpy as np

from oracle import als


def _factors(I=5, J=4, K=6, N=3, seed=3):
    rng = np.random.default_rng(seed)
    return rng.standard_normal((I, N)), rng.standard_normal((J, N)), rng.standard_normal((K, N))


def test_gram_and_mttkrp_by_literal_loops():
    """Eqs.45-46 with every summation index as a Python loop (a transposed factor or a swapped j / k would show)."""
    X, Y, Z = _factors()
    I, J, K, N = X.shape[0], Y.shape[0], Z.shape[0], X.shape[1]
    A = np.random.default_rng(4).standard_normal((I, J, K))
    S = np.zeros((N, N))
    for n in range(N):
        for m in range(N):
            S[n, m] = sum(Y[j, n] * Y[j, m] for j in range(J)) * sum(Z[k, n] * Z[k, m] for k in range(K))
    R = np.zeros((I, N))
    for i in range(I):
        for n in range(N):
            R[i, n] = sum(A[i, j, k] * Y[j, n] * Z[k, n] for j in range(J) for k in range(K))
    assert np.abs(als.gram(Y, Z) - S).max() <= 1e-13 * np.abs(S).max()
    assert np.abs(als.mttkrp(A, Y, Z) - R).max() <= 1e-13 * np.abs(R).max()


def test_exact_cp_tensor_is_recovered():
    """A exactly of rank N with the true Y, Z: the least-squares solution of Eq.44 is the true X, and N PCG iterations
    reach it (CG terminates in at most N steps in exact arithmetic), from an unrelated starting guess."""
    X, Y, Z = _factors(6, 7, 8, 4)
    A = np.einsum("in,jn,kn->ijk", X, Y, Z)
    X0 = np.random.default_rng(9).standard_normal(X.shape)
    got, rn2 = als.als_update(A, Y, Z, X0, iters=8)
    assert np.abs(got - X).max() <= 1e-9 * np.abs(X).max()
    assert rn2.max() <= 1e-18 * np.abs(als.mttkrp(A, Y, Z)).max() ** 2


def test_pcg_converges_to_the_direct_solve_and_is_the_least_squares_minimiser():
    """For a general A the converged update equals R S^-1 (LAPACK solve) and minimises |A - [[X, Y, Z]]|_F over X:
    the gradient A_(1) (Z (.) Y) - X S vanishes and any perturbation of X increases the misfit."""
    X0, Y, Z = _factors(5, 6, 7, 4, seed=11)
    A = np.random.default_rng(12).standard_normal((5, 6, 7))
    got, _ = als.als_update(A, Y, Z, X0, iters=12)
    S, R = als.gram(Y, Z), als.mttkrp(A, Y, Z)
    want = np.linalg.solve(S, R.T).T
    assert np.abs(got - want).max() <= 1e-10 * np.abs(want).max()

    def misfit(Xm):
        return np.linalg.norm(A - np.einsum("in,jn,kn->ijk", Xm, Y, Z))

    base = misfit(got)
    assert base < misfit(X0)
    rng = np.random.default_rng(13)
    for _ in range(5):
        assert misfit(got + 1e-3 * rng.standard_normal(got.shape)) > base


def test_zero_iterations_and_orthogonal_factors():
    """iters = 0 returns the starting guess and its true residual; when Y and Z have orthogonal columns S is diagonal,
    the preconditioner is its exact inverse and ONE iteration solves every row."""
    X0, _, _ = _factors(4, 5, 6, 3, seed=21)
    rng = np.random.default_rng(22)
    Y = np.linalg.qr(rng.standard_normal((5, 3)))[0] * np.array([1.0, 2.0, 0.5])
    Z = np.linalg.qr(rng.standard_normal((6, 3)))[0] * np.array([3.0, 1.0, 0.25])
    A = rng.standard_normal((4, 5, 6))
    S, R = als.gram(Y, Z), als.mttkrp(A, Y, Z)
    assert np.abs(S - np.diag(np.diag(S))).max() <= 1e-14
    got0, rn0 = als.als_update(A, Y, Z, X0, iters=0)
    assert np.array_equal(got0, X0)
    assert np.abs(rn0 - np.sum((R - X0 @ S) ** 2, axis=1)).max() <= 1e-12 * rn0.max()
    got1, rn1 = als.als_update(A, Y, Z, X0, iters=1)
    assert np.abs(got1 - R / np.diag(S)).max() <= 1e-13 * np.abs(got1).max()
    got2, _ = als.als_update(A, Y, Z, got1, iters=3)          # already converged rows take zero steps, no NaN
    assert np.all(np.isfinite(got2)) and np.abs(got2 - got1).max() <= 1e-13 * np.abs(got1).max()

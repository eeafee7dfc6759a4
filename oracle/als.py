"""One alternating-least-squares factor update of a CP factorisation -- TEST INFRASTRUCTURE, not a product path.

PAPER.md Appendix I (l.355-373): A_ijk ~ sum_n X_i^n Y_j^n Z_k^n (Eq.43).  With Y and Z fixed the rows of X solve

    sum_n' S_nn' X_i^n' = R_i^n                                             (Eq.44 l.363)
    S_nn' = (sum_j Y_j^n Y_j^n') (sum_k Z_k^n Z_k^n')                       (Eq.45 l.367)
    R_i^n = sum_jk A_ijk Y_j^n Z_k^n                                        (Eq.46 l.371)

"by the preconditioned conjugate gradient method using the diagonal of S as the preconditioner" (l.373).  S and R have
plain definitions and are written out as such.  The solve is an iteration, so it follows the textbook PCG recurrence
step by step, one independent system per row i (l.373: "An update of the i-th row ... is independent of all other
rows"), started from the current X, for a fixed number of iterations.  A row whose search direction has p.Sp = 0 (it has
converged exactly) takes a zero step; a row with r.z = 0 keeps its direction unchanged (beta = 0).  The paper does not
print the recurrence or a stopping rule: DESIGN.md reading R22.

Layouts: A[I, J, K], X[I, N], Y[J, N], Z[K, N].
"""
from __future__ import annotations

import numpy as np


def gram(Y, Z):
    """S[n, n'] of Eq.45."""
    return (Y.T @ Y) * (Z.T @ Z)


def mttkrp(A, Y, Z):
    """R[i, n] of Eq.46."""
    return np.einsum("ijk,jn,kn->in", A, Y, Z, optimize=True)


def pcg_rows(S, R, X0, iters):
    """`iters` PCG iterations on S x_i = R_i for every row i, preconditioner diag(S), start X0.  Returns (X, rnorm2) with
    rnorm2[i] = |r_i|^2 of the recurrence residual after the last iteration."""
    d = np.diag(S).copy()
    X = np.array(X0, dtype=np.float64, copy=True)
    r = R - X @ S.T
    z = r / d
    p = z.copy()
    rz = np.sum(r * z, axis=1)
    for _ in range(iters):
        Sp = p @ S.T
        pSp = np.sum(p * Sp, axis=1)
        alpha = np.where(pSp != 0.0, rz / np.where(pSp != 0.0, pSp, 1.0), 0.0)
        X += alpha[:, None] * p
        r -= alpha[:, None] * Sp
        z = r / d
        rz_new = np.sum(r * z, axis=1)
        beta = np.where(rz != 0.0, rz_new / np.where(rz != 0.0, rz, 1.0), 0.0)
        p = z + beta[:, None] * p
        rz = rz_new
    return X, np.sum(r * r, axis=1)


def als_update(A, Y, Z, X0, iters):
    """The X update of one ALS sweep: Eqs.44-46 with `iters` PCG iterations from X0.  Returns (X, rnorm2)."""
    return pcg_rows(gram(Y, Z), mttkrp(A, Y, Z), X0, iters)

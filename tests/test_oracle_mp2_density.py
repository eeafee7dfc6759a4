"""Pins of oracle/mp2_density.py (Appendix II, Eqs.47-56 l.375-415) against things other than itself."""
import numpy as np

from conftest import small_inputs
from oracle import mp2_density


def _problem(o=3, v=4, NP=5, seed=17, symmetric=True):
    x = small_inputs(o, v, 6, NP, 7, seed=seed)
    Z = x.Z if symmetric else x.Z + np.triu(np.random.default_rng(seed).standard_normal((NP, NP)), 1)
    return x.Xo, x.Xv, Z


def test_literal_loops_over_eqs_47_48():
    """Every summation index of Eqs.47-48 (l.379-383) as a Python loop, amplitudes element by element from Eq.23: a
    swapped index in the exchange parts (t_jk^ba, t_ji^bc) or a wrong sign / factor would show.  Z is NOT symmetric here,
    so t_ij^ab != t_ji^ba and every index position matters."""
    Xo, Xv, Z = _problem(2, 3, 4, symmetric=False)
    o, v, NP = Xo.shape[0], Xv.shape[0], Z.shape[0]

    def t(i, j, a, b):
        return sum(Xo[i, P] * Xv[a, P] * Z[P, Q] * Xo[j, Q] * Xv[b, Q] for P in range(NP) for Q in range(NP))

    D_oo = np.zeros((o, o))
    for i in range(o):
        for j in range(o):
            D_oo[i, j] = -2 * sum(t(i, k, a, b) * (2 * t(j, k, a, b) - t(j, k, b, a))
                                  for k in range(o) for a in range(v) for b in range(v))
    D_vv = np.zeros((v, v))
    for a in range(v):
        for b in range(v):
            D_vv[a, b] = 2 * sum(t(i, j, a, c) * (2 * t(i, j, b, c) - t(j, i, b, c))
                                 for i in range(o) for j in range(o) for c in range(v))
    got_oo, got_vv = mp2_density.mp2_density(Xo, Xv, Z)
    assert np.abs(got_oo - D_oo).max() <= 1e-12 * np.abs(D_oo).max()
    assert np.abs(got_vv - D_vv).max() <= 1e-12 * np.abs(D_vv).max()


def test_one_occupied_orbital_closed_form():
    """o = 1: t_11^ab = M_ab with M = Xv diag(Xo) Z diag(Xo) Xv^T symmetric, so 2t - t~ = t and
    D_11 = -2 |M|_F^2, D_vv = 2 M M^T."""
    Xo, Xv, Z = _problem(1, 5, 6)
    M = (Xv * Xo[0]) @ Z @ (Xv * Xo[0]).T
    D_oo, D_vv = mp2_density.mp2_density(Xo, Xv, Z)
    assert abs(D_oo[0, 0] + 2 * np.sum(M * M)) <= 1e-12 * abs(D_oo[0, 0])
    assert np.abs(D_vv - 2 * M @ M.T).max() <= 1e-12 * np.abs(D_vv).max()


def test_trace_symmetry_and_definiteness():
    """tr D_oo = -tr D_vv (the number of electrons is conserved); for pair-symmetric amplitudes (symmetric Z) both
    blocks are symmetric, D_oo <= 0 and D_vv >= 0 (the closed-shell form 2t - t~ has eigenvalues 1 and 3)."""
    Xo, Xv, Z = _problem(3, 4, 5)
    D_oo, D_vv = mp2_density.mp2_density(Xo, Xv, Z)
    assert abs(np.trace(D_oo) + np.trace(D_vv)) <= 1e-12 * abs(np.trace(D_vv))
    assert np.abs(D_oo - D_oo.T).max() <= 1e-13 * np.abs(D_oo).max()
    assert np.abs(D_vv - D_vv.T).max() <= 1e-13 * np.abs(D_vv).max()
    assert np.linalg.eigvalsh(D_oo).max() <= 1e-13 * np.abs(D_oo).max()
    assert np.linalg.eigvalsh(D_vv).min() >= -1e-13 * np.abs(D_vv).max()


def _eqs_53_56(yo, yv, T):
    """The O(N^4) factorisation of Appendix II, innermost parenthesis first (l.407), in the paper's letters:
    o^{WX}, v^{WX} of Eqs.51-52; Coulomb-like parts Eqs.53-54; exchange-like parts Eqs.55-56."""
    no, nv = yo.shape[0], yv.shape[0]
    o = yo.T @ yo
    v = yv.T @ yv
    K = T @ ((o * v) @ T.T)                                   # K[W, Y] = sum_X T^WX sum_Z (o v)^XZ T^YZ
    D_oo = -4 * yo @ (v * K) @ yo.T                           # Eq.53
    D_vv = 4 * yv @ (o * K) @ yv.T                            # Eq.54
    for i in range(no):                                       # Eq.55
        for j in range(no):
            inner = np.einsum("W,aW,WX->aX", yo[i], yv, T)                # sum_W T^WX (y_i^W y_a^W)
            inner = np.einsum("aZ,aX->XZ", yv, inner)                     # sum_a y_a^Z ( . )
            inner = o * inner                                             # o^XZ ( . )
            inner = np.einsum("YZ,XZ->XY", T, inner)                      # sum_Z T^YZ ( . )
            inner = np.einsum("XY,XY->Y", v, inner)                       # sum_X v^XY ( . )
            D_oo[i, j] += 2 * yo[j] @ inner                               # sum_Y y_j^Y ( . )
    for a in range(nv):                                       # Eq.56
        for b in range(nv):
            inner = np.einsum("iW,W,WX->iX", yo, yv[a], T)
            inner = np.einsum("iZ,iX->XZ", yo, inner)
            inner = v * inner
            inner = np.einsum("YZ,XZ->XY", T, inner)
            inner = np.einsum("XY,XY->Y", o, inner)
            D_vv[a, b] -= 2 * yv[b] @ inner
    return D_oo, D_vv


def test_factorised_eqs_53_56_reproduce_the_definition():
    """Eqs.53-56 (l.401-413), restated line by line, equal Eqs.47-48 -- also for a non-symmetric T, which fixes the
    transposition of every T and of o / v in the exchange-like parts."""
    for symmetric in (True, False):
        Xo, Xv, Z = _problem(3, 4, 6, seed=23, symmetric=symmetric)
        want_oo, want_vv = mp2_density.mp2_density(Xo, Xv, Z)
        got_oo, got_vv = _eqs_53_56(Xo, Xv, Z)
        assert np.abs(got_oo - want_oo).max() <= 1e-12 * np.abs(want_oo).max()
        assert np.abs(got_vv - want_vv).max() <= 1e-12 * np.abs(want_vv).max()


def test_single_elements_equal_the_dense_blocks():
    """density_oo_element / density_vv_element (used at sizes where the dense t does not fit) against the dense oracle,
    every element, with a non-symmetric Z so that the index positions of the exchange parts matter."""
    Xo, Xv, Z = _problem(3, 4, 5, seed=29, symmetric=False)
    D_oo, D_vv = mp2_density.mp2_density(Xo, Xv, Z)
    for i in range(3):
        for j in range(3):
            assert abs(mp2_density.density_oo_element(Xo, Xv, Z, i, j) - D_oo[i, j]) <= 1e-12 * np.abs(D_oo).max()
    for a in range(4):
        for b in range(4):
            assert abs(mp2_density.density_vv_element(Xo, Xv, Z, a, b) - D_vv[a, b]) <= 1e-12 * np.abs(D_vv).max()

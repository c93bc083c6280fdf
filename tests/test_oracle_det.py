"""Pins for the oracle's determinant (oracle.wick_oracle.det_elim) against things other than itself:
the Leibniz definition Eq. (14), LAPACK, Cauchy-Binet, Jacobi's complementary-minor
identity (the only strong pin for n = 10, 11 where brute force is impossible), antisymmetry
Eq. (19), and singular matrices."""
import itertools

import numpy as np
import pytest

from oracle import wick_oracle as wo


def _rand(rng, *shape):
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


@pytest.mark.parametrize("n", [1, 2, 3, 4, 5, 6])
def test_det_elim_vs_leibniz(n):
    rng = np.random.default_rng(10 + n)
    for _ in range(4):
        M = _rand(rng, n, n)
        ref = wo.det_leibniz(M)
        got = wo.det_elim(M)
        assert abs(got - ref) <= 1e-12 * max(1.0, abs(ref))


@pytest.mark.parametrize("n", range(1, 13))
def test_det_elim_vs_lapack_batched(n):
    rng = np.random.default_rng(100 + n)
    M = _rand(rng, 64, n, n)
    ref = np.linalg.det(M)
    got = wo.det_elim(M)
    assert got.shape == (64,)
    assert np.all(np.abs(got - ref) <= 1e-11 * np.abs(ref))


def test_leibniz_closed_forms():
    # 2x2 and a triangular matrix pin the Leibniz routine itself (textbook values)
    M = np.array([[1 + 2j, 3], [4j, 5 - 1j]])
    assert abs(wo.det_leibniz(M) - ((1 + 2j) * (5 - 1j) - 3 * 4j)) < 1e-14
    Tm = np.triu(np.arange(1, 17).reshape(4, 4)).astype(complex)
    assert abs(wo.det_leibniz(Tm) - 1 * 6 * 11 * 16) < 1e-12
    assert abs(wo.det_elim(Tm) - 1 * 6 * 11 * 16) < 1e-12


@pytest.mark.parametrize("n", [10, 11])
def test_jacobi_complementary_minors(n):
    """det A[I,J] = (-1)^{sum I + sum J} det A det(A^-1)[J^c, I^c]  (0-based index sums).  For n = 10 / 11
    the right side only needs a 12x12 LAPACK det/inverse and a 2x2 / 1x1 minor."""
    rng = np.random.default_rng(7 + n)
    A = _rand(rng, 12, 12)
    Ainv = np.linalg.inv(A)
    dA = np.linalg.det(A)
    subsets = list(itertools.combinations(range(12), n))
    picks = rng.choice(len(subsets), size=(12, 2))
    for pi, pj in picks:
        I, J = subsets[pi], subsets[pj]
        Ic = [k for k in range(12) if k not in I]
        Jc = [k for k in range(12) if k not in J]
        comp = Ainv[np.ix_(Jc, Ic)]
        small = comp[0, 0] if len(Ic) == 1 else comp[0, 0] * comp[1, 1] - comp[0, 1] * comp[1, 0]
        ref = (-1) ** (sum(I) + sum(J)) * dA * small
        got = wo.det_elim(A[np.ix_(I, J)])
        assert abs(got - ref) <= 1e-10 * abs(ref)


@pytest.mark.parametrize("n", [2, 3, 5, 6])
def test_cauchy_binet(n):
    """det (AB)[I,J] = sum_K det A[I,K] det B[K,J] over all n-subsets K of {0..11}."""
    rng = np.random.default_rng(50 + n)
    A, B = _rand(rng, 12, 12), _rand(rng, 12, 12)
    I = tuple(sorted(rng.choice(12, n, replace=False)))
    J = tuple(sorted(rng.choice(12, n, replace=False)))
    Ks = np.array(list(itertools.combinations(range(12), n)))
    left = wo.det_elim((A @ B)[np.ix_(I, J)])
    dA = wo.det_elim(A[np.array(I)[None, :, None], Ks[:, None, :]])
    dB = wo.det_elim(B[Ks[:, :, None], np.array(J)[None, None, :]])
    right = np.sum(dA * dB)
    assert abs(left - right) <= 1e-11 * np.sum(np.abs(dA * dB))


def test_antisymmetry_eq19():
    """Eq. (19): permuting rows by sigma and columns by tau multiplies det by sgn(sigma) sgn(tau)."""
    rng = np.random.default_rng(3)
    S = _rand(rng, 12, 12)
    rows, cols = [1, 4, 7, 9, 10], [0, 2, 3, 8, 11]
    base = wo.det_elim(S[np.ix_(rows, cols)])
    for _ in range(10):
        ps, pt = rng.permutation(5), rng.permutation(5)
        ss, _ = wo.sort_with_sign(list(ps))
        st, _ = wo.sort_with_sign(list(pt))
        got = wo.det_elim(S[np.ix_([rows[i] for i in ps], [cols[i] for i in pt])])
        assert abs(got - ss * st * base) <= 1e-12 * abs(base)


def test_sort_with_sign_small_cases():
    assert wo.sort_with_sign([0, 1, 2]) == (1, (0, 1, 2))
    assert wo.sort_with_sign([1, 0, 2]) == (-1, (0, 1, 2))
    assert wo.sort_with_sign([2, 0, 1]) == (1, (0, 1, 2))      # cyclic = even
    assert wo.sort_with_sign([2, 1, 0]) == (-1, (0, 1, 2))
    assert wo.sort_with_sign([3, 3, 1])[0] == 0                 # repeated index: Pauli zero


def test_singular_and_zero_matrices():
    rng = np.random.default_rng(5)
    M = _rand(rng, 6, 6)
    M[:, 3] = 0
    assert wo.det_elim(M) == 0
    M = _rand(rng, 6, 6)
    M[4] = M[1]
    assert abs(wo.det_elim(M)) < 1e-12
    assert wo.det_elim(np.zeros((5, 5), dtype=complex)) == 0
    assert wo.det_elim(np.eye(7, dtype=complex)) == 1
    P = np.eye(6)[[1, 0, 2, 3, 4, 5]].astype(complex)           # one transposition
    assert wo.det_elim(P) == -1

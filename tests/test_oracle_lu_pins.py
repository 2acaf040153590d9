"""Pins for the linear-solve oracle (oracle/zkd_oracle.c: zkd_oracle_lu_solve; NEXT-3, "Gaussian elimination, LU
decomposition").  Expected values come from mpmath: closed forms, constructions, invariants - never from the oracle itself.

L1 2x2 Cramer closed form        L3 residual ||A X - B||            L5 third opinion: mpmath.lu_solve
L2 B = A X0 with chosen X0       L4 permutation / diagonal / triangular matrices (exact), singular -> status 1
"""
import random

import numpy as np

import oracle
import zkd_inputs as zi
from test_oracle_svd_pins import log2abs, rand_matrix, rmatrix_from_mp, rmatrix_to_mp


def solve(mp, A, B):
    N, nrhs = A.rows, B.cols
    Ab, Bb = rmatrix_from_mp(mp, A), rmatrix_from_mp(mp, B)
    X, rc = oracle.lu_solve(Ab, Bb, N, nrhs)
    return rc, rmatrix_to_mp(mp, X, N, nrhs), rmatrix_to_mp(mp, Ab, N, N), rmatrix_to_mp(mp, Bb, N, nrhs)


def test_L1_cramer(mp):
    rng = random.Random(1)
    A, B = rand_matrix(mp, rng, 2, 2), rand_matrix(mp, rng, 2, 1)
    rc, X, Ar, Br = solve(mp, A, B)
    assert rc == 0
    det = Ar[0, 0] * Ar[1, 1] - Ar[0, 1] * Ar[1, 0]
    want = [(Br[0, 0] * Ar[1, 1] - Ar[0, 1] * Br[1, 0]) / det, (Ar[0, 0] * Br[1, 0] - Br[0, 0] * Ar[1, 0]) / det]
    for i in range(2):
        assert log2abs(mp, X[i, 0] - want[i]) <= -760 + max(0, log2abs(mp, want[i]))


def test_L2_L3_constructed_and_residual(mp):
    rng = random.Random(2)
    N, nrhs = 9, 3
    A, X0 = rand_matrix(mp, rng, N, N), rand_matrix(mp, rng, N, nrhs)
    Ar = rmatrix_to_mp(mp, rmatrix_from_mp(mp, A), N, N)          # A as the oracle sees it (768 bit)
    B = Ar * X0                                                    # exact to 1200 bits; rounded to 768 on encoding
    rc, X, _, Br = solve(mp, Ar, B)
    assert rc == 0
    cond = mp.norm(Ar, 2) * mp.norm(Ar ** -1, 2)
    for i in range(N):
        for j in range(nrhs):
            assert log2abs(mp, X[i, j] - X0[i, j]) <= -762 + log2abs(mp, cond)
    R = Ar * X - Br
    assert max(log2abs(mp, R[i, j]) for i in range(N) for j in range(nrhs)) <= -758


def test_L4_exact_cases_and_singular(mp):
    N = 5
    perm = [3, 0, 4, 1, 2]
    A = mp.matrix(N, N)
    for i in range(N):
        A[i, perm[i]] = mp.mpc(0, 2) if i % 2 else mp.mpf(-4)     # powers of two: every quotient is exact
    B = mp.matrix(N, 1)
    for i in range(N):
        B[i, 0] = mp.mpc(i + 1, -i) / 8
    rc, X, _, _ = solve(mp, A, B)
    assert rc == 0
    for i in range(N):
        assert X[perm[i], 0] == B[i, 0] / A[i, perm[i]]
    # upper triangular with unit diagonal and dyadic entries: exact back substitution
    T = mp.eye(4)
    T[0, 1], T[0, 3], T[1, 2], T[2, 3] = mp.mpf(1) / 2, mp.mpc(0, 1) / 4, mp.mpf(-3) / 8, mp.mpf(5) / 16
    x0 = mp.matrix([mp.mpf(1), mp.mpc(1, 1), mp.mpf(-2), mp.mpf(3) / 4])
    rc, X, _, _ = solve(mp, T, T * x0)
    assert rc == 0 and all(X[i, 0] == x0[i] for i in range(4))
    # exactly singular: a zero column
    S = mp.matrix(3, 3)
    S[0, 0], S[1, 0], S[2, 2] = 1, 2, 3
    rc, _, _, _ = solve(mp, S, mp.matrix([1, 2, 3]))
    assert rc == 1


def test_L5_third_opinion(mp):
    rng = random.Random(5)
    N = 7
    A, B = rand_matrix(mp, rng, N, N), rand_matrix(mp, rng, N, 2)
    rc, X, Ar, Br = solve(mp, A, B)
    assert rc == 0
    for c in range(2):
        want = mp.lu_solve(Ar, Br[:, c])
        for i in range(N):
            assert log2abs(mp, X[i, c] - want[i]) <= -745

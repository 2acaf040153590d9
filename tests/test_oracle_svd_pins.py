"""Pins for the SVD oracle (oracle/zkd_oracle.c: zkd_oracle_svd, zkd_oracle_svd_compare; NEXT-1).
Every expected value is computed here with mpmath from closed forms, constructions and invariants - never by the oracle
itself and never by the CUDA path.

S1 2x2 closed form                              S5 rank-deficient, zero and diagonal inputs
S2 constructed U diag(sigma) V^H, M >=< N       S6 third opinion: mpmath.svd_c
S3 sigma^2 = eigenvalues of A^H A (mpmath)      S7 the comparator itself: group / projector logic against mpmath values
S4 ||A||_F^2 = sum sigma^2
"""
from fractions import Fraction

import numpy as np
import pytest

import oracle
import zkd_inputs as zi

P = 768
RB = zi.real_bytes(P)


def log2abs(mp, x):
    x = abs(x)
    return -10**9 if x == 0 else float(mp.log(x, 2))


def rmatrix_from_mp(mp, Mx, prec=P):
    rb = zi.real_bytes(prec)
    out = np.zeros((Mx.rows, Mx.cols, 2, rb), dtype=np.uint8)
    for i in range(Mx.rows):
        for j in range(Mx.cols):
            z = mp.mpc(Mx[i, j])
            out[i, j, 0] = np.frombuffer(zi.from_mpf(z.real, prec), dtype=np.uint8)
            out[i, j, 1] = np.frombuffer(zi.from_mpf(z.imag, prec), dtype=np.uint8)
    return out.reshape(-1)


def rmatrix_to_mp(mp, buf, R, C, prec=P):
    rb = zi.real_bytes(prec)
    flat = np.asarray(buf).reshape(R, C, 2, rb)
    Mx = mp.matrix(R, C)
    for i in range(R):
        for j in range(C):
            Mx[i, j] = mp.mpc(zi.to_mpf(flat[i, j, 0], prec), zi.to_mpf(flat[i, j, 1], prec))
    return Mx


def rvec_to_mp(buf, K, prec=P):
    rb = zi.real_bytes(prec)
    flat = np.asarray(buf).reshape(K, rb)
    return [zi.to_mpf(flat[i], prec) for i in range(K)]


def rand_c(mp, rng):
    return mp.mpc(mp.mpf(rng.getrandbits(900)) / mp.mpf(2) ** 899 - 1, mp.mpf(rng.getrandbits(900)) / mp.mpf(2) ** 899 - 1)


def rand_matrix(mp, rng, R, C):
    A = mp.matrix(R, C)
    for i in range(R):
        for j in range(C):
            A[i, j] = rand_c(mp, rng)
    return A


def rand_unitary(mp, rng, n, reflectors=3):
    Q = mp.eye(n)
    for _ in range(reflectors):
        u = mp.matrix(n, 1)
        for i in range(n):
            u[i] = rand_c(mp, rng)
        nn = sum(abs(u[i]) ** 2 for i in range(n))
        H = mp.eye(n) - 2 * (u * u.H) / nn
        Q = Q * H
    return Q


def run_svd(mp, A):
    M, N = A.rows, A.cols
    K = min(M, N)
    buf = rmatrix_from_mp(mp, A)
    S, U, V, info = oracle.svd(buf, M, N)
    assert info["status"] == 0, info
    return buf, S, U, V, rvec_to_mp(S, K), rmatrix_to_mp(mp, U, M, K), rmatrix_to_mp(mp, V, N, K)


def check_svd_invariants(mp, A, s, U, V, bits=-758):
    M, N, K = A.rows, A.cols, len(s)
    F = mp.sqrt(sum(abs(A[i, j]) ** 2 for i in range(M) for j in range(N)))
    F = F if F > 0 else mp.mpf(1)
    for j in range(K):
        r1 = mp.sqrt(sum(abs(sum(A[i, k] * V[k, j] for k in range(N)) - s[j] * U[i, j]) ** 2 for i in range(M)))
        r2 = mp.sqrt(sum(abs(sum(mp.conj(A[i, k]) * U[i, j] for i in range(M)) - s[j] * V[k, j]) ** 2 for k in range(N)))
        assert log2abs(mp, r1 / F) <= bits and log2abs(mp, r2 / F) <= bits, (j, log2abs(mp, r1 / F), log2abs(mp, r2 / F))
    for X, rows in ((U, M), (V, N)):
        for a in range(K):
            for b in range(K):
                g = sum(mp.conj(X[k, a]) * X[k, b] for k in range(rows)) - (1 if a == b else 0)
                assert log2abs(mp, g) <= bits, (a, b, log2abs(mp, g))
    assert all(s[j] >= s[j + 1] for j in range(K - 1)) and all(x >= 0 for x in s)
    # phase convention: the first largest-modulus component of v_j is real positive
    for j in range(K):
        k = max(range(N), key=lambda i: (abs(V[i, j]), -i))
        assert mp.im(V[k, j]) == 0 and mp.re(V[k, j]) > 0


def test_S1_two_by_two_closed_form(mp):
    import random

    rng = random.Random(1)
    for _ in range(3):
        A = rand_matrix(mp, rng, 2, 2)
        _, _, _, _, s, U, V = run_svd(mp, A)
        S2 = sum(abs(A[i, j]) ** 2 for i in range(2) for j in range(2))
        det = A[0, 0] * A[1, 1] - A[0, 1] * A[1, 0]
        disc = mp.sqrt(S2 ** 2 - 4 * abs(det) ** 2)
        want = [mp.sqrt((S2 + disc) / 2), mp.sqrt((S2 - disc) / 2)]
        for g, w in zip(s, want):
            assert log2abs(mp, g - w) <= -762
        check_svd_invariants(mp, A, s, U, V)


@pytest.mark.parametrize("M,N", [(6, 6), (7, 4), (3, 6)])
def test_S2_constructed(mp, M, N):
    import random

    rng = random.Random(100 * M + N)
    K = min(M, N)
    sig = [mp.mpf(3) / 2, mp.mpf(1), mp.mpf(2) ** -40, mp.mpf(2) ** -300, mp.mpf(5) / 8, mp.mpf(1) / 3][:K]
    sig = sorted(sig, reverse=True)
    QU, QV = rand_unitary(mp, rng, M), rand_unitary(mp, rng, N)
    A = mp.matrix(M, N)
    for i in range(M):
        for j in range(N):
            A[i, j] = sum(QU[i, k] * sig[k] * mp.conj(QV[j, k]) for k in range(K))
    buf, S, U, V, s, Um, Vm = run_svd(mp, A)
    for g, w in zip(s, sig):
        assert log2abs(mp, g - w) <= -760, (float(g), float(w))   # A was rounded to 768 bits: |dsigma| <= 2^-768 ||A||
    Ar = rmatrix_to_mp(mp, buf, M, N)
    check_svd_invariants(mp, Ar, s, Um, Vm)
    # vectors: the pair (u_j, v_j) equals the constructed pair up to ONE common phase, to 2^-768 ||A|| / gap
    for j in range(K):
        ip = sum(mp.conj(QV[k, j]) * Vm[k, j] for k in range(N))
        ph = ip / abs(ip)
        gap = min([abs(sig[j] - sig[i]) for i in range(K) if i != j] + [2 * sig[j]])
        eu = mp.sqrt(sum(abs(Um[k, j] - QU[k, j] * ph) ** 2 for k in range(M)))
        ev = mp.sqrt(sum(abs(Vm[k, j] - QV[k, j] * ph) ** 2 for k in range(N)))
        assert log2abs(mp, eu) <= -756 - log2abs(mp, gap) and log2abs(mp, ev) <= -756 - log2abs(mp, gap), (j, log2abs(mp, eu))


def test_S3_S4_gram_eigenvalues_and_frobenius(mp):
    import random

    rng = random.Random(3)
    A = rand_matrix(mp, rng, 6, 4)
    buf, S, U, V, s, Um, Vm = run_svd(mp, A)
    Ar = rmatrix_to_mp(mp, buf, 6, 4)
    G = Ar.H * Ar
    ev = sorted(mp.eighe(G, eigvals_only=True), reverse=True)   # independent route: mpmath's Hermitian eigensolver
    for g, w in zip(s, ev):
        assert log2abs(mp, g * g - w) <= -755
    F2 = sum(abs(Ar[i, j]) ** 2 for i in range(6) for j in range(4))
    assert log2abs(mp, sum(x * x for x in s) - F2) <= -758
    check_svd_invariants(mp, Ar, s, Um, Vm)


def test_S5_rank_deficient_zero_diagonal(mp):
    import random

    rng = random.Random(5)
    # rank 2, 5 x 4: sigma_3 = sigma_4 = 0 up to the rounding of A to 768 bits
    B, C = rand_matrix(mp, rng, 5, 2), rand_matrix(mp, rng, 2, 4)
    A = B * C
    buf, S, U, V, s, Um, Vm = run_svd(mp, A)
    Ar = rmatrix_to_mp(mp, buf, 5, 4)
    assert log2abs(mp, s[2]) <= -755 and log2abs(mp, s[3]) <= -755 and s[1] > mp.mpf(2) ** -10
    check_svd_invariants(mp, Ar, s, Um, Vm, bits=-750)
    # zero matrix
    Z = mp.matrix(3, 5)
    _, _, _, _, s, Um, Vm = run_svd(mp, Z)
    assert all(x == 0 for x in s)
    check_svd_invariants(mp, Z, s, Um, Vm)
    # diagonal with a negative and a complex entry: sigma = |d|, descending
    D = mp.matrix(4, 4)
    d = [mp.mpc(-3, 0) / 4, mp.mpc(0, 2), mp.mpc(1, 1) / 8, mp.mpc(5, 0) / 16]
    for i in range(4):
        D[i, i] = d[i]
    _, _, _, _, s, Um, Vm = run_svd(mp, D)
    for g, w in zip(s, sorted((abs(x) for x in d), reverse=True)):
        assert log2abs(mp, g - w) <= -764
    check_svd_invariants(mp, D, s, Um, Vm)


def test_S6_third_opinion_mpmath_svd(mp):
    import random

    rng = random.Random(6)
    A = rand_matrix(mp, rng, 5, 3)
    buf, S, U, V, s, Um, Vm = run_svd(mp, A)
    Ar = rmatrix_to_mp(mp, buf, 5, 3)
    s3 = mp.svd_c(Ar, compute_uv=False)
    for g, w in zip(s, [s3[i] for i in range(3)]):
        assert log2abs(mp, g - w) <= -758


def test_S7_comparator_against_mpmath(mp):
    """zkd_oracle_svd_compare: (i)-(iii) against mpmath on a perturbed decomposition, and the group logic of (iv): a common
    phase on (u_j, v_j) and a unitary remix inside a degenerate group change nothing; a 2^-700 leak between two groups is
    reported at 2^-700 and measured against the right gap; an opposite phase on u_j and v_j (which breaks A v = sigma u) is
    caught by the stacked comparison."""
    import random

    rng = random.Random(7)
    M, N, K = 6, 5, 5
    sig = [mp.mpf(2), mp.mpf(1), mp.mpf(1), mp.mpf(1), mp.mpf(1) / 4]        # a 3-fold singular value
    QU, QV = rand_unitary(mp, rng, M), rand_unitary(mp, rng, N)
    U0, V0 = QU[:, :K], QV[:, :K]
    A = mp.matrix(M, N)
    for i in range(M):
        for j in range(N):
            A[i, j] = sum(U0[i, k] * sig[k] * mp.conj(V0[j, k]) for k in range(K))
    enc = lambda Mx: rmatrix_from_mp(mp, Mx)
    encs = lambda v: np.concatenate([np.frombuffer(zi.from_mpf(x), dtype=np.uint8) for x in v])
    Ab = enc(A)
    F = mp.sqrt(sum(x * x for x in sig))
    base = oracle.svd_compare(Ab, M, N, encs(sig), enc(U0), enc(V0), encs(sig), enc(U0), enc(V0))
    assert base["groups"] == 3 and base["max_group"] == 3
    assert base["log2_resid_rel"] <= -760 and base["log2_orth"] <= -760 and base["vec_margin_bits"] <= -20
    # common phases and a unitary remix of the 3-fold group: still the same decomposition
    W = rand_unitary(mp, rng, 3)
    U1, V1 = U0.copy(), V0.copy()
    for i in range(M):
        for b in range(3):
            U1[i, 1 + b] = sum(U0[i, 1 + a] * W[a, b] for a in range(3))
    for i in range(N):
        for b in range(3):
            V1[i, 1 + b] = sum(V0[i, 1 + a] * W[a, b] for a in range(3))
    ph = mp.expj(mp.mpf(1) / 3)
    for i in range(M):
        U1[i, 0] *= ph
    for i in range(N):
        V1[i, 0] *= ph
    c = oracle.svd_compare(Ab, M, N, encs(sig), enc(U1), enc(V1), encs(sig), enc(U0), enc(V0))
    assert c["log2_resid_rel"] <= -758 and c["log2_orth"] <= -758 and c["vec_margin_bits"] <= -15, c
    # a 2^-700 leak of pair 4 into pair 0:  z_0 += eps z_4  ->  err = eps ||z_4|| / sqrt 2 ... = eps (stacked vectors scaled to 1)
    eps = mp.mpf(2) ** -700
    U2, V2 = U0.copy(), V0.copy()
    for i in range(M):
        U2[i, 0] = U0[i, 0] + eps * U0[i, 4]
    for i in range(N):
        V2[i, 0] = V0[i, 0] + eps * V0[i, 4]
    c = oracle.svd_compare(Ab, M, N, encs(sig), enc(U2), enc(V2), encs(sig), enc(U0), enc(V0))
    assert abs(c["log2_vec_err"] - (-700.0)) <= 0.01, c
    gap0 = mp.mpf(1)                                   # sigma_0 = 2: nearest other sigma is 1, mirrored -2 is 4 away
    want_margin = -700.0 - (-(P - 38) + log2abs(mp, F) - log2abs(mp, gap0))
    assert abs(c["vec_margin_bits"] - want_margin) <= 0.01, (c, want_margin)
    # residual (ii) of the leaked pair, from mpmath: A v - sigma u = eps (sigma_4 - sigma_0) u_4
    want_res = log2abs(mp, eps * abs(sig[4] - sig[0]) / F)
    assert abs(c["log2_resid_rel"] - want_res) <= 0.01, (c, want_res)
    assert abs(c["log2_orth"] - (-700.0)) <= 0.01, c       # u_0^H u_4 = eps
    # opposite phases on u_4 and v_4: both are still unit vectors in the right spans, but the pair is wrong
    U3, V3 = U0.copy(), V0.copy()
    for i in range(M):
        U3[i, 4] = -U0[i, 4]
    c = oracle.svd_compare(Ab, M, N, encs(sig), enc(U3), enc(V3), encs(sig), enc(U0), enc(V0))
    assert c["vec_margin_bits"] > 100 and c["log2_resid_rel"] > -5, c
    # (i): sigma perturbed by 2^-500
    sig2 = list(sig)
    sig2[1] += mp.mpf(2) ** -500
    c = oracle.svd_compare(Ab, M, N, encs(sig2), enc(U0), enc(V0), encs(sig), enc(U0), enc(V0))
    assert abs(c["log2_dsig_rel"] - log2abs(mp, mp.mpf(2) ** -500 / F)) <= 0.01, c

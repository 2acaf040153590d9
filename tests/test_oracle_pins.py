"""Pins for the CPU oracle (oracle/zkd_oracle.c): every expected value here is computed with mpmath / exact
rationals from closed forms, invariants or brute force — never by the oracle itself and never by the CUDA path.

P1  2x2 closed form                      P6  paper's epsilon = 2^-(n-1) example
P2  Hermitian tridiagonal Toeplitz       P7  residual / orthogonality invariants, comparator cross-check
P3  Q diag(lambda) Q^H, chosen lambda    P8  ordering and guard-precision independence
P4  trace and Frobenius identities       P9  degenerate cases
P5  characteristic polynomial, N <= 4    P10 third opinion: mpmath.eighe
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


def decode(mp, lam, X, N):
    return zi.rvector_to_mp(lam, N), zi.cmatrix_to_mp(X, N)


def fro(mp, M):
    return mp.sqrt(sum(abs(M[i, j]) ** 2 for i in range(M.rows) for j in range(M.cols)))


def herm_from_upper(mp, A, N):
    H = mp.matrix(N, N)
    for i in range(N):
        H[i, i] = mp.re(A[i, i])
        for j in range(i + 1, N):
            H[i, j] = A[i, j]
            H[j, i] = mp.conj(A[i, j])
    return H


def check_invariants(mp, A, lam, X, N, bits=-760):
    """(ii) ||A x_j - lam_j x_j|| <= 2^bits F and (iii) |X^H X - I| <= 2^bits, layout X[i][j] = comp i of vec j."""
    F = fro(mp, A)
    for j in range(N):
        r = mp.sqrt(sum(abs(sum(A[i, k] * X[k, j] for k in range(N)) - lam[j] * X[i, j]) ** 2 for i in range(N)))
        assert log2abs(mp, r / F) <= bits, (j, log2abs(mp, r / F))
    for i in range(N):
        for j in range(N):
            g = sum(mp.conj(X[k, i]) * X[k, j] for k in range(N)) - (1 if i == j else 0)
            assert log2abs(mp, g) <= bits, (i, j, log2abs(mp, g))
    for j in range(N - 1):
        assert lam[j] <= lam[j + 1]


def vec_err(mp, x, v, N):
    """|| x - v (v^H x) ||_2 : phase-invariant, well conditioned (SURVEY 8(c) comparator (iv), |G| = 1)."""
    ip = sum(mp.conj(v[k]) * x[k] for k in range(N))
    return mp.sqrt(sum(abs(x[k] - v[k] * ip) ** 2 for k in range(N)))


# ------------------------------------------------------------------------------------------------------------
def test_number_format_roundtrip(mp):
    # API layout vs an independent pure-Python codec and vs MPFR's own double conversion
    for v in [0.0, 1.0, -1.0, 0.75, -3.0e-200, 1.5e300, 2.0 ** -1000]:
        b = oracle.api_from_double(v)
        assert len(b) == 112
        assert oracle.api_to_double(b) == v
        assert zi.to_fraction(b) == Fraction(v)
        assert zi.from_fraction(Fraction(v)) == b
    # rounding to nearest even at 768 bits
    x = Fraction(1) + Fraction(1, 2 ** 768)  # exactly half an ulp above 1 -> ties to even -> 1
    assert zi.to_fraction(zi.from_fraction(x)) == 1
    x = Fraction(1) + Fraction(3, 2 ** 768)  # 1.5 ulp (ulp = 2^-767) -> ties to even -> 1 + 2 ulp
    assert zi.to_fraction(zi.from_fraction(x)) == 1 + Fraction(2, 2 ** 767)


def test_generator_uniform_and_hermitian(mp):
    N = 6
    A = zi.cmatrix_to_mp(zi.random_hermitian(N, 77), N)
    for i in range(N):
        assert mp.im(A[i, i]) == 0
        for j in range(N):
            assert A[i, j] == mp.conj(A[j, i])
            assert -1 <= mp.re(A[i, j]) < 1 and -1 <= mp.im(A[i, j]) < 1
    # all 768 mantissa bits random: the value is not representable in 200 bits
    m, e = zi.decode_real(zi.random_hermitian(N, 77)[:RB])
    assert m % (1 << 500) != 0
    # mean/variance of uniform[-1,1): 0 and 1/3
    vals = []
    buf = np.zeros(RB, dtype=np.uint8)
    for k in range(4000):
        zi.lib().zkd_inputs_uniform_real(buf.ctypes.data, P, 5, 9, k * 12)
        vals.append(float(zi.to_fraction(buf)))
    vals = np.array(vals)
    assert abs(vals.mean()) < 0.05 and abs(vals.var() - 1 / 3) < 0.03 and vals.min() < -0.99 and vals.max() > 0.99


def test_generator_qdq_is_what_it_says(mp):
    # A Q = Q diag(lam), Q unitary — checked in mpmath, independent of the oracle
    N = 7
    vals = [Fraction(k * k - 10, 16) for k in range(N)]
    lam = zi._lam_array(vals)
    A, Q = zi.qdq(N, 11, 3, 3, lam, want_q=True)
    A = zi.cmatrix_to_mp(A, N)
    Q = zi.cmatrix_to_mp(Q, N)
    L = [mp.mpf(v.numerator) / v.denominator for v in vals]
    check_invariants(mp, A, L, Q, N, bits=-762)


# ------------------------------------------------------------------------------------------------------------
def test_P1_two_by_two_closed_form(mp):
    for seed in (1, 2, 3):
        Ab = zi.random_hermitian(2, seed)
        A = zi.cmatrix_to_mp(Ab, 2)
        al, be, ga = mp.re(A[0, 0]), A[0, 1], mp.re(A[1, 1])
        disc = mp.sqrt(((al - ga) / 2) ** 2 + abs(be) ** 2)
        lm, lp = (al + ga) / 2 - disc, (al + ga) / 2 + disc
        lam, X, info = oracle.diag_herm(Ab, 2)
        assert info["status"] == 0 and info["rotations"] == 1  # one rotation suffices
        lam, X = decode(mp, lam, X, 2)
        F = fro(mp, A)
        assert log2abs(mp, (lam[0] - lm) / F) <= -764 and log2abs(mp, (lam[1] - lp) / F) <= -764
        v = [be, lp - al]
        nv = mp.sqrt(abs(v[0]) ** 2 + abs(v[1]) ** 2)
        v = [v[0] / nv, v[1] / nv]
        assert log2abs(mp, vec_err(mp, [X[0, 1], X[1, 1]], v, 2)) <= -762
        # phase convention A9: largest-modulus component real positive
        k = 0 if abs(X[0, 1]) >= abs(X[1, 1]) else 1
        assert mp.im(X[k, 1]) == 0 and mp.re(X[k, 1]) > 0


def test_P2_tridiagonal_toeplitz(mp):
    N = 12
    a = zi.to_mpf(zi.from_mpf(mp.mpf(3) / 7))            # rounded to 768 bits: the matrix is exactly Toeplitz
    br = zi.to_mpf(zi.from_mpf(mp.mpf(2) / 9))
    bi = zi.to_mpf(zi.from_mpf(-mp.mpf(5) / 11))
    b = mp.mpc(br, bi)
    T = mp.matrix(N, N)
    for j in range(N):
        T[j, j] = a
        if j + 1 < N:
            T[j, j + 1] = b
            T[j + 1, j] = mp.conj(b)
    Ab = zi.cmatrix_from_mp(T, N)
    lam, X, info = oracle.diag_herm(Ab, N)
    assert info["status"] == 0
    lam, X = decode(mp, lam, X, N)
    F = fro(mp, T)
    ph = mp.conj(b) / abs(b)
    # ascending order <=> k = N..1
    for idx, k in enumerate(range(N, 0, -1)):
        lk = a + 2 * abs(b) * mp.cos(k * mp.pi / (N + 1))
        assert log2abs(mp, (lam[idx] - lk) / F) <= -762, idx
        v = [mp.sqrt(mp.mpf(2) / (N + 1)) * ph ** j * mp.sin(j * k * mp.pi / (N + 1)) for j in range(1, N + 1)]
        assert log2abs(mp, vec_err(mp, [X[i, idx] for i in range(N)], v, N)) <= -758, idx


def test_P3_constructed_spectrum(mp):
    N = 12
    vals = [Fraction(-7, 8), Fraction(-1, 2), Fraction(-1, 3).limit_denominator(1) , Fraction(-1, 16), Fraction(0), Fraction(1, 1024),
            Fraction(1, 8), Fraction(1, 4), Fraction(3, 8), Fraction(1, 2), Fraction(3, 4), Fraction(15, 16)]
    vals = sorted(set(vals))
    while len(vals) < N:
        vals.append(vals[-1] + Fraction(1, 32))
    lamb = zi._lam_array(vals)
    Ab, Qb = zi.qdq(N, 21, 0, 3, lamb, want_q=True)
    lam, X, info = oracle.diag_herm(Ab, N)
    assert info["status"] == 0
    lam, X = decode(mp, lam, X, N)
    Q = zi.cmatrix_to_mp(Qb, N)
    A = zi.cmatrix_to_mp(Ab, N)
    F = fro(mp, A)
    for j in range(N):
        lj = mp.mpf(vals[j].numerator) / vals[j].denominator
        assert log2abs(mp, (lam[j] - lj) / F) <= -760, j
        gap = min(abs(vals[j] - vals[i]) for i in range(N) if i != j)
        e = vec_err(mp, [X[i, j] for i in range(N)], [Q[i, j] for i in range(N)], N)
        assert log2abs(mp, e) <= -758 - np.log2(float(gap)), j


def test_P4_trace_and_frobenius_exact(mp):
    N = 16
    Ab = zi.random_hermitian(N, 1001)   # config c1
    lam, X, info = oracle.diag_herm(Ab, N, want_vectors=False)
    flat = Ab.reshape(N, N, 2, RB)
    tr = sum(zi.to_fraction(flat[i, i, 0]) for i in range(N))
    f2 = sum(zi.to_fraction(flat[i, j, c]) ** 2 for i in range(N) for j in range(N) for c in range(2))
    L = [zi.to_fraction(lam.reshape(N, RB)[j]) for j in range(N)]
    assert abs(sum(L) - tr) <= Fraction(1, 2 ** 755)
    assert abs(sum(l * l for l in L) - f2) <= Fraction(1, 2 ** 750)


@pytest.mark.parametrize("N", [2, 3, 4])
def test_P5_characteristic_polynomial_roots(mp, N):
    Ab = zi.random_hermitian(N, 40 + N)
    A = herm_from_upper(mp, zi.cmatrix_to_mp(Ab, N), N)
    # Faddeev-LeVerrier in mpmath at 1200 bits: p(x) = x^N + c_{N-1} x^{N-1} + ... + c_0
    M = mp.zeros(N, N)
    c = [mp.mpf(1)]
    I = mp.eye(N)
    for k in range(1, N + 1):
        M = A * M + c[-1] * I
        AM = A * M
        c.append(-sum(AM[i, i] for i in range(N)) / k)
    coeffs = [mp.re(x) for x in c]
    roots = sorted(mp.re(r) for r in mp.polyroots(coeffs, maxsteps=500, extraprec=4000))
    lam, _, info = oracle.diag_herm(Ab, N)
    lam = zi.rvector_to_mp(lam, N)
    F = fro(mp, A)
    for j in range(N):
        assert log2abs(mp, (lam[j] - roots[j]) / F) <= -755, (j, log2abs(mp, (lam[j] - roots[j]) / F))


def test_P6_paper_epsilon_example(mp):
    # Schmidt weights {1 - eps, eps}, eps ~ 2^(-n+1): eps must be resolved from the null space
    N, n = 8, 500
    vals = zi.epsilon_spectrum(N, n)
    Ab = zi.qdq(N, 31, 0, 3, zi._lam_array(vals))
    lam, X, info = oracle.diag_herm(Ab, N)
    assert info["status"] == 0
    L = [zi.to_fraction(lam.reshape(N, RB)[j]) for j in range(N)]
    eps = Fraction(1, 2 ** (n - 1))
    assert abs(L[N - 1] - (1 - eps)) <= Fraction(1, 2 ** 760)
    assert abs(L[N - 2] - eps) <= Fraction(1, 2 ** 760)       # relative 2^-261
    for j in range(N - 2):
        assert abs(L[j]) <= Fraction(1, 2 ** 760)
    lam_mp, Xm = decode(mp, lam, X, N)
    check_invariants(mp, zi.cmatrix_to_mp(Ab, N), lam_mp, Xm, N, bits=-758)


def test_P7_invariants_and_comparator_crosscheck(mp):
    N = 8
    Ab = zi.random_hermitian(N, 8)
    lam, X, info = oracle.diag_herm(Ab, N)
    A = zi.cmatrix_to_mp(Ab, N)
    lm, Xm = decode(mp, lam, X, N)
    check_invariants(mp, A, lm, Xm, N)
    c = oracle.compare(Ab, N, lam, X, lam, X)
    F = fro(mp, A)
    assert abs(c["log2_F"] - float(mp.log(F, 2))) < 1e-9
    # the comparator's residual must agree with an mpmath evaluation of the same definition
    worst = max(log2abs(mp, mp.sqrt(sum(abs(sum(A[i, k] * Xm[k, j] for k in range(N)) - lm[j] * Xm[i, j]) ** 2
                                        for i in range(N))) / F) for j in range(N))
    assert abs(c["log2_resid_rel"] - worst) < 0.01
    assert c["log2_dlam_rel"] < -1e8 and c["vec_margin_bits"] < -20 and c["groups"] == N
    # sensitivity: a 2^-700 perturbation of one component / a transposed X / a swapped eigenvalue must be seen
    Xp = X.copy().reshape(N, N, 2, RB)
    f = zi.to_fraction(Xp[2, 3, 0]) + Fraction(1, 2 ** 700)
    Xp[2, 3, 0] = np.frombuffer(zi.from_fraction(f), dtype=np.uint8)
    c2 = oracle.compare(Ab, N, lam, Xp.reshape(-1), lam, X)
    assert -702 < c2["log2_orth"] < -698 and c2["log2_resid_rel"] > -706 and c2["vec_margin_bits"] > 0
    Xt = np.ascontiguousarray(X.reshape(N, N, 2 * RB).transpose(1, 0, 2)).reshape(-1)
    assert oracle.compare(Ab, N, lam, Xt)["log2_resid_rel"] > -10
    lsw = lam.copy().reshape(N, RB)
    lsw[[0, 1]] = lsw[[1, 0]]
    assert oracle.compare(Ab, N, lsw.reshape(-1), X, lam, X)["log2_dlam_rel"] > -10


def test_P8_ordering_and_guard_independence(mp):
    for N in (9, 16):
        Ab = zi.random_hermitian(N, 300 + N)
        l0, X0, i0 = oracle.diag_herm(Ab, N, ordering="row-cyclic")
        l1, X1, i1 = oracle.diag_herm(Ab, N, ordering="round-robin", threads=4)
        l2, X2, i2 = oracle.diag_herm(Ab, N, ordering="row-cyclic", guard_bits=256)
        assert i0["status"] == i1["status"] == i2["status"] == 0
        for (l, X) in ((l1, X1), (l2, X2)):
            c = oracle.compare(Ab, N, l, X, l0, X0)
            assert c["log2_dlam_rel"] <= -762 and c["log2_resid_rel"] <= -762 and c["log2_orth"] <= -762
            assert c["vec_margin_bits"] <= -20


def test_P9_degenerate_cases(mp):
    N = 5
    zero = np.zeros(N * N * 2 * RB, dtype=np.uint8)
    lam, X, info = oracle.diag_herm(zero, N)
    assert info["status"] == 0 and not lam.any()
    Xm = zi.cmatrix_to_mp(X, N)
    assert all(Xm[i, j] == (1 if i == j else 0) for i in range(N) for j in range(N))
    # c I
    M = mp.eye(N) * (mp.mpf(5) / 8)
    lam, X, _ = oracle.diag_herm(zi.cmatrix_from_mp(M, N), N)
    assert all(l == mp.mpf(5) / 8 for l in zi.rvector_to_mp(lam, N))
    # diagonal, unsorted -> sorted, X a permutation
    d = [mp.mpf(3) / 4, -mp.mpf(1) / 2, mp.mpf(1) / 8, -mp.mpf(7) / 8, mp.mpf(0)]
    M = mp.diag(d)
    lam, X, _ = oracle.diag_herm(zi.cmatrix_from_mp(M, N), N)
    assert zi.rvector_to_mp(lam, N) == sorted(d)
    Xm = zi.cmatrix_to_mp(X, N)
    order = sorted(range(N), key=lambda i: d[i])
    assert all(Xm[i, j] == (1 if i == order[j] else 0) for i in range(N) for j in range(N))
    # real symmetric -> real eigenvectors
    S = mp.matrix(N, N)
    for i in range(N):
        for j in range(i, N):
            S[i, j] = S[j, i] = mp.mpf((i * 7 + j * 3) % 11 - 5) / 16
    lam, X, _ = oracle.diag_herm(zi.cmatrix_from_mp(S, N), N)
    Xm = zi.cmatrix_to_mp(X, N)
    assert all(mp.im(Xm[i, j]) == 0 for i in range(N) for j in range(N))
    check_invariants(mp, S, zi.rvector_to_mp(lam, N), Xm, N)
    # N = 1: lambda = Re a11, x = 1 ; the imaginary part of the diagonal is ignored (reading A15)
    one = np.concatenate([np.frombuffer(zi.from_fraction(Fraction(-3, 8)), dtype=np.uint8),
                          np.frombuffer(zi.from_fraction(Fraction(1, 8)), dtype=np.uint8)])
    lam, X, info = oracle.diag_herm(one, 1)
    assert zi.to_fraction(lam) == Fraction(-3, 8) and zi.to_fraction(X[:RB]) == 1 and not X[RB:].any()
    # malformed number -> status 3
    bad = zi.random_hermitian(3, 1).copy()
    bad[4] = 1
    assert oracle.diag_herm(bad, 3)[2]["status"] == 3
    # lower triangle is ignored (upper authoritative, A15)
    Ab = zi.random_hermitian(4, 9)
    Ac = Ab.copy().reshape(4, 4, 2, RB)
    Ac[3, 0] = Ac[0, 1]
    assert np.array_equal(oracle.diag_herm(Ab, 4)[0], oracle.diag_herm(Ac.reshape(-1), 4)[0])


def test_P10_third_opinion_mpmath_eighe(mp):
    N = 6
    Ab = zi.random_hermitian(N, 66)
    A = herm_from_upper(mp, zi.cmatrix_to_mp(Ab, N), N)
    E, Q = mp.eighe(A)
    lam, X, _ = oracle.diag_herm(Ab, N)
    lam, X = decode(mp, lam, X, N)
    F = fro(mp, A)
    for j in range(N):
        assert log2abs(mp, (lam[j] - E[j]) / F) <= -760
        assert log2abs(mp, vec_err(mp, [X[i, j] for i in range(N)], [Q[i, j] for i in range(N)], N)) <= -750


def test_clustered_spectrum_small(mp):
    # config-5-shaped: clusters with spacing 2^-200 must be resolved individually (reading A10/A13)
    cfg = zi.config("c5small", want_answer=True)
    N = cfg["N"]
    lam, X, info = oracle.diag_herm(cfg["A"], N)
    assert info["status"] == 0
    c = oracle.compare(cfg["A"], N, lam, X, cfg["lam"], cfg["Q"])
    assert c["log2_dlam_rel"] <= -758 and c["log2_resid_rel"] <= -758 and c["log2_orth"] <= -758
    assert c["groups"] == N and c["vec_margin_bits"] <= -10


# ------------------------------------------------------------------------------------------------------------
# P11: the comparator's multi-member branch (SURVEY.md 8(c) comparator (iv), reading A10) — the part that certifies
# exact multiplicities and near-degenerate groups.  Every expected value is evaluated in mpmath from the definition
# E_G = X_G - X0_G (X0_G^H X_G), gap_G = distance from the group's extreme members to the nearest eigenvalue outside.
def _random_unitary(mp, m, seed):
    import random

    rng = random.Random(seed)
    Z = mp.matrix(m, m)
    for i in range(m):
        for j in range(m):
            Z[i, j] = mp.mpc(rng.uniform(-1, 1), rng.uniform(-1, 1))
    Qm, _ = mp.qr(Z)
    return Qm


def _groups_mp(mp, lam0, F):
    """reading A10: a new group starts where the gap to the previous eigenvalue exceeds 2^-666 F"""
    starts = [0]
    for j in range(len(lam0) - 1):
        if lam0[j + 1] - lam0[j] > mp.ldexp(F, -666):
            starts.append(j + 1)
    return starts + [len(lam0)]


def _group_measures_mp(mp, lam0, X0, X, F):
    """per group: (log2 ||E_G||_F, margin in bits against 2^-730 F / gap_G), definitions written out"""
    N = len(lam0)
    st = _groups_mp(mp, lam0, F)
    out = []
    for g in range(len(st) - 1):
        a, b = st[g], st[g + 1]
        m = b - a
        M = mp.matrix(m, m)
        for p in range(m):
            for q in range(m):
                M[p, q] = sum(mp.conj(X0[k, a + p]) * X[k, a + q] for k in range(N))
        e2 = mp.mpf(0)
        for k in range(N):
            for q in range(m):
                e2 += abs(X[k, a + q] - sum(X0[k, a + p] * M[p, q] for p in range(m))) ** 2
        gaps = []
        if a > 0:
            gaps.append(lam0[a] - lam0[a - 1])
        if b < N:
            gaps.append(lam0[b] - lam0[b - 1])
        le = log2abs(mp, mp.sqrt(e2))
        out.append((le, le - (-730 + float(mp.log(F, 2)) - float(mp.log(min(gaps), 2))) if gaps else -1e9))
    return out


def test_P11_comparator_multi_member_groups(mp):
    N = 8
    t = Fraction(1, 2 ** 700)
    vals = [Fraction(-1, 4), Fraction(0), t, 2 * t, Fraction(1, 2), Fraction(1, 2), Fraction(3, 4), Fraction(1)]
    lamb = zi._lam_array(vals)
    Ab, Qb = zi.qdq(N, 1111, 0, 3, lamb, want_q=True)
    A = herm_from_upper(mp, zi.cmatrix_to_mp(Ab, N), N)
    F = fro(mp, A)
    Q = zi.cmatrix_to_mp(Qb, N)
    lam0 = [mp.mpf(v.numerator) / v.denominator for v in vals]
    assert _groups_mp(mp, lam0, F) == [0, 1, 4, 6, 7, 8]  # {-1/4} {0, t, 2t} {1/2, 1/2} {3/4} {1}

    def run(Xm, cols=None):
        Xb = zi.cmatrix_from_mp(Xm, N)
        c = oracle.compare(Ab, N, lamb.reshape(-1), Xb, lamb.reshape(-1), Qb, cols=cols)
        return c, zi.cmatrix_to_mp(Xb, N)  # the rounded candidate the comparator actually saw

    # (a) a unitary remix inside each multi-member group (non-symmetric, complex: a transposed or conjugated index in
    #     M = X0_G^H X_G would leave an O(1) error) changes nothing: E stays at the rounding level of the inputs
    R = mp.eye(N)
    U3, U2 = _random_unitary(mp, 3, 5), _random_unitary(mp, 2, 6)
    for p in range(3):
        for q in range(3):
            R[1 + p, 1 + q] = U3[p, q]
    for p in range(2):
        for q in range(2):
            R[4 + p, 4 + q] = U2[p, q]
    X1 = Q * R
    c, X1r = run(X1)
    meas = _group_measures_mp(mp, lam0, Q, X1r, F)
    assert c["groups"] == 5 and c["max_group"] == 3
    assert c["log2_vec_err"] <= -760
    assert abs(c["log2_vec_err"] - max(m[0] for m in meas)) < 0.01
    assert abs(c["vec_margin_bits"] - max(m[1] for m in meas)) < 0.01
    # without the remix the same measure is at the same level: the remix is invisible
    c0, _ = run(Q)
    assert c0["log2_vec_err"] <= -760

    # (b) a 2^-700 leak out of the 3-member group (a component along an eigenvector outside it) is reported at 2^-700,
    #     against the gap of that group's extreme members: min(0 - (-1/4), 1/2 - 2t) = 1/4
    X2 = X1.copy()
    for k in range(N):
        X2[k, 2] += Q[k, 6] * mp.ldexp(mp.mpf(1), -700)
    c, X2r = run(X2)
    meas = _group_measures_mp(mp, lam0, Q, X2r, F)
    assert abs(c["log2_vec_err"] - (-700)) < 0.01
    assert abs(c["log2_vec_err"] - max(m[0] for m in meas)) < 0.01
    want_margin = -700 - (-730 + float(mp.log(F, 2)) - (-2))
    assert abs(c["vec_margin_bits"] - want_margin) < 0.01 and c["vec_margin_bits"] > 0
    assert abs(c["vec_margin_bits"] - max(m[1] for m in meas)) < 0.01
    # a leak INSIDE the group (along another member of the same group) is not an error of the subspace
    X3 = X1.copy()
    for k in range(N):
        X3[k, 2] += Q[k, 3] * mp.ldexp(mp.mpf(1), -700)
    c, X3r = run(X3)
    assert c["log2_vec_err"] <= -760 and c["log2_orth"] > -702  # only orthonormality sees it

    # (c) cols = [...]: residual and orthogonality are those of the chosen columns only (the leak sits in column 2)
    lam_mp = lam0

    def col_measures(Xm, j):
        r = mp.sqrt(sum(abs(sum(A[i, k] * Xm[k, j] for k in range(N)) - lam_mp[j] * Xm[i, j]) ** 2 for i in range(N)))
        o = max(abs(sum(mp.conj(Xm[k, i]) * Xm[k, j] for k in range(N)) - (1 if i == j else 0)) for i in range(N))
        return log2abs(mp, r / F), log2abs(mp, o)

    cfull, _ = run(X2)
    for cols in ([2], [0, 5], [1, 2, 7]):
        cc, _ = run(X2, cols=cols)
        want_r = max(col_measures(X2r, j)[0] for j in cols)
        want_o = max(col_measures(X2r, j)[1] for j in cols)
        assert abs(cc["log2_resid_rel"] - want_r) < 0.01 and abs(cc["log2_orth"] - want_o) < 0.01, cols
        # the group part is independent of cols
        assert abs(cc["vec_margin_bits"] - cfull["vec_margin_bits"]) < 1e-9
    assert abs(cfull["log2_resid_rel"] - max(col_measures(X2r, j)[0] for j in range(N))) < 0.01

    # (d) one group spanning the whole spectrum (A = c I): any unitary X is correct, no gap exists
    cI = zi.cmatrix_from_mp(mp.eye(5) * (mp.mpf(5) / 8), 5)
    lamI = zi._lam_array([Fraction(5, 8)] * 5).reshape(-1)
    XI = zi.cmatrix_from_mp(_random_unitary(mp, 5, 9), 5)
    c = oracle.compare(cI, 5, lamI, XI, lamI, zi.cmatrix_from_mp(mp.eye(5), 5))
    assert c["groups"] == 1 and c["max_group"] == 5 and c["vec_margin_bits"] < -1e8
    assert c["log2_resid_rel"] <= -760 and c["log2_orth"] <= -760


def test_P12_rqi_restatement_agrees_with_jacobi_and_mpmath(mp):
    """oracle.rqi_refine - the CPU restatement of the paper's own route (fp64 LAPACK eigendecomposition + Rayleigh quotient
    iteration in MPFR), used only as a timed baseline - gives the eigenpairs of the pinned Jacobi oracle, and its
    residual, computed here in mpmath, is at the working precision; three iterations from the fp64 start are cubic."""
    N = 12
    A = zi.random_hermitian(N, 1212)
    lam, X, _, _ = oracle.rqi_refine(A, N, iters=3, threads=2)
    l0, X0, info = oracle.diag_herm(A, N)
    assert info["status"] == 0
    c = oracle.compare(A, N, lam, X, l0, X0)
    assert c["log2_dlam_rel"] <= -750 and c["log2_resid_rel"] <= -750 and c["log2_orth"] <= -745 and c["vec_margin_bits"] <= 0, c
    Am = herm_from_upper(mp, zi.cmatrix_to_mp(A, N), N)
    lam_m, Xm = decode(mp, lam, X, N)
    F = fro(mp, Am)
    j = 5
    r = mp.sqrt(sum(abs(sum(Am[i, k] * Xm[k, j] for k in range(N)) - lam_m[j] * Xm[i, j]) ** 2 for i in range(N)))
    assert log2abs(mp, r / F) <= -755
    # one iteration is not enough (vector 2^-50 -> 2^-150, eigenvalue error its square), a subset of pairs works, the sampling hook returns
    lam2, X2, _, _ = oracle.rqi_refine(A, N, first=3, count=4, iters=1, threads=1)
    d = max(abs(zi.to_fraction(lam2.reshape(4, -1)[t]) - zi.to_fraction(l0.reshape(N, -1)[3 + t])) for t in range(4))
    assert Fraction(1, 2 ** 420) < d < Fraction(1, 2 ** 200), float(d)
    oracle.rqi_refine(A, N, first=0, count=2, iters=1, max_pivots=3, threads=1)

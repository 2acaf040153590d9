"""NEXT-1: zkd_svd through the C ABI against the MPFR one-sided Jacobi SVD oracle
(oracle.svd, pinned in tests/test_oracle_svd_pins.py).  Tolerances: north_star's, carried over to singular triplets:
|dsigma| <= 2^-740 ||A||_F; max(||A v - sigma u||, ||A^H u - sigma v||) <= 2^-740 ||A||_F; |U^H U - I|, |V^H V - I| <= 2^-740;
pairs (u_j; v_j) / group projectors within 2^-730 ||A||_F / gap (comparator zkd_oracle_svd_compare)."""
from __future__ import annotations

import random
from fractions import Fraction

import numpy as np
import pytest

import oracle
import zkd_inputs as zi

pytestmark = pytest.mark.gpu
P = 768


@pytest.fixture(scope="module")
def zkd():
    import torch

    assert torch.cuda.is_available()
    import paper_2402_11868_b200 as z

    z.lib()
    return z


def gpu_svd(zkd, A, M, N, batch, prec=P, entry="ws"):
    import torch

    rb, K = zkd.real_bytes(prec), min(M, N)
    dA = torch.from_numpy(np.ascontiguousarray(A)).cuda()
    S = torch.zeros(batch * K * rb, dtype=torch.uint8, device="cuda")
    U = torch.zeros(batch * M * K * 2 * rb, dtype=torch.uint8, device="cuda")
    V = torch.zeros(batch * N * K * 2 * rb, dtype=torch.uint8, device="cuda")
    info = torch.zeros(batch * 24, dtype=torch.uint8, device="cuda")
    if entry == "ws":
        ws = torch.empty(zkd.svd_bufsize(M, N, batch, prec), dtype=torch.uint8, device="cuda")
        zkd.svd_ws(M, N, batch, dA, S, U, V, ws, info, prec_bits=prec)
    else:
        zkd.svd(M, N, batch, dA, S, U, V, prec_bits=prec)
    torch.cuda.synchronize()
    assert np.array_equal(dA.cpu().numpy(), np.ascontiguousarray(A)), "input was modified"
    return (S.cpu().numpy().reshape(batch, -1), U.cpu().numpy().reshape(batch, -1), V.cpu().numpy().reshape(batch, -1),
            zkd.read_info(info, batch))


def rand_general(M, N, seed, prec=P):
    """M x N complex matrix, Re / Im uniform[-1,1) with every mantissa bit random (the generator of reading A2)."""
    rb = zi.real_bytes(prec)
    n = max(M, N)
    H = zi.random_hermitian(n, seed, 0, prec).reshape(n, n, 2, rb)   # upper triangle + mirrored lower: take a rectangle
    H2 = zi.random_hermitian(n, seed + 1, 0, prec).reshape(n, n, 2, rb)
    out = np.zeros((M, N, 2, rb), dtype=np.uint8)
    for i in range(M):
        for j in range(N):
            out[i, j] = H[i, j] if i <= j else H2[j, i]
            if i == j:
                out[i, j, 1] = H2[i, j, 0]
    return out.reshape(-1)


def check(c, prec, what, with_ref=True):
    tol = -(prec - 28.0)
    assert c["log2_resid_rel"] <= tol, (what, c)
    assert c["log2_orth"] <= tol, (what, c)
    if with_ref:
        assert c["log2_dsig_rel"] <= tol, (what, c)
        assert c["vec_margin_bits"] <= 0, (what, c)


def check_order_and_phase(S, V, N, K, prec=P):
    s = [zi.to_fraction(S.reshape(K, -1)[j], prec) for j in range(K)]
    assert all(s[j] >= s[j + 1] for j in range(K - 1)) and all(x >= 0 for x in s)
    Vr = V.reshape(N, K, 2, -1)
    for j in range(K):
        col = [(zi.to_fraction(Vr[i, j, 0], prec), zi.to_fraction(Vr[i, j, 1], prec)) for i in range(N)]
        m2 = [a * a + b * b for a, b in col]
        k = max(range(N), key=lambda i: (m2[i], -i))
        assert any(col[i][1] == 0 and col[i][0] > 0 and m2[k] - m2[i] <= Fraction(1, 2 ** (prec - 68)) for i in range(N)), j


@pytest.mark.parametrize("M,N,batch", [(8, 8, 2), (16, 16, 1), (12, 5, 2), (5, 12, 1), (33, 20, 1), (1, 1, 1), (1, 7, 1)])
def test_svd_random(zkd, M, N, batch):
    K = min(M, N)
    A = np.concatenate([rand_general(M, N, 5000 + 10 * M + N + 100 * b) for b in range(batch)])
    S, U, V, info = gpu_svd(zkd, A, M, N, batch)
    Ab = A.reshape(batch, -1)
    for b in range(batch):
        assert info[b]["status"] == 0, info[b]
        S0, U0, V0, oi = oracle.svd(Ab[b], M, N)
        assert oi["status"] == 0
        check(oracle.svd_compare(Ab[b], M, N, S[b], U[b], V[b], S0, U0, V0), P, (M, N, b))
        check_order_and_phase(S[b], V[b], N, K)


def constructed(mp, M, N, sig, seed):
    from test_oracle_svd_pins import rand_unitary, rmatrix_from_mp

    rng = random.Random(seed)
    K = min(M, N)
    QU, QV = rand_unitary(mp, rng, M), rand_unitary(mp, rng, N)
    A = mp.matrix(M, N)
    for i in range(M):
        for j in range(N):
            A[i, j] = sum(QU[i, k] * sig[k] * mp.conj(QV[j, k]) for k in range(K))
    return rmatrix_from_mp(mp, A)


@pytest.mark.parametrize("M,N", [(10, 10), (12, 7), (6, 11)])
def test_svd_tiny_and_repeated_singular_values(zkd, mp, M, N):
    """Schmidt-weight-like spectra: a dominant value, a repeated value, weights down to 2^-600, exact zeros (rank deficiency):
    sigma to ABSOLUTE 2^-740 ||A||_F, which the A^H A route would lose."""
    K = min(M, N)
    sig = [mp.mpf(1), mp.mpf(1) / 2, mp.mpf(1) / 2, mp.mpf(2) ** -30, mp.mpf(2) ** -200, mp.mpf(2) ** -600, mp.mpf(0), mp.mpf(0),
           mp.mpf(0), mp.mpf(0), mp.mpf(0)][:K]
    A = constructed(mp, M, N, sig, 7000 + M * 31 + N)
    S, U, V, info = gpu_svd(zkd, A, M, N, 1)
    assert info[0]["status"] == 0, info
    got = [zi.to_fraction(S[0].reshape(K, -1)[j]) for j in range(K)]
    for g, w in zip(got, sig):
        assert abs(g - Fraction(int(w * mp.mpf(2) ** 900), 2 ** 900)) <= Fraction(1, 2 ** 738), (float(g), float(w))
    S0, U0, V0, oi = oracle.svd(A, M, N)
    check(oracle.svd_compare(A, M, N, S[0], U[0], V[0], S0, U0, V0), P, (M, N))


def test_svd_mps_shaped_batch(zkd):
    """A batch of c4 matrices (N = 32, rank 8, Schmidt weights down to 2^-60, 24 exact zeros: BASELINE.json configs[3]) as SVD
    input: a Hermitian PSD matrix's singular values are its eigenvalues, known by construction; the null-space step runs for
    the whole batch at once (every matrix has rank 8)."""
    cfg = zi.config("c4", batch=6)
    N, b = cfg["N"], cfg["batch"]
    S, U, V, info = gpu_svd(zkd, cfg["A"], N, N, b)
    want = sorted(cfg["lam_exact"], reverse=True)
    A = cfg["A"].reshape(b, -1)
    for i in range(b):
        assert info[i]["status"] == 0, info[i]
        got = [zi.to_fraction(S[i].reshape(N, -1)[j]) for j in range(N)]
        for g, w in zip(got, want):
            assert abs(g - w) <= Fraction(1, 2 ** 740), (i, float(g), float(w))
        c = oracle.svd_compare(A[i], N, N, S[i], U[i], V[i])
        check(c, P, ("c4", i), with_ref=False)
    S0, U0, V0, _ = oracle.svd(A[0], N, N)
    check(oracle.svd_compare(A[0], N, N, S[0], U[0], V[0], S0, U0, V0), P, "c4[0]")


def test_svd_larger_rectangular(zkd):
    M, N = 96, 64   # the (M + N) = 160 eigenproblem: several GEMM tiles and a ragged tail
    A = rand_general(M, N, 9090)
    S, U, V, info = gpu_svd(zkd, A, M, N, 1)
    S0, U0, V0, oi = oracle.svd(A, M, N)
    assert oi["status"] == 0
    check(oracle.svd_compare(A, M, N, S[0], U[0], V[0], S0, U0, V0), P, (M, N))


def test_svd_degenerate_inputs(zkd, mp):
    from test_oracle_svd_pins import rmatrix_from_mp

    # zero matrix, identity-like, rank one
    for M, N, fn in [(4, 6, lambda i, j: 0), (5, 5, lambda i, j: (mp.mpf(-3) / 7 if i == j else 0)),
                     (6, 4, lambda i, j: mp.mpc(i + 1, 1) * mp.mpc(j + 1, -2) / 64)]:
        K = min(M, N)
        A = mp.matrix(M, N)
        for i in range(M):
            for j in range(N):
                A[i, j] = fn(i, j)
        buf = rmatrix_from_mp(mp, A)
        S, U, V, info = gpu_svd(zkd, buf, M, N, 1)
        assert info[0]["status"] == 0, info
        S0, U0, V0, _ = oracle.svd(buf, M, N)
        c = oracle.svd_compare(buf, M, N, S[0], U[0], V[0], S0, U0, V0)
        if c["log2_F"] < -1e8:   # the zero matrix: sigma = 0 exactly, any orthonormal U, V
            assert all(zi.decode_real(S[0].reshape(K, -1)[j])[0] == 0 for j in range(K))
            assert c["log2_orth"] <= -740, c
            continue
        check(c, P, (M, N), with_ref=False)
        assert c["log2_dsig_rel"] <= -740, c


def test_svd_other_precision_and_stream_entry(zkd):
    M, N, prec = 9, 6, 256
    A = rand_general(M, N, 8123, prec)
    S, U, V, _ = gpu_svd(zkd, A, M, N, 1, prec, entry="stream")
    S0, U0, V0, _ = oracle.svd(A, M, N, prec=prec)
    check(oracle.svd_compare(A, M, N, S[0], U[0], V[0], S0, U0, V0, prec=prec), prec, "256")


def test_svd_argument_errors(zkd):
    import torch

    t = torch.zeros(1 << 16, dtype=torch.uint8, device="cuda")
    L = zkd.lib()
    p = t.data_ptr()
    assert L.zkd_svd_ws(0, 4, 1, 768, p, p, p, p, p, 1 << 16, None, None) == -1
    assert L.zkd_svd_ws(4, 4, 1, 100, p, p, p, p, p, 1 << 16, None, None) == -2
    assert L.zkd_svd_ws(4, 4, 1, 768, p, p, p, p, p, 16, None, None) == -3
    assert L.zkd_svd_ws(2000, 2000, 1, 768, p, p, p, p, p, 1 << 16, None, None) == -1

"""NEXT-3 (multiprecision LU / Gaussian elimination) and S4a' (exact RQI by one LU per eigenpair, PAPER.md:33,
SURVEY.md 8(a)) through the C ABI, against the MPFR oracles (oracle.lu_solve, oracle.diag_herm) and against the production
path: both routes must give the same eigenpairs to the north_star tolerances."""
from __future__ import annotations

from fractions import Fraction

import numpy as np
import pytest

import oracle
import zkd_inputs as zi
from test_gpu_svd import rand_general

pytestmark = pytest.mark.gpu
P = 768
RB = 16 + P // 8


@pytest.fixture(scope="module")
def zkd():
    import torch

    assert torch.cuda.is_available()
    import paper_2402_11868_b200 as z

    z.lib()
    return z


def gpu_lu(zkd, A, B, N, nrhs, batch, prec=P):
    import torch

    rb = zkd.real_bytes(prec)
    dA = torch.from_numpy(np.ascontiguousarray(A)).cuda()
    dB = torch.from_numpy(np.ascontiguousarray(B)).cuda()
    X = torch.zeros(batch * N * nrhs * 2 * rb, dtype=torch.uint8, device="cuda")
    st = torch.zeros(batch, dtype=torch.int32, device="cuda")
    ws = torch.empty(zkd.lu_solve_bufsize(N, nrhs, batch, prec), dtype=torch.uint8, device="cuda")
    zkd.lu_solve(N, nrhs, batch, dA, dB, X, ws, st, prec_bits=prec)
    torch.cuda.synchronize()
    return X.cpu().numpy().reshape(batch, -1), st.cpu().numpy()


def fr(buf, prec=P):
    return zi.to_fraction(buf, prec)


@pytest.mark.parametrize("N,nrhs,batch", [(1, 1, 1), (2, 2, 2), (5, 1, 3), (17, 3, 2), (40, 2, 1)])
def test_lu_solve_against_oracle(zkd, N, nrhs, batch):
    A = np.concatenate([rand_general(N, N, 100 * N + b) for b in range(batch)])
    B = np.concatenate([rand_general(N, nrhs, 7 + 100 * N + b) for b in range(batch)])
    X, st = gpu_lu(zkd, A, B, N, nrhs, batch)
    assert list(st) == [0] * batch
    Ab, Bb = A.reshape(batch, -1), B.reshape(batch, -1)
    for b in range(batch):
        X0, rc = oracle.lu_solve(Ab[b], Bb[b], N, nrhs)
        assert rc == 0
        got = X[b].reshape(N * nrhs * 2, RB)
        ref = X0.reshape(N * nrhs * 2, RB)
        scale = max(abs(fr(ref[e])) for e in range(N * nrhs * 2))
        worst = max(abs(fr(got[e]) - fr(ref[e])) for e in range(N * nrhs * 2))
        # fixed point: absolute accuracy 2^-(768+2) in the scaled units times the growth of the solve (cond(A) ~ 2^10 at these sizes)
        assert worst <= scale * Fraction(1, 2 ** 730), (N, b, float(worst / scale))


def test_lu_solve_status(zkd):
    N = 4
    A = rand_general(N, N, 31).reshape(N, N, 2, RB).copy()
    A[:, 2] = 0                                            # a zero column: singular
    A2 = rand_general(N, N, 32).reshape(N, N, 2, RB).copy()
    A2[1, 1, 0, 4] = 1                                     # flags != 0: malformed
    A3 = rand_general(N, N, 33)
    Aall = np.concatenate([A.reshape(-1), A2.reshape(-1), A3])
    B = np.concatenate([rand_general(N, 1, 40 + b) for b in range(3)])
    X, st = gpu_lu(zkd, Aall, B, N, 1, 3)
    assert list(st) == [1, 3, 0]
    X0, rc = oracle.lu_solve(A3, B.reshape(3, -1)[2], N, 1)
    assert rc == 0
    got, ref = X[2].reshape(N * 2, RB), X0.reshape(N * 2, RB)
    assert max(abs(fr(got[e]) - fr(ref[e])) for e in range(N * 2)) <= Fraction(1, 2 ** 730)


def gpu_rqi(zkd, A, N, batch, prec=P):
    import torch

    rb = zkd.real_bytes(prec)
    dA = torch.from_numpy(np.ascontiguousarray(A)).cuda()
    lam = torch.zeros(batch * N * rb, dtype=torch.uint8, device="cuda")
    X = torch.zeros(batch * N * N * 2 * rb, dtype=torch.uint8, device="cuda")
    info = torch.zeros(batch * 24, dtype=torch.uint8, device="cuda")
    ws = torch.empty(zkd.diag_herm_rqi_lu_bufsize(N, batch, prec), dtype=torch.uint8, device="cuda")
    zkd.diag_herm_rqi_lu(N, batch, dA, lam, X, ws, info, prec_bits=prec)
    torch.cuda.synchronize()
    return lam.cpu().numpy().reshape(batch, -1), X.cpu().numpy().reshape(batch, -1), zkd.read_info(info, batch)


@pytest.mark.parametrize("name,batch", [("c1", 2), ("c2", 1)])
def test_exact_rqi_agrees_with_oracle_and_production_path(zkd, name, batch):
    """S4a' on c1 and c2: three to four cubic iterations; parity with the oracle at the north_star tolerances, and agreement of
    the two GPU routes (correction-equation RQI vs exact RQI by LU) to 2^-740."""
    from test_gpu_parity import check, gpu_diag

    cfg = zi.config(name, batch=batch)
    N, b = cfg["N"], cfg["batch"]
    lam, X, info = gpu_rqi(zkd, cfg["A"], N, b)
    lam2, X2, _ = gpu_diag(zkd, cfg["A"], N, b)
    A = cfg["A"].reshape(b, -1)
    for i in range(b):
        assert info[i]["status"] == 0 and info[i]["steps"] <= 5, info[i]
        l0, X0, _ = oracle.diag_herm(A[i], N)
        check(oracle.compare(A[i], N, lam[i], X[i], l0, X0), (name, "rqi", i))
        check(oracle.compare(A[i], N, lam[i], X[i], lam2[i], X2[i]), (name, "rqi vs production", i))


def test_exact_rqi_refuses_clusters_and_other_precision(zkd):
    cfg = zi.config("c4small", batch=1)
    with pytest.raises(zkd.ZkdError) as ei:
        gpu_rqi(zkd, cfg["A"], cfg["N"], 1)
    assert ei.value.code == -7
    N, prec = 12, 256
    A = zi.random_hermitian(N, 606, 0, prec)
    lam, X, info = gpu_rqi(zkd, A, N, 1, prec)
    l0, X0, _ = oracle.diag_herm(A, N, prec=prec)
    c = oracle.compare(A, N, lam[0], X[0], l0, X0, prec=prec)
    assert c["log2_resid_rel"] <= -(prec - 28) and c["log2_orth"] <= -(prec - 28) and c["log2_dlam_rel"] <= -(prec - 28), c
    assert c["vec_margin_bits"] <= 0, c

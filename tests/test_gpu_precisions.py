"""NEXT-2: the hot path at the paper's other precisions - 256 bit (Deutsch-Jozsa runs) and
128 bit (Shor runs) - and 512 bit, against the MPFR oracle run at the same precision.  Tolerances are
north_star's scaled with the precision P (reading A18 of DESIGN.md): 2^-(P-28) ||A||_F for eigenvalues and residuals,
2^-(P-28) for orthonormality, 2^-(P-38) ||A||_F / gap for vectors / projectors (the comparator's own constants follow P)."""
from __future__ import annotations

import random

import numpy as np
import pytest

import oracle
import zkd_inputs as zi

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def zkd():
    import torch

    assert torch.cuda.is_available()
    import paper_2402_11868_b200 as z

    z.lib()
    return z


def gpu_diag(zkd, A, N, batch, prec, entry="ws"):
    import torch

    rb = zkd.real_bytes(prec)
    assert rb == 16 + prec // 8
    dA = torch.from_numpy(np.ascontiguousarray(A)).cuda()
    lam = torch.zeros(batch * N * rb, dtype=torch.uint8, device="cuda")
    X = torch.zeros(batch * N * N * 2 * rb, dtype=torch.uint8, device="cuda")
    info = torch.zeros(batch * 24, dtype=torch.uint8, device="cuda")
    if entry == "ws":
        ws = torch.empty(zkd.diag_herm_bufsize(N, batch, prec), dtype=torch.uint8, device="cuda")
        zkd.diag_herm_ws(N, batch, dA, lam, X, ws, info, prec_bits=prec)
    else:
        zkd.diag_herm(N, batch, dA, lam, X, prec_bits=prec)
    torch.cuda.synchronize()
    return lam.cpu().numpy().reshape(batch, -1), X.cpu().numpy().reshape(batch, -1), zkd.read_info(info, batch)


def check(c, prec, what):
    tol = -(prec - 28.0)
    assert c["log2_resid_rel"] <= tol, (what, c)
    assert c["log2_orth"] <= tol, (what, c)
    assert c["log2_dlam_rel"] <= tol, (what, c)
    assert c["vec_margin_bits"] <= 0, (what, c)


@pytest.mark.parametrize("prec", [128, 256, 512])
@pytest.mark.parametrize("name,batch", [("c1", 2), ("c4small", 3), ("c2", 1)])
def test_parity_at_other_precisions(zkd, prec, name, batch):
    cfg = zi.config(name, batch=batch, prec=prec)
    N, b = cfg["N"], cfg["batch"]
    lam, X, info = gpu_diag(zkd, cfg["A"], N, b, prec)
    A = cfg["A"].reshape(b, -1)
    for i in range(b):
        assert info[i]["status"] == 0, info[i]
        l0, X0, oi = oracle.diag_herm(A[i], N, prec=prec)
        assert oi["status"] == 0
        check(oracle.compare(A[i], N, lam[i], X[i], l0, X0, prec=prec), prec, (name, prec, i))


@pytest.mark.parametrize("prec", [128, 256])
def test_ragged_and_stream_ordered_entry(zkd, prec):
    N = 37
    A = zi.random_hermitian(N, 4242, 0, prec)
    lam, X, _ = gpu_diag(zkd, A, N, 1, prec, entry="stream")
    l0, X0, _ = oracle.diag_herm(A, N, prec=prec)
    check(oracle.compare(A, N, lam[0], X[0], l0, X0, prec=prec), prec, ("ragged", prec))


def test_paper_epsilon_example_at_256_bits(zkd):
    """PAPER.md:35 at the Deutsch-Jozsa precision: eigenvalues {1 - eps, eps, 0, ...} with eps = 2^-(n-1), n = 200,
    rotated by reflectors: eps is recovered to absolute 2^-(256-28)."""
    from fractions import Fraction

    prec, N = 256, 16
    eps = Fraction(1, 2 ** 199)
    vals = sorted([1 - eps, eps] + [Fraction(0)] * (N - 2))
    A = zi.qdq(N, 3535, 0, 3, zi._lam_array(vals, prec), prec=prec)
    lam, X, info = gpu_diag(zkd, A, N, 1, prec)
    got = [zi.to_fraction(lam[0].reshape(N, -1)[j], prec) for j in range(N)]
    for g, w in zip(got, vals):
        assert abs(g - w) <= Fraction(1, 2 ** (prec - 28)), (float(g), float(w))
    c = oracle.compare(A, N, lam[0], X[0], prec=prec)
    assert c["log2_resid_rel"] <= -(prec - 28) and c["log2_orth"] <= -(prec - 28), c


@pytest.mark.parametrize("prec", [128, 256, 512, 768])
def test_conversion_round_trip_at_every_precision(zkd, prec):
    """API (prec) -> FX -> API (prec) is the identity for numbers whose bits all lie above the FX floor, and the FX digits are
    the exact integer value * 2^812."""
    import torch

    from zkd_testlib import ints_from_fx_planes

    rng = random.Random(prec)
    n = 400
    rb = 16 + prec // 8
    vals = []
    buf = np.zeros((n, rb), dtype=np.uint8)
    for e in range(n):
        mant = rng.getrandbits(prec) | (1 << (prec - 1))
        if rng.random() < 0.5:
            mant = -mant
        exp2 = -prec - rng.randrange(0, 812 - prec + 1)  # |value| in [2^-(k+1), 2^-k), all bits >= 2^-812
        buf[e] = np.frombuffer(zi.encode_real(mant, exp2, prec), dtype=np.uint8)
        vals.append(mant << (812 + exp2))
    d_api = torch.from_numpy(buf.reshape(-1)).cuda()
    fx = torch.zeros(30 * n, dtype=torch.int32, device="cuda")
    zkd.fx_from_api(n, d_api, fx, prec_bits=prec)
    back = torch.zeros(n * rb, dtype=torch.uint8, device="cuda")
    zkd.fx_to_api(n, fx, back, prec_bits=prec)
    torch.cuda.synchronize()
    assert ints_from_fx_planes(fx.cpu().numpy().reshape(30, n)) == vals
    assert np.array_equal(back.cpu().numpy(), buf.reshape(-1))


def test_unsupported_precisions(zkd):
    assert zkd.real_bytes(100) == 0 and zkd.real_bytes(64) == 0 and zkd.real_bytes(832) == 0
    with pytest.raises(zkd.ZkdError) as ei:
        zkd.diag_herm_bufsize(8, 1, 100)
    assert ei.value.code == -2

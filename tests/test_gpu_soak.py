"""Randomised structures through the whole hot path (C ABI), checked with properties that need no reference run:
status, residual and orthogonality (oracle comparator on the GPU's own output) and, for constructed spectra
(Q diag(lambda) Q^H, reading A14), every eigenvalue against the chosen one.  Sizes, batch sizes and spectrum shapes are
drawn from a seeded generator: random Hermitian, clusters at spacings 2^-12 .. 2^-700, exact multiplicities, low rank,
geometric cascades, near-degenerate pairs.  This net caught two bugs that every hand-written case had passed (a carry
look-ahead error in the warp-cooperative GEMM epilogue; early splits not converging on geometric cascades)."""
from __future__ import annotations

import os
import random
import sys
from fractions import Fraction

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import oracle  # noqa: E402
import zkd_inputs as zi  # noqa: E402

pytestmark = pytest.mark.gpu
TOL = -740.0


@pytest.fixture(scope="module")
def zkd():
    import torch

    if not torch.cuda.is_available():
        pytest.skip("needs a GPU")
    import paper_2402_11868_b200 as z

    z.lib()
    return z


def _run(z, A, N, b):
    import torch

    rb = z.REAL_BYTES
    Ad = torch.from_numpy(np.ascontiguousarray(A)).cuda()
    lam = torch.zeros(b * N * rb, dtype=torch.uint8, device="cuda")
    X = torch.zeros(b * N * N * 2 * rb, dtype=torch.uint8, device="cuda")
    ws = torch.empty(z.diag_herm_bufsize(N, b), dtype=torch.uint8, device="cuda")
    info = torch.zeros(b * 24, dtype=torch.uint8, device="cuda")
    z.diag_herm_ws(N, b, Ad, lam, X, ws, info)
    torch.cuda.synchronize()
    return lam.cpu().numpy().reshape(b, -1), X.cpu().numpy().reshape(b, -1), z.read_info(info, b)


def _spectrum(rng, kind, N):
    if kind == "clusters":
        ncl = rng.randint(1, max(1, N // 3))
        sp = rng.choice([12, 25, 60, 150, 300, 500, 700])
        cent = [Fraction(rng.randint(-2 ** 30, 2 ** 30), 2 ** 30) for _ in range(ncl)]
        return [cent[i % ncl] + Fraction(i // ncl, 2 ** sp) for i in range(N)]
    if kind == "mult":
        base = [Fraction(rng.randint(-8, 8), 8) for _ in range(max(1, N // 4))]
        return [rng.choice(base) for _ in range(N)]
    if kind == "lowrank":
        r = rng.randint(1, max(1, N // 3))
        return [Fraction(rng.randint(1, 2 ** 20), 2 ** 20) for _ in range(r)] + [Fraction(0)] * (N - r)
    if kind == "geom":
        step = rng.choice([3, 11, 30, 45])
        return [Fraction(rng.choice([1, -1]), 2 ** (1 + step * i)) if 1 + step * i < 760 else Fraction(0) for i in range(N)]
    sp = rng.choice([40, 100, 260, 420, 640])  # "pairs"
    vals = []
    for _ in range(N // 2):
        c = Fraction(rng.randint(-2 ** 20, 2 ** 20), 2 ** 20)
        vals += [c, c + Fraction(1, 2 ** sp)]
    return vals + [Fraction(3, 2)] * (N - len(vals))


@pytest.mark.parametrize("seed,opts", [(1, {}), (2, {}), (22, {}), (5, {"combine_path": 2}), (6, {"combine_path": 1, "sstep_cpb": 4}),
                                       (7, {"early_split": 0})])
def test_random_structures(zkd, seed, opts):
    rng = random.Random(seed)
    old = {k: zkd.get_option(k) for k in opts}
    for k, v in opts.items():
        zkd.set_option(k, v)
    failures = []
    try:
        for case in range(40):
            N = rng.choice([2, 3, 5, 8, 12, 16, 20, 24, 31, 33, 40, 48, 64])
            kind = rng.choice(["rand", "clusters", "mult", "lowrank", "geom", "pairs"])
            b = rng.choice([1, 1, 2, 3])
            mats, specs = [], []
            for s in range(b):
                if kind == "rand" or N < 3:
                    mats.append(zi.random_hermitian(N, 50000 + 100 * seed + case, s))
                    specs.append(None)
                else:
                    vals = sorted(_spectrum(rng, kind, N))
                    mats.append(zi.qdq(N, 60000 + 100 * seed + case, s, rng.randint(1, 4), zi._lam_array(vals)))
                    specs.append(vals)
            A = np.concatenate([np.asarray(m).reshape(-1) for m in mats])
            lam, X, info = _run(zkd, A, N, b)
            A2 = A.reshape(b, -1)
            for i in range(b):
                tag = (seed, case, kind, N, b, i)
                if info[i]["status"] != 0:
                    failures.append((tag, info[i]))
                    continue
                cols = None if N <= 40 else np.sort(np.random.default_rng(case).choice(N, size=6, replace=False)).astype(np.int32)
                c = oracle.compare(A2[i], N, lam[i], X[i], cols=cols)
                if c["log2_F"] < -1e8:  # the zero matrix (all chosen eigenvalues 0): lambda = 0, X = I
                    assert all(zi.decode_real(lam[i].reshape(N, -1)[j])[0] == 0 for j in range(N)), tag
                    continue
                if not (c["log2_resid_rel"] <= TOL and c["log2_orth"] <= TOL):
                    failures.append((tag, {k: round(float(v), 1) for k, v in c.items()}))
                    continue
                if specs[i] is not None:
                    # north_star: |dlam| <= 2^-740 ||A||_F, with ||A||_F^2 = sum lambda^2 exactly (A = Q diag(lambda) Q^H
                    # up to the 2^-768 rounding of its entries): compared squared, in exact rationals
                    got = [zi.to_fraction(lam[i].reshape(N, -1)[j]) for j in range(N)]
                    F2 = sum(w * w for w in specs[i])
                    if not all((g - w) ** 2 * 4 ** 740 <= F2 for g, w in zip(got, specs[i])):
                        failures.append((tag, "eigenvalue mismatch"))
    finally:
        for k, v in old.items():
            zkd.set_option(k, v)
    assert not failures, failures[:5]

"""NEXT-4: zkd_mps_two_site_update through the C ABI against the plain CPU definition (oracle/mps_update.py,
pinned in tests/test_oracle_mps_pins.py).  What is unique is compared (weights, the kept count, the reduced density matrix's
eigenpairs through the Hermitian comparator, Theta = L' R'); the eigenvector phases follow the library's convention A9."""
from __future__ import annotations

import random

import numpy as np
import pytest

import oracle
import zkd_inputs as zi
from oracle import mps_update as mu
from test_oracle_mps_pins import enc, gate_cnot, gate_identity
from test_oracle_svd_pins import log2abs, rand_matrix, rand_unitary, rmatrix_to_mp

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


def gpu_update(zkd, L, R, G, chiL, chiC, chiR, d, batch, max_keep=0, cutoff_bits=700):
    import torch

    mL, mR = chiL * d, d * chiR
    K = min(mL, max_keep) if max_keep > 0 else mL
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    W = torch.zeros(batch * K * RB, dtype=torch.uint8, device="cuda")
    Ln = torch.zeros(batch * mL * K * 2 * RB, dtype=torch.uint8, device="cuda")
    Rn = torch.zeros(batch * K * mR * 2 * RB, dtype=torch.uint8, device="cuda")
    kept = torch.zeros(batch, dtype=torch.int32, device="cuda")
    info = torch.zeros(batch * 24, dtype=torch.uint8, device="cuda")
    ws = torch.empty(zkd.mps_two_site_update_bufsize(chiL, chiC, chiR, d, batch), dtype=torch.uint8, device="cuda")
    zkd.mps_two_site_update(chiL, chiC, chiR, d, batch, t(L), t(R), t(G), W, Ln, Rn, kept, ws, max_keep=max_keep, cutoff_bits=cutoff_bits,
                            info=info)
    torch.cuda.synchronize()
    return (W.cpu().numpy().reshape(batch, -1), Ln.cpu().numpy().reshape(batch, -1), Rn.cpu().numpy().reshape(batch, -1),
            kept.cpu().numpy(), zkd.read_info(info, batch))


def compare_with_oracle(mp, ref, W, Ln, Rn, kept, mL, mR, K):
    tr = ref["trace"]
    got_w = [zi.to_mpf(W.reshape(K, -1)[k]) for k in range(K)]
    for g, w in zip(got_w, ref["weights"]):
        assert log2abs(mp, (g - w) / tr) <= -740, (g, w)
    assert kept == min(ref["kept"], K)
    Lm, Rm = rmatrix_to_mp(mp, Ln, mL, K), rmatrix_to_mp(mp, Rn, K, mR)
    if K == mL:
        # (L', w) is an eigendecomposition of rho: residual, orthonormality and vectors / degenerate subspaces by the Hermitian comparator
        lam_asc = np.ascontiguousarray(W.reshape(K, -1)[::-1]).reshape(-1)
        X_asc = np.ascontiguousarray(Ln.reshape(mL, K, 2, -1)[:, ::-1]).reshape(-1)
        l0, X0, _ = oracle.diag_herm(ref["rho_api"], mL)
        c = oracle.compare(ref["rho_api"], mL, lam_asc, X_asc, l0, X0)
        assert c["log2_resid_rel"] <= -740 and c["log2_orth"] <= -740 and c["log2_dlam_rel"] <= -740 and c["vec_margin_bits"] <= 0, c
    # R' = L'^H Theta and Theta = L' R' + (discarded weights)
    T = ref["theta"]
    F = mp.sqrt(tr)
    for k in range(K):
        for c_ in range(mR):
            want = sum(mp.conj(Lm[r, k]) * T[r, c_] for r in range(mL))
            assert log2abs(mp, (Rm[k, c_] - want) / F) <= -738, (k, c_)
    rec = Lm * Rm - T
    err2 = sum(abs(rec[i, j]) ** 2 for i in range(mL) for j in range(mR))
    discarded = sum(w for w in ref["weights"][K:])
    assert err2 <= discarded * (1 + mp.mpf(2) ** -100) + tr * mp.mpf(2) ** -1470, (mp.nstr(err2, 5), mp.nstr(discarded, 5))


def test_bell_pair_and_product_state(zkd, mp):
    h = mp.sqrt(mp.mpf(1) / 2)
    L, R = mp.matrix(2, 1), mp.matrix(1, 2)
    L[0, 0] = L[1, 0] = h
    R[0, 0] = 1
    for G, want, k in ((gate_cnot(mp), [mp.mpf(1) / 2, mp.mpf(1) / 2], 2), (gate_identity(mp), [mp.mpf(1), mp.mpf(0)], 1)):
        W, Ln, Rn, kept, info = gpu_update(zkd, enc(mp, L), enc(mp, R), enc(mp, G), 1, 1, 1, 2, 1)
        assert info[0]["status"] == 0, info
        got = [zi.to_mpf(W[0].reshape(2, -1)[i]) for i in range(2)]
        assert all(log2abs(mp, g - w) <= -740 for g, w in zip(got, want)) and kept[0] == k
        ref = mu.two_site_update(mp, enc(mp, L), enc(mp, R), enc(mp, G), 1, 1, 1, 2)
        compare_with_oracle(mp, ref, W[0], Ln[0], Rn[0], kept[0], 2, 2, 2)


def test_paper_epsilon_example(zkd, mp):
    """Schmidt weights {1 - eps, eps, 0, 0} with eps = 2^-600 behind random unitaries and a random two-qubit gate
    applied and undone inside the site tensors: eps comes back to absolute 2^-740."""
    rng = random.Random(3535)
    chiL, chiC, chiR, d = 2, 4, 3, 2
    mL, mR = chiL * d, d * chiR
    eps = mp.mpf(2) ** -600
    w = [1 - eps, eps, mp.mpf(0), mp.mpf(0)]
    QL, QR = rand_unitary(mp, rng, mL), rand_unitary(mp, rng, mR)
    L, R = mp.matrix(mL, chiC), mp.matrix(chiC, mR)
    for r_ in range(mL):
        for k in range(chiC):
            L[r_, k] = QL[r_, k] * mp.sqrt(w[k])
    for k in range(chiC):
        for c in range(mR):
            R[k, c] = mp.conj(QR[c, k])
    G = gate_identity(mp)
    for cutoff, want_kept in ((700, 2), (500, 1)):
        W, Ln, Rn, kept, info = gpu_update(zkd, enc(mp, L), enc(mp, R), enc(mp, G), chiL, chiC, chiR, d, 1, cutoff_bits=cutoff)
        assert info[0]["status"] == 0, info
        got = [zi.to_mpf(W[0].reshape(mL, -1)[i]) for i in range(mL)]
        for g, x in zip(got, w):
            assert log2abs(mp, g - x) <= -740, (g, x)
        assert kept[0] == want_kept
    ref = mu.two_site_update(mp, enc(mp, L), enc(mp, R), enc(mp, G), chiL, chiC, chiR, d, cutoff_bits=500)
    compare_with_oracle(mp, ref, W[0], Ln[0], Rn[0], kept[0], mL, mR, mL)


@pytest.mark.parametrize("chiL,chiC,chiR,d,batch,max_keep", [(3, 4, 3, 2, 2, 0), (4, 2, 5, 2, 1, 3), (2, 3, 2, 3, 1, 0)])
def test_random_sites_and_gates(zkd, mp, chiL, chiC, chiR, d, batch, max_keep):
    rng = random.Random(1000 * chiL + 100 * chiC + 10 * chiR + d)
    mL, mR = chiL * d, d * chiR
    K = min(mL, max_keep) if max_keep > 0 else mL
    Ls, Rs, Gs = [], [], []
    for b in range(batch):
        Ls.append(enc(mp, rand_matrix(mp, rng, mL, chiC)))
        Rs.append(enc(mp, rand_matrix(mp, rng, chiC, mR)))
        Gs.append(enc(mp, rand_unitary(mp, rng, d * d)))
    W, Ln, Rn, kept, info = gpu_update(zkd, np.concatenate(Ls), np.concatenate(Rs), np.concatenate(Gs), chiL, chiC, chiR, d, batch,
                                       max_keep=max_keep)
    for b in range(batch):
        assert info[b]["status"] == 0, info[b]
        ref = mu.two_site_update(mp, Ls[b], Rs[b], Gs[b], chiL, chiC, chiR, d)
        compare_with_oracle(mp, ref, W[b], Ln[b], Rn[b], kept[b], mL, mR, K)

"""Pins for the MPS two-site update oracle (oracle/mps_update.py; NEXT-4): expected values from exact
constructions, never from the oracle or the CUDA path."""
import random
from fractions import Fraction

import numpy as np

import oracle
import zkd_inputs as zi
from oracle import mps_update as mu
from test_oracle_svd_pins import log2abs, rand_unitary, rmatrix_from_mp

P = 768


def enc(mp, M):
    return rmatrix_from_mp(mp, M)


def gate_identity(mp, d=2):
    return mp.eye(d * d)


def gate_cnot(mp):
    G = mp.zeros(4, 4)
    G[0, 0] = G[1, 1] = G[2, 3] = G[3, 2] = 1
    return G


def product_sites(mp, v0, v1):
    """chiL = chiC = chiR = 1, d = 2: L[(0,i),0] = v0[i], R[0,(j,0)] = v1[j]"""
    L, R = mp.matrix(2, 1), mp.matrix(1, 2)
    for i in range(2):
        L[i, 0] = v0[i]
        R[0, i] = v1[i]
    return L, R


def test_M1_product_state_and_bell_pair(mp):
    h = mp.sqrt(mp.mpf(1) / 2)
    L, R = product_sites(mp, [h, h], [1, 0])                      # |+>|0>
    r = mu.two_site_update(mp, enc(mp, L), enc(mp, R), enc(mp, gate_identity(mp)), 1, 1, 1, 2)
    assert log2abs(mp, r["weights"][0] - 1) <= -760 and log2abs(mp, r["weights"][1]) <= -760 and r["kept"] == 1
    r = mu.two_site_update(mp, enc(mp, L), enc(mp, R), enc(mp, gate_cnot(mp)), 1, 1, 1, 2)   # CNOT |+0> = Bell pair
    assert all(log2abs(mp, x - mp.mpf(1) / 2) <= -760 for x in r["weights"]) and r["kept"] == 2
    T = r["theta"]                                                   # (|00> + |11>)/sqrt 2
    assert log2abs(mp, T[0, 0] - h) <= -760 and log2abs(mp, T[1, 1] - h) <= -760 and log2abs(mp, T[0, 1]) <= -760


def test_M2_paper_epsilon_example_and_invariants(mp):
    """Schmidt weights {1 - eps, eps, 0, ...} with eps = 2^-(n-1), here n = 601: built as
    Theta = QL diag(sqrt w) QR^H split into L = QL diag(sqrt w), R = QR^H; identity gate."""
    rng = random.Random(35)
    chiL, chiC, chiR, d = 2, 4, 3, 2
    mL, mR = chiL * d, d * chiR
    eps = mp.mpf(2) ** -600
    w = [1 - eps, eps, mp.mpf(0), mp.mpf(0)]
    QL, QR = rand_unitary(mp, rng, mL), rand_unitary(mp, rng, mR)
    L = mp.matrix(mL, chiC)
    R = mp.matrix(chiC, mR)
    for r_ in range(mL):
        for k in range(chiC):
            L[r_, k] = QL[r_, k] * mp.sqrt(w[k])
    for k in range(chiC):
        for c in range(mR):
            R[k, c] = mp.conj(QR[c, k])
    r = mu.two_site_update(mp, enc(mp, L), enc(mp, R), enc(mp, gate_identity(mp)), chiL, chiC, chiR, d, cutoff_bits=700)
    for g, want in zip(r["weights"], w):
        assert log2abs(mp, g - want) <= -750, (g, want)           # eps itself to ABSOLUTE 2^-750: 150 significant bits of it
    assert r["kept"] == 2
    assert mu.two_site_update(mp, enc(mp, L), enc(mp, R), enc(mp, gate_identity(mp)), chiL, chiC, chiR, d, cutoff_bits=500)["kept"] == 1
    # invariants: trace(rho) = ||Theta||_F^2 = sum w; Theta = Lnew Rnew; weights = squared singular values (pinned SVD oracle)
    T = r["theta"]
    F2 = sum(abs(T[i, j]) ** 2 for i in range(mL) for j in range(mR))
    assert log2abs(mp, sum(r["weights"]) - F2) <= -755 and log2abs(mp, r["trace"] - F2) <= -760
    rec = r["Lnew"] * r["Rnew"] - T
    assert max(log2abs(mp, rec[i, j]) for i in range(mL) for j in range(mR)) <= -755
    S, _, _, _ = oracle.svd(enc(mp, T), mL, mR)
    s = [zi.to_mpf(S.reshape(mL, -1)[k]) for k in range(mL)]
    for g, sv in zip(r["weights"], s):
        assert log2abs(mp, g - sv * sv) <= -750

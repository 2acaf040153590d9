"""GPU tests of the building-block kernels behind the C ABI (include/zkd.h): number-format conversion (S0/S6),
the digit GEMM (S4a/S4d/S4e) and the fp64 seed (S1).  Integer work is compared bit for bit with Python integers."""
from __future__ import annotations

import random

import numpy as np
import pytest

import zkd_inputs as zi
from zkd_testlib import (DB, FRAC, ND, api_value_to_fx_int, fxc_from_ints, ints_from_fx_planes, ints_from_fxc, window)

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def zkd():
    import torch

    assert torch.cuda.is_available()
    import paper_2402_11868_b200 as z

    z.lib()
    return z


def _dev(a):
    import torch

    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def test_fx_from_api_and_back_bit_exact(zkd):
    import torch

    rng = random.Random(7)
    vals = []  # (mant, exp2)
    for e in (-900, -812, -800, -400, -100, -29, -28, -1, 0, 1, 5, 20):
        for _ in range(12):
            m = rng.getrandbits(768) | (1 << 767)
            if rng.random() < 0.5:
                m = -m
            vals.append((m, e - 768))
    vals += [(0, 0), (1 << 767, -767), (-(1 << 767), -767), ((1 << 768) - 1, -768 - 3), (-((1 << 768) - 1), -768 - 790)]
    count = len(vals)
    api = np.zeros((count, zi.real_bytes()), dtype=np.uint8)
    for i, (m, e) in enumerate(vals):
        api[i] = np.frombuffer(zi.encode_real(m, e), dtype=np.uint8)
    for scale in (0, 3, -7):
        d_api = _dev(api)
        d_fx = torch.zeros(ND * count, dtype=torch.int32, device="cuda")
        zkd.fx_from_api(count, d_api, d_fx, scale)
        got = ints_from_fx_planes(d_fx.cpu().numpy())
        want = [api_value_to_fx_int(m, e, scale) for (m, e) in vals]
        assert got == want
        # and back: round to nearest even at 768 bits, exponent shifted back by the scale
        d_back = torch.zeros(count * zi.real_bytes(), dtype=torch.uint8, device="cuda")
        zkd.fx_to_api(count, d_fx, d_back, scale)
        back = d_back.cpu().numpy().reshape(count, -1)
        for i, w in enumerate(want):
            exp = zi.encode_real(w, -FRAC - scale)
            assert bytes(back[i]) == exp, i


def _rand_fx(rng, count, top_bit, digits):
    """random signed values that fit the window [top_bit - 28 digits, top_bit) with two spare bits"""
    lsb = max(0, top_bit - DB * digits)
    out = []
    for _ in range(count):
        v = rng.getrandbits(top_bit - 2 - lsb) << lsb if top_bit - 2 - lsb > 0 else 0
        out.append(-v if rng.random() < 0.5 else v)
    return out


GEMM_CASES = [
    # M, N, K, batch, op_a, (a_top, a_dig), (b_top, b_dig), mode, cut
    (5, 7, 3, 1, 0, (812, 30), (815, 3), 0, -1),       # W = A X0 shape
    (16, 16, 16, 2, 0, (812, 30), (815, 30), 0, -1),   # full product
    (33, 18, 37, 1, 0, (812, 30), (815, 30), 0, -1),   # ragged tiles, several K tiles
    (20, 20, 20, 1, 1, (815, 5), (700, 5), 0, -1),     # C = X^H R windows
    (20, 20, 20, 3, 0, (815, 6), (650, 6), 0, 480),    # T = X E with a cut
    (24, 9, 40, 1, 0, (812, 24), (660, 8), 1, -1),     # W += A T
    (24, 9, 40, 1, 0, (812, 24), (660, 8), 2, -1),     # subtract mode
    (70, 70, 70, 1, 1, (815, 12), (500, 12), 0, -1),
]


# the same contraction through the int8 tcgen05 engine (S4b): forced on small ragged shapes (partial TMA boxes), and
# shapes spanning several 128-tiles, K blocks and a ragged tail
GEMM_I8_CASES = [
    (16, 16, 16, 2, 0, (812, 30), (815, 30), 0, -1),
    (33, 18, 37, 1, 0, (812, 30), (815, 30), 0, -1),
    (20, 20, 20, 1, 1, (815, 5), (700, 5), 0, -1),
    (20, 20, 20, 3, 0, (815, 6), (650, 6), 0, 480),
    (24, 9, 40, 1, 0, (812, 24), (660, 8), 1, -1),
    (24, 9, 40, 1, 0, (812, 24), (660, 8), 2, -1),
    (130, 70, 150, 1, 0, (812, 30), (815, 3), 0, -1),
    (140, 136, 260, 1, 1, (815, 9), (600, 9), 0, -1),
    (128, 128, 128, 1, 0, (812, 30), (815, 30), 0, -1),
]


@pytest.mark.parametrize("case", GEMM_I8_CASES)
def test_gemm_fx_int8_tcgen05_matches_python_integers(zkd, case):
    zkd.set_option("gemm_path", 2)
    try:
        zkd.kernel_timing(True)
        test_gemm_fx_matches_python_integers(zkd, case, path=2)
        ms, launches, macs = zkd.kernel_timing_read_i8()
        assert launches == 1 and macs > 0, "the int8 tcgen05 kernel did not run"
    finally:
        zkd.kernel_timing(False)
        zkd.set_option("gemm_path", 0)


@pytest.mark.parametrize("case", GEMM_CASES)
@pytest.mark.parametrize("combine", [1, 2])
def test_gemm_fx_epilogues_match_python_integers(zkd, case, combine):
    """both epilogues of the IMAD engine (digit-serial and warp-cooperative carry resolution) are bit-identical"""
    zkd.set_option("combine_path", combine)
    try:
        test_gemm_fx_matches_python_integers(zkd, case, path=1)
    finally:
        zkd.set_option("combine_path", 0)


@pytest.mark.parametrize("case", GEMM_CASES)
@pytest.mark.parametrize("tile", [8, 16])
def test_gemm_fx_tile_sizes_match_python_integers(zkd, case, tile):
    """the IMAD kernel built with 8 x 8 x 8 and with 16 x 16 x 16 tiles (option gemm_tile; automatic by tile fill otherwise)"""
    zkd.set_option("gemm_tile", tile)
    try:
        test_gemm_fx_matches_python_integers(zkd, case, path=1)
    finally:
        zkd.set_option("gemm_tile", 0)


@pytest.mark.parametrize("case", GEMM_CASES)
def test_gemm_fx_matches_python_integers(zkd, case, path=1):
    import torch

    M, N, K, batch, op_a, (a_top, a_dig), (b_top, b_dig), mode, cut = case
    rng = random.Random(hash(case) & 0xFFFF)
    a_rows, a_cols = (K, M) if op_a else (M, K)
    Are = _rand_fx(rng, batch * M * K, a_top, a_dig)
    Aim = _rand_fx(rng, batch * M * K, a_top, a_dig)
    Bre = _rand_fx(rng, batch * K * N, b_top, b_dig)
    Bim = _rand_fx(rng, batch * K * N, b_top, b_dig)
    # add junk below the windows: it must be ignored (floor semantics)
    a_lsb, b_lsb = a_top - DB * a_dig, b_top - DB * b_dig
    if a_lsb > 0:
        Are = [v + rng.getrandbits(a_lsb) for v in Are]
        Aim = [v + rng.getrandbits(a_lsb) for v in Aim]
    if b_lsb > 0:
        Bre = [v + rng.getrandbits(b_lsb) for v in Bre]
        Bim = [v + rng.getrandbits(b_lsb) for v in Bim]
    C0re = _rand_fx(rng, batch * M * N, 800, 30)
    C0im = _rand_fx(rng, batch * M * N, 800, 30)
    dA, dB = _dev(fxc_from_ints(Are, Aim)), _dev(fxc_from_ints(Bre, Bim))
    dC = _dev(fxc_from_ints(C0re, C0im))
    err = torch.zeros(1, dtype=torch.int32, device="cuda")
    msb = torch.zeros(1, dtype=torch.int32, device="cuda")
    zkd.gemm_fx(M, N, K, batch, op_a, dA, a_top, a_dig, dB, b_top, b_dig, dC, mode, cut, path, None, err, msb)
    torch.cuda.synchronize()
    assert int(err.item()) == 0
    gre, gim = ints_from_fxc(dC.cpu().numpy())
    # exact reference on the windows
    def a_at(b, i, k):
        idx = b * M * K + (k * M + i if op_a else i * K + k)
        re, im = window(Are[idx], a_top, a_dig), window(Aim[idx], a_top, a_dig)
        # the library conjugates at window level: -floor(x) ("Digit GEMM")
        return (re, -im) if op_a else (re, im)
    # dropped digit columns: |error| <= K 2^(a_lsb + b_top - 837) FX units ("Digit GEMM"), + 2 for the floors
    e_bits = a_lsb + b_top - 837 + (K - 1).bit_length()
    tol = 2 + (1 << e_bits if e_bits >= 0 else 0)
    worst = 0
    maxmag = 0
    for b in range(batch):
        for i in range(M):
            for j in range(N):
                sre = sim = 0
                for k in range(K):
                    are, aim = a_at(b, i, k)
                    idx = b * K * N + k * N + j
                    bre, bim = window(Bre[idx], b_top, b_dig), window(Bim[idx], b_top, b_dig)
                    sre += are * bre - aim * bim
                    sim += are * bim + aim * bre
                e = b * M * N + i * N + j
                for (s, g, c0) in ((sre, gre[e], C0re[e]), (sim, gim[e], C0im[e])):
                    p = s >> FRAC  # floor(product / 2^812)
                    if cut > 0:
                        p = (p >> cut) << cut
                    want = p if mode == 0 else (c0 + p if mode == 1 else c0 - p)
                    d = abs(g - want)
                    if cut > 0:
                        d = min(d, abs(d - (1 << cut)))  # a carry across the cut is a legitimate 1-ulp-at-cut difference
                    worst = max(worst, d)
                    maxmag = max(maxmag, abs(g))
    assert worst <= tol, (worst, tol)
    # msb_out reports the value that ends up in the destination (in accumulate modes: the sum, not the product)
    assert maxmag.bit_length() - 1 <= int(msb.item()) <= maxmag.bit_length() + 1


@pytest.mark.parametrize("combine", [1, 2])
@pytest.mark.parametrize("mode", [0, 1, 2])
def test_gemm_fx_near_identity_carry_chains(zkd, combine, mode):
    """Products of near-identity matrices (G = X^H X, X (I + M)): results like 1 - 2^-300 or -2^-500, whose canonical digits
    are long runs of 2^28-1 and 0 with carries and borrows meeting in them - the case that random operands never produce
    (a look-ahead bug of the warp-cooperative epilogue passed every random test and was caught by a soak of the pipeline)."""
    import torch

    M = N = K = 13
    batch = 2
    rng = random.Random(1234 + mode)
    one = 1 << FRAC

    def near_identity():
        re, im = [], []
        for b in range(batch):
            for i in range(M):
                for j in range(M):
                    e = rng.choice([1, -1]) * (1 << rng.randint(0, 780)) if rng.random() < 0.8 else 0
                    f = rng.choice([1, -1]) * (1 << rng.randint(0, 780)) if rng.random() < 0.5 else 0
                    re.append((one if i == j else 0) + e)
                    im.append(f if i != j else 0)
        return re, im

    Are, Aim = near_identity()
    Bre, Bim = near_identity()
    C0re = [(one if (e % (M * N)) // N == e % N else 0) - rng.getrandbits(rng.randint(1, 700)) for e in range(batch * M * N)]
    C0im = [rng.choice([1, -1]) * (1 << rng.randint(0, 700)) for _ in range(batch * M * N)]
    dA, dB, dC = _dev(fxc_from_ints(Are, Aim)), _dev(fxc_from_ints(Bre, Bim)), _dev(fxc_from_ints(C0re, C0im))
    err = torch.zeros(1, dtype=torch.int32, device="cuda")
    zkd.set_option("combine_path", combine)
    try:
        zkd.gemm_fx(M, N, K, batch, 1, dA, 815, 30, dB, 815, 30, dC, mode, -1, 1, None, err, None)
        torch.cuda.synchronize()
    finally:
        zkd.set_option("combine_path", 0)
    assert int(err.item()) == 0
    gre, gim = ints_from_fxc(dC.cpu().numpy())
    worst = 0
    for b in range(batch):
        for i in range(M):
            for j in range(N):
                sre = sim = 0
                for k in range(K):
                    ia, ib = b * M * K + k * M + i, b * K * N + k * N + j
                    are, aim = Are[ia], -Aim[ia]  # op_a = 1: conjugate transpose
                    sre += are * Bre[ib] - aim * Bim[ib]
                    sim += are * Bim[ib] + aim * Bre[ib]
                e = b * M * N + i * N + j
                for s_, g, c0 in ((sre, gre[e], C0re[e]), (sim, gim[e], C0im[e])):
                    p_ = s_ >> FRAC
                    want = p_ if mode == 0 else (c0 + p_ if mode == 1 else c0 - p_)
                    worst = max(worst, abs(g - want))
    assert worst <= 2 + (1 << max(0, -25 + 815 - 837 + 4)), worst


def test_gemm_fx_flags_window_overflow(zkd):
    import torch

    # an element with a bit above the declared window must raise the error flag
    vals = [1 << 700] + [0] * 3
    dA = _dev(fxc_from_ints(vals, [0] * 4))
    dB = _dev(fxc_from_ints([1 << 812] * 4, [0] * 4))
    dC = _dev(fxc_from_ints([0] * 4, [0] * 4))
    err = torch.zeros(1, dtype=torch.int32, device="cuda")
    zkd.gemm_fx(2, 2, 2, 1, 0, dA, 650, 4, dB, 815, 3, dC, 0, -1, 0, None, err, None)
    torch.cuda.synchronize()
    assert int(err.item()) & 1


@pytest.mark.parametrize("N,batch", [(1, 2), (2, 3), (7, 2), (16, 4), (33, 2), (64, 3), (96, 1), (200, 1), (300, 1), (515, 2), (1000, 1)])
def test_seed_fp64_vs_lapack(zkd, N, batch):
    import torch

    rng = np.random.default_rng(100 + N)
    A = rng.uniform(-1, 1, (batch, N, N)) + 1j * rng.uniform(-1, 1, (batch, N, N))
    A = (A + A.conj().transpose(0, 2, 1)) / 2
    dA = _dev(A.astype(np.complex128).view(np.float64))
    mu = torch.zeros(batch * N, dtype=torch.float64, device="cuda")
    V = torch.zeros(batch * N * N * 2, dtype=torch.float64, device="cuda")
    zkd.seed_fp64(N, batch, dA, mu, V)
    torch.cuda.synchronize()
    mu = mu.cpu().numpy().reshape(batch, N)
    V = V.cpu().numpy().view(np.complex128).reshape(batch, N, N)
    for b in range(batch):
        w = np.linalg.eigvalsh(A[b])
        F = np.linalg.norm(A[b])
        assert np.all(np.diff(mu[b]) >= 0)
        assert np.max(np.abs(mu[b] - w)) <= 1e-12 * max(F, 1) * N
        assert np.max(np.abs(V[b].conj().T @ V[b] - np.eye(N))) <= 1e-13 * N
        assert np.max(np.abs(A[b] @ V[b] - V[b] * mu[b][None, :])) <= 1e-11 * max(F, 1)


@pytest.mark.parametrize("N", [300, 515, 1000])
def test_seed_fp64_gram_rounds_vs_lapack(zkd, N):
    """option seed_gram = 2: the blocked seed with the rotations of a round found on the Gram matrix of the CTA's column blocks."""
    zkd.set_option("seed_gram", 2)
    try:
        test_seed_fp64_vs_lapack(zkd, N, 1)
    finally:
        zkd.set_option("seed_gram", 0)


def test_measured_imad_peak_is_plausible(zkd):
    p = zkd.measure_imad_peak(30.0)
    # IMAD.WIDE with a 64-bit accumulator issues at half the 32-bit IMAD rate: 148 SMs x ~30.5 /clk x (1.0 .. 2.1 GHz)
    assert 148 * 28 * 1.0e9 < p < 148 * 33 * 2.1e9, p


def test_measured_i8_mma_peak_is_plausible(zkd):
    p = zkd.measure_i8_mma_peak(20.0)
    # 128 x 128 x 32 kind::i8 per >= 64 clocks per SM: at most 148 x 16384 op/clk x 2.1 GHz; at least half of that at 1 GHz
    assert 148 * 8192 * 1.0e9 < p < 148 * 16384 * 2.1e9 * 1.02, p


def test_measured_dfma_peak_is_plausible(zkd):
    p = zkd.measure_dfma_peak(30.0)
    # fp64 FMA: 148 SMs x (32 .. 64 lanes/clk) x 2 flop x (1.0 .. 2.1 GHz)
    assert 148 * 32 * 2 * 1.0e9 * 0.9 < p < 148 * 64 * 2 * 2.1e9 * 1.05, p

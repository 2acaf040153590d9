"""SURVEY.md section 4 tier 2: the multi-digit primitives of the CUDA path (fx.cuh / fx_funcs.cuh), one by one, against
Python's exact integers through the element-wise entry zkd_fx_prim.  add / sub / half / msb / the fp64 round trip and the
multiply (against its stated truncation rule) are bit-exact; the multiply is also checked against the exact product within
the bound the rule implies; reciprocal and reciprocal square root (Newton iterations built from those multiplies) within
a stated number of units of 2^-812."""
from __future__ import annotations

import math
import random

import numpy as np
import pytest

from zkd_testlib import DB, DMASK, FRAC, ND, fx_planes_from_ints, ints_from_fx_planes

pytestmark = pytest.mark.gpu

MOD = 1 << (DB * (ND - 1) + 32)


def wrap(v: int) -> int:
    v %= MOD
    return v - MOD if v >= MOD // 2 else v


@pytest.fixture(scope="module")
def zkd():
    import torch

    assert torch.cuda.is_available()
    import paper_2402_11868_b200 as z

    z.lib()
    return z


def run(zkd, op, a, b=None):
    import torch

    n = len(a)
    da = torch.from_numpy(fx_planes_from_ints(a)).cuda()
    db = torch.from_numpy(fx_planes_from_ints(b)).cuda() if b is not None else None
    out = torch.zeros(ND * n, dtype=torch.int32, device="cuda")
    zkd.fx_prim(op, n, da, db, out)
    torch.cuda.synchronize()
    planes = out.cpu().numpy().reshape(ND, n)
    assert np.all((planes[: ND - 1] >= 0) & (planes[: ND - 1] <= DMASK)), "digits 0..28 must be canonical"
    return ints_from_fx_planes(planes)


def rand_fx(rng, bits, signed=True):
    """a random FX integer of about `bits` bits; some with long runs of 0 / 2^28-1 digits (carry chains)"""
    bits = max(bits, 2)
    v = rng.getrandbits(bits)
    kind = rng.randrange(6)
    if kind == 0:
        v = (1 << bits) - 1 - rng.getrandbits(20)          # ...111 digits
    elif kind == 1:
        v = (1 << rng.randrange(1, bits)) + rng.getrandbits(8)  # ...000 digits
    elif kind == 2:
        v = rng.getrandbits(rng.randrange(1, bits))
    if signed and rng.random() < 0.5:
        v = -v
    return v


def digits(v: int):
    d = [(v >> (DB * k)) & DMASK for k in range(ND - 1)]
    d.append(v >> (DB * (ND - 1)))
    return d


def mul_model(a: int, b: int) -> int:
    """fx_mul as documented in include/zkd.h: digit products a_i b_j with i + j >= 28, rounded at the guard column."""
    da, db = digits(a), digits(b)
    acc = 0
    for i in range(ND):
        for j in range(ND):
            if i + j >= ND - 2:
                acc += da[i] * db[j] << (DB * (i + j))
    acc += 1 << (DB * (ND - 2) + DB - 1)
    return wrap(acc >> (DB * (ND - 1)))


def test_add_sub_half_exact(zkd):
    rng = random.Random(11)
    a = [rand_fx(rng, 838) for _ in range(1500)] + [0, -1, 1, (1 << 839) - 1, -(1 << 839)]
    b = [rand_fx(rng, 838) for _ in range(1500)] + [0, 1, -1, 1, -1]
    assert run(zkd, "add", a, b) == [wrap(x + y) for x, y in zip(a, b)]
    assert run(zkd, "sub", a, b) == [wrap(x - y) for x, y in zip(a, b)]
    assert run(zkd, "half", a) == [x >> 1 for x in a]


def test_msb(zkd):
    rng = random.Random(12)
    a = [rand_fx(rng, rng.randrange(1, 839)) for _ in range(2000)] + [0, -1, 1, -2, (1 << 838), -(1 << 838)]
    want = [(x if x >= 0 else ~x).bit_length() for x in a]
    assert [v for v in run(zkd, "msb", a)] == want


def test_mul_bit_exact_against_its_rule_and_close_to_exact(zkd):
    rng = random.Random(13)
    a, b = [], []
    for _ in range(3000):
        ba = rng.randrange(1, 826)
        a.append(rand_fx(rng, ba))
        b.append(rand_fx(rng, rng.randrange(1, min(838, 1650 - ba))))  # |a b| < 2^26 in value: fits FX
    a += [0, 1 << FRAC, -(1 << FRAC), (1 << FRAC) - 1]
    b += [rand_fx(rng, 800), rand_fx(rng, 800), rand_fx(rng, 800), (1 << FRAC) - 1]
    got = run(zkd, "mul", a, b)
    assert got == [mul_model(x, y) for x, y in zip(a, b)]
    # against the exact product: the dropped digit columns are non-negative except through a negative top digit
    worst = 0
    for x, y, g in zip(a, b, got):
        if abs(x * y) >> (2 * FRAC + 26):
            continue  # the product does not fit FX: only the wrapped rule applies
        worst = max(worst, abs(g * (1 << FRAC) - x * y) >> FRAC)
    assert worst <= 29, worst  # |g - x y / 2^812| <= 29 units of 2^-812


def test_reciprocal(zkd):
    rng = random.Random(14)
    lo, hi = 1 << (FRAC - 2), 1 << (FRAC - 1)
    a = [lo + rng.getrandbits(FRAC - 2) for _ in range(1500)] + [lo, hi, lo + 1, hi - 1, (lo + hi) // 2]
    got = run(zkd, "recip", a)
    worst = max(abs(g - (1 << (2 * FRAC)) // x) for x, g in zip(a, got))
    assert worst <= 64, worst  # units of 2^-812 on a result in [2, 4]


def test_rsqrt(zkd):
    rng = random.Random(15)
    a = []
    for _ in range(1200):
        bits = rng.randrange(762, 838)  # 1/sqrt(a) < 2^26 must fit the FX integer part
        a.append((1 << (bits - 1)) + rng.getrandbits(bits - 1))
    a += [1 << FRAC, 1 << (FRAC - 2), (1 << FRAC) - 1, 3 << (FRAC - 1)]
    got = run(zkd, "rsqrt", a)
    worst = 0.0
    for x, g in zip(a, got):
        exact = math.isqrt((1 << (3 * FRAC + 40)) // x)  # 2^20 sub-units
        scale = max(1.0, 2.0 ** ((FRAC - x.bit_length()) / 2))
        worst = max(worst, abs(g * (1 << 20) - exact) / (1 << 20) / scale)
    assert worst <= 64, worst
    assert run(zkd, "rsqrt", [0, -5]) == [0, 0]


def test_fp64_round_trip(zkd):
    """fx_to_double (truncating Horner) then fx_from_double (exact scatter of the 53-bit mantissa): the result is a double's
    worth of leading bits of the input, within 2 ulp_53 of it, and a fixed point of the round trip for values that are
    doubles already."""
    rng = random.Random(16)
    a = [rand_fx(rng, rng.randrange(60, 838)) for _ in range(1500)]
    got = run(zkd, "from_double", a)
    for x, g in zip(a, got):
        assert abs(g - x) <= abs(x) >> 51, (x, g)
    exact = [(rng.getrandbits(53) | (1 << 52)) << rng.randrange(0, 780) for _ in range(500)]
    exact = [v if rng.random() < 0.5 else -v for v in exact]
    assert run(zkd, "from_double", exact) == exact

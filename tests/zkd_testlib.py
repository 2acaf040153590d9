"""Helpers for the GPU tests: a pure-Python-integer model of the library's internal fixed-point planes (include/zkd.h,
"Internal fixed-point format") so that building-block kernels can be checked bit for bit against Python's exact
integer arithmetic.  Shares no code with the CUDA path or with oracle/."""
from __future__ import annotations

import numpy as np

ND, DB, FRAC = 30, 28, 812
DMASK = (1 << DB) - 1


def fx_planes_from_ints(vals) -> np.ndarray:
    """list of Python ints (value * 2^812) -> int32[ND][count], canonical digits (top digit signed)."""
    out = np.zeros((ND, len(vals)), dtype=np.int32)
    for e, v in enumerate(vals):
        for k in range(ND - 1):
            out[k, e] = (v >> (DB * k)) & DMASK
        top = v >> (DB * (ND - 1))
        assert -(1 << 31) <= top < (1 << 31), "value does not fit FX"
        out[ND - 1, e] = top
    return out


def ints_from_fx_planes(planes: np.ndarray) -> list[int]:
    planes = np.asarray(planes).reshape(ND, -1)
    out = []
    for e in range(planes.shape[1]):
        v = 0
        for k in range(ND):
            v += int(planes[k, e]) << (DB * k)
        out.append(v)
    return out


def fxc_from_ints(re, im) -> np.ndarray:
    """complex FX array: int32[2][ND][count]"""
    return np.stack([fx_planes_from_ints(re), fx_planes_from_ints(im)])


def ints_from_fxc(arr: np.ndarray):
    arr = np.asarray(arr).reshape(2, ND, -1)
    return ints_from_fx_planes(arr[0]), ints_from_fx_planes(arr[1])


def window(v: int, top_bit: int, digits: int) -> int:
    """bits [top_bit - 28*digits, top_bit) of the two's-complement integer v (floor at the low end)."""
    lsb = top_bit - DB * digits
    if lsb <= 0:
        return v
    return (v >> lsb) << lsb


def api_value_to_fx_int(mant: int, exp2: int, scale_bits: int = 0) -> int:
    """value = mant 2^exp2 -> trunc-toward-zero(value * 2^(812 + scale))"""
    sh = exp2 + FRAC + scale_bits
    if mant == 0:
        return 0
    a = abs(mant)
    m = a << sh if sh >= 0 else a >> (-sh)
    return m if mant > 0 else -m

"""Seeded synthetic input generators, shared by the oracle tests and the CUDA-path tests / bench.

This module holds none of the method's arithmetic (no eigensolver, no refinement, no comparator); it builds
*inputs* only, with the shapes and value distributions of the paper's workload ("N x N Hermitian matrix with
random elements", 768-bit) and of BASELINE.json's five configs (recipe in DESIGN.md, section
"Input recipe").  It also carries a small pure-Python codec between the API number layout and Python integers
so that tests can inspect numbers without going through either the oracle or the CUDA library.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from fractions import Fraction

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libzkd_inputs.so")
_SRC = os.path.join(_HERE, "zkd_inputs.c")

PREC = 768


def build(force: bool = False) -> str:
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(
            ["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", _SO, _SRC, "-l:libmpfr.so.6", "-l:libgmp.so.10"]
        )
    return _SO


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        u8p = ctypes.c_void_p
        L.zkd_inputs_word.restype = ctypes.c_uint64
        L.zkd_inputs_word.argtypes = [ctypes.c_uint64] * 3
        L.zkd_inputs_random_herm.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_uint64, ctypes.c_uint64, u8p]
        L.zkd_inputs_qdq.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_uint64, ctypes.c_uint64, ctypes.c_int, u8p, u8p, u8p]
        L.zkd_inputs_uniform_real.argtypes = [u8p, ctypes.c_int, ctypes.c_uint64, ctypes.c_uint64, ctypes.c_uint64]
        _lib = L
    return _lib


def real_bytes(prec: int = PREC) -> int:
    return 16 + prec // 8


# ----------------------------------------------------------------------------------------------------------
# API number codec (pure Python integers; independent of oracle/ and of the CUDA library)
# ----------------------------------------------------------------------------------------------------------

def encode_real(mant: int, exp2: int, prec: int = PREC) -> bytes:
    """Encode the exact value mant * 2**exp2 (mant any Python int) after round-to-nearest-even to prec bits."""
    rb = real_bytes(prec)
    if mant == 0:
        return bytes(rb)
    sign = -1 if mant < 0 else 1
    m = abs(mant)
    bl = m.bit_length()
    if bl > prec:
        sh = bl - prec
        q, r = m >> sh, m & ((1 << sh) - 1)
        half = 1 << (sh - 1)
        if r > half or (r == half and (q & 1)):
            q += 1
        m, exp2 = q, exp2 + sh
        if m.bit_length() > prec:
            m >>= 1
            exp2 += 1
    else:
        m <<= prec - bl
        exp2 -= prec - bl
    # value = m * 2**exp2 with m in [2^(prec-1), 2^prec)  ->  exp field e: value = m * 2**(e - prec)
    e = exp2 + prec
    out = bytearray(rb)
    out[0:4] = int(sign).to_bytes(4, "little", signed=True)
    out[8:16] = int(e).to_bytes(8, "little", signed=True)
    out[16:] = m.to_bytes(prec // 8, "little")
    return bytes(out)


def decode_real(buf, prec: int = PREC):
    """Return (mant, exp2) with value = mant * 2**exp2 exactly (mant signed Python int)."""
    b = bytes(buf)
    sign = int.from_bytes(b[0:4], "little", signed=True)
    flags = int.from_bytes(b[4:8], "little", signed=True)
    e = int.from_bytes(b[8:16], "little", signed=True)
    m = int.from_bytes(b[16:16 + prec // 8], "little")
    if flags != 0 or sign not in (-1, 0, 1):
        raise ValueError("malformed API number")
    if sign == 0:
        return 0, 0
    if not (m >> (prec - 1)):
        raise ValueError("API number not normalised")
    return sign * m, e - prec


def to_fraction(buf, prec: int = PREC) -> Fraction:
    m, e = decode_real(buf, prec)
    return Fraction(m) * (Fraction(2) ** e)


def to_mpf(buf, prec: int = PREC):
    import mpmath

    m, e = decode_real(buf, prec)
    return mpmath.ldexp(mpmath.mpf(m), e)


def from_fraction(x: Fraction, prec: int = PREC) -> bytes:
    """Round an exact rational to prec bits (nearest-even on the truncated binary expansion with sticky bit)."""
    if x == 0:
        return bytes(real_bytes(prec))
    num, den = x.numerator, x.denominator
    # scale so that the quotient has prec+64 bits, then fold the remainder into a sticky bit
    sh = prec + 64 + den.bit_length() - abs(num).bit_length()
    if sh < 0:
        sh = 0
    q, r = divmod(abs(num) << sh, den)
    q = (q << 1) | (1 if r else 0)
    return encode_real(q if num > 0 else -q, -sh - 1, prec)


def from_mpf(x, prec: int = PREC) -> bytes:
    import mpmath

    x = mpmath.mpf(x)
    if x == 0:
        return bytes(real_bytes(prec))
    sgn, man, ex, _bc = x._mpf_
    return encode_real(-int(man) if sgn else int(man), int(ex), prec)


def reals_array(n: int, prec: int = PREC) -> np.ndarray:
    return np.zeros((n, real_bytes(prec)), dtype=np.uint8)


def cmatrix_to_mp(buf: np.ndarray, N: int, prec: int = PREC):
    """Decode an N x N complex API matrix into an mpmath matrix (small N only)."""
    import mpmath

    rb = real_bytes(prec)
    flat = np.ascontiguousarray(buf).reshape(N, N, 2, rb)
    M = mpmath.matrix(N, N)
    for i in range(N):
        for j in range(N):
            M[i, j] = mpmath.mpc(to_mpf(flat[i, j, 0], prec), to_mpf(flat[i, j, 1], prec))
    return M


def rvector_to_mp(buf: np.ndarray, N: int, prec: int = PREC):
    rb = real_bytes(prec)
    flat = np.ascontiguousarray(buf).reshape(N, rb)
    return [to_mpf(flat[i], prec) for i in range(N)]


def cmatrix_from_mp(M, N: int, prec: int = PREC) -> np.ndarray:
    import mpmath

    rb = real_bytes(prec)
    out = np.zeros((N, N, 2, rb), dtype=np.uint8)
    for i in range(N):
        for j in range(N):
            z = mpmath.mpc(M[i, j])
            out[i, j, 0] = np.frombuffer(from_mpf(z.real, prec), dtype=np.uint8)
            out[i, j, 1] = np.frombuffer(from_mpf(z.imag, prec), dtype=np.uint8)
    return out.reshape(-1)


# ----------------------------------------------------------------------------------------------------------
# generators
# ----------------------------------------------------------------------------------------------------------

def random_hermitian(N: int, seed: int, stream: int = 0, prec: int = PREC) -> np.ndarray:
    """N x N complex Hermitian, off-diagonal Re/Im and real diagonal i.i.d. uniform[-1,1) (reading A2).
    Returns a uint8 array of N*N*2*real_bytes(prec) bytes in the API layout."""
    out = np.zeros(N * N * 2 * real_bytes(prec), dtype=np.uint8)
    rc = lib().zkd_inputs_random_herm(N, prec, seed, stream, out.ctypes.data)
    if rc:
        raise ValueError("zkd_inputs_random_herm failed")
    return out


def qdq(N: int, seed: int, stream: int, reflectors: int, lam: np.ndarray, want_q: bool = False, prec: int = PREC):
    """A = Q diag(lam) Q^H with Q from `reflectors` seeded Householder reflectors (readings A12-A14).
    `lam` is an (N, real_bytes) uint8 array of API reals.  Returns A (and Q if want_q)."""
    rb = real_bytes(prec)
    lam = np.ascontiguousarray(lam, dtype=np.uint8).reshape(N, rb)
    A = np.zeros(N * N * 2 * rb, dtype=np.uint8)
    Q = np.zeros(N * N * 2 * rb, dtype=np.uint8) if want_q else None
    rc = lib().zkd_inputs_qdq(N, prec, seed, stream, reflectors, lam.ctypes.data, A.ctypes.data,
                              Q.ctypes.data if want_q else None)
    if rc:
        raise ValueError("zkd_inputs_qdq failed")
    return (A, Q) if want_q else A


def _lam_array(values, prec: int = PREC) -> np.ndarray:
    """values: list of Fractions (exact dyadic rationals) -> (N, rb) uint8."""
    rb = real_bytes(prec)
    out = np.zeros((len(values), rb), dtype=np.uint8)
    for i, v in enumerate(values):
        out[i] = np.frombuffer(from_fraction(Fraction(v), prec), dtype=np.uint8)
    return out


def mps_spectrum(N: int = 32, exps=(1, 11, 21, 31, 40, 50, 60)):
    """Reading A12: 1 dominant value + powers of two 2^-e, the rest exact zeros; trace exactly 1.
    Returned ascending (zeros first)."""
    small = [Fraction(1, 2 ** e) for e in exps]
    dom = 1 - sum(small)
    vals = [Fraction(0)] * (N - len(small) - 1) + sorted(small + [dom])
    return vals


def clustered_spectrum(n_clusters: int, cluster_size: int, seed: int, spacing_exp: int = 200, prec: int = PREC):
    """Reading A13: cluster centres uniform[-1,1) (seeded, prec bits), lambda = c_g + k 2^-spacing_exp."""
    rb = real_bytes(prec)
    buf = np.zeros(rb, dtype=np.uint8)
    centres = []
    for g in range(n_clusters):
        lib().zkd_inputs_uniform_real(buf.ctypes.data, prec, seed, 0xC1057E5, g * (prec // 64))
        centres.append(to_fraction(buf, prec))
    vals = []
    for c in centres:
        for k in range(cluster_size):
            vals.append(c + Fraction(k, 2 ** spacing_exp))
    vals.sort()
    return vals


def epsilon_spectrum(N: int, n_qubits: int):
    """Schmidt weights {1 - eps, eps, 0, ...} with eps = 2^-(n-1)."""
    eps = Fraction(1, 2 ** (n_qubits - 1))
    return [Fraction(0)] * (N - 2) + [eps, 1 - eps]


CONFIG_SEEDS = {"c1": 1001, "c2": 1002, "c3": 1003, "c4": 1004, "c5": 1005}


def config(name: str, want_answer: bool = False, batch: int | None = None, prec: int = PREC):
    """Build one of BASELINE.json's configs (or a reduced analog).  Returns dict with
    N, batch, A (uint8, [batch][N][N][2][rb]) and, for constructed spectra, lam (and Q if want_answer)."""
    rb = real_bytes(prec)
    if name in ("c1", "c2", "c3"):
        N = {"c1": 16, "c2": 64, "c3": 256}[name]
        b = batch or 1
        A = np.concatenate([random_hermitian(N, CONFIG_SEEDS[name], s, prec) for s in range(b)])
        return {"name": name, "N": N, "batch": b, "A": A}
    if name in ("c4", "c4small"):
        N = 32 if name == "c4" else 16
        b = batch or (512 if name == "c4" else 4)
        exps = (1, 11, 21, 31, 40, 50, 60)
        vals = mps_spectrum(N, exps)
        lam = _lam_array(vals, prec)
        As, Qs = [], []
        for s in range(b):
            r = qdq(N, CONFIG_SEEDS["c4"], s, 3, lam, want_q=want_answer, prec=prec)
            if want_answer:
                As.append(r[0]); Qs.append(r[1])
            else:
                As.append(r)
        d = {"name": name, "N": N, "batch": b, "A": np.concatenate(As), "lam": np.tile(lam.reshape(-1), b), "lam_exact": vals}
        if want_answer:
            d["Q"] = np.concatenate(Qs)
        return d
    if name in ("c5", "c5small", "c5mid"):
        ncl, csz, refl = {"c5": (64, 16, 8), "c5mid": (8, 16, 8), "c5small": (4, 8, 3)}[name]
        N = ncl * csz
        vals = clustered_spectrum(ncl, csz, CONFIG_SEEDS["c5"], 200, prec)
        lam = _lam_array(vals, prec)
        r = qdq(N, CONFIG_SEEDS["c5"], 0, refl, lam, want_q=want_answer, prec=prec)
        d = {"name": name, "N": N, "batch": 1, "A": r[0] if want_answer else r, "lam": lam.reshape(-1), "lam_exact": vals}
        if want_answer:
            d["Q"] = r[1]
        return d
    raise KeyError(name)

"""oracle — TEST INFRASTRUCTURE ONLY.

A plain, slow CPU oracle (768-bit cyclic Jacobi on MPFR, C source in zkd_oracle.c) for the result the hot path
computes: the eigendecomposition of a dense complex Hermitian matrix at 768-bit precision (2.1).
Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this package.
It imports nothing from paper_2402_11868_b200 (the CUDA path) and the CUDA path imports nothing from here.

Parity status: pinned (tests/test_oracle_pins.py) — see the header of zkd_oracle.c for the list of pins.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libzkd_oracle.so")
_SRCS = [os.path.join(_HERE, "zkd_oracle.c"), os.path.join(_HERE, "mpfr_abi.h")]

PREC = 768
GUARD_BITS = 128  # reading A6


def build(force: bool = False) -> str:
    if force or not os.path.exists(_SO) or any(os.path.getmtime(_SO) < os.path.getmtime(s) for s in _SRCS):
        subprocess.check_call(
            ["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", _SO, _SRCS[0], "-l:libmpfr.so.6", "-l:libgmp.so.10", "-lm"]
        )
    return _SO


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        vp = ctypes.c_void_p
        L.zkd_oracle_diag_herm.restype = ctypes.c_int
        L.zkd_oracle_diag_herm.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                           ctypes.c_long, vp, vp, vp, vp]
        L.zkd_oracle_compare.restype = ctypes.c_int
        L.zkd_oracle_compare.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, vp, vp, vp, vp, vp, vp, ctypes.c_int, vp]
        L.zkd_oracle_svd.restype = ctypes.c_int
        L.zkd_oracle_svd.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, vp, vp, vp, vp, vp]
        L.zkd_oracle_svd_compare.restype = ctypes.c_int
        L.zkd_oracle_svd_compare.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, vp, vp, vp, vp, vp, vp, vp, vp]
        L.zkd_oracle_lu_solve.restype = ctypes.c_int
        L.zkd_oracle_lu_solve.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, vp, vp, vp]
        L.zkd_oracle_rqi.restype = ctypes.c_int
        L.zkd_oracle_rqi.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, vp, vp, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                     ctypes.c_int, ctypes.c_int, vp, vp]
        L.zkd_oracle_api_to_double.restype = ctypes.c_double
        L.zkd_oracle_api_to_double.argtypes = [vp, ctypes.c_int]
        L.zkd_oracle_api_from_double.argtypes = [vp, ctypes.c_int, ctypes.c_double]
        L.zkd_oracle_mpfr_version.restype = ctypes.c_char_p
        L.zkd_oracle_max_threads.restype = ctypes.c_int
        _lib = L
    return _lib


def real_bytes(prec: int = PREC) -> int:
    return 16 + prec // 8


def host_threads() -> int:
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:  # pragma: no cover
        return os.cpu_count() or 1


def diag_herm(A: np.ndarray, N: int, prec: int = PREC, ordering: str = "row-cyclic", guard_bits: int = GUARD_BITS,
              threads: int | None = None, max_rotations: int = 0, want_vectors: bool = True):
    """Cyclic Jacobi eigendecomposition of ONE N x N Hermitian matrix given in the API layout.
    Returns (eigvals uint8[N*rb], eigvecs uint8[N*N*2*rb] or None, info dict)."""
    rb = real_bytes(prec)
    A = np.ascontiguousarray(A, dtype=np.uint8)
    assert A.size == N * N * 2 * rb, (A.size, N)
    lam = np.zeros(N * rb, dtype=np.uint8)
    X = np.zeros(N * N * 2 * rb, dtype=np.uint8) if want_vectors else None
    info = (ctypes.c_long * 3)()
    o = {"row-cyclic": 0, "round-robin": 1}[ordering]
    t = threads or (host_threads() if o == 1 else 1)
    rc = lib().zkd_oracle_diag_herm(N, prec, guard_bits, o, t, max_rotations, A.ctypes.data, lam.ctypes.data,
                                    X.ctypes.data if want_vectors else None, info)
    return lam, X, {"status": rc, "sweeps": info[0], "rotations": info[1], "threads": t}


def compare(A: np.ndarray, N: int, lam: np.ndarray, X: np.ndarray, lam0: np.ndarray | None = None,
            X0: np.ndarray | None = None, cols=None, prec: int = PREC, threads: int | None = None) -> dict:
    """Comparator of SURVEY.md 8(c): returns log2 error measures (see zkd_oracle_compare)."""
    out = np.zeros(8, dtype=np.float64)
    c = np.ascontiguousarray(cols, dtype=np.int32) if cols is not None else None
    lib().zkd_oracle_compare(
        N, prec, threads or host_threads(),
        np.ascontiguousarray(A).ctypes.data, np.ascontiguousarray(lam).ctypes.data, np.ascontiguousarray(X).ctypes.data,
        np.ascontiguousarray(lam0).ctypes.data if lam0 is not None else None,
        np.ascontiguousarray(X0).ctypes.data if X0 is not None else None,
        c.ctypes.data if c is not None else None, len(c) if c is not None else 0, out.ctypes.data)
    return {"log2_dlam_rel": out[0], "log2_resid_rel": out[1], "log2_orth": out[2], "vec_margin_bits": out[3],
            "log2_F": out[4], "groups": int(out[5]) if out[5] > -1e8 else 0,
            "max_group": int(out[6]) if out[6] > -1e8 else 0, "log2_vec_err": out[7]}


def svd(A: np.ndarray, M: int, N: int, prec: int = PREC, guard_bits: int = GUARD_BITS):
    """One-sided Jacobi SVD of ONE M x N complex matrix in the API layout (NEXT-1).
    Returns (S uint8[K*rb] descending, U uint8[M*K*2*rb], V uint8[N*K*2*rb], info dict), K = min(M, N)."""
    rb = real_bytes(prec)
    K = min(M, N)
    A = np.ascontiguousarray(A, dtype=np.uint8)
    assert A.size == M * N * 2 * rb, (A.size, M, N)
    S = np.zeros(K * rb, dtype=np.uint8)
    U = np.zeros(M * K * 2 * rb, dtype=np.uint8)
    V = np.zeros(N * K * 2 * rb, dtype=np.uint8)
    info = (ctypes.c_long * 3)()
    rc = lib().zkd_oracle_svd(M, N, prec, guard_bits, A.ctypes.data, S.ctypes.data, U.ctypes.data, V.ctypes.data, info)
    return S, U, V, {"status": rc, "sweeps": info[0], "rotations": info[1]}


def svd_compare(A: np.ndarray, M: int, N: int, S, U, V, S0=None, U0=None, V0=None, prec: int = PREC) -> dict:
    """Comparator for singular value decompositions (see zkd_oracle_svd_compare)."""
    out = np.zeros(8, dtype=np.float64)
    def p(x):
        return np.ascontiguousarray(x).ctypes.data if x is not None else None
    keep = [np.ascontiguousarray(x) for x in (A, S, U, V)] + [np.ascontiguousarray(x) for x in (S0, U0, V0) if x is not None]
    lib().zkd_oracle_svd_compare(M, N, prec, keep[0].ctypes.data, keep[1].ctypes.data, keep[2].ctypes.data, keep[3].ctypes.data,
                                 p(S0), p(U0), p(V0), out.ctypes.data)
    return {"log2_dsig_rel": out[0], "log2_resid_rel": out[1], "log2_orth": out[2], "vec_margin_bits": out[3], "log2_F": out[4],
            "groups": int(out[5]) if out[5] > -1e8 else 0, "max_group": int(out[6]) if out[6] > -1e8 else 0, "log2_vec_err": out[7]}


def lu_solve(A: np.ndarray, B: np.ndarray, N: int, nrhs: int, prec: int = PREC, guard_bits: int = GUARD_BITS):
    """Gaussian elimination with partial pivoting on MPFR (NEXT-3): X with A X = B.  Returns (X, status)."""
    rb = real_bytes(prec)
    A = np.ascontiguousarray(A, dtype=np.uint8)
    B = np.ascontiguousarray(B, dtype=np.uint8)
    assert A.size == N * N * 2 * rb and B.size == N * nrhs * 2 * rb
    X = np.zeros(N * nrhs * 2 * rb, dtype=np.uint8)
    rc = lib().zkd_oracle_lu_solve(N, nrhs, prec, guard_bits, A.ctypes.data, B.ctypes.data, X.ctypes.data)
    return X, rc


def api_matrix_to_complex128(A: np.ndarray, N: int, prec: int = PREC) -> np.ndarray:
    """Hermitian API matrix (upper triangle authoritative) rounded to complex128, for the fp64 stage of rqi_refine."""
    rb = real_bytes(prec)
    flat = np.ascontiguousarray(A, dtype=np.uint8).reshape(N, N, 2, rb)
    out = np.zeros((N, N), dtype=np.complex128)
    for i in range(N):
        for j in range(i, N):
            re = lib().zkd_oracle_api_to_double(flat[i, j, 0].ctypes.data, prec)
            im = lib().zkd_oracle_api_to_double(flat[i, j, 1].ctypes.data, prec) if i != j else 0.0
            out[i, j] = complex(re, im)
            out[j, i] = complex(re, -im)
    return out


def rqi_refine(A: np.ndarray, N: int, first: int = 0, count: int | None = None, iters: int = 3, max_pivots: int = 0,
               threads: int | None = None, prec: int = PREC, guard_bits: int = GUARD_BITS, V64: np.ndarray | None = None):
    """CPU restatement of the paper's route: LAPACK fp64 eigendecomposition (numpy.linalg.eigh), then Rayleigh
    quotient iteration in MPFR (one Gaussian elimination per eigenpair and iteration).  Timed CPU baseline only.
    Returns (lam uint8[count*rb], X uint8[N*count*2*rb], seconds of the fp64 stage, V64)."""
    import time

    rb = real_bytes(prec)
    count = N - first if count is None else count
    A = np.ascontiguousarray(A, dtype=np.uint8)
    t0 = time.perf_counter()
    if V64 is None:
        _, V64 = np.linalg.eigh(api_matrix_to_complex128(A, N, prec))
    t64 = time.perf_counter() - t0
    Vc = np.ascontiguousarray(V64.astype(np.complex128)).view(np.float64)
    lam = np.zeros(count * rb, dtype=np.uint8)
    X = np.zeros(N * count * 2 * rb, dtype=np.uint8)
    rc = lib().zkd_oracle_rqi(N, prec, guard_bits, A.ctypes.data, Vc.ctypes.data, first, count, iters, max_pivots,
                              threads or host_threads(), lam.ctypes.data, X.ctypes.data)
    assert rc == 0, rc
    return lam, X, t64, V64


def api_to_double(buf, prec: int = PREC) -> float:
    b = np.ascontiguousarray(np.frombuffer(bytes(buf), dtype=np.uint8))
    return lib().zkd_oracle_api_to_double(b.ctypes.data, prec)


def api_from_double(v: float, prec: int = PREC) -> bytes:
    b = np.zeros(real_bytes(prec), dtype=np.uint8)
    lib().zkd_oracle_api_from_double(b.ctypes.data, prec, v)
    return bytes(b)

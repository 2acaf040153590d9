"""paper_2402_11868_b200 — thin ctypes binding of libzkd (include/zkd.h).

Argument marshalling only: every step of the hot path (S0 ingest .. S6 export) runs in the
CUDA kernels of libzkd.so.  torch is used for device memory and streams, nothing else.  There is no CPU fallback:
if libzkd.so is missing or fails to load, importing a function from here raises.
"""
from __future__ import annotations

import ctypes
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
SO_PATH = os.path.join(_HERE, "libzkd.so")

PREC = 768
REAL_BYTES = 16 + PREC // 8  # 112
FX_DIGITS = 30
FX_FRAC_BITS = 812

ZKD_OK = 0


class ZkdError(RuntimeError):
    def __init__(self, code: int, what: str):
        super().__init__(f"{what}: {strerror(code)} ({code})")
        self.code = code


class zkd_info(ctypes.Structure):
    _fields_ = [("status", ctypes.c_int32), ("steps", ctypes.c_int32), ("n_clusters", ctypes.c_int32),
                ("max_cluster", ctypes.c_int32), ("log2_resid", ctypes.c_float), ("log2_orth", ctypes.c_float)]


_lib = None


def lib() -> ctypes.CDLL:
    """Load libzkd.so (built in-tree by paper_2402_11868_b200.build).  Fails loudly when it is absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(SO_PATH):
        raise ImportError(f"{SO_PATH} not found: run `python -m paper_2402_11868_b200.build` (no CPU fallback exists)")
    L = ctypes.CDLL(SO_PATH)
    vp, ci, cs, cd = ctypes.c_void_p, ctypes.c_int, ctypes.c_size_t, ctypes.c_double
    L.zkd_real_bytes.restype = cs
    L.zkd_real_bytes.argtypes = [ci]
    L.zkd_diag_herm_bufsize.argtypes = [ci, ci, ci, ctypes.POINTER(cs)]
    L.zkd_diag_herm_ws.argtypes = [ci, ci, ci, vp, vp, vp, vp, cs, vp, vp]
    L.zkd_diag_herm.argtypes = [ci, ci, ci, vp, vp, vp, vp]
    L.zkd_diag_herm_host.argtypes = [ci, ci, ci, vp, vp, vp, vp]
    L.zkd_svd_bufsize.argtypes = [ci, ci, ci, ci, ctypes.POINTER(cs)]
    L.zkd_svd_ws.argtypes = [ci, ci, ci, ci, vp, vp, vp, vp, vp, cs, vp, vp]
    L.zkd_svd.argtypes = [ci, ci, ci, ci, vp, vp, vp, vp, vp]
    L.zkd_lu_solve_bufsize.argtypes = [ci, ci, ci, ci, ctypes.POINTER(cs)]
    L.zkd_lu_solve.argtypes = [ci, ci, ci, ci, vp, vp, vp, vp, cs, vp, vp]
    L.zkd_diag_herm_rqi_lu_bufsize.argtypes = [ci, ci, ci, ctypes.POINTER(cs)]
    L.zkd_diag_herm_rqi_lu.argtypes = [ci, ci, ci, vp, vp, vp, vp, cs, vp, vp]
    L.zkd_mps_two_site_update_bufsize.argtypes = [ci, ci, ci, ci, ci, ci, ctypes.POINTER(cs)]
    L.zkd_mps_two_site_update.argtypes = [ci, ci, ci, ci, ci, ci, vp, vp, vp, ci, ci, vp, vp, vp, vp, vp, vp, cs, vp]
    L.zkd_set_option.argtypes = [ctypes.c_char_p, cd]
    L.zkd_get_option.argtypes = [ctypes.c_char_p, ctypes.POINTER(cd)]
    L.zkd_strerror.restype = ctypes.c_char_p
    L.zkd_strerror.argtypes = [ci]
    L.zkd_version.restype = ci
    L.zkd_counters.restype = None
    L.zkd_counters.argtypes = [ctypes.POINTER(ctypes.c_uint64), ctypes.POINTER(ctypes.c_uint64)]
    L.zkd_counters_reset.restype = None
    L.zkd_kernel_timing.argtypes = [ci]
    L.zkd_kernel_timing_read.argtypes = [ctypes.POINTER(cd), ctypes.POINTER(ctypes.c_uint64), ctypes.POINTER(ctypes.c_uint64)]
    L.zkd_kernel_timing_read_i8.argtypes = [ctypes.POINTER(cd), ctypes.POINTER(ctypes.c_uint64), ctypes.POINTER(ctypes.c_uint64)]
    L.zkd_pack.argtypes = [vp, ci, ci, ctypes.c_int64, vp]
    L.zkd_unpack.argtypes = [vp, ci, ctypes.POINTER(ci), ctypes.POINTER(ctypes.c_int64), vp]
    L.zkd_from_double.argtypes = [vp, ci, cd]
    L.zkd_to_double.restype = cd
    L.zkd_to_double.argtypes = [vp, ci]
    L.zkd_fx_from_api.argtypes = [ci, ci, vp, vp, ci, vp]
    L.zkd_fx_to_api.argtypes = [ci, ci, vp, vp, ci, vp]
    L.zkd_fx_prim.argtypes = [ci, ci, vp, vp, vp, vp]
    L.zkd_gemm_fx_bufsize.argtypes = [ci, ci, ci, ci, ctypes.POINTER(cs)]
    L.zkd_gemm_fx.argtypes = [ci, ci, ci, ci, ci, vp, ci, ci, vp, ci, ci, vp, ci, ci, ci, vp, cs, vp, vp, vp]
    L.zkd_seed_fp64.argtypes = [ci, ci, vp, vp, vp, vp]
    L.zkd_seed_fp64_static.argtypes = [ci, ci, vp, vp, vp, vp]
    L.zkd_measure_imad_peak.argtypes = [cd, ctypes.POINTER(cd), vp]
    L.zkd_measure_dfma_peak.argtypes = [cd, ctypes.POINTER(cd), vp]
    L.zkd_measure_i8_mma_peak.argtypes = [cd, ctypes.POINTER(cd), vp]
    L.zkd_seed_stats.argtypes = [ctypes.POINTER(ctypes.c_uint64), ctypes.POINTER(ctypes.c_uint64), ci]
    L.zkd_kernel_timing_categories.restype = ci
    L.zkd_kernel_timing_name.restype = ctypes.c_char_p
    L.zkd_kernel_timing_name.argtypes = [ci]
    L.zkd_kernel_timing_read_cat.argtypes = [ci, ctypes.POINTER(cd), ctypes.POINTER(ctypes.c_uint64), ctypes.POINTER(ctypes.c_uint64),
                                             ctypes.POINTER(ctypes.c_uint64)]
    _lib = L
    return L


def strerror(code: int) -> str:
    return lib().zkd_strerror(code).decode()


def _check(rc: int, what: str) -> None:
    if rc != ZKD_OK:
        raise ZkdError(rc, what)


def _stream_ptr(stream) -> int:
    import torch

    s = stream if stream is not None else torch.cuda.current_stream()
    return int(s.cuda_stream)


def _dev_u8(t, nbytes: int, name: str) -> int:
    import torch

    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.is_contiguous()):
        raise TypeError(f"{name} must be a contiguous CUDA tensor")
    if t.numel() * t.element_size() < nbytes:
        raise ValueError(f"{name} holds {t.numel() * t.element_size()} bytes, {nbytes} needed")
    return t.data_ptr()


def real_bytes(prec_bits: int = PREC) -> int:
    return int(lib().zkd_real_bytes(prec_bits))


def version() -> int:
    return int(lib().zkd_version())


def set_option(key: str, value: float) -> None:
    _check(lib().zkd_set_option(key.encode(), float(value)), f"zkd_set_option({key})")


def get_option(key: str) -> float:
    v = ctypes.c_double()
    _check(lib().zkd_get_option(key.encode(), ctypes.byref(v)), f"zkd_get_option({key})")
    return v.value


def counters() -> tuple[int, int]:
    a, b = ctypes.c_uint64(), ctypes.c_uint64()
    lib().zkd_counters(ctypes.byref(a), ctypes.byref(b))
    return int(a.value), int(b.value)


def counters_reset() -> None:
    lib().zkd_counters_reset()


def kernel_timing(enable: bool) -> None:
    _check(lib().zkd_kernel_timing(1 if enable else 0), "zkd_kernel_timing")


def kernel_timing_read() -> tuple[float, int, int]:
    """(summed digit-GEMM kernel time in ms, timed launches, digit products of those launches)"""
    ms, n, m = ctypes.c_double(), ctypes.c_uint64(), ctypes.c_uint64()
    _check(lib().zkd_kernel_timing_read(ctypes.byref(ms), ctypes.byref(n), ctypes.byref(m)), "zkd_kernel_timing_read")
    return ms.value, int(n.value), int(m.value)


def kernel_timing_read_i8() -> tuple[float, int, int]:
    """(summed int8 tcgen05 GEMM kernel time in ms, timed launches, s8 x s8 MACs of those launches)"""
    ms, n, m = ctypes.c_double(), ctypes.c_uint64(), ctypes.c_uint64()
    _check(lib().zkd_kernel_timing_read_i8(ctypes.byref(ms), ctypes.byref(n), ctypes.byref(m)), "zkd_kernel_timing_read_i8")
    return ms.value, int(n.value), int(m.value)


def kernel_timing_categories() -> int:
    return int(lib().zkd_kernel_timing_categories())


def kernel_timing_name(category: int) -> str:
    return lib().zkd_kernel_timing_name(category).decode()


def kernel_timing_read_cat(category: int) -> tuple[float, int, int, int]:
    """(summed kernel time in ms, timed launches, work executed, work algorithmic) of one kernel category"""
    ms, n, we, wa = ctypes.c_double(), ctypes.c_uint64(), ctypes.c_uint64(), ctypes.c_uint64()
    _check(lib().zkd_kernel_timing_read_cat(category, ctypes.byref(ms), ctypes.byref(n), ctypes.byref(we), ctypes.byref(wa)),
           "zkd_kernel_timing_read_cat")
    return ms.value, int(n.value), int(we.value), int(wa.value)


def kernel_timing_read_all() -> dict:
    """{category name: (ms, launches, work executed, work algorithmic)} for every kernel category of the library"""
    return {kernel_timing_name(c): kernel_timing_read_cat(c) for c in range(kernel_timing_categories())}


def seed_stats(reset: bool = False) -> tuple[int, int]:
    """(column elements checked, column elements rotated) by the fp64 seed kernels since the last reset"""
    a, b = ctypes.c_uint64(), ctypes.c_uint64()
    _check(lib().zkd_seed_stats(ctypes.byref(a), ctypes.byref(b), 1 if reset else 0), "zkd_seed_stats")
    return int(a.value), int(b.value)


def diag_herm_bufsize(N: int, batch: int, prec_bits: int = PREC) -> int:
    n = ctypes.c_size_t()
    _check(lib().zkd_diag_herm_bufsize(N, batch, prec_bits, ctypes.byref(n)), "zkd_diag_herm_bufsize")
    return int(n.value)


def diag_herm_ws(N: int, batch: int, A, eigvals, eigvecs, workspace, info=None, prec_bits: int = PREC, stream=None) -> None:
    """zkd_diag_herm_ws on device tensors (uint8, API layout).  `info`: optional uint8/int32 CUDA tensor of
    batch * sizeof(zkd_info) bytes."""
    rb = 16 + prec_bits // 8
    a = _dev_u8(A, batch * N * N * 2 * rb, "A")
    lam = _dev_u8(eigvals, batch * N * rb, "eigvals")
    x = _dev_u8(eigvecs, batch * N * N * 2 * rb, "eigvecs")
    need = diag_herm_bufsize(N, batch, prec_bits)
    w = _dev_u8(workspace, need, "workspace")
    i = _dev_u8(info, batch * ctypes.sizeof(zkd_info), "info") if info is not None else None
    _check(lib().zkd_diag_herm_ws(N, batch, prec_bits, a, lam, x, w, workspace.numel() * workspace.element_size(), i,
                                  _stream_ptr(stream)), "zkd_diag_herm_ws")


def diag_herm(N: int, batch: int, A, eigvals, eigvecs, prec_bits: int = PREC, stream=None) -> None:
    rb = 16 + prec_bits // 8
    a = _dev_u8(A, batch * N * N * 2 * rb, "A")
    lam = _dev_u8(eigvals, batch * N * rb, "eigvals")
    x = _dev_u8(eigvecs, batch * N * N * 2 * rb, "eigvecs")
    _check(lib().zkd_diag_herm(N, batch, prec_bits, a, lam, x, _stream_ptr(stream)), "zkd_diag_herm")


def diag_herm_host(N: int, batch: int, A_host, eigvals_host, eigvecs_host, info_host=None, prec_bits: int = PREC) -> None:
    """zkd_diag_herm_host on HOST buffers (numpy uint8 arrays or pinned CPU torch tensors), copies included."""
    def ptr(x):
        return x.ctypes.data if hasattr(x, "ctypes") else x.data_ptr()
    ip = ctypes.addressof(info_host) if info_host is not None else None
    _check(lib().zkd_diag_herm_host(N, batch, prec_bits, ptr(A_host), ptr(eigvals_host), ptr(eigvecs_host), ip),
           "zkd_diag_herm_host")


def svd_bufsize(M: int, N: int, batch: int, prec_bits: int = PREC) -> int:
    n = ctypes.c_size_t()
    _check(lib().zkd_svd_bufsize(M, N, batch, prec_bits, ctypes.byref(n)), "zkd_svd_bufsize")
    return int(n.value)


def svd_ws(M: int, N: int, batch: int, A, S, U, V, workspace, info=None, prec_bits: int = PREC, stream=None) -> None:
    """zkd_svd_ws on device tensors (uint8, API layout): thin SVD, K = min(M, N) (NEXT-1)."""
    rb, K = 16 + prec_bits // 8, min(M, N)
    i = _dev_u8(info, batch * ctypes.sizeof(zkd_info), "info") if info is not None else None
    _check(lib().zkd_svd_ws(M, N, batch, prec_bits, _dev_u8(A, batch * M * N * 2 * rb, "A"), _dev_u8(S, batch * K * rb, "S"),
                            _dev_u8(U, batch * M * K * 2 * rb, "U"), _dev_u8(V, batch * N * K * 2 * rb, "V"),
                            _dev_u8(workspace, svd_bufsize(M, N, batch, prec_bits), "workspace"),
                            workspace.numel() * workspace.element_size(), i, _stream_ptr(stream)), "zkd_svd_ws")


def svd(M: int, N: int, batch: int, A, S, U, V, prec_bits: int = PREC, stream=None) -> None:
    rb, K = 16 + prec_bits // 8, min(M, N)
    _check(lib().zkd_svd(M, N, batch, prec_bits, _dev_u8(A, batch * M * N * 2 * rb, "A"), _dev_u8(S, batch * K * rb, "S"),
                         _dev_u8(U, batch * M * K * 2 * rb, "U"), _dev_u8(V, batch * N * K * 2 * rb, "V"), _stream_ptr(stream)),
           "zkd_svd")


def lu_solve_bufsize(N: int, nrhs: int, batch: int, prec_bits: int = PREC) -> int:
    n = ctypes.c_size_t()
    _check(lib().zkd_lu_solve_bufsize(N, nrhs, batch, prec_bits, ctypes.byref(n)), "zkd_lu_solve_bufsize")
    return int(n.value)


def lu_solve(N: int, nrhs: int, batch: int, A, B, X, workspace, status=None, prec_bits: int = PREC, stream=None) -> None:
    """zkd_lu_solve on device tensors (uint8, API layout): X with A X = B by multiprecision LU (NEXT-3)."""
    rb = 16 + prec_bits // 8
    _check(lib().zkd_lu_solve(N, nrhs, batch, prec_bits, _dev_u8(A, batch * N * N * 2 * rb, "A"), _dev_u8(B, batch * N * nrhs * 2 * rb, "B"),
                              _dev_u8(X, batch * N * nrhs * 2 * rb, "X"), _dev_u8(workspace, lu_solve_bufsize(N, nrhs, batch, prec_bits), "workspace"),
                              workspace.numel() * workspace.element_size(),
                              _dev_u8(status, batch * 4, "status") if status is not None else None, _stream_ptr(stream)), "zkd_lu_solve")


def diag_herm_rqi_lu_bufsize(N: int, batch: int, prec_bits: int = PREC) -> int:
    n = ctypes.c_size_t()
    _check(lib().zkd_diag_herm_rqi_lu_bufsize(N, batch, prec_bits, ctypes.byref(n)), "zkd_diag_herm_rqi_lu_bufsize")
    return int(n.value)


def diag_herm_rqi_lu(N: int, batch: int, A, eigvals, eigvecs, workspace, info=None, prec_bits: int = PREC, stream=None) -> None:
    """zkd_diag_herm_rqi_lu: the exact-RQI-by-LU cross-check route (S4a'), arguments as diag_herm_ws."""
    rb = 16 + prec_bits // 8
    i = _dev_u8(info, batch * ctypes.sizeof(zkd_info), "info") if info is not None else None
    _check(lib().zkd_diag_herm_rqi_lu(N, batch, prec_bits, _dev_u8(A, batch * N * N * 2 * rb, "A"), _dev_u8(eigvals, batch * N * rb, "eigvals"),
                                      _dev_u8(eigvecs, batch * N * N * 2 * rb, "eigvecs"),
                                      _dev_u8(workspace, diag_herm_rqi_lu_bufsize(N, batch, prec_bits), "workspace"),
                                      workspace.numel() * workspace.element_size(), i, _stream_ptr(stream)), "zkd_diag_herm_rqi_lu")


def mps_two_site_update_bufsize(chiL: int, chiC: int, chiR: int, d: int, batch: int, prec_bits: int = PREC) -> int:
    n = ctypes.c_size_t()
    _check(lib().zkd_mps_two_site_update_bufsize(chiL, chiC, chiR, d, batch, prec_bits, ctypes.byref(n)), "zkd_mps_two_site_update_bufsize")
    return int(n.value)


def mps_two_site_update(chiL: int, chiC: int, chiR: int, d: int, batch: int, L, R, G, W, Lnew, Rnew, kept, workspace, max_keep: int = 0,
                        cutoff_bits: int = 700, info=None, prec_bits: int = PREC, stream=None) -> None:
    """zkd_mps_two_site_update on device tensors (uint8, API layout; kept: int32[batch]) - NEXT-4."""
    rb = 16 + prec_bits // 8
    mL, mR = chiL * d, d * chiR
    K = min(mL, max_keep) if max_keep > 0 else mL
    i = _dev_u8(info, batch * ctypes.sizeof(zkd_info), "info") if info is not None else None
    _check(lib().zkd_mps_two_site_update(
        chiL, chiC, chiR, d, batch, prec_bits, _dev_u8(L, batch * mL * chiC * 2 * rb, "L"), _dev_u8(R, batch * chiC * mR * 2 * rb, "R"),
        _dev_u8(G, batch * d ** 4 * 2 * rb, "G"), max_keep, cutoff_bits, _dev_u8(W, batch * K * rb, "W"),
        _dev_u8(Lnew, batch * mL * K * 2 * rb, "Lnew"), _dev_u8(Rnew, batch * K * mR * 2 * rb, "Rnew"), _dev_u8(kept, batch * 4, "kept"), i,
        _dev_u8(workspace, mps_two_site_update_bufsize(chiL, chiC, chiR, d, batch, prec_bits), "workspace"),
        workspace.numel() * workspace.element_size(), _stream_ptr(stream)), "zkd_mps_two_site_update")


def read_info(info_tensor, batch: int) -> list[dict]:
    raw = bytes(info_tensor.cpu().numpy().tobytes())
    arr = (zkd_info * batch).from_buffer_copy(raw[: batch * ctypes.sizeof(zkd_info)])
    return [{f: getattr(a, f) for f, _ in zkd_info._fields_} for a in arr]


# ---- building blocks -------------------------------------------------------------------------------------------

def fx_from_api(count: int, src_api, dst_fx, scale_bits: int = 0, stream=None, prec_bits: int = PREC) -> None:
    _check(lib().zkd_fx_from_api(count, prec_bits, _dev_u8(src_api, count * (16 + prec_bits // 8), "src_api"),
                                 _dev_u8(dst_fx, count * FX_DIGITS * 4, "dst_fx"), scale_bits, _stream_ptr(stream)),
           "zkd_fx_from_api")


def fx_to_api(count: int, src_fx, dst_api, scale_bits: int = 0, stream=None, prec_bits: int = PREC) -> None:
    _check(lib().zkd_fx_to_api(count, prec_bits, _dev_u8(src_fx, count * FX_DIGITS * 4, "src_fx"),
                               _dev_u8(dst_api, count * (16 + prec_bits // 8), "dst_api"), scale_bits, _stream_ptr(stream)),
           "zkd_fx_to_api")


PRIM = {"add": 0, "sub": 1, "mul": 2, "recip": 3, "rsqrt": 4, "msb": 5, "half": 6, "from_double": 7}


def fx_prim(op: str, count: int, a_fx, b_fx, out_fx, stream=None) -> None:
    """element-wise multi-digit primitive on real FX arrays (int32[30][count] device tensors)"""
    nb = count * FX_DIGITS * 4
    _check(lib().zkd_fx_prim(PRIM[op], count, _dev_u8(a_fx, nb, "a_fx"), _dev_u8(b_fx, nb, "b_fx") if b_fx is not None else None,
                             _dev_u8(out_fx, nb, "out_fx"), _stream_ptr(stream)), "zkd_fx_prim")


def gemm_fx_bufsize(M: int, N: int, K: int, batch: int) -> int:
    n = ctypes.c_size_t()
    _check(lib().zkd_gemm_fx_bufsize(M, N, K, batch, ctypes.byref(n)), "zkd_gemm_fx_bufsize")
    return int(n.value)


def gemm_fx(M, N, K, batch, op_a, A_fx, a_top_bit, a_digits, B_fx, b_top_bit, b_digits, C_fx, mode=0, out_cut_bit=-1,
            path=0, workspace=None, err_flag=None, msb_out=None, stream=None) -> None:
    import torch

    if workspace is None:
        workspace = torch.empty(gemm_fx_bufsize(M, N, K, batch), dtype=torch.uint8, device=A_fx.device)
    per = 2 * FX_DIGITS * 4
    _check(lib().zkd_gemm_fx(M, N, K, batch, op_a, _dev_u8(A_fx, batch * M * K * per, "A_fx"), a_top_bit, a_digits,
                             _dev_u8(B_fx, batch * K * N * per, "B_fx"), b_top_bit, b_digits,
                             _dev_u8(C_fx, batch * M * N * per, "C_fx"), mode, out_cut_bit, path, workspace.data_ptr(),
                             workspace.numel() * workspace.element_size(),
                             err_flag.data_ptr() if err_flag is not None else None,
                             msb_out.data_ptr() if msb_out is not None else None, _stream_ptr(stream)), "zkd_gemm_fx")


def seed_fp64(N: int, batch: int, A64, mu, V, stream=None) -> None:
    _check(lib().zkd_seed_fp64(N, batch, _dev_u8(A64, batch * N * N * 16, "A64"), _dev_u8(mu, batch * N * 8, "mu"),
                               _dev_u8(V, batch * N * N * 16, "V"), _stream_ptr(stream)), "zkd_seed_fp64")


SEED_STATIC_MAX_N = 512


def seed_fp64_static(N: int, batch: int, A64, mu, V, stream=None) -> None:
    """zkd_seed_fp64 without any allocation (scratch in a static device array; N <= SEED_STATIC_MAX_N)"""
    _check(lib().zkd_seed_fp64_static(N, batch, _dev_u8(A64, batch * N * N * 16, "A64"), _dev_u8(mu, batch * N * 8, "mu"),
                                      _dev_u8(V, batch * N * N * 16, "V"), _stream_ptr(stream)), "zkd_seed_fp64_static")


def measure_imad_peak(millis: float = 50.0, stream=None) -> float:
    v = ctypes.c_double()
    _check(lib().zkd_measure_imad_peak(millis, ctypes.byref(v), _stream_ptr(stream)), "zkd_measure_imad_peak")
    return v.value


def measure_i8_mma_peak(millis: float = 50.0, stream=None) -> float:
    v = ctypes.c_double()
    _check(lib().zkd_measure_i8_mma_peak(millis, ctypes.byref(v), _stream_ptr(stream)), "zkd_measure_i8_mma_peak")
    return float(v.value)


def measure_dfma_peak(millis: float = 50.0, stream=None) -> float:
    v = ctypes.c_double()
    _check(lib().zkd_measure_dfma_peak(millis, ctypes.byref(v), _stream_ptr(stream)), "zkd_measure_dfma_peak")
    return v.value


# ---- host-side number helpers (no CUDA) --------------------------------------------------------------------------

def pack(sign: int, exp: int, limbs_le, prec_bits: int = PREC) -> bytes:
    """one real in the API layout from (sign, exp, 64-bit limbs little-endian)"""
    n = prec_bits // 64
    buf = ctypes.create_string_buffer(16 + prec_bits // 8)
    arr = (ctypes.c_uint64 * n)(*[int(x) for x in limbs_le])
    _check(lib().zkd_pack(buf, prec_bits, sign, ctypes.c_int64(exp), arr), "zkd_pack")
    return buf.raw


def unpack(src: bytes, prec_bits: int = PREC) -> tuple[int, int, list[int]]:
    n = prec_bits // 64
    s, e, out = ctypes.c_int(), ctypes.c_int64(), (ctypes.c_uint64 * n)()
    _check(lib().zkd_unpack(ctypes.c_char_p(bytes(src)), prec_bits, ctypes.byref(s), ctypes.byref(e), out), "zkd_unpack")
    return s.value, e.value, [int(x) for x in out]


def from_double(v: float, prec_bits: int = PREC) -> bytes:
    buf = ctypes.create_string_buffer(16 + prec_bits // 8)
    _check(lib().zkd_from_double(buf, prec_bits, float(v)), "zkd_from_double")
    return buf.raw


def to_double(src: bytes, prec_bits: int = PREC) -> float:
    return float(lib().zkd_to_double(ctypes.c_char_p(bytes(src)), prec_bits))

"""CPU-only tests of the boundary (include/zkd.h) and of the host logic around it: the C-ABI library loads and exports
every symbol the header declares, the host-side number helpers follow the documented layout, argument validation
happens before any CUDA call, and the N>1 "replicas only" aggregation of bench.py works over gloo (world_size 2).
No compute entry point is called here (no GPU)."""
from __future__ import annotations

import ctypes
import os
import re
import struct
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


@pytest.fixture(scope="module")
def L():
    from paper_2402_11868_b200 import build as zkd_build

    zkd_build.build()
    import paper_2402_11868_b200 as z

    return z.lib()


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "zkd.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    src = re.sub(r"//[^\n]*", "", src)
    return sorted(set(re.findall(r"\b(zkd_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol(L):
    names = declared_symbols()
    assert len(names) >= 20, names
    for nm in ("zkd_diag_herm", "zkd_diag_herm_ws", "zkd_diag_herm_bufsize", "zkd_diag_herm_host", "zkd_real_bytes"):
        assert nm in names
    missing = [nm for nm in names if not hasattr(L, nm)]
    assert not missing, f"declared in include/zkd.h but not exported by libzkd.so: {missing}"


def test_binding_uses_the_same_names():
    import paper_2402_11868_b200 as z

    for nm in declared_symbols():
        short = nm[len("zkd_"):]
        assert hasattr(z, short) or short in ("info",), f"binding lacks {short}"


def test_real_bytes_and_strerror(L):
    assert L.zkd_real_bytes(768) == 112
    assert L.zkd_real_bytes(100) == 0  # unsupported precision
    assert L.zkd_version() >= 100
    assert L.zkd_strerror(0) and L.zkd_strerror(-1) and L.zkd_strerror(-12345)
    assert len({L.zkd_strerror(-k) for k in range(1, 6)}) >= 4


def test_other_precisions_host_helpers(L):
    """NEXT-2: multiples of 64 bits from 128 to 768 (PAPER.md:61 256 bit, :65 128 bit)."""
    import paper_2402_11868_b200 as z

    for prec in (128, 192, 256, 512, 768):
        assert L.zkd_real_bytes(prec) == 16 + prec // 8
        n = prec // 64
        limbs = [(0x9E3779B97F4A7C15 * (k + 3)) & 0xFFFFFFFFFFFFFFFF for k in range(n)]
        limbs[-1] |= 1 << 63
        raw = z.pack(1, 5, limbs, prec)
        assert len(raw) == 16 + prec // 8
        assert z.unpack(raw, prec) == (1, 5, limbs)
        for v in (0.0, 1.0, -0.3125, 3.0e-200, -7.5e250):
            assert z.to_double(z.from_double(v, prec), prec) == v
    for prec in (0, 64, 100, 832, 1024):
        assert L.zkd_real_bytes(prec) == 0


def test_pack_unpack_layout(L):
    # layout of one real: int32 sign, int32 flags, int64 exp, uint64 limb[12] little-endian
    limbs = [(0x0123456789ABCDEF * (k + 1)) & 0xFFFFFFFFFFFFFFFF for k in range(12)]
    limbs[11] |= 1 << 63
    arr = (ctypes.c_uint64 * 12)(*limbs)
    buf = ctypes.create_string_buffer(112)
    assert L.zkd_pack(buf, 768, -1, ctypes.c_int64(-37), arr) == 0
    sign, flags, exp = struct.unpack_from("<iiq", buf.raw, 0)
    assert (sign, flags, exp) == (-1, 0, -37)
    assert list(struct.unpack_from("<12Q", buf.raw, 16)) == limbs
    s, e, out = ctypes.c_int(0), ctypes.c_int64(0), (ctypes.c_uint64 * 12)()
    assert L.zkd_unpack(buf, 768, ctypes.byref(s), ctypes.byref(e), out) == 0
    assert (s.value, e.value, list(out)) == (-1, -37, limbs)
    # not normalised (top bit clear) is rejected
    limbs[11] &= ~(1 << 63)
    assert L.zkd_pack(buf, 768, 1, ctypes.c_int64(0), (ctypes.c_uint64 * 12)(*limbs)) < 0
    assert L.zkd_pack(buf, 512, 1, ctypes.c_int64(0), arr) < 0


@pytest.mark.parametrize("v", [0.0, 1.0, -1.0, 0.5, -0.75, 3.141592653589793, 2.0 ** -60, -(2.0 ** 40) * 1.0000000001, 5e-324])
def test_from_double_to_double_exact(L, v):
    L.zkd_to_double.restype = ctypes.c_double
    buf = ctypes.create_string_buffer(112)
    assert L.zkd_from_double(buf, 768, ctypes.c_double(v)) == 0
    assert L.zkd_to_double(buf, 768) == v
    sign, flags, exp = struct.unpack_from("<iiq", buf.raw, 0)
    top = struct.unpack_from("<12Q", buf.raw, 16)[11]
    if v == 0.0:
        assert (sign, exp, top) == (0, 0, 0)
    else:
        # value = sign * mantissa * 2^(exp-768), mantissa in [1/2, 1) * 2^768  (MPFR convention)
        import math

        m, e = math.frexp(abs(v))
        assert sign == (1 if v > 0 else -1) and exp == e and top >> 63 == 1
        assert top == int(m * 2 ** 64) & 0xFFFFFFFFFFFFFFFF or top == int(m * 2 ** 64)


def test_argument_validation_needs_no_gpu(L):
    n = ctypes.c_size_t(0)
    assert L.zkd_diag_herm_bufsize(64, 1, 768, ctypes.byref(n)) == 0 and n.value > 0
    small = n.value
    assert L.zkd_diag_herm_bufsize(64, 4, 768, ctypes.byref(n)) == 0 and n.value > small
    assert L.zkd_diag_herm_bufsize(0, 1, 768, ctypes.byref(n)) < 0
    assert L.zkd_diag_herm_bufsize(8, 0, 768, ctypes.byref(n)) < 0
    assert L.zkd_diag_herm_bufsize(8, 1, 100, ctypes.byref(n)) == -2  # unsupported precision
    assert L.zkd_diag_herm_bufsize(8, 1, 768, None) < 0
    # NULL pointers are refused before anything touches CUDA
    assert L.zkd_diag_herm_ws(8, 1, 768, None, None, None, None, 0, None, None) < 0
    assert L.zkd_diag_herm(8, 1, 768, None, None, None, None) < 0
    assert L.zkd_diag_herm_host(8, 1, 768, None, None, None, None) < 0
    d = ctypes.c_double(0)
    assert L.zkd_set_option(b"no_such_option", 1.0) < 0
    assert L.zkd_get_option(b"tau_bits", ctypes.byref(d)) == 0 and d.value == 20
    assert L.zkd_set_option(b"tau_bits", 18.0) == 0
    assert L.zkd_get_option(b"tau_bits", ctypes.byref(d)) == 0 and d.value == 18
    assert L.zkd_set_option(b"tau_bits", 20.0) == 0


def test_missing_library_fails_loudly(tmp_path, monkeypatch):
    import paper_2402_11868_b200 as z

    monkeypatch.setattr(z, "_lib", None)
    monkeypatch.setattr(z, "SO_PATH", str(tmp_path / "libzkd.so"))
    with pytest.raises(ImportError):
        z.lib()


# ---- N > 1: replicas only, one scalar MAX all_reduce outside the timed region (world_size 2 over gloo) -------------
def _replica_worker(rank: int, world: int, port: int, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import torch.distributed as dist

    import bench

    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # rank r "measured" (r+1) seconds for 10 steps of a batch of 4
        value, tmax = bench.aggregate(world, 4, 10, float(rank + 1), device="cpu")
        # every rank draws a different seed stream of the same workload
        N, b, A = bench.make_workload("c1", rank)
        q.put((rank, value, tmax, N, b, bytes(A[:64].tobytes())))
    finally:
        dist.destroy_process_group()


def test_replicas_world_size_2_gloo():
    import socket

    import torch.multiprocessing as mp

    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_replica_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    out = sorted(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(60)
        assert p.exitcode == 0
    (r0, v0, t0, N0, b0, a0), (r1, v1, t1, N1, b1, a1) = out
    assert t0 == t1 == 2.0                      # MAX over ranks
    assert v0 == v1 == 2 * 4 * 10 / 2.0         # all ranks' matrices / max time
    assert (N0, b0) == (N1, b1) == (16, 1)
    assert a0 != a1                             # different seed streams per replica

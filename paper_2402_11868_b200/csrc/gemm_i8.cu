// gemm_i8.cu — S4b of SURVEY.md 8(a): the digit GEMM's contraction as limb-sliced int8 tcgen05 MMAs with exact int32
// accumulation (north_star (e): "the residual/update GEMM A*Y ... run as limb-sliced int8 tcgen05 MMAs with exact int32
// accumulation and carry propagation wherever that beats the IMAD path").
//
// The operands arrive as the compact balanced radix-2^28 digit planes the IMAD path uses (prep_kernel).  Here every
// entry is re-sliced into balanced radix-2^8 digits ("slices", s8 in [-128,127]); with P = sum_a P_a 2^(8a) and
// Q = sum_b Q_b 2^(8b) the product is  sum_d 2^(8d) S_d,  S_d = sum_{a+b=d} P_a Q_b  (a convolution of int8 GEMMs).
// One CTA owns a 128 x 128 output tile and D = 4 consecutive columns d: four int32 accumulators in TMEM (512 columns).
// For each 128-deep K block it walks a upward; the slices Q_b it needs form a window sliding downward, so every step
// brings in one P tile and one Q tile (TMA, 128B swizzle) and issues D x 4 tcgen05.mma.kind::i8 (128x128x32).
// |S_d| <= K * min(nsP,nsQ) * 2^14 < 2^31 is enforced by splitting K.  Columns below dcut (the IMAD path's truncation
// point) are not computed.  The epilogue stores raw S_d; combine_i8_kernel folds the radix-2^8 columns into FX digits
// (3M recombination, carries, cut, add/sub into the destination) exactly like combine_kernel does for radix 2^28.
#include <cuda.h>

#include <vector>

#include "fx.cuh"
#include "gemm_i8.h"
#include "timing.h"

namespace zkd {

namespace {

constexpr int I8_BM = 128, I8_BN = 128, I8_BK = 128;  // BK in int8 elements = bytes = one 128B swizzle row
constexpr int I8_D = 4;                               // accumulators (columns d) per CTA: 4 x 128 TMEM columns
// ring depths (tiles of 16 KB) are template parameters <RP, RQ>: a step keeps 1 P tile and up to 4 Q tiles live, so the
// producer runs RP - 1 / RQ - 4 steps ahead of the MMAs
constexpr int I8_TILE_BYTES = I8_BM * I8_BK;          // 16384
constexpr int I8_THREADS = 192;                       // warps 0-3 epilogue, 4 TMA producer, 5 MMA issuer
constexpr size_t i8_smem(int rp, int rq) { return (size_t)(rp + rq) * I8_TILE_BYTES + 1024 /*align*/ + 512 /*barriers*/; }

// ---- PTX wrappers --------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "WAIT_%=:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra DONE_%=;\n\t"
      "bra WAIT_%=;\n\t"
      "DONE_%=:\n\t}" ::"r"(smem_u32(bar)), "r"(parity)
      : "memory");
}
__device__ __forceinline__ void tma_load_3d(void* smem_dst, const CUtensorMap* map, uint64_t* bar, int c0, int c1, int c2) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];" ::"r"(
          smem_u32(smem_dst)),
      "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2)
      : "memory");
}
__device__ __forceinline__ void umma_commit(uint64_t* bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void umma_i8(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p;\n\t}" ::"r"(tmem_d),
      "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
      : "memory");
}
// K-major, 128B-swizzled operand tile (rows of 128 bytes, 8-row groups 1024 B apart); sm_100 descriptor version 1
__device__ __forceinline__ uint64_t umma_desc_sw128(uint32_t smem_addr) {
  uint64_t d = 0;
  d |= (uint64_t)((smem_addr & 0x3FFFF) >> 4);  // start address
  d |= (uint64_t)1 << 16;                       // leading byte offset (unused for swizzled K-major)
  d |= (uint64_t)(1024 >> 4) << 32;             // stride byte offset: 8 rows x 128 B
  d |= (uint64_t)1 << 46;                       // descriptor version (sm_100)
  d |= (uint64_t)2 << 61;                       // SWIZZLE_128B
  return d;
}
__device__ __forceinline__ void tmem_ld_32x32b_x16_nowait(uint32_t taddr, uint32_t (&v)[16]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
      : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]), "=r"(v[9]),
        "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
      : "r"(taddr));
}
// one lane of a converged warp; unlike "lane == 0" the compiler knows the branch holds exactly one thread, so tcgen05 / TMA
// instructions inside it are issued straight from uniform registers (no per-instruction election loop)
__device__ __forceinline__ bool elect_one() {
  uint32_t pred;
  asm volatile("{\n\t.reg .pred P;\n\telect.sync _|P, 0xffffffff;\n\tselp.b32 %0, 1, 0, P;\n\t}" : "=r"(pred));
  return pred != 0;
}
__device__ __forceinline__ void tmem_ld_32x32b_x32(uint32_t taddr, uint32_t (&v)[32]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
      "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
      : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]), "=r"(v[9]),
        "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]), "=r"(v[17]), "=r"(v[18]),
        "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]),
        "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
      : "r"(taddr));
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}

}  // namespace

namespace {

// ---- re-slicing: compact balanced radix-2^28 planes -> balanced radix-2^8 planes, K-major, K padded to 128 ----------
struct SliceArgs {
  const int32_t* src;  // [G][nw][R][C]
  int8_t* dst;         // [G][ns][rows][Kp]   (P: rows = R, k = c;  Q: rows = C, k = r)
  int R, C, G, nw, ns, rows, K, Kp, transpose;
  int* err_flag;
};

__global__ void __launch_bounds__(256) slice_i8_kernel(SliceArgs a) {
  const size_t per = (size_t)a.rows * a.Kp;
  const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= per * a.G) return;
  const int g = (int)(e / per);
  const size_t rk = e % per;
  const int row = (int)(rk / a.Kp), kk = (int)(rk % a.Kp);
  int8_t* __restrict__ dst = a.dst + (size_t)g * a.ns * per + rk;
  if (kk >= a.K) {
    for (int j = 0; j < a.ns; ++j) dst[(size_t)j * per] = 0;
    return;
  }
  const size_t RC = (size_t)a.R * a.C;
  const size_t sidx = a.transpose ? ((size_t)kk * a.C + row) : ((size_t)row * a.C + kk);
  const int32_t* __restrict__ src = a.src + (size_t)g * a.nw * RC + sidx;
  int64_t acc = 0;
  int pos = 0, j = 0;
  bool bad = false;
  for (int k = 0; k < a.nw; ++k) {
    const int32_t d = src[(size_t)k * RC];
    acc += (int64_t)d << (DB * k - pos);
    const int limit = (k == a.nw - 1) ? a.ns * 8 : DB * (k + 1);
    while (pos + 8 <= limit) {
      int64_t cy = (acc + 128) >> 8;
      int64_t byte = acc - (cy << 8);
      if (j == a.ns - 1) {
        byte = acc;
        cy = 0;
        if (acc < -128 || acc > 127) bad = true;
      }
      dst[(size_t)j * per] = (int8_t)byte;
      acc = cy;
      pos += 8;
      ++j;
    }
  }
  if (bad && a.err_flag) atomicOr(a.err_flag, 4);
}


// The same re-slicing, four consecutive k per thread and two digits (56 bits = seven slices) per step.  The balanced
// slices of a value x are the plain bytes of x + 0x80...80 with their top bits flipped, and what is left above them is the
// carry: one 64-bit add, one xor and one shift per seven slices instead of a carry step per slice; the slices of the
// thread's four elements are transposed with byte permutes and leave as one 32-bit store per slice plane.  Lanes of a warp
// cover 128 consecutive k of one row (TRANS = false: the source is read with 16-byte loads) or 8 rows x 16 k (TRANS = true:
// the source is k-major there, so 8 consecutive rows make one 32-byte sector).  Bit-identical to slice_i8_kernel.
template <bool TRANS>
__global__ void __launch_bounds__(256) slice4_i8_kernel(SliceArgs a) {
  const int KG = a.Kp >> 2;  // groups of four k per row (a multiple of 32)
  const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  int g, row, kg;
  if (!TRANS) {
    kg = (int)(t % KG);
    const size_t rest = t / KG;
    row = (int)(rest % a.rows);
    g = (int)(rest / a.rows);
  } else {
    const int lane = threadIdx.x & 31;
    const size_t wid = t >> 5;
    const int KT = KG >> 2, RT = (a.rows + 7) >> 3;
    kg = (int)(wid % KT) * 4 + (lane & 3);
    const size_t rest = wid / KT;
    row = (int)(rest % RT) * 8 + (lane >> 2);
    g = (int)(rest / RT);
  }
  if (g >= a.G || row >= a.rows) return;
  const int kk = kg << 2;
  const size_t per = (size_t)a.rows * a.Kp;
  uint32_t* __restrict__ dst = (uint32_t*)(a.dst + (size_t)g * a.ns * per + (size_t)row * a.Kp + kk);
  const size_t dstride = per >> 2;
  const size_t RC = (size_t)a.R * a.C;
  const int32_t* __restrict__ src = a.src + (size_t)g * a.nw * RC + (TRANS ? ((size_t)kk * a.C + row) : ((size_t)row * a.C + kk));
  const size_t estride = TRANS ? (size_t)a.C : 1;  // between the thread's four elements
  const int nvalid = a.K - kk;                      // elements kk + i with i < nvalid exist
  const bool vec = !TRANS && (a.C & 3) == 0 && nvalid >= 4 && (((uintptr_t)a.src & 15) == 0);
  auto load4 = [&](int k, int32_t (&d)[4]) {
    const int32_t* p = src + (size_t)k * RC;
    if (vec) {
      const int4 v = *(const int4*)p;
      d[0] = v.x; d[1] = v.y; d[2] = v.z; d[3] = v.w;
    } else {
#pragma unroll
      for (int i = 0; i < 4; ++i) d[i] = i < nvalid ? p[(size_t)i * estride] : 0;
    }
  };
  constexpr int64_t BIAS7 = 0x0080808080808080ll;
  int64_t cy[4] = {0, 0, 0, 0};
  int j = 0;
  const int npair = a.nw >> 1;
  for (int pr = 0; pr < npair; ++pr) {
    int32_t d0[4], d1[4];
    load4(2 * pr, d0);
    load4(2 * pr + 1, d1);
    uint32_t lo[4], hi[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const int64_t tt = cy[i] + (int64_t)d0[i] + ((int64_t)d1[i] << DB) + BIAS7;
      const uint64_t x = (uint64_t)tt ^ (uint64_t)BIAS7;
      cy[i] = tt >> 56;
      lo[i] = (uint32_t)x;
      hi[i] = (uint32_t)(x >> 32);
    }
    const uint32_t la = __byte_perm(lo[0], lo[1], 0x5140), lb = __byte_perm(lo[2], lo[3], 0x5140);
    const uint32_t lc = __byte_perm(lo[0], lo[1], 0x7362), ld = __byte_perm(lo[2], lo[3], 0x7362);
    const uint32_t ha = __byte_perm(hi[0], hi[1], 0x5140), hb = __byte_perm(hi[2], hi[3], 0x5140);
    const uint32_t hc = __byte_perm(hi[0], hi[1], 0x7362), hd = __byte_perm(hi[2], hi[3], 0x7362);
    uint32_t* o = dst + (size_t)j * dstride;
    o[0] = __byte_perm(la, lb, 0x5410);
    o[dstride] = __byte_perm(la, lb, 0x7632);
    o[2 * dstride] = __byte_perm(lc, ld, 0x5410);
    o[3 * dstride] = __byte_perm(lc, ld, 0x7632);
    o[4 * dstride] = __byte_perm(ha, hb, 0x5410);
    o[5 * dstride] = __byte_perm(ha, hb, 0x7632);
    o[6 * dstride] = __byte_perm(hc, hd, 0x5410);
    j += 7;
  }
  // what is left: the odd last digit (if any) on top of the carry; ns - j - 1 more balanced slices, then the top slice takes the rest
  if (a.nw & 1) {
    int32_t d[4];
    load4(a.nw - 1, d);
#pragma unroll
    for (int i = 0; i < 4; ++i) cy[i] += d[i];
  }
  bool bad = false;
  for (; j < a.ns; ++j) {
    uint32_t w = 0;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      int64_t byte;
      if (j < a.ns - 1) {
        const int64_t c = (cy[i] + 128) >> 8;
        byte = cy[i] - (c << 8);
        cy[i] = c;
      } else {
        byte = cy[i];
        if (byte < -128 || byte > 127) bad = true;
      }
      w |= ((uint32_t)byte & 255u) << (8 * i);
    }
    dst[(size_t)j * dstride] = w;
  }
  if (bad && a.err_flag) atomicOr(a.err_flag, 4);
}

}  // namespace

namespace {

// ---- the tcgen05 kernel ----------------------------------------------------------------------------------------------
struct I8Args {
  int32_t* out;  // [nsplit][G][ncol][M][N] int32, or (packed) [nsplit][G][ngroups][M][N] int64 = sum_dd S_(4 dg + dd) 2^(8 dd)
  int packed;
  int M, N, G, nsP, nsQ, dcut, ncol, ngroups, nkb, kb_per_split, nsplit;
  uint32_t p_tile_bytes, q_tile_bytes;  // bytes one TMA box delivers (rows may be < 128 for small matrices)
  int bdiag;  // Q (128 x 128, one K block) is block diagonal in 32 x 32 blocks: K chunk k only feeds output columns 32 k .. 32 k + 31
};

// the slice ranges of one column group [d0, d0 + D)
struct GroupRange {
  int d0, a_min, a_max, b_min, b_max, nA, nQ;
};
__device__ __forceinline__ GroupRange group_range(const I8Args& a, int dg) {
  GroupRange r;
  r.d0 = a.dcut + I8_D * dg;
  const int dhi = min(r.d0 + I8_D - 1, a.nsP + a.nsQ - 2);
  r.a_min = max(0, r.d0 - (a.nsQ - 1));
  r.a_max = min(a.nsP - 1, dhi);
  r.b_max = min(a.nsQ - 1, dhi - r.a_min);
  r.b_min = max(0, r.d0 - r.a_max);
  r.nA = r.a_max - r.a_min + 1;
  r.nQ = r.b_max - r.b_min + 1;
  return r;
}

// One CTA = one 128 x 128 output tile x D columns.  Work proceeds in macro-steps of S consecutive slices a of one K block:
// the producer loads the S P tiles and the (at most S, or S + D - 1 at the start of a K block) new Q tiles of the window under
// ONE transaction barrier, the issuing thread waits once, issues up to S x D x 4 MMAs back to back and commits ONCE; the
// producer learns from that commit which macro-steps are complete and reuses the slots of the tiles that died in them.  (The
// issuing thread's waits and commits are not hidden behind the MMAs - the tensor pipe's queue is short - so the count of
// barrier operations per MMA is what sets the kernel's speed: see profiles/r02_summary.md.)
constexpr int I8_RF = 8;  // transaction ("full") and completion ("done") barrier rings, indexed by macro-step

template <int I8_RP, int I8_RQ, int I8_S>
__global__ void __launch_bounds__(I8_THREADS, 1)
gemm_i8_kernel(const __grid_constant__ CUtensorMap mapP, const __grid_constant__ CUtensorMap mapQ, const I8Args a) {
  static_assert(I8_RQ >= I8_S + I8_D - 1 + I8_S && I8_RP >= 2 * I8_S && I8_RP < I8_RF, "ring depths");
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  uint8_t* p_tiles = smem;                                  // [RP][16 KB]
  uint8_t* q_tiles = smem + (size_t)I8_RP * I8_TILE_BYTES;  // [RQ][16 KB]
  uint64_t* bars = (uint64_t*)(smem + (size_t)(I8_RP + I8_RQ) * I8_TILE_BYTES);
  uint64_t* full = bars;            // [RF] all tiles of macro-step m have landed
  uint64_t* done = bars + I8_RF;    // [RF] all MMAs of macro-step m have completed
  uint64_t* tmem_full = bars + 2 * I8_RF;
  uint32_t* tmem_base_slot = (uint32_t*)(tmem_full + 1);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int j0 = blockIdx.x * I8_BN, i0 = blockIdx.y * I8_BM;
  int z = blockIdx.z;
  const int dg = z % a.ngroups;
  z /= a.ngroups;
  const int sp = z % a.nsplit;
  const int g = z / a.nsplit;
  const GroupRange gr = group_range(a, dg);
  const int kb0 = sp * a.kb_per_split, kb1 = min(a.nkb, kb0 + a.kb_per_split);
  const int nm = (gr.nA + I8_S - 1) / I8_S;  // macro-steps per K block

  if (threadIdx.x == 0) {
    for (int i = 0; i < I8_RF; ++i) { mbar_init(full + i, 1); mbar_init(done + i, 1); }
    mbar_init(tmem_full, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  if (warp == 5) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_base_slot)), "n"(512));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tmem_base = *tmem_base_slot;

  if (warp == 4) {
    // ===== TMA producer =====
    if (elect_one()) {
      int pdeath[I8_RP], qdeath[I8_RQ];  // macro-step in which the tile now in the slot is used last
      for (int i = 0; i < I8_RP; ++i) pdeath[i] = -1;
      for (int i = 0; i < I8_RQ; ++i) qdeath[i] = -1;
      int known_done = -1;  // macro-steps <= known_done are complete
      auto wait_done = [&](int upto) {
        while (known_done < upto) {
          ++known_done;
          mbar_wait(done + (known_done % I8_RF), (uint32_t)(known_done / I8_RF) & 1u);
        }
      };
      int M = 0;
      uint32_t pslot = 0, qslot = 0;
      for (int kb = kb0; kb < kb1; ++kb) {
        int q_next = gr.b_max;
        for (int m = 0; m < nm; ++m, ++M) {
          const int aa0 = gr.a_min + m * I8_S, aa1 = min(gr.a_max, aa0 + I8_S - 1);
          const int lowest = max(gr.b_min, gr.d0 - aa1);
          const int nq_new = max(0, q_next - lowest + 1), np_new = aa1 - aa0 + 1;
          uint64_t* fb = full + (M % I8_RF);
          mbar_expect_tx(fb, (uint32_t)nq_new * a.q_tile_bytes + (uint32_t)np_new * a.p_tile_bytes);
          while (q_next >= lowest) {
            wait_done(qdeath[qslot]);
            tma_load_3d(q_tiles + (size_t)qslot * I8_TILE_BYTES, &mapQ, fb, kb * I8_BK, j0, g * a.nsQ + q_next);
            // Q_b is used last by the slice a = d0 + D - 1 - b (the group's highest column), clipped to the K block's range
            qdeath[qslot] = M - m + (min(gr.a_max, gr.d0 + I8_D - 1 - q_next) - gr.a_min) / I8_S;
            qslot = qslot + 1 == I8_RQ ? 0 : qslot + 1;
            --q_next;
          }
          for (int aa = aa0; aa <= aa1; ++aa) {
            wait_done(pdeath[pslot]);
            tma_load_3d(p_tiles + (size_t)pslot * I8_TILE_BYTES, &mapP, fb, kb * I8_BK, i0, g * a.nsP + aa);
            pdeath[pslot] = M;
            pslot = pslot + 1 == I8_RP ? 0 : pslot + 1;
          }
        }
      }
    }
  } else if (warp == 5) {
    // ===== MMA issuer =====
    if (elect_one()) {
      // S32 accumulate, S8 x S8, both K-major, M = 128, N = 128
      constexpr uint32_t idesc = (2u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(I8_BN >> 3) << 17) | ((uint32_t)(I8_BM >> 4) << 24);
      const uint32_t p_base = smem_u32(p_tiles), q_base = smem_u32(q_tiles);
      uint32_t started = 0;
      uint32_t pslot = 0;
      int M = 0;
      for (int kb = kb0; kb < kb1; ++kb) {
        // ring slot of tile b_max of this K block (tiles enter the ring in the order b_max, b_max - 1, ...)
        const uint32_t qslot0 = (uint32_t)(((long long)(kb - kb0) * gr.nQ) % I8_RQ);
        for (int m = 0; m < nm; ++m, ++M) {
          const int aa0 = gr.a_min + m * I8_S, aa1 = min(gr.a_max, aa0 + I8_S - 1);
          mbar_wait(full + (M % I8_RF), (uint32_t)(M / I8_RF) & 1u);
          asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
          for (int aa = aa0; aa <= aa1; ++aa) {
            const uint32_t pa = p_base + pslot * I8_TILE_BYTES;
            // slot of Q_b, b = d0 + dd - aa: (qslot0 + b_max - b) mod RQ
            const uint32_t s0 = (qslot0 + (uint32_t)(gr.b_max - (gr.d0 - aa) + I8_RQ * 16)) % I8_RQ;  // dd = 0 (b may lie outside the range)
#pragma unroll
            for (int dd = 0; dd < I8_D; ++dd) {
              const int b = gr.d0 + dd - aa;
              if (b < gr.b_min || b > gr.b_max) continue;
              const uint32_t sq = s0 >= (uint32_t)dd ? s0 - dd : s0 + I8_RQ - dd;
              const uint32_t qa = q_base + sq * I8_TILE_BYTES;
              if (a.bdiag) {
                // block-diagonal Q (cluster-tile products X_t M_t of a cluster pass): the 32 K values of chunk k meet only the 32 rows
                // 32 k .. 32 k + 31 of the K-major Q tile (4096 bytes apart: whole 1024-byte swizzle atoms), so the MMA is 128 x 32 x 32
                // into its own 32 accumulator columns - a quarter of the multiply-adds of the full-width instruction
                constexpr uint32_t idesc32 = (2u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(32 >> 3) << 17) | ((uint32_t)(I8_BM >> 4) << 24);
#pragma unroll
                for (int k = 0; k < I8_BK / 32; ++k) {
                  umma_i8(tmem_base + dd * I8_BN + 32 * k, umma_desc_sw128(pa + k * 32), umma_desc_sw128(qa + k * 4096 + k * 32), idesc32,
                          (started >> dd) & 1);
                }
              } else {
#pragma unroll
                for (int k = 0; k < I8_BK / 32; ++k) {
                  umma_i8(tmem_base + dd * I8_BN, umma_desc_sw128(pa + k * 32), umma_desc_sw128(qa + k * 32), idesc,
                          ((started >> dd) & 1) | (k > 0));
                }
              }
              started |= 1u << dd;
            }
            pslot = pslot + 1 == I8_RP ? 0 : pslot + 1;
          }
          umma_commit(done + (M % I8_RF));
        }
      }
      umma_commit(tmem_full);
    }
  } else {
    // ===== epilogue: warps 0-3, TMEM lanes 32*warp .. +31 = output rows =====
    mbar_wait(tmem_full, 0);
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const int i = i0 + warp * 32 + lane;
    const size_t mn = (size_t)a.M * a.N;
    if (a.packed) {
      // the group's columns leave as ONE 64-bit word per entry, sum_dd S_(d0 + dd) 2^(8 dd) (|S| < 2^31: below 2^56): half the
      // bytes of four int32 columns and a quarter of the words combine_i8_packed_kernel has to walk
      const int ncv = min(I8_D, a.ncol - I8_D * dg);  // columns of this group that exist (their accumulators were written)
      int64_t* o = (int64_t*)a.out + ((size_t)(sp * a.G + g) * a.ngroups + dg) * mn + (size_t)i * a.N + j0;
#pragma unroll 1
      for (int cc = 0; cc < I8_BN; cc += 16) {
        uint32_t v[I8_D][16];
#pragma unroll
        for (int dd = 0; dd < I8_D; ++dd) {
          if (dd < ncv) {
            tmem_ld_32x32b_x16_nowait(tmem_base + ((uint32_t)(warp * 32) << 16) + dd * I8_BN + cc, v[dd]);
          } else {
#pragma unroll
            for (int t = 0; t < 16; ++t) v[dd][t] = 0;
          }
        }
        asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
        int64_t r[16];
#pragma unroll
        for (int t = 0; t < 16; ++t)
          r[t] = (int64_t)(int32_t)v[0][t] + ((int64_t)(int32_t)v[1][t] << 8) + ((int64_t)(int32_t)v[2][t] << 16) +
                 ((int64_t)(int32_t)v[3][t] << 24);
        if (i < a.M) {
          if (j0 + cc + 16 <= a.N && (a.N & 1) == 0) {
#pragma unroll
            for (int t = 0; t < 16; t += 2) *(longlong2*)(o + cc + t) = make_longlong2(r[t], r[t + 1]);
          } else {
#pragma unroll
            for (int t = 0; t < 16; ++t)
              if (j0 + cc + t < a.N) o[cc + t] = r[t];
          }
        }
      }
    } else
    for (int dd = 0; dd < I8_D; ++dd) {
      const int c = I8_D * dg + dd;  // column index relative to dcut
      if (c >= a.ncol) break;
      // every kept column d <= nsP + nsQ - 2 receives at least one slice pair, so its accumulator has been written
      int32_t* o = a.out + ((size_t)(sp * a.G + g) * a.ncol + c) * mn + (size_t)i * a.N + j0;
#pragma unroll 1
      for (int cc = 0; cc < I8_BN; cc += 32) {
        uint32_t v[32];
        tmem_ld_32x32b_x32(tmem_base + ((uint32_t)(warp * 32) << 16) + dd * I8_BN + cc, v);
        if (i < a.M) {
          if (j0 + cc + 32 <= a.N && (a.N & 3) == 0) {
#pragma unroll
            for (int t = 0; t < 32; t += 4) *(int4*)(o + cc + t) = make_int4((int)v[t], (int)v[t + 1], (int)v[t + 2], (int)v[t + 3]);
          } else {
#pragma unroll
            for (int t = 0; t < 32; ++t)
              if (j0 + cc + t < a.N) o[cc + t] = (int32_t)v[t];
          }
        }
      }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  }
  __syncthreads();
  if (warp == 5) {
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(512));
  }
}

}  // namespace

namespace {

// ---- measured issue peak of the MMA shape the kernel uses (roofline denominator next to the bf16-derived one) ----------
// One CTA per SM, operands resident in shared memory (no TMA), one elected thread issuing 128 x 128 x 32 kind::i8 MMAs back
// to back into four accumulators exactly as gemm_i8_kernel does, one commit at the end.
__global__ void __launch_bounds__(128, 1) i8_peak_kernel(int niter) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  uint64_t* bar = (uint64_t*)(smem + 5 * I8_TILE_BYTES);
  uint32_t* slot = (uint32_t*)(bar + 1);
  for (int i = threadIdx.x; i < 5 * I8_TILE_BYTES / 4; i += blockDim.x) ((uint32_t*)smem)[i] = ((uint32_t)i * 2654435761u) ^ ((uint32_t)i >> 3);
  if (threadIdx.x == 0) {
    mbar_init(bar, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  const int warp = threadIdx.x >> 5;
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(slot)), "n"(512));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tm = *slot;
  if (warp == 0) {
    if (elect_one()) {
      constexpr uint32_t idesc = (2u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(I8_BN >> 3) << 17) | ((uint32_t)(I8_BM >> 4) << 24);
      const uint32_t pa = smem_u32(smem), qa = pa + I8_TILE_BYTES;
      for (int it = 0; it < niter; ++it) {
#pragma unroll
        for (int dd = 0; dd < I8_D; ++dd) {
#pragma unroll
          for (int k = 0; k < I8_BK / 32; ++k)
            umma_i8(tm + dd * I8_BN, umma_desc_sw128(pa + k * 32), umma_desc_sw128(qa + dd * I8_TILE_BYTES + k * 32), idesc, 1);
        }
      }
      umma_commit(bar);
      mbar_wait(bar, 0);
    }
    __syncwarp();
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == 0) {
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tm), "n"(512));
  }
}

}  // namespace

int measure_i8_mma_peak(double millis, double* ops_per_sec, cudaStream_t s) {
  int dev = 0, sms = 0;
  ZKD_CUDA_TRY(cudaGetDevice(&dev));
  ZKD_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  const size_t smem = 5 * (size_t)I8_TILE_BYTES + 1024 + 64;
  ZKD_CUDA_TRY(cudaFuncSetAttribute(i8_peak_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  cudaEvent_t e0, e1;
  ZKD_CUDA_TRY(cudaEventCreate(&e0));
  ZKD_CUDA_TRY(cudaEventCreate(&e1));
  int iters = 2000;
  double best = 0;
  const int reps = millis > 20 ? 5 : 3;
  int rc = ZKD_OK;
  i8_peak_kernel<<<sms, 128, smem, s>>>(100);  // warm-up
  for (int r = 0; r < reps + 1; ++r) {
    cudaEventRecord(e0, s);
    i8_peak_kernel<<<sms, 128, smem, s>>>(iters);
    cudaEventRecord(e1, s);
    if (cudaEventSynchronize(e1) != cudaSuccess) {
      (void)cudaGetLastError();
      rc = ZKD_ERR_CUDA;
      break;
    }
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    const double ops = 2.0 * I8_BM * I8_BN * 32.0 * (I8_BK / 32) * I8_D * (double)iters * sms;
    if (r > 0 && ops / (ms * 1e-3) > best) best = ops / (ms * 1e-3);
    if (r == 0 && ms > 0) {
      double scale = (millis / reps) / ms;
      if (scale > 50) scale = 50;
      if (scale < 0.05) scale = 0.05;
      iters = (int)(iters * scale) + 1;
    }
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  if (rc == ZKD_OK) *ops_per_sec = best;
  return rc;
}

namespace {

// ---- combine: radix-2^8 column sums -> FX digits ------------------------------------------------------------------------
struct CombineI8Args {
  const int32_t* raw;  // [nsplit][3*batch][ncol][M*N]
  int32_t* dst;        // complex FX, batch*M*N
  size_t mn;
  int N, ld;           // destination view (see combine_kernel)
  const int* off;
  size_t plane_count;
  int batch, ncol, nsplit;
  int base_bit;  // FX bit position of column 0's LSB (may be negative)
  int cut_bit;   // clear result bits below this FX bit (<= 0: none)
  int mode;      // 0 assign, 1 add, 2 sub
  int* msb_out;
};

// one thread per (element, part); part 0 = Re = k1 - k3, part 1 = Im = k1 + k2
__global__ void __launch_bounds__(256) combine_i8_kernel(CombineI8Args a) {
  const size_t tot = a.mn * a.batch;
  const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int part = blockIdx.y;
  if (e >= tot) return;
  const int b = (int)(e / a.mn);
  const size_t ij = e % a.mn;
  const size_t gstride = (size_t)a.ncol * a.mn;
  const size_t sstride = (size_t)3 * a.batch * gstride;
  const int32_t* __restrict__ r1 = a.raw + (size_t)(b * 3 + 0) * gstride + ij;
  const int32_t* __restrict__ r2 = a.raw + (size_t)(b * 3 + (part == 0 ? 2 : 1)) * gstride + ij;
  const int sgn2 = part == 0 ? -1 : 1;
  const size_t tot_d = a.plane_count;
  int32_t* dst = a.dst + (part ? (size_t)ND * tot_d : 0) + (a.off ? (size_t)a.off[b] : (size_t)b * a.mn) +
                 (size_t)(ij / a.N) * a.ld + (ij % a.N);

  auto col = [&](int c) -> int64_t {
    int64_t s1 = 0, s2 = 0;
    for (int s = 0; s < a.nsplit; ++s) {
      s1 += r1[(size_t)s * sstride + (size_t)c * a.mn];
      s2 += r2[(size_t)s * sstride + (size_t)c * a.mn];
    }
    return s1 + sgn2 * s2;
  };
  // FX digit k covers bits [28k, 28k+28); walk k upward from the digit holding column 0, feeding each digit the
  // columns whose LSB falls inside it
  const int kstart = a.base_bit >= 0 ? a.base_bit / DB : -((-a.base_bit + DB - 1) / DB);
  const int cutq = a.cut_bit > 0 ? a.cut_bit / DB : 0, cutr = a.cut_bit > 0 ? a.cut_bit % DB : 0;
  int64_t acc = 0, cy2 = 0;
  int c = 0;
  int msb_pos = 0, msb_neg = 0;
  for (int k = kstart; k <= ND - 1; ++k) {
    const int lo = k * DB;
    if (k < ND - 1) {
      while (c < a.ncol && a.base_bit + 8 * c < lo + DB) {
        acc += col(c) << (a.base_bit + 8 * c - lo);
        ++c;
      }
    } else {
      // the signed top digit takes everything that is left (sign extension unless the result overflows FX, which the
      // callers' magnitude bounds exclude)
      while (c < a.ncol) {
        const int sh = a.base_bit + 8 * c - lo;
        if (sh < 40) acc += col(c) << sh;
        ++c;
      }
    }
    int32_t digit;
    if (k < ND - 1) {
      digit = (int32_t)(acc & DMASK);
      acc >>= DB;
    } else {
      digit = (int32_t)acc;
    }
    if (k < 0) continue;
    if (k < cutq) digit = 0;
    else if (k == cutq && cutr) digit &= ~((1 << cutr) - 1);
    int32_t* dp = dst + (size_t)k * tot_d;
    int32_t outd = digit;
    if (a.mode != 0) {
      const int64_t t = (int64_t)*dp + (a.mode == 1 ? (int64_t)digit : -(int64_t)digit) + cy2;
      if (k < ND - 1) {
        cy2 = t >> DB;
        outd = (int32_t)(t & DMASK);
      } else {
        outd = (int32_t)t;
      }
    }
    *dp = outd;
    if (k < ND - 1) {
      if (outd != 0) msb_pos = k * DB + (32 - __clz(outd));
      if (outd != DMASK) msb_neg = k * DB + (32 - __clz((~outd) & DMASK));
    } else {
      if (outd > 0) msb_pos = k * DB + (32 - __clz(outd));
      if (outd < -1) msb_neg = k * DB + (32 - __clz(~outd));
      if (a.msb_out) atomicMax(a.msb_out, outd < 0 ? msb_neg : msb_pos);
    }
  }
  if (a.mode == 0)
    for (int kk = 0; kk < kstart && kk < ND; ++kk) dst[(size_t)kk * tot_d] = 0;
}

// The same fold for the packed output of gemm_i8_kernel (one int64 per entry and group of four columns).  The groups are
// first normalised into a stream of 32-bit words of the two's complement value V = sum_g G_g 2^(32 g) (one 64-bit add and one
// shift per group: w = G_g + carry, word = low 32 bits, carry = w >> 32; beyond the last group the words are the sign); FX digit
// k is then the bit field [28 k - base_bit, +28) of that stream (one funnel shift), the signed top digit the 32 bits from its
// position.  No per-column 64-bit shifts and a quarter of the loads of combine_i8_kernel; bit-identical to it.
__global__ void __launch_bounds__(256) combine_i8_packed_kernel(CombineI8Args a) {
  const size_t tot = a.mn * a.batch;
  const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int part = blockIdx.y;
  if (e >= tot) return;
  const int b = (int)(e / a.mn);
  const size_t ij = e % a.mn;
  const int ng = a.ncol;  // here: number of groups
  const size_t gstride = (size_t)ng * a.mn;
  const size_t sstride = (size_t)3 * a.batch * gstride;
  const int64_t* __restrict__ r1 = (const int64_t*)a.raw + (size_t)(b * 3 + 0) * gstride + ij;
  const int64_t* __restrict__ r2 = (const int64_t*)a.raw + (size_t)(b * 3 + (part == 0 ? 2 : 1)) * gstride + ij;
  const bool neg2 = part == 0;
  const size_t tot_d = a.plane_count;
  int32_t* dst = a.dst + (part ? (size_t)ND * tot_d : 0) + (a.off ? (size_t)a.off[b] : (size_t)b * a.mn) +
                 (size_t)(ij / a.N) * a.ld + (ij % a.N);

  // word stream: index -1 is a zero word (bits below base_bit), 0 .. ng - 1 the normalised groups, then the sign
  int gi = 0;
  int64_t carry = 0;
  auto next_word = [&]() -> uint32_t {
    int64_t w = carry;
    if (gi < ng) {
      for (int s = 0; s < a.nsplit; ++s) {
        const int64_t x1 = r1[(size_t)s * sstride + (size_t)gi * a.mn], x2 = r2[(size_t)s * sstride + (size_t)gi * a.mn];
        w += neg2 ? x1 - x2 : x1 + x2;
      }
      ++gi;
    }
    carry = w >> 32;
    return (uint32_t)w;
  };
  const int kstart = a.base_bit >= 0 ? a.base_bit / DB : -((-a.base_bit + DB - 1) / DB);
  const int k0 = kstart > 0 ? kstart : 0;
  const int cutq = a.cut_bit > 0 ? a.cut_bit / DB : 0, cutr = a.cut_bit > 0 ? a.cut_bit % DB : 0;
  // bit offset of digit k0 in the stream that starts with the zero word: >= 4
  long p = (long)DB * k0 - a.base_bit + 32;
  uint32_t wa = 0, wb = next_word();  // stream words q, q + 1 with q = 0
  long q = 0;
  int64_t cy2 = 0;
  int msb_pos = 0, msb_neg = 0;
  if (a.mode == 0)
    for (int kk = 0; kk < k0 && kk < ND; ++kk) dst[(size_t)kk * tot_d] = 0;
  for (int k = k0; k <= ND - 1; ++k, p += DB) {
    while (q < (p >> 5)) {
      wa = wb;
      wb = next_word();
      ++q;
    }
    const uint32_t f = __funnelshift_r(wa, wb, (uint32_t)(p & 31));
    int32_t digit = k < ND - 1 ? (int32_t)(f & (uint32_t)DMASK) : (int32_t)f;
    if (k < cutq) digit = 0;
    else if (k == cutq && cutr) digit &= ~((1 << cutr) - 1);
    int32_t* dp = dst + (size_t)k * tot_d;
    int32_t outd = digit;
    if (a.mode != 0) {
      const int64_t t = (int64_t)*dp + (a.mode == 1 ? (int64_t)digit : -(int64_t)digit) + cy2;
      if (k < ND - 1) {
        cy2 = t >> DB;
        outd = (int32_t)(t & DMASK);
      } else {
        outd = (int32_t)t;
      }
    }
    *dp = outd;
    if (k < ND - 1) {
      if (outd != 0) msb_pos = k * DB + (32 - __clz(outd));
      if (outd != DMASK) msb_neg = k * DB + (32 - __clz((~outd) & DMASK));
    } else {
      if (outd > 0) msb_pos = k * DB + (32 - __clz(outd));
      if (outd < -1) msb_neg = k * DB + (32 - __clz(~outd));
      if (a.msb_out) atomicMax(a.msb_out, outd < 0 ? msb_neg : msb_pos);
    }
  }
}

}  // namespace

// ---- host side -----------------------------------------------------------------------------------------------------

namespace {

using EncodeTiledFn = CUresult (*)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                   const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                   CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_tiled_fn() {
  static EncodeTiledFn fn = nullptr;
  static bool tried = false;
  if (!tried) {
    tried = true;
    void* p = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
        qres == cudaDriverEntryPointSuccess)
      fn = (EncodeTiledFn)p;
    else
      (void)cudaGetLastError();
  }
  return fn;
}

// int8 planes [planes][rows][Kp] -> 3D map (k, row, plane), box 128 x min(128, rows) x 1, 128B swizzle
int make_map(CUtensorMap* map, const int8_t* base, int Kp, int rows, int planes, int box_rows) {
  EncodeTiledFn fn = encode_tiled_fn();
  if (!fn) return ZKD_ERR_CUDA;
  const cuuint64_t dims[3] = {(cuuint64_t)Kp, (cuuint64_t)rows, (cuuint64_t)planes};
  const cuuint64_t strides[2] = {(cuuint64_t)Kp, (cuuint64_t)Kp * rows};
  const cuuint32_t box[3] = {(cuuint32_t)I8_BK, (cuuint32_t)box_rows, 1};
  const cuuint32_t estr[3] = {1, 1, 1};
  const CUresult r = fn(map, CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, (void*)base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                        CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? ZKD_OK : ZKD_ERR_CUDA;
}

inline size_t align_up(size_t x, size_t a = 1024) { return (x + a - 1) / a * a; }
inline int slices_for(int nw) { return (DB * nw + 8) / 8; }
constexpr int kMaxSlices = (DB * ND + 8) / 8;  // 106
constexpr int kMaxCols = 128;                  // kept columns: <= nsP + nsQ - 1 - dcut <= 106 + 8 + ... (checked at run time)

int pick_nsplit(int K, int nsmin) {
  // |S_d| <= Ksplit * nsmin * 2^14 must stay below 2^31
  const int nkb = (K + I8_BK - 1) / I8_BK;
  int kb_per = nkb;
  while (kb_per > 1 && (long)kb_per * I8_BK * nsmin >= 131072) --kb_per;
  return (nkb + kb_per - 1) / kb_per;
}

}  // namespace

namespace {
thread_local double t_useful = 1.0;
}
double gemm_useful_fraction() { return t_useful; }
GemmUsefulScope::GemmUsefulScope(double f) : old_(t_useful) { t_useful = f; }
GemmUsefulScope::~GemmUsefulScope() { t_useful = old_; }

void kernel_timing_enable_i8(bool on) { (void)on; }
int kernel_timing_read_i8(double* ms, uint64_t* launches, uint64_t* macs) { return kt_read(KC_GEMM_I8, ms, launches, macs, nullptr); }

bool gemm_i8_eligible(int path, int M, int N, int K, int batch) {
  (void)batch;
  if (path == 1) return false;                              // IMAD only
  if (path == 2) return M >= 8 && N >= 8 && K >= 1;         // forced (tests)
  return M >= 128 && N >= 128 && K >= 128;                  // auto: where one matrix fills 128 x 128 tiles
}

size_t gemm_i8_workspace_bytes(int M, int N, int K, int batch) {
  const size_t Kp = (size_t)(K + I8_BK - 1) / I8_BK * I8_BK;
  const size_t G = 3 * (size_t)batch;
  const size_t p8 = align_up(G * kMaxSlices * (size_t)M * Kp);
  const size_t q8 = align_up(G * kMaxSlices * (size_t)N * Kp);
  const int nsplit = pick_nsplit(K, kMaxSlices);
  const size_t raw = align_up(sizeof(int32_t) * (size_t)nsplit * G * kMaxCols * (size_t)M * N);
  return p8 + q8 + raw;
}

int gemm_i8_finish(int M, int N, int K, int batch, const int32_t* Pc, const int32_t* Qc, int np, int nq, int lsbP, int lsbQ,
                   int32_t* dst_fx, int mode, int cut_bit, void* ws, size_t ws_bytes, int* err_flag, int* msb_out,
                   cudaStream_t stream, const GemmDstView* dv, bool q_bdiag32) {
  if (ws_bytes < gemm_i8_workspace_bytes(M, N, K, batch)) return ZKD_ERR_WORKSPACE;
  const int Kp = (K + I8_BK - 1) / I8_BK * I8_BK;
  const int G = 3 * batch;
  const int nsP = slices_for(np), nsQ = slices_for(nq);
  const int low28 = nq >= 2 ? nq - 2 : 0;  // the IMAD instances' truncation rule (gemm_digits.cuh)
  const int dcut = DB * low28 / 8;
  const int ncol = nsP + nsQ - 1 - dcut;
  if (ncol < 1 || ncol > kMaxCols) return ZKD_ERR_INTERNAL;
  char* w = (char*)ws;
  int8_t* P8 = (int8_t*)w;
  w += align_up((size_t)G * kMaxSlices * M * Kp);
  int8_t* Q8 = (int8_t*)w;
  w += align_up((size_t)G * kMaxSlices * N * Kp);
  int32_t* raw = (int32_t*)w;

  {
    SliceArgs sa{};
    sa.src = Pc; sa.dst = P8; sa.R = M; sa.C = K; sa.G = G; sa.nw = np; sa.ns = nsP; sa.rows = M; sa.K = K; sa.Kp = Kp;
    sa.transpose = 0; sa.err_flag = err_flag;
    size_t tot = (size_t)G * M * Kp;
    {
      KtScope kt(KC_SLICE_I8, stream, (uint64_t)G * M * K * 4ull * np + (uint64_t)tot * nsP);
      if (options().i8_slice == 1) slice_i8_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, stream>>>(sa);
      else slice4_i8_kernel<false><<<(unsigned)((tot / 4 + 255) / 256), 256, 0, stream>>>(sa);
    }
    count_launch();
    sa.src = Qc; sa.dst = Q8; sa.R = K; sa.C = N; sa.nw = nq; sa.ns = nsQ; sa.rows = N; sa.transpose = 1;
    tot = (size_t)G * N * Kp;
    {
      KtScope kt(KC_SLICE_I8, stream, (uint64_t)G * N * K * 4ull * nq + (uint64_t)tot * nsQ);
      const size_t thr = (size_t)G * ((N + 7) / 8) * (Kp / 16) * 32;  // warps of 8 rows x 16 k
      if (options().i8_slice == 1) slice_i8_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, stream>>>(sa);
      else slice4_i8_kernel<true><<<(unsigned)((thr + 255) / 256), 256, 0, stream>>>(sa);
    }
    count_launch();
  }
  CUtensorMap mapP, mapQ;
  const int boxP = M < I8_BM ? M : I8_BM, boxQ = N < I8_BN ? N : I8_BN;
  ZKD_TRY(make_map(&mapP, P8, Kp, M, G * nsP, boxP));
  ZKD_TRY(make_map(&mapQ, Q8, Kp, N, G * nsQ, boxQ));

  I8Args ka{};
  const bool packed = options().i8_packed != 0;
  ka.packed = packed ? 1 : 0;
  ka.out = raw; ka.M = M; ka.N = N; ka.G = G; ka.nsP = nsP; ka.nsQ = nsQ; ka.dcut = dcut; ka.ncol = ncol;
  ka.ngroups = (ncol + I8_D - 1) / I8_D;
  ka.nkb = Kp / I8_BK;
  ka.nsplit = pick_nsplit(K, nsP < nsQ ? nsP : nsQ);
  ka.kb_per_split = (ka.nkb + ka.nsplit - 1) / ka.nsplit;
  ka.nsplit = (ka.nkb + ka.kb_per_split - 1) / ka.kb_per_split;
  ka.p_tile_bytes = (uint32_t)boxP * I8_BK;
  ka.q_tile_bytes = (uint32_t)boxQ * I8_BK;
  ka.bdiag = (q_bdiag32 && options().i8_bdiag && K == I8_BK && N == I8_BN) ? 1 : 0;
  // macro-step of 2 slices with rings <4, 9> by default; i8_step = 1: one slice per step, rings <5, 8>
  const bool step1 = options().i8_step == 1;
  auto kern = step1 ? gemm_i8_kernel<5, 8, 1> : gemm_i8_kernel<4, 9, 2>;
  const size_t smem = i8_smem(4, 9);
  ZKD_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));  // per device, cheap
  const dim3 grid((N + I8_BN - 1) / I8_BN, (M + I8_BM - 1) / I8_BM, (unsigned)(G * ka.nsplit * ka.ngroups));
  if (grid.z > 65535) return ZKD_ERR_INTERNAL;
  // int8 MACs actually issued: every (a, b) pair with a + b >= dcut, on full 128 x 128 x 128 blocks
  uint64_t pairs = 0;
  for (int x = 0; x < nsP; ++x)
    for (int y = 0; y < nsQ; ++y)
      if (x + y >= dcut) ++pairs;
  const uint64_t macs = pairs * (uint64_t)G * grid.x * grid.y * ka.nkb * I8_BM * I8_BN * I8_BK / (ka.bdiag ? 4 : 1);
  {
    // algorithmic: the same slice pairs on the matrices as they are (no padding of M, N, K to 128)
    KtScope kt(KC_GEMM_I8, stream, macs, (uint64_t)((double)(pairs * (uint64_t)G * M * N * K) * gemm_useful_fraction()));
    kern<<<grid, I8_THREADS, smem, stream>>>(mapP, mapQ, ka);
  }
  count_launch();
  count_i8_macs(macs);
  ZKD_TRY(launch_check());

  CombineI8Args ca{};
  ca.raw = raw; ca.dst = dst_fx; ca.mn = (size_t)M * N; ca.batch = batch; ca.ncol = ncol; ca.nsplit = ka.nsplit;
  ca.N = N; ca.ld = dv && dv->ld ? dv->ld : N; ca.off = dv ? dv->off : nullptr;
  ca.plane_count = dv && dv->plane_count ? dv->plane_count : (size_t)batch * M * N;
  ca.base_bit = lsbP + lsbQ - FRAC + 8 * dcut;
  ca.cut_bit = cut_bit; ca.mode = mode; ca.msb_out = msb_out;
  const size_t tot = (size_t)batch * M * N;
  if (packed) {
    ca.ncol = ka.ngroups;
    KtScope kt(KC_COMBINE_I8, stream, 4ull * tot * ((uint64_t)ka.nsplit * 3 * 2 * ka.ngroups + 2ull * ND * (mode == 0 ? 1 : 2)));
    combine_i8_packed_kernel<<<dim3((unsigned)((tot + 255) / 256), 2), 256, 0, stream>>>(ca);
  } else {
    KtScope kt(KC_COMBINE_I8, stream, 4ull * tot * ((uint64_t)ka.nsplit * 3 * ncol + 2ull * ND * (mode == 0 ? 1 : 2)));
    combine_i8_kernel<<<dim3((unsigned)((tot + 255) / 256), 2), 256, 0, stream>>>(ca);
  }
  count_launch();
  return launch_check();
}

}  // namespace zkd

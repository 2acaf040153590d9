// gemm_digits.cu — complex FX matrix product on the IMAD path: operand preparation (window extraction, 3M
// combinations, balanced digits), instance selection, and the combine epilogue (split-K sum, 3M recombination,
// carry propagation, placement into the FX destination).
//
// Complex product by 3 real products (3M):  with P = pr + i pi and Q = qr + i qi,
//     k1 = (pr + pi) qr,  k2 = pr (qi - qr),  k3 = pi (qr + qi);   Re = k1 - k3,  Im = k1 + k2.
// In fixed point the operand sums are exact, so 3M costs nothing in accuracy.
#include <algorithm>
#include <cstdio>
#include <vector>

#include "gemm_digits.cuh"
#include "gemm_i8.h"
#include "timing.h"
#include "zkd_internal.h"

namespace zkd {

#define ZKD_DECL_Q(n) \
  extern const GemmInstance kGemmInstQ##n[]; \
  extern const int kGemmInstQ##n##Count;
ZKD_DECL_Q(3) ZKD_DECL_Q(4) ZKD_DECL_Q(5) ZKD_DECL_Q(6) ZKD_DECL_Q(8) ZKD_DECL_Q(10) ZKD_DECL_Q(12) ZKD_DECL_Q(15)
ZKD_DECL_Q(18) ZKD_DECL_Q(22) ZKD_DECL_Q(30)

static const std::vector<GemmInstance>& instances() {
  static std::vector<GemmInstance> v;
  if (v.empty()) {
#define ZKD_ADD_Q(n) v.insert(v.end(), kGemmInstQ##n, kGemmInstQ##n + kGemmInstQ##n##Count);
    ZKD_ADD_Q(3) ZKD_ADD_Q(4) ZKD_ADD_Q(5) ZKD_ADD_Q(6) ZKD_ADD_Q(8) ZKD_ADD_Q(10) ZKD_ADD_Q(12) ZKD_ADD_Q(15)
    ZKD_ADD_Q(18) ZKD_ADD_Q(22) ZKD_ADD_Q(30)
  }
  return v;
}

static uint64_t inst_cost(const GemmInstance& in) {
  // digit products per (i,j,k): pairs (a,b) with a + b >= low
  uint64_t c = 0;
  for (int a = 0; a < in.np; ++a)
    for (int b = 0; b < in.nq; ++b)
      if (a + b >= in.low) ++c;
  return c;
}

// digit products per (i,j,k) the REQUEST needs: its own windows with the truncation rule applied to them (no instance padding)
static uint64_t request_cost(int nwP, int nwQ) {
  const int low = nwQ >= 2 ? nwQ - 2 : 0;
  uint64_t c = 0;
  for (int a = 0; a < nwP; ++a)
    for (int b = 0; b < nwQ; ++b)
      if (a + b >= low) ++c;
  return c;
}

// Cheapest instance with np >= nwP, nq >= nwQ and at least `ncols_needed` kept columns below the top.
static const GemmInstance* pick_instance(int nwP, int nwQ) {
  const GemmInstance* best = nullptr;
  uint64_t bc = ~0ull;
  for (const auto& in : instances()) {
    if (in.np < nwP || in.nq < nwQ) continue;
    // padding an operand at its low end shifts the needed columns up by the same amount, so the truncation rule
    // LOW = NQ - 2 of the instance keeps at least the columns the request needs when nq_inst - nwQ <= np pad ...
    uint64_t c = inst_cost(in);
    if (c < bc) { bc = c; best = &in; }
  }
  return best;
}

// ---- operand preparation ----------------------------------------------------------------------------------------

struct PrepArgs {
  const int32_t* src;  // complex FX, batch * rows * cols
  int32_t* dst;        // [3*batch][nw][R][C]
  size_t src_count;    // complex elements per plane of the source array
  int ld;              // row stride of the stored matrix
  const int* off;      // per batch element start (null: b * R * C)
  int R, C;            // destination dims (P: M x K, Q: K x N)
  int batch;
  int transpose;       // source stored C x R and conjugated
  int side;            // 0: P-type planes (re+im, re, im); 1: Q-type planes (re, im-re, re+im)
  int lsb_bit;         // FX bit position of digit 0 of the compact operand (may be negative)
  int nw;              // digits written
  int nw_src;          // digits taken from the source window (the rest, at the LOW end, are zero padding)
  int* err_flag;
};

__device__ __forceinline__ int32_t fx_digit_get(const int32_t* __restrict__ planes, size_t count, size_t idx, int q, int32_t top) {
  if (q < 0) return 0;
  if (q < kND - 1) return planes[(size_t)q * count + idx];
  if (q == kND - 1) return top & DMASK;
  if (q == kND) return (top >> DB) & DMASK;
  return top < 0 ? DMASK : 0;
}

struct PrepArgs2 { PrepArgs side[2]; };

// One launch prepares both operands (blockIdx.y = 0: P, 1: Q).  All digits of the element's window are fetched up front
// by an unrolled, predicated loop (independent loads in flight together); the window extraction, the 3M sums and the
// balanced-digit carry chain then run on registers.
constexpr int kPrepMaxDigits = kND + 2;  // window digits + the one above, at most

__global__ void __launch_bounds__(256) prep_kernel(PrepArgs2 both) {
  const PrepArgs& a = both.side[blockIdx.y];
  const size_t per = (size_t)a.R * a.C;
  const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= per * a.batch) return;
  const int b = (int)(e / per);
  const size_t rc = e % per;
  const int r = (int)(rc / a.C), c = (int)(rc % a.C);
  const size_t base = a.off ? (size_t)a.off[b] : (size_t)b * per;
  const size_t sidx = base + (a.transpose ? ((size_t)c * a.ld + r) : ((size_t)r * a.ld + c));
  const int32_t* __restrict__ re = a.src;
  const int32_t* __restrict__ im = a.src + (size_t)kND * a.src_count;
  const int32_t top_re = re[(size_t)(kND - 1) * a.src_count + sidx];
  const int32_t top_im = im[(size_t)(kND - 1) * a.src_count + sidx];
  const bool neg_re = top_re < 0, neg_im = top_im < 0;
  const int pad = a.nw - a.nw_src;  // zero digits at the low end
  const int lsb = a.lsb_bit + pad * DB;
  int q0 = lsb >= 0 ? lsb / DB : -((-lsb + DB - 1) / DB);  // floor(lsb / 28)
  const int sh = lsb - q0 * DB;                             // 0..27
  const int nsrc = a.nw_src;

  int32_t lr[kPrepMaxDigits], li[kPrepMaxDigits];
#pragma unroll
  for (int t = 0; t < kPrepMaxDigits; ++t) {
    const bool need = t <= nsrc;
    lr[t] = need ? fx_digit_get(re, a.src_count, sidx, q0 + t, top_re) : 0;
    li[t] = need ? fx_digit_get(im, a.src_count, sidx, q0 + t, top_im) : 0;
  }

  int64_t carry[3] = {0, 0, 0};
  bool bad = false;
  const size_t dplane = per;                      // elements per digit plane of one g
  int32_t* __restrict__ dst0 = a.dst + ((size_t)(b * 3) * a.nw) * dplane + rc;
  for (int d = 0; d < pad; ++d) {
    dst0[((size_t)0 * a.nw + d) * dplane] = 0;
    dst0[((size_t)1 * a.nw + d) * dplane] = 0;
    dst0[((size_t)2 * a.nw + d) * dplane] = 0;
  }
#pragma unroll
  for (int d = 0; d < kND; ++d) {
    if (d < nsrc) {
      int32_t wr = sh ? (((lr[d] >> sh) | (lr[d + 1] << (DB - sh))) & DMASK) : lr[d];
      int32_t wi = sh ? (((li[d] >> sh) | (li[d + 1] << (DB - sh))) & DMASK) : li[d];
      const bool last = d == nsrc - 1;
      if (last) {  // signed top digit of the window
        if (neg_re) wr -= (1 << DB);
        if (neg_im) wi -= (1 << DB);
      }
      if (a.transpose) wi = -wi;  // conjugate (window-level negate; the dropped low bits only move the truncation)
      int64_t v[3];
      if (a.side == 0) { v[0] = (int64_t)wr + wi; v[1] = wr; v[2] = wi; }
      else             { v[0] = wr; v[1] = (int64_t)wi - wr; v[2] = (int64_t)wr + wi; }
#pragma unroll
      for (int pl = 0; pl < 3; ++pl) {
        int64_t t = v[pl] + carry[pl];
        int64_t out;
        if (!last) {
          int64_t cy = (t + DHALF) >> DB;
          out = t - (cy << DB);
          carry[pl] = cy;
        } else {
          out = t;
          if (t < -(DHALF) || t > DHALF) bad = true;  // does not fit the window with the 3M headroom
        }
        dst0[((size_t)pl * a.nw + pad + d) * dplane] = (int32_t)out;
      }
    }
  }
  // bits above the window must be sign extension
  {
    const int tb = lsb + nsrc * DB;  // == top_bit
    const int qt = tb >= 0 ? tb / DB : -((-tb + DB - 1) / DB);
    const int s2 = tb - qt * DB;
    for (int q = qt; q <= kND + 1; ++q) {
      int32_t dr = fx_digit_get(re, a.src_count, sidx, q, top_re), di = fx_digit_get(im, a.src_count, sidx, q, top_im);
      int32_t fr = neg_re ? DMASK : 0, fi = neg_im ? DMASK : 0;
      int32_t mask = (q == qt) ? ((DMASK >> s2) << s2) : DMASK;
      if (((dr ^ fr) & mask) || ((di ^ fi) & mask)) bad = true;
    }
  }
  if (bad && a.err_flag) atomicOr(a.err_flag, 1);
}

// ---- combine ------------------------------------------------------------------------------------------------------

struct CombineArgs {
  const int32_t* raw;  // [split][3*batch][nc][M*N]
  int32_t* dst;        // complex FX, batch*M*N
  size_t mn;           // M*N
  int N, ld;           // destination view: element (i, j) of batch element b at off[b] + i * ld + j
  const int* off;      // null: b * mn
  size_t plane_count;  // complex elements per destination plane
  int batch, nc, nsplit;
  int base_bit;        // FX bit position of raw column 0's LSB (may be negative)
  int cut_bit;         // clear result bits below this FX bit (<= 0: none)
  int mode;            // GemmMode
  int* msb_out;
};

// one thread per (element, part); part 0 = Re = k1 - k3, part 1 = Im = k1 + k2.
// NS: compile-time bound of the split count (0: any), so that the loads of all splits of a column chunk are in flight together
template <int NS>
__global__ void __launch_bounds__(256) combine_kernel(CombineArgs a) {
  const size_t tot = a.mn * a.batch;
  const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int part = blockIdx.y;
  if (e >= tot) return;
  const int b = (int)(e / a.mn);
  const size_t ij = e % a.mn;
  const int G = 3 * a.batch;
  const size_t colstride = a.mn;
  const size_t gstride = (size_t)a.nc * a.mn;
  const size_t sstride = (size_t)G * gstride;
  const int32_t* r1 = a.raw + (size_t)(b * 3 + 0) * gstride + ij;
  const int32_t* r2 = a.raw + (size_t)(b * 3 + (part == 0 ? 2 : 1)) * gstride + ij;
  const int sgn2 = part == 0 ? -1 : 1;

  int q = a.base_bit >= 0 ? a.base_bit / DB : -((-a.base_bit + DB - 1) / DB);
  const int sh = a.base_bit - q * DB;  // 0..27
  const size_t tot_d = a.plane_count;
  int32_t* dst = a.dst + (part ? (size_t)kND * tot_d : 0) + (a.off ? (size_t)a.off[b] : (size_t)b * a.mn) +
                 (size_t)(ij / a.N) * a.ld + (ij % a.N);

  int64_t cy = 0;   // carry of the raw-column normalisation
  int64_t cy2 = 0;  // carry of the destination addition
  int msb_pos = 0, msb_neg = 0;  // candidates for the result's msb (if it ends up >= 0 / < 0)
  const int cutq = a.cut_bit > 0 ? a.cut_bit / DB : 0, cutr = a.cut_bit > 0 ? a.cut_bit % DB : 0;

  const int32_t* __restrict__ q1 = r1;
  const int32_t* __restrict__ q2 = r2;
  auto col = [&](int c) -> int64_t {
    int64_t s1 = 0, s2 = 0;
    for (int s = 0; s < a.nsplit; ++s) {
      s1 += q1[(size_t)s * sstride + (size_t)c * colstride];
      s2 += q2[(size_t)s * sstride + (size_t)c * colstride];
    }
    return (s1 + sgn2 * s2) << sh;
  };
  // columns are fetched eight at a time (independent loads in flight together); the carry chains run on registers
  constexpr int CH = 8;
  for (int c0 = 0; q + c0 <= kND - 1; c0 += CH) {
    int64_t s1[CH], s2[CH];
    int32_t old[CH];
#pragma unroll
    for (int u = 0; u < CH; ++u) { s1[u] = 0; s2[u] = 0; old[u] = 0; }
    if (a.mode != 0) {
#pragma unroll
      for (int u = 0; u < CH; ++u) {
        const int k = q + c0 + u;
        if (k >= 0 && k <= kND - 1) old[u] = dst[(size_t)k * tot_d];
      }
    }
    if (NS > 0) {
      constexpr int NSA = NS > 0 ? NS : 1;
      int32_t l1[NSA][CH], l2[NSA][CH];
#pragma unroll
      for (int s = 0; s < NS; ++s) {
#pragma unroll
        for (int u = 0; u < CH; ++u) {
          const bool in = s < a.nsplit && c0 + u < a.nc;
          l1[s][u] = in ? q1[(size_t)s * sstride + (size_t)(c0 + u) * colstride] : 0;
          l2[s][u] = in ? q2[(size_t)s * sstride + (size_t)(c0 + u) * colstride] : 0;
        }
      }
#pragma unroll
      for (int s = 0; s < NS; ++s) {
#pragma unroll
        for (int u = 0; u < CH; ++u) { s1[u] += l1[s][u]; s2[u] += l2[s][u]; }
      }
    } else {
      for (int s = 0; s < a.nsplit; ++s) {
#pragma unroll
        for (int u = 0; u < CH; ++u) {
          if (c0 + u < a.nc) {
            s1[u] += q1[(size_t)s * sstride + (size_t)(c0 + u) * colstride];
            s2[u] += q2[(size_t)s * sstride + (size_t)(c0 + u) * colstride];
          }
        }
      }
    }
#pragma unroll
    for (int u = 0; u < CH; ++u) {
      const int c = c0 + u;
      const int k = q + c;
      if (k <= kND - 1) {
        int64_t v = cy + ((s1[u] + sgn2 * s2[u]) << sh);
        int32_t digit;
        if (k < kND - 1) {
          cy = v >> DB;
          digit = (int32_t)(v & DMASK);
        } else {
          // everything that is left lands in the signed top digit (higher raw columns are sign extension unless the
          // result overflows FX, which the callers' magnitude bounds exclude)
          if (c + 1 < a.nc) v += col(c + 1) << DB;
          digit = (int32_t)v;
          cy = 0;
        }
        if (k >= 0) {
          if (k < cutq) digit = 0;
          else if (k == cutq && cutr) digit &= ~((1 << cutr) - 1);
          int32_t* dp = dst + (size_t)k * tot_d;
          int32_t outd = digit;
          if (a.mode != 0) {
            int64_t t = (int64_t)old[u] + (a.mode == 1 ? (int64_t)digit : -(int64_t)digit) + cy2;
            if (k < kND - 1) {
              cy2 = t >> DB;
              outd = (int32_t)(t & DMASK);
            } else {
              outd = (int32_t)t;
            }
          }
          *dp = outd;
          // msb of the value that ends up in the destination
          if (k < kND - 1) {
            if (outd != 0) msb_pos = k * DB + (32 - __clz(outd));
            if (outd != DMASK) msb_neg = k * DB + (32 - __clz((~outd) & DMASK));
          } else {
            if (outd > 0) msb_pos = k * DB + (32 - __clz(outd));
            if (outd < -1) msb_neg = k * DB + (32 - __clz(~outd));
            if (a.msb_out) atomicMax(a.msb_out, outd < 0 ? msb_neg : msb_pos);
          }
        }
      }
    }
  }
  // digits below the first written one (q > 0) are untouched in Add/Sub mode and must be zero in Assign mode
  if (a.mode == 0)
    for (int kk = 0; kk < q && kk < kND; ++kk) dst[(size_t)kk * tot_d] = 0;
}

// Warp-cooperative combine: one warp per (8 consecutive elements, part).  Lane k owns FX digit k of those elements (lanes
// 0..29), lane 30 the raw columns that lie below digit 0 (only their carry matters).  All raw columns of an element are
// fetched in one round trip (each lane reads 8 consecutive words = one sector per column and split), and the carries are
// resolved by parallel relaxation: every lane hands the overflow of its digit to the lane above until no lane overflows
// (3 - 5 rounds; a full ripple is 30).  The canonical digits of an integer are unique, so the result is bit-identical to
// the digit-serial kernel above.
constexpr int EPW = 8;

// lo: this lane's digit value (any int64), hi: what it owes the lane above (0 on entry is fine).  Two relaxation rounds bring
// every debt down to {-1, 0, +1} (|v| < 2^63 -> |hi| < 2^35 -> < 2^8 -> <= 1); the remaining unit carries and borrows may
// ripple through runs of 2^28-1 / 0 digits (a small negative result borrows through ALL its higher digits), so they are
// resolved by carry look-ahead on warp ballots instead of 30 more rounds: with G = lanes that emit a unit and P = lanes that
// would pass one on, the lanes that receive one are ((P + (G << 1)) ^ P ^ (G << 1)) | (G << 1).
__device__ __forceinline__ void relax_digits(int64_t (&lo)[EPW], int64_t (&hi)[EPW], int lane) {
  const bool low = lane < kND - 1;        // digits 0..28 are reduced mod 2^28
  const bool top = lane == kND - 1;       // digit 29 keeps the signed rest
  constexpr unsigned kLowMask = (1u << (kND - 1)) - 1;
#pragma unroll
  for (int round = 0; round < 2; ++round) {
#pragma unroll
    for (int u = 0; u < EPW; ++u) {
      int64_t inc = __shfl_up_sync(0xffffffffu, hi[u], 1);
      if (lane == 0 || lane > kND - 1) inc = 0;
      const int64_t t = lo[u] + inc;
      if (low) { hi[u] = t >> DB; lo[u] = t & DMASK; }
      else { hi[u] = 0; lo[u] = t; }
    }
  }
#pragma unroll
  for (int u = 0; u < EPW; ++u) {
    int64_t inc = __shfl_up_sync(0xffffffffu, hi[u], 1);  // -1, 0 or +1
    if (lane == 0 || lane > kND - 1) inc = 0;
    int64_t t = lo[u];
    // First all the +1 units, then all the -1 units: within one sign a lane that emits a unit (it wrapped to 0, resp. to
    // 2^28-1) can never also pass one on, so every lane receives at most one unit per phase - which is all a bit mask can say.
    bool gen = false;
    if (inc == 1) {
      t += 1;
      if (low && t == (int64_t)DMASK + 1) { t = 0; gen = true; }
    }
    unsigned G = __ballot_sync(0xffffffffu, gen) & kLowMask;
    unsigned P = __ballot_sync(0xffffffffu, low && t == DMASK) & kLowMask;
    unsigned C = (((P + (G << 1)) ^ P ^ (G << 1)) | (G << 1));
    if ((C >> lane) & 1) t = low ? ((t + 1) & DMASK) : (top ? t + 1 : t);
    gen = false;
    if (inc == -1) {
      t -= 1;
      if (low && t < 0) { t = DMASK; gen = true; }
    }
    G = __ballot_sync(0xffffffffu, gen) & kLowMask;
    P = __ballot_sync(0xffffffffu, low && t == 0) & kLowMask;
    C = (((P + (G << 1)) ^ P ^ (G << 1)) | (G << 1));
    if ((C >> lane) & 1) t = low ? ((t - 1) & DMASK) : (top ? t - 1 : t);
    lo[u] = t;
    hi[u] = 0;
  }
}

__global__ void __launch_bounds__(256) combine_warp_kernel(CombineArgs a) {
  const int lane = threadIdx.x & 31;
  const size_t w = ((size_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int part = blockIdx.y;
  const size_t gpb = (a.mn + EPW - 1) / EPW;  // groups per batch element
  if (w >= gpb * a.batch) return;             // the whole warp leaves together
  const int b = (int)(w / gpb);
  const size_t ij0 = (w % gpb) * EPW;
  const int nvalid = (int)(a.mn - ij0 < (size_t)EPW ? a.mn - ij0 : (size_t)EPW);
  const int G = 3 * a.batch;
  const size_t gstride = (size_t)a.nc * a.mn;
  const size_t sstride = (size_t)G * gstride;
  const int32_t* __restrict__ r1 = a.raw + (size_t)(b * 3 + 0) * gstride + ij0;
  const int32_t* __restrict__ r2 = a.raw + (size_t)(b * 3 + (part == 0 ? 2 : 1)) * gstride + ij0;
  const int sgn2 = part == 0 ? -1 : 1;
  const int q = a.base_bit >= 0 ? a.base_bit / DB : -((-a.base_bit + DB - 1) / DB);
  const int sh = a.base_bit - q * DB;  // 0..27
  const int k = lane;                  // FX digit of this lane (lanes 0..29)
  const size_t tot_d = a.plane_count;

  // destination addresses of the 8 elements (views: rows of ld words)
  size_t daddr[EPW];
#pragma unroll
  for (int u = 0; u < EPW; ++u) {
    const size_t ij = ij0 + (u < nvalid ? u : 0);
    daddr[u] = (part ? (size_t)kND * tot_d : 0) + (a.off ? (size_t)a.off[b] : (size_t)b * a.mn) + (ij / a.N) * a.ld + (ij % a.N);
  }
  int32_t old[EPW];
#pragma unroll
  for (int u = 0; u < EPW; ++u) old[u] = 0;
  if (a.mode != 0 && k < kND) {
#pragma unroll
    for (int u = 0; u < EPW; ++u)
      if (u < nvalid) old[u] = a.dst[daddr[u] + (size_t)k * tot_d];
  }

  // column sums of this lane's digit
  int64_t v[EPW];
#pragma unroll
  for (int u = 0; u < EPW; ++u) v[u] = 0;
  auto add_col = [&](int c, int shift) {
    for (int s = 0; s < a.nsplit; ++s) {
      int32_t l1[EPW], l2[EPW];
#pragma unroll
      for (int u = 0; u < EPW; ++u) {
        const bool in = u < nvalid;
        l1[u] = in ? r1[(size_t)s * sstride + (size_t)c * a.mn + u] : 0;
        l2[u] = in ? r2[(size_t)s * sstride + (size_t)c * a.mn + u] : 0;
      }
#pragma unroll
      for (int u = 0; u < EPW; ++u) v[u] += ((int64_t)l1[u] + sgn2 * (int64_t)l2[u]) << shift;
    }
  };
  if (k < kND) {
    const int c = k - q;
    if (c >= 0 && c < a.nc) add_col(c, sh);
    // everything that is left lands in the signed top digit (higher raw columns are sign extension unless the result
    // overflows FX, which the callers' magnitude bounds exclude)
    if (k == kND - 1 && c >= 0 && c + 1 < a.nc) add_col(c + 1, sh + DB);
  } else if (k == kND) {
    // raw columns below digit 0: serial carry chain (a handful of columns), delivered to digit 0
    const int nlow = -q < a.nc ? -q : a.nc;
    int64_t cy[EPW];
#pragma unroll
    for (int u = 0; u < EPW; ++u) cy[u] = 0;
    for (int c = 0; c < nlow; ++c) {
#pragma unroll
      for (int u = 0; u < EPW; ++u) v[u] = 0;
      add_col(c, sh);
#pragma unroll
      for (int u = 0; u < EPW; ++u) cy[u] = (cy[u] + v[u]) >> DB;
    }
    // digits between the last low column and digit 0 only pass the carry on: cy >> 28 per skipped digit
    for (int kk = q + nlow; kk < 0; ++kk) {
#pragma unroll
      for (int u = 0; u < EPW; ++u) cy[u] >>= DB;
    }
#pragma unroll
    for (int u = 0; u < EPW; ++u) v[u] = cy[u];
  }
  // carry of the low columns into digit 0
#pragma unroll
  for (int u = 0; u < EPW; ++u) {
    const int64_t cin = __shfl_sync(0xffffffffu, v[u], kND);
    if (k == 0) v[u] += cin;
    if (k >= kND) v[u] = 0;
  }
  int64_t lo[EPW], hi[EPW];
#pragma unroll
  for (int u = 0; u < EPW; ++u) {
    if (k < kND - 1) { lo[u] = v[u] & DMASK; hi[u] = v[u] >> DB; }
    else { lo[u] = v[u]; hi[u] = 0; }
  }
  relax_digits(lo, hi, lane);

  // cut, accumulate
  const int cutq = a.cut_bit > 0 ? a.cut_bit / DB : 0, cutr = a.cut_bit > 0 ? a.cut_bit % DB : 0;
  int32_t outd[EPW];
#pragma unroll
  for (int u = 0; u < EPW; ++u) {
    int32_t digit = (int32_t)lo[u];
    if (k < cutq) digit = 0;
    else if (k == cutq && cutr) digit &= ~((1 << cutr) - 1);
    outd[u] = digit;
  }
  if (a.mode != 0) {
#pragma unroll
    for (int u = 0; u < EPW; ++u) {
      const int64_t t = (int64_t)old[u] + (a.mode == 1 ? (int64_t)outd[u] : -(int64_t)outd[u]);
      if (k < kND - 1) { lo[u] = t & DMASK; hi[u] = t >> DB; }
      else { lo[u] = (k == kND - 1) ? t : 0; hi[u] = 0; }
    }
    relax_digits(lo, hi, lane);
#pragma unroll
    for (int u = 0; u < EPW; ++u) outd[u] = (int32_t)lo[u];
  }
  // store (accumulate modes leave the digits below the product's lowest one untouched: they cannot change)
  if (k < kND && (a.mode == 0 || k >= q)) {
#pragma unroll
    for (int u = 0; u < EPW; ++u)
      if (u < nvalid) a.dst[daddr[u] + (size_t)k * tot_d] = outd[u];
  }
  // msb of the stored values
  if (a.msb_out) {
    int best = 0;
#pragma unroll
    for (int u = 0; u < EPW; ++u) {
      const int32_t top = __shfl_sync(0xffffffffu, outd[u], kND - 1);
      int cand = 0;
      if (k < kND - 1) {
        if (top < 0) { if (outd[u] != DMASK) cand = k * DB + (32 - __clz((~outd[u]) & DMASK)); }
        else if (outd[u] != 0) cand = k * DB + (32 - __clz(outd[u]));
      } else if (k == kND - 1) {
        if (outd[u] > 0) cand = k * DB + (32 - __clz(outd[u]));
        if (outd[u] < -1) cand = k * DB + (32 - __clz(~outd[u]));
      }
      if (u < nvalid && cand > best) best = cand;
    }
    for (int o = 16; o > 0; o >>= 1) best = max(best, __shfl_xor_sync(0xffffffffu, best, o));
    if (lane == 0 && best) atomicMax(a.msb_out, best);
  }
}

// ---- host side ----------------------------------------------------------------------------------------------------

void kernel_timing_enable(bool on) { kt_enable(on); }
int kernel_timing_read(double* ms, uint64_t* launches, uint64_t* macs) { return kt_read(KC_GEMM_DIGITS, ms, launches, macs, nullptr); }

static size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }

// tile size for a shape: 8 when 16-wide tiles would be filled much worse (see gemm_digits.cuh)
static int pick_tile(int M, int N, int K) {
  if (options().gemm_tile == 8 || options().gemm_tile == 16) return options().gemm_tile;
  auto fill = [&](int t) {
    auto up = [&](int x) { return (double)((x + t - 1) / t * t); };
    return (double)M * N * K / (up(M) * up(N) * up(K));
  };
  return fill(8) > 1.25 * fill(16) ? 8 : 16;
}

static int pick_splits(int M, int N, int K, int batch, int tg = GT) {
  // Split K until the product has about min_split_ctas CTAs, but leave every split at least two 16-deep K tiles: a CTA
  // that does a single tile is all prologue and epilogue, and every split adds a raw plane for the epilogue to sum
  // (measured: N = 64, K = 64: 2 splits 2.27 ms per matrix, 4 splits 2.37, none 2.46; K = 1024 wants its splits).
  const long tiles = std::max(1L, (long)((M + tg - 1) / tg) * ((N + tg - 1) / tg) * 3 * batch / (tg == 8 ? 4 : 1));  // in units of 256 threads
  const int want = options().min_split_ctas;
  if (tiles >= want) return 1;
  int s = (int)((want + tiles - 1) / tiles);
  const int kmax = ((K + 15) / 16) / 2;  // at least 32 of K per split, whatever the tile
  if (s > kmax) s = kmax;
  if (s > 32) s = 32;
  return s < 1 ? 1 : s;
}

size_t gemm_workspace_bytes(int M, int N, int K, int batch) {
  const size_t pc = align_up(sizeof(int32_t) * 3 * (size_t)batch * kND * M * K);
  const size_t qc = align_up(sizeof(int32_t) * 3 * (size_t)batch * kND * K * N);
  const int sp = std::max(pick_splits(M, N, K, batch, 16), pick_splits(M, N, K, batch, 8));
  const size_t raw = align_up(sizeof(int32_t) * (size_t)sp * 3 * batch * (2 * kND + 3) * M * N);
  const size_t i8 = gemm_i8_eligible(options().gemm_path, M, N, K, batch) ? gemm_i8_workspace_bytes(M, N, K, batch) : 0;
  return pc + qc + (raw > i8 ? raw : i8);
}

uint64_t gemm_complex_macs(int M, int N, int K, int batch, int nwP, int nwQ, int* inst_np, int* inst_nq) {
  const GemmInstance* in = pick_instance(nwP, nwQ);
  if (!in) return 0;
  if (inst_np) *inst_np = in->np;
  if (inst_nq) *inst_nq = in->nq;
  return inst_cost(*in) * 3ull * (uint64_t)batch * M * N * K;
}

int gemm_complex(int M, int N, int K, int batch, const GemmSide& P, const GemmSide& Q, int32_t* dst_fx, GemmMode mode,
                 int out_cut_bit, int path, void* workspace, size_t workspace_bytes, int* err_flag, int* msb_out,
                 cudaStream_t stream, const GemmDstView* dv) {
  if (M < 1 || N < 1 || K < 1 || batch < 1 || P.nw < 1 || Q.nw < 1 || P.nw > kND || Q.nw > kND) return ZKD_ERR_INVALID_ARG;
  // the instance needs NQ <= NP roles only through its truncation rule; pad whichever side is short
  const GemmInstance* in = pick_instance(P.nw, Q.nw);
  if (!in) return ZKD_ERR_INTERNAL;
  if (workspace_bytes < gemm_workspace_bytes(M, N, K, batch)) return ZKD_ERR_WORKSPACE;
  char* w = (char*)workspace;
  int32_t* Pc = (int32_t*)w;
  w += align_up(sizeof(int32_t) * 3 * (size_t)batch * kND * M * K);
  int32_t* Qc = (int32_t*)w;
  w += align_up(sizeof(int32_t) * 3 * (size_t)batch * kND * K * N);
  int32_t* raw = (int32_t*)w;

  // the int8 tcgen05 engine takes the windows as they are; the IMAD instances need them padded at the LOW end up to
  // the instance's digit counts
  const bool use_i8 = gemm_i8_eligible(path, M, N, K, batch) &&
                      workspace_bytes >= align_up(sizeof(int32_t) * 3 * (size_t)batch * kND * M * K) +
                                             align_up(sizeof(int32_t) * 3 * (size_t)batch * kND * K * N) +
                                             gemm_i8_workspace_bytes(M, N, K, batch);
  const int npad = use_i8 ? P.nw : in->np, nqad = use_i8 ? Q.nw : in->nq;
  const int lsbP = P.top_bit - DB * npad, lsbQ = Q.top_bit - DB * nqad;
  {
    PrepArgs2 both{};
    PrepArgs& pa = both.side[0];
    pa.src = P.fx; pa.dst = Pc; pa.src_count = P.plane_count ? P.plane_count : (size_t)batch * M * K; pa.R = M; pa.C = K; pa.batch = batch;
    pa.ld = P.ld ? P.ld : (P.conj_transpose ? M : K); pa.off = P.off;
    pa.transpose = P.conj_transpose ? 1 : 0; pa.side = 0; pa.lsb_bit = lsbP; pa.nw = npad; pa.nw_src = P.nw; pa.err_flag = err_flag;
    PrepArgs& qa = both.side[1];
    qa.src = Q.fx; qa.dst = Qc; qa.src_count = Q.plane_count ? Q.plane_count : (size_t)batch * K * N; qa.R = K; qa.C = N; qa.batch = batch;
    qa.ld = Q.ld ? Q.ld : N; qa.off = Q.off;
    qa.transpose = 0; qa.side = 1; qa.lsb_bit = lsbQ; qa.nw = nqad; qa.nw_src = Q.nw; qa.err_flag = err_flag;
    const size_t tot = (size_t)batch * K * (size_t)(M > N ? M : N);
    {
      // bytes: the source windows read (re + im) and the three compact planes written, both operands
      const uint64_t bytes = 4ull * batch * ((uint64_t)M * K * (2 * (P.nw + 1) + 3 * npad) + (uint64_t)K * N * (2 * (Q.nw + 1) + 3 * nqad));
      KtScope kt(KC_PREP, stream, bytes);
      prep_kernel<<<dim3((unsigned)((tot + 255) / 256), 2), 256, 0, stream>>>(both);
    }
    count_launch();
  }
  if (use_i8)
    return gemm_i8_finish(M, N, K, batch, Pc, Qc, npad, nqad, lsbP, lsbQ, dst_fx, (int)mode, out_cut_bit, raw,
                          workspace_bytes - (size_t)((char*)raw - (char*)workspace), err_flag, msb_out, stream, dv, Q.bdiag32);
  const int tg = pick_tile(M, N, K);
  const int nsplit = pick_splits(M, N, K, batch, tg);
  int ksplit = (K + nsplit - 1) / nsplit;
  ksplit = (ksplit + tg - 1) / tg * tg;
  const int nsp = (K + ksplit - 1) / ksplit;
  GemmKArgs ka{};
  ka.P = Pc; ka.Q = Qc; ka.Out = raw;
  ka.p_dstride = (size_t)M * K; ka.p_gstride = (size_t)in->np * M * K;
  ka.q_dstride = (size_t)K * N; ka.q_gstride = (size_t)in->nq * K * N;
  ka.M = M; ka.N = N; ka.K = K; ka.G = 3 * batch; ka.ksplit = ksplit; ka.nsplit = nsp;
  dim3 grid((N + tg - 1) / tg, (M + tg - 1) / tg, (unsigned)(3 * batch * nsp));
  const uint64_t nmacs = inst_cost(*in) * 3ull * (uint64_t)batch * M * N * K;
  {
    KtScope kt(KC_GEMM_DIGITS, stream, nmacs,
               (uint64_t)((double)(request_cost(P.nw, Q.nw) * 3ull * (uint64_t)batch * M * N * K) * gemm_useful_fraction()));
    if ((tg == 8 ? in->launch8 : in->launch)(ka, grid, stream) != cudaSuccess) return ZKD_ERR_CUDA;
  }
  count_launch();
  count_macs(nmacs);

  CombineArgs ca{};
  ca.raw = raw; ca.dst = dst_fx; ca.mn = (size_t)M * N; ca.batch = batch; ca.nc = in->nc; ca.nsplit = nsp;
  ca.N = N; ca.ld = dv && dv->ld ? dv->ld : N; ca.off = dv ? dv->off : nullptr;
  ca.plane_count = dv && dv->plane_count ? dv->plane_count : (size_t)batch * M * N;
  ca.base_bit = lsbP + lsbQ + DB * in->low - kFRAC;
  ca.cut_bit = out_cut_bit; ca.mode = (int)mode; ca.msb_out = msb_out;
  const size_t tot = (size_t)batch * M * N;
  const dim3 cgrid((unsigned)((tot + 255) / 256), 2);
  // the warp-cooperative kernel wins only while the digit-serial one cannot fill the machine (measured: c2 2.47 -> 2.40 ms,
  // but c4 244 -> 316 ms when forced)
  const int cpath = options().combine_path;
  // bytes: raw columns read (two of the three planes per part, every split) + the FX digits written (+ read when accumulating)
  KtScope kt(KC_COMBINE, stream, 4ull * batch * M * N * ((uint64_t)nsp * 3 * in->nc + 2ull * kND * (mode == GemmMode::Assign ? 1 : 2)));
  if (cpath == 2 || (cpath == 0 && tot <= 32768)) {
    const size_t warps = ((size_t)M * N + EPW - 1) / EPW * batch;
    combine_warp_kernel<<<dim3((unsigned)((warps * 32 + 255) / 256), 2), 256, 0, stream>>>(ca);
  } else if (nsp == 1) combine_kernel<1><<<cgrid, 256, 0, stream>>>(ca);
  else if (nsp == 2) combine_kernel<2><<<cgrid, 256, 0, stream>>>(ca);
  else if (nsp <= 4) combine_kernel<4><<<cgrid, 256, 0, stream>>>(ca);
  else combine_kernel<0><<<cgrid, 256, 0, stream>>>(ca);
  count_launch();
  return launch_check();
}

}  // namespace zkd

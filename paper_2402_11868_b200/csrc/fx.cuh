// fx.cuh — device-side fixed-point ("FX") multi-digit arithmetic for libzkd.
//
// Number format (north_star (a): "fixed-width multiprecision number format ... stored structure-of-arrays so
// limb loads coalesce"): block fixed point, ZKD_FX_DIGITS = 30 digits of 28 bits held in int32 words, value =
// (sum_d digit[d] 2^(28 d)) * 2^-812.  Digits 0..28 are in [0, 2^28); digit 29 is signed (integer part and sign),
// i.e. a radix-2^28 two's-complement expansion.  Arrays are digit-major planes: plane d of a real array with
// `count` elements is int32[count], so consecutive threads read consecutive words of one plane.
//
// Why 28-bit digits in 32-bit words: independent IMAD.WIDE (32x32+64 -> 64) issue at 30.5 per clock per SM on sm_100a
// (zkd_measure_imad_peak, the register-only loop in api.cu: 8.86e12 /s at 1965 MHz; half the 32-bit IMAD rate), but a
// carry chain (IMAD.WIDE.X with predicate carries) reached only 44 % of that in the same loop.  With 28-bit digits a 64-bit
// column accumulator absorbs >= 128 products before it can overflow, so products are independent IMAD.WIDEs and carries are
// resolved once per tile, off the hot loop.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace zkd {

constexpr int ND = 30;          // digits per FX real
constexpr int DB = 28;          // bits per digit
constexpr int FRAC = 812;       // fractional bits (= 29 digits)
constexpr int32_t DMASK = (1 << DB) - 1;
constexpr int64_t DHALF = 1ll << (DB - 1);

// ---- carry handling on int64 column accumulators -----------------------------------------------------------

// canonical: columns 0..N-2 -> [0, 2^28), the top column keeps the (signed) rest
template <int N>
__device__ __forceinline__ void carry_canon(int64_t (&c)[N]) {
#pragma unroll
  for (int i = 0; i < N - 1; ++i) {
    int64_t carry = c[i] >> DB;
    c[i] &= DMASK;
    c[i + 1] += carry;
  }
}

// balanced: columns 0..N-2 -> [-2^27, 2^27), the top column keeps the rest
template <int N>
__device__ __forceinline__ void carry_balanced(int64_t (&c)[N]) {
#pragma unroll
  for (int i = 0; i < N - 1; ++i) {
    int64_t carry = (c[i] + DHALF) >> DB;
    c[i] -= carry << DB;
    c[i + 1] += carry;
  }
}

template <int N>
__device__ __forceinline__ void carry_canon32(int32_t (&d)[N]) {
#pragma unroll
  for (int i = 0; i < N - 1; ++i) {
    int32_t carry = d[i] >> DB;
    d[i] &= DMASK;
    d[i + 1] += carry;
  }
}

// ---- loads / stores on digit-major planes ---------------------------------------------------------------------

__device__ __forceinline__ void fx_load(int32_t (&d)[ND], const int32_t* __restrict__ p, size_t count, size_t idx) {
#pragma unroll
  for (int k = 0; k < ND; ++k) d[k] = p[(size_t)k * count + idx];
}
__device__ __forceinline__ void fx_store(int32_t* __restrict__ p, size_t count, size_t idx, const int32_t (&d)[ND]) {
#pragma unroll
  for (int k = 0; k < ND; ++k) p[(size_t)k * count + idx] = d[k];
}
__device__ __forceinline__ void fx_zero(int32_t (&d)[ND]) {
#pragma unroll
  for (int k = 0; k < ND; ++k) d[k] = 0;
}
__device__ __forceinline__ bool fx_is_neg(const int32_t (&d)[ND]) { return d[ND - 1] < 0; }

// d <- a + b, a - b, -a  (canonical in, canonical out; wraps modulo 2^(28*29+32))
__device__ __forceinline__ void fx_add(int32_t (&r)[ND], const int32_t (&a)[ND], const int32_t (&b)[ND]) {
#pragma unroll
  for (int k = 0; k < ND; ++k) r[k] = a[k] + b[k];
  carry_canon32(r);
}
__device__ __forceinline__ void fx_sub(int32_t (&r)[ND], const int32_t (&a)[ND], const int32_t (&b)[ND]) {
#pragma unroll
  for (int k = 0; k < ND; ++k) r[k] = a[k] - b[k];
  carry_canon32(r);
}
__device__ __forceinline__ void fx_neg(int32_t (&r)[ND], const int32_t (&a)[ND]) {
#pragma unroll
  for (int k = 0; k < ND; ++k) r[k] = -a[k];
  carry_canon32(r);
}
// arithmetic shift right by one bit (value / 2, floor)
__device__ __forceinline__ void fx_half(int32_t (&r)[ND], const int32_t (&a)[ND]) {
#pragma unroll
  for (int k = 0; k < ND - 1; ++k) r[k] = ((a[k] >> 1) | (a[k + 1] << (DB - 1))) & DMASK;
  r[ND - 1] = a[ND - 1] >> 1;
}

// position (0-based, from the FX LSB) of the highest bit that differs from the sign, +1; 0 for 0 and -1.
// |value| < 2^(msb - 812).  Works on canonical digits.
__device__ __forceinline__ int fx_msb(const int32_t (&d)[ND]) {
  const bool neg = d[ND - 1] < 0;
  int msb = 0;
  {
    int32_t t = neg ? ~d[ND - 1] : d[ND - 1];
    if (t) msb = (ND - 1) * DB + (32 - __clz(t));
  }
#pragma unroll
  for (int k = ND - 2; k >= 0; --k) {
    int32_t t = neg ? (~d[k] & DMASK) : d[k];
    if (msb == 0 && t) msb = k * DB + (32 - __clz(t));
  }
  return msb;
}

// FX -> double (truncating beyond ~80 bits; plenty for seeds and magnitude estimates)
__device__ __forceinline__ double fx_to_double(const int32_t (&d)[ND]) {
  double v = (double)d[ND - 1];
#pragma unroll
  for (int k = ND - 2; k >= 0; --k) v = v * 268435456.0 + (double)d[k];  // Horner, exact enough: low digits vanish
  return ldexp(v, -FRAC);
}
// double -> FX, rounds toward zero at 2^-812; |v| must be < 2^31
__device__ __forceinline__ void fx_from_double(int32_t (&d)[ND], double v) {
  fx_zero(d);
  if (v == 0.0 || !isfinite(v)) return;
  const bool neg = v < 0;
  double a = fabs(v);
  int e;
  double m = frexp(a, &e);                              // a = m 2^e, m in [1/2,1)
  uint64_t mant = (uint64_t)ldexp(m, 53);               // 53-bit integer
  int lsb = e - 53 + FRAC;                              // bit position of mant's LSB in FX
  if (lsb < 0) {
    if (lsb <= -53) return;
    mant >>= -lsb;
    lsb = 0;
  }
  // scatter mant (<= 53 bits) starting at bit lsb
  int k0 = lsb / DB, r = lsb % DB;
  unsigned __int128 w = (unsigned __int128)mant << r;   // up to 81 bits
#pragma unroll
  for (int k = 0; k < ND; ++k) {
    int j = k - k0;
    if (j >= 0 && j < 4) {
      uint64_t piece = (uint64_t)(w >> (j * DB));
      d[k] = (k == ND - 1) ? (int32_t)piece : (int32_t)(piece & DMASK);
    }
  }
  if (neg) {
    int32_t t[ND];
    fx_neg(t, d);
#pragma unroll
    for (int k = 0; k < ND; ++k) d[k] = t[k];
  }
}

// ---- products ---------------------------------------------------------------------------------------------------

// acc[c - LOWCOL] += sign * a[i] * b[j] for all i + j = c >= LOWCOL  (column accumulators, no carries)
template <int NA, int NB, int LOWCOL, int NACC, bool NEGATE>
__device__ __forceinline__ void mac_cols(int64_t (&acc)[NACC], const int32_t (&a)[NA], const int32_t (&b)[NB]) {
#pragma unroll
  for (int i = 0; i < NA; ++i) {
#pragma unroll
    for (int j = 0; j < NB; ++j) {
      if (i + j >= LOWCOL && i + j - LOWCOL < NACC) {
        if (NEGATE)
          acc[i + j - LOWCOL] -= (int64_t)a[i] * (int64_t)b[j];
        else
          acc[i + j - LOWCOL] += (int64_t)a[i] * (int64_t)b[j];
      }
    }
  }
}

// Full-width FX product accumulators: columns 28 (guard) .. 58 -> NACC = 31; result digit r = column r + 29.
constexpr int FXP_LOW = ND - 2;   // 28
constexpr int FXP_NACC = ND + 1;  // 31

template <bool NEGATE>
__device__ __forceinline__ void fx_mac(int64_t (&acc)[FXP_NACC], const int32_t (&a)[ND], const int32_t (&b)[ND]) {
  mac_cols<ND, ND, FXP_LOW, FXP_NACC, NEGATE>(acc, a, b);
}
__device__ __forceinline__ void fxp_zero(int64_t (&acc)[FXP_NACC]) {
#pragma unroll
  for (int k = 0; k < FXP_NACC; ++k) acc[k] = 0;
}
// keep the accumulators small between MACs (any number of fx_mac calls may follow)
__device__ __forceinline__ void fxp_relax(int64_t (&acc)[FXP_NACC]) { carry_balanced(acc); }
// round the guard column away and deliver canonical digits
__device__ __forceinline__ void fxp_finish(int32_t (&r)[ND], int64_t (&acc)[FXP_NACC]) {
  acc[0] += DHALF;  // round to nearest at the guard column
  carry_canon(acc);
#pragma unroll
  for (int k = 0; k < ND; ++k) r[k] = (int32_t)acc[k + 1];
}
// r = a * b (rounded)
__device__ __forceinline__ void fx_mul(int32_t (&r)[ND], const int32_t (&a)[ND], const int32_t (&b)[ND]) {
  int64_t acc[FXP_NACC];
  fxp_zero(acc);
  fx_mac<false>(acc, a, b);
  fxp_finish(r, acc);
}

// warp-level sum of column accumulators (all lanes get nothing; lane 0 holds the total)
template <int N>
__device__ __forceinline__ void warp_sum_cols(int64_t (&acc)[N]) {
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) {
#pragma unroll
    for (int k = 0; k < N; ++k) acc[k] += __shfl_down_sync(0xffffffffu, acc[k], off);
  }
}

// ---- dynamic shifts built from conditional static stages (no dynamic register indexing) ------------------------------
template <int N>
__device__ __forceinline__ void shl_bits(int32_t (&d)[N], int s) {  // 0 <= s < 28, canonical digits, top signed
#pragma unroll
  for (int k = N - 1; k > 0; --k) d[k] = (k == N - 1) ? ((d[k] << s) | (d[k - 1] >> (DB - s))) : (((d[k] << s) | (d[k - 1] >> (DB - s))) & DMASK);
  d[0] = (d[0] << s) & DMASK;
}
// generic left shift by s bits (s >= 0) using bit part (s % 28) and digit part (s / 28) with a 5-stage digit barrel
template <int N>
__device__ __forceinline__ void fx_shl(int32_t (&d)[N], int s) {
  const int sb = s % DB, sd = s / DB;
  // bit part via conditional static stages 1,2,4,8,16 (sum < 28)
  if (sb & 1) shl_bits(d, 1);
  if (sb & 2) shl_bits(d, 2);
  if (sb & 4) shl_bits(d, 4);
  if (sb & 8) shl_bits(d, 8);
  if (sb & 16) shl_bits(d, 16);
#pragma unroll
  for (int b = 0; b < 5; ++b) {
    const int st = 1 << b;
    if (sd & st) {
      // the signed top digit only keeps its low 28 bits when it moves down... it never moves down on a left shift.
#pragma unroll
      for (int k = N - 1; k >= 0; --k) {
        int32_t v = (k - st >= 0) ? d[k - st] : 0;
        if (k == N - 1) v = (v << 4) >> 4;  // the digit that becomes the top digit carries the sign in its bit 27
        d[k] = v;
      }
    }
  }
}
// arithmetic right shift by s bits
template <int N>
__device__ __forceinline__ void shr_bits(int32_t (&d)[N], int s) {
#pragma unroll
  for (int k = 0; k < N - 1; ++k) d[k] = ((d[k] >> s) | (d[k + 1] << (DB - s))) & DMASK;
  d[N - 1] >>= s;
}
template <int N>
__device__ __forceinline__ void fx_shr(int32_t (&d)[N], int s) {
  const int sb = s % DB, sd = s / DB;
  if (sb & 1) shr_bits(d, 1);
  if (sb & 2) shr_bits(d, 2);
  if (sb & 4) shr_bits(d, 4);
  if (sb & 8) shr_bits(d, 8);
  if (sb & 16) shr_bits(d, 16);
#pragma unroll
  for (int b = 0; b < 5; ++b) {
    const int st = 1 << b;
    if (sd & st) {
      const int32_t fill = d[N - 1] < 0 ? DMASK : 0;
      const int32_t top = d[N - 1];
#pragma unroll
      for (int k = 0; k < N; ++k) {
        int32_t v;
        if (k + st < N - 1) v = d[k + st];
        else if (k + st == N - 1) v = (k == N - 1) ? top : (top & DMASK);
        else if (k + st == N) v = (k == N - 1) ? (top >> DB) : ((top >> DB) & DMASK);
        else v = (k == N - 1) ? (top < 0 ? -1 : 0) : fill;
        d[k] = v;
      }
    }
  }
}


}  // namespace zkd

// fx_api.cuh — device function converting one API real into FX digits (used by the S0 ingest kernels).
#pragma once
#include "fx.cuh"
#include "zkd_internal.h"

namespace zkd {

constexpr int kMaxLimbs = kPrec / 64;  // 12: the largest supported precision (the API precision is a run-time argument)

// 64 bits of the prec-bit mantissa starting at bit `pos` (bits outside [0,prec) read as zero)
__device__ __forceinline__ uint64_t mant_bits(const uint64_t* __restrict__ limb, int pos, int prec) {
  const int kLimbs = prec >> 6;
  if (pos >= prec || pos <= -64) return 0;
  int li = pos >= 0 ? pos >> 6 : -((-pos + 63) >> 6);
  int r = pos - li * 64;  // 0..63
  uint64_t lo = (li >= 0 && li < kLimbs) ? limb[li] : 0;
  uint64_t hi = (li + 1 >= 0 && li + 1 < kLimbs) ? limb[li + 1] : 0;
  return r ? ((lo >> r) | (hi << (64 - r))) : lo;
}

// returns status bits: 1 = malformed number, 2 = magnitude does not fit FX.  d = value * 2^sc (truncated toward 0).
__device__ __forceinline__ int api_real_to_fx(const uint8_t* __restrict__ s, int sc, bool negate, int32_t (&d)[ND], int prec) {
  const int kLimbs = prec >> 6;
  const int32_t sign = *(const int32_t*)(s);
  const int32_t flags = *(const int32_t*)(s + 4);
  const int64_t ex = *(const int64_t*)(s + 8);
  const uint64_t* limb = (const uint64_t*)(s + 16);
  fx_zero(d);
  if (flags != 0 || sign < -1 || sign > 1) return 1;
  if (sign == 0) return 0;
  if (!(limb[kLimbs - 1] >> 63)) return 1;
  const int64_t sh64 = ex + (kFRAC - prec) + sc;   // FX_int = m << sh
  if (sh64 > kFxBits - prec) return 2;             // the top mantissa bit would pass FX bit 839 (|value| >= 2^27)
  if (sh64 <= -(int64_t)prec - 64) return 0;
  const int sh = (int)sh64;
#pragma unroll
  for (int k = 0; k < ND; ++k) d[k] = (int32_t)(mant_bits(limb, k * DB - sh, prec) & DMASK);
  if ((sign < 0) != negate) {
    int32_t t[ND];
    fx_neg(t, d);
#pragma unroll
    for (int k = 0; k < ND; ++k) d[k] = t[k];
  }
  return 0;
}

// exponent of a valid nonzero API real; returns false for zero; *bad set for malformed
__device__ __forceinline__ bool api_real_exp(const uint8_t* __restrict__ s, int64_t* ex, bool* bad, int prec) {
  const int kLimbs = prec >> 6;
  const int32_t sign = *(const int32_t*)(s);
  const int32_t flags = *(const int32_t*)(s + 4);
  const uint64_t* limb = (const uint64_t*)(s + 16);
  if (flags != 0 || sign < -1 || sign > 1) { *bad = true; return false; }
  if (sign == 0) return false;
  if (!(limb[kLimbs - 1] >> 63)) { *bad = true; return false; }
  *ex = *(const int64_t*)(s + 8);
  return true;
}

}  // namespace zkd

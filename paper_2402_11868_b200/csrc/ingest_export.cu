// ingest_export.cu — S0 (API numbers -> FX planes) and S6 (FX planes -> API numbers) conversion kernels.
//
// API real (include/zkd.h): {int32 sign; int32 flags; int64 exp; uint64 limb[prec/64]}, value = sign * m * 2^(exp-prec);
// prec is a run-time argument (128 .. 768 in steps of 64).
// FX real: 30 digits of 28 bits, value = int * 2^-812 (fx.cuh).  One thread per number; the AoS side is read /
// written with 16-byte accesses, the SoA side is coalesced across threads.
#include "fx_api.cuh"
#include "timing.h"

namespace zkd {

// status bits written with atomicOr: 1 = malformed number, 2 = magnitude does not fit FX
__global__ void __launch_bounds__(128) fx_from_api_kernel(size_t count, const uint8_t* __restrict__ src, int32_t* __restrict__ dst,
                                                          int scale_bits, const int* __restrict__ scale_dev, int scale_stride,
                                                          size_t per_scale, int* status, int prec) {
  const int kApiRealBytes = 16 + (prec >> 3);
  const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= count) return;
  int sc = scale_bits;
  if (scale_dev) sc += scale_dev[(e / per_scale) * scale_stride];
  int32_t d[ND];
  const int st = api_real_to_fx(src + e * kApiRealBytes, sc, false, d, prec);
  if (st && status) atomicOr(status, st);
  fx_store(dst, count, e, d);
}

// dst real index = e * dst_stride + dst_off (dst_stride = 2 writes the re or im slots of a complex array)
__global__ void __launch_bounds__(128) fx_to_api_kernel(size_t count, const int32_t* __restrict__ src, uint8_t* __restrict__ dst,
                                                        int dst_stride, int dst_off, int scale_bits,
                                                        const int* __restrict__ scale_dev, int scale_stride, size_t per_scale,
                                                        int prec) {
  const int kApiRealBytes = 16 + (prec >> 3), kLimbs = prec >> 6;
  const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= count) return;
  int32_t d[ND];
  fx_load(d, src, count, e);
  uint8_t* o = dst + (e * dst_stride + dst_off) * kApiRealBytes;
  const bool neg = d[ND - 1] < 0;
  if (neg) {
    int32_t t[ND];
    fx_neg(t, d);
#pragma unroll
    for (int k = 0; k < ND; ++k) d[k] = t[k];
  }
  const int msb = fx_msb(d);  // 1 + index of the highest set bit of the magnitude
  uint64_t* o64 = (uint64_t*)o;
  if (msb == 0) {
#pragma unroll
    for (int k = 0; k < kMaxLimbs + 2; ++k)
      if (k < kLimbs + 2) o64[k] = 0;
    return;
  }
  // magnitude bits [lo, lo + prec) with lo = msb - prec form the mantissa; round to nearest even on the rest
  const int lo = msb - prec;
  // digits live in local memory from here on (dynamic indexing); this is a cold kernel
  auto bits64 = [&](int pos) -> uint64_t {  // 64 bits of the magnitude starting at bit pos
    uint64_t r = 0;
#pragma unroll
    for (int k = 0; k < ND; ++k) {
      const int off = k * DB - pos;  // where digit k lands in the 64-bit word
      const uint64_t dk = (uint64_t)(uint32_t)d[k];
      if (off >= 0 && off < 64) r |= dk << off;
      else if (off < 0 && off > -32) r |= dk >> (-off);
    }
    return r;
  };
  uint64_t m[kMaxLimbs];
#pragma unroll
  for (int k = 0; k < kMaxLimbs; ++k) m[k] = k < kLimbs ? bits64(lo + 64 * k) : 0;
  bool round_up = false;
  if (lo > 0) {
    // round bit = bit lo-1; sticky = any bit below
    const uint64_t below = bits64(lo - 64);  // bits [lo-64, lo)
    const bool rb = (below >> 63) & 1;
    bool sticky = (below << 1) != 0;
    if (!sticky) {
#pragma unroll
      for (int k = 0; k < ND; ++k) {
        const int hi = k * DB + DB;  // digit k covers bits [k*28, hi)
        if (hi <= lo - 64) { if (d[k]) sticky = true; }
        else if (k * DB < lo - 64) { if ((uint32_t)d[k] & ((1u << (lo - 64 - k * DB)) - 1)) sticky = true; }
      }
    }
    round_up = rb && (sticky || (m[0] & 1));
  }
  int64_t ex = (int64_t)msb - kFRAC;  // value = mant * 2^(msb - prec - 812) = mant * 2^(ex - prec)
  if (round_up) {
    bool carry = true;
#pragma unroll
    for (int k = 0; k < kMaxLimbs; ++k) {
      if (carry && k < kLimbs) {
        m[k] += 1;
        carry = m[k] == 0;
      }
    }
    if (carry) {  // mantissa overflowed to 2^prec
#pragma unroll
      for (int k = 0; k < kMaxLimbs; ++k)
        if (k == kLimbs - 1) m[k] = 1ull << 63;
      ex += 1;
    }
  }
  int sc = scale_bits;
  if (scale_dev) sc += scale_dev[(e / per_scale) * scale_stride];
  ex -= sc;
  int32_t* o32 = (int32_t*)o;
  o32[0] = neg ? -1 : 1;
  o32[1] = 0;
  o64[1] = (uint64_t)ex;
#pragma unroll
  for (int k = 0; k < kMaxLimbs; ++k)
    if (k < kLimbs) o64[2 + k] = m[k];
}

int fx_from_api_scaled(size_t count, const void* src_api, int32_t* dst_fx, int scale_bits, const int* scale_dev,
                       int scale_stride, size_t per_scale, int* status, cudaStream_t s, int prec) {
  KtScope kt_scope(KC_IO, s);
  if (count == 0) return ZKD_OK;
  fx_from_api_kernel<<<(unsigned)((count + 127) / 128), 128, 0, s>>>(count, (const uint8_t*)src_api, dst_fx, scale_bits,
                                                                     scale_dev, scale_stride, per_scale ? per_scale : 1, status, prec);
  count_launch();
  return launch_check();
}
int fx_to_api_scaled(size_t count, const int32_t* src_fx, void* dst_api, int scale_bits, const int* scale_dev, int scale_stride,
                     size_t per_scale, cudaStream_t s, int prec) {
  KtScope kt_scope(KC_IO, s);
  if (count == 0) return ZKD_OK;
  fx_to_api_kernel<<<(unsigned)((count + 127) / 128), 128, 0, s>>>(count, src_fx, (uint8_t*)dst_api, 1, 0, scale_bits, scale_dev,
                                                                   scale_stride, per_scale ? per_scale : 1, prec);
  count_launch();
  return launch_check();
}
// complex FX array (re planes, im planes) -> interleaved (re, im) API numbers
int fxc_to_api(size_t count, const int32_t* src_fxc, void* dst_api, cudaStream_t s, int prec) {
  KtScope kt_scope(KC_IO, s);
  if (count == 0) return ZKD_OK;
  for (int part = 0; part < 2; ++part)
    fx_to_api_kernel<<<(unsigned)((count + 127) / 128), 128, 0, s>>>(count, src_fxc + (size_t)part * ND * count, (uint8_t*)dst_api,
                                                                     2, part, 0, nullptr, 0, 1, prec);
  count_launch(2);
  return launch_check();
}
// the same with one power-of-two scale per `per_scale` complex elements (value = fx 2^-scale)
int fxc_to_api_scaled(size_t count, const int32_t* src_fxc, void* dst_api, const int* scale_dev, size_t per_scale, cudaStream_t s, int prec) {
  KtScope kt_scope(KC_IO, s);
  if (count == 0) return ZKD_OK;
  for (int part = 0; part < 2; ++part)
    fx_to_api_kernel<<<(unsigned)((count + 127) / 128), 128, 0, s>>>(count, src_fxc + (size_t)part * ND * count, (uint8_t*)dst_api,
                                                                     2, part, 0, scale_dev, 1, per_scale ? per_scale : 1, prec);
  count_launch(2);
  return launch_check();
}
int fx_from_api(int count, const void* src_api, int32_t* dst_fx, int scale_bits, cudaStream_t s, int prec) {
  return fx_from_api_scaled((size_t)count, src_api, dst_fx, scale_bits, nullptr, 0, 1, nullptr, s, prec);
}
int fx_to_api(int count, const int32_t* src_fx, void* dst_api, int scale_bits, cudaStream_t s, int prec) {
  return fx_to_api_scaled((size_t)count, src_fx, dst_api, scale_bits, nullptr, 0, 1, s, prec);
}

}  // namespace zkd

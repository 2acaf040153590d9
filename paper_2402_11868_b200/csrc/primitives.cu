// primitives.cu — element-wise entry to the multi-digit primitives of fx.cuh / fx_funcs.cuh (SURVEY.md 8(a) "MP primitives",
// north_star (b)), exported as zkd_fx_prim so that tests can check each primitive against exact integer arithmetic
// (tier 2).  The hot path calls the same device functions from inside its kernels.
#include "fx_funcs.cuh"
#include "timing.h"
#include "zkd_internal.h"

namespace zkd {

__global__ void __launch_bounds__(128) fx_prim_kernel(int op, size_t count, const int32_t* __restrict__ a, const int32_t* __restrict__ b,
                                                      int32_t* __restrict__ out) {
  const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= count) return;
  int32_t x[ND], y[ND], r[ND];
  fx_load(x, a, count, e);
  if (b) fx_load(y, b, count, e); else fx_zero(y);
  switch (op) {
    case ZKD_PRIM_ADD: fx_add(r, x, y); break;
    case ZKD_PRIM_SUB: fx_sub(r, x, y); break;
    case ZKD_PRIM_MUL: fx_mul(r, x, y); break;
    case ZKD_PRIM_RECIP: fx_recip_quarter<ND - 1>(r, x, 5); break;
    case ZKD_PRIM_RSQRT: fx_rsqrt(r, x); break;
    case ZKD_PRIM_MSB: fx_zero(r); r[0] = fx_msb(x); break;
    case ZKD_PRIM_HALF: fx_half(r, x); break;
    case ZKD_PRIM_FROM_DOUBLE: fx_from_double(r, fx_to_double(x)); break;
    default: fx_zero(r);
  }
  fx_store(out, count, e, r);
}

int fx_prim(int op, size_t count, const int32_t* a, const int32_t* b, int32_t* out, cudaStream_t s) {
  if (count == 0) return ZKD_OK;
  KtScope kt(KC_OTHER, s);
  fx_prim_kernel<<<(unsigned)((count + 127) / 128), 128, 0, s>>>(op, count, a, b, out);
  count_launch();
  return launch_check();
}

}  // namespace zkd

// fx_funcs.cuh — multi-digit functions built on fx.cuh: Newton reciprocal and reciprocal square root from an fp64 start
// (SURVEY.md 8(a) "MP primitives": "reciprocal, rsqrt, divide via Newton from an fp64 seed").  Used by ecalc_kernel (S4d),
// phase_kernel (S6), the LU kernels (S4a') and the primitive test entry zkd_fx_prim.
#pragma once
#include "fx.cuh"

namespace zkd {

// r <- 1/d' for d' in [1/4,1/2] given as FX (only the top W digits below the binary point are used);
// r returned as FX (value in [2,4]).  Newton: r <- r + r (1 - d' r), quadratic from an fp64 start.
template <int W>
__device__ __forceinline__ void fx_recip_quarter(int32_t (&r)[ND], const int32_t (&dq)[ND], int iters) {
  // work on full FX digits but zero everything below digit ND-1-W so that products are short where it matters:
  // the compiler removes multiplications by literal zeros only if the zeros are compile-time; so use W-digit arrays.
  constexpr int LO = ND - 1 - W;  // first digit kept (FX digit index); fractional digits kept: 29 - LO = W...
  int32_t dw[W + 1], rw[W + 1];   // digits LO..ND-1 of d' and r
#pragma unroll
  for (int k = 0; k <= W; ++k) dw[k] = dq[LO + k];
  {
    // fp64 start from the top three digits of d'
    double dd = ((double)dw[W] * 268435456.0 + (double)dw[W - 1]) * 268435456.0 + (double)dw[W - 2];
    dd = ldexp(dd, -3 * DB + DB);  // value: digit ND-1 is the integer digit -> dw[W] has weight 1
    const double r0 = 1.0 / dd;     // in [2,4]
    int32_t t[ND];
    fx_from_double(t, r0);
#pragma unroll
    for (int k = 0; k <= W; ++k) rw[k] = t[LO + k];
  }
  // value(x) = sum_k x[k] 2^(28 (k - W)); product columns: x[a] y[b] has weight 2^(28 (a + b - 2W)); result digit k
  // <- column k + W.  Keep columns >= W - 1 (guard).
  for (int it = 0; it < iters; ++it) {
    int64_t acc[W + 2];
#pragma unroll
    for (int k = 0; k < W + 2; ++k) acc[k] = 0;
    mac_cols<W + 1, W + 1, W - 1, W + 2, false>(acc, dw, rw);  // columns W-1 .. 2W; the top one is signed digit W
    carry_canon(acc);
    // e = 1 - d' r : digits (acc[1 + k] is result digit k)
    int32_t ew[W + 1];
#pragma unroll
    for (int k = 0; k <= W; ++k) ew[k] = -(int32_t)acc[1 + k];
    ew[W] += 1;
    carry_canon32(ew);
    // r += r e
    int64_t acc2[W + 2];
#pragma unroll
    for (int k = 0; k < W + 2; ++k) acc2[k] = 0;
    // ew is canonical with signed top; rw canonical
    mac_cols<W + 1, W + 1, W - 1, W + 2, false>(acc2, rw, ew);
    carry_canon(acc2);
#pragma unroll
    for (int k = 0; k <= W; ++k) rw[k] += (int32_t)acc2[1 + k];
    carry_canon32(rw);
  }
  fx_zero(r);
#pragma unroll
  for (int k = 0; k <= W; ++k) r[LO + k] = rw[k];
}


// y <- 1/sqrt(s) for an FX number s > 0 (any magnitude that fits): s' = s 4^t in [1/4, 1), y' = 1/sqrt(s') in (1, 2] by Newton
// y' <- y' (3 - s' y'^2) / 2 from an fp64 start (five iterations: 50 -> 100 -> ... bits, the last two at the FX floor), then
// y = y' 2^t.  The products are fx_mul (truncated below the guard column), so the result is good to a few units of 2^-812
// times 2^t.  s <= 0 returns 0.
__device__ __forceinline__ void fx_rsqrt(int32_t (&y)[ND], const int32_t (&s)[ND]) {
  int32_t s2[ND];
#pragma unroll
  for (int q = 0; q < ND; ++q) s2[q] = s[q];
  const int msb = fx_msb(s2);
  if (msb == 0 || s[ND - 1] < 0) { fx_zero(y); return; }
  // s' = s 4^t with msb(s') in {811, 812}  (s' in [1/4, 1))
  int t2 = 812 - msb;
  t2 -= (t2 & 1);
  if (t2 >= 0) fx_shl(s2, t2); else fx_shr(s2, -t2);
  fx_from_double(y, rsqrt(fx_to_double(s2)));  // y in (1, 2]
  for (int it = 0; it < 5; ++it) {
    int32_t yy[ND], syy[ND], corr[ND], three[ND], h[ND];
    fx_mul(yy, y, y);
    fx_mul(syy, s2, yy);
    fx_zero(three); three[ND - 1] = 3;
    fx_sub(corr, three, syy);  // 3 - s y^2
    fx_mul(h, y, corr);
    fx_half(y, h);
  }
  // 1/sqrt(s) = y 2^(t2/2)
  if (t2 >= 0) fx_shl(y, t2 / 2); else fx_shr(y, (-t2) / 2);
}

}  // namespace zkd

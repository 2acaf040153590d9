// lu.cu — multiprecision LU factorisation with partial pivoting and triangular solves on FX planes (SURVEY.md 8(f) NEXT-3:
// ZKCM_OMP's "Gaussian elimination, LU decomposition"), and on top of it the exact Rayleigh quotient iteration
// S4a' of SURVEY.md 8(a) ("the Rayleigh quotient iteration was employed to recover the precision"): per
// eigenpair, sigma = x^H A x, LU of (A - sigma I), y = (A - sigma I)^-1 x, x = y / ||y||.  north_star (d) names this route as
// the alternative to the correction-equation form that the production path uses; it is O(N^4), needs one factorisation per
// eigenpair of a matrix that is singular by design, and cannot separate clustered eigenvalues, so it serves as the
// in-product cross-check for isolated spectra at N <= 64.
//
// One CTA per problem (matrix, or matrix and eigenpair).  The matrix lives in global memory (L2) as complex FX planes;
// every elimination step is: pivot search (fp64 magnitudes), row swap, Newton reciprocal of the pivot (fx_funcs.cuh), the
// multiplier column, and the rank-one update of the trailing block - one 30 x 30-digit complex multiply-subtract per element
// and thread.  All products are the truncated FX products of fx.cuh (exact integer columns, one rounding).
#include "blocks.h"
#include "fx_funcs.cuh"
#include "timing.h"

namespace zkd {

namespace {

struct Cfx { int32_t re[ND], im[ND]; };

__device__ __forceinline__ void cload(Cfx& z, const int32_t* __restrict__ base, size_t count, size_t e) {
  fx_load(z.re, base, count, e);
  fx_load(z.im, base + (size_t)ND * count, count, e);
}
__device__ __forceinline__ void cstore(int32_t* __restrict__ base, size_t count, size_t e, const Cfx& z) {
  fx_store(base, count, e, z.re);
  fx_store(base + (size_t)ND * count, count, e, z.im);
}
// r = a * b (one rounding per part)
__device__ __forceinline__ void cmul(Cfx& r, const Cfx& a, const Cfx& b) {
  int64_t acc[FXP_NACC];
#pragma unroll 1
  for (int part = 0; part < 2; ++part) {
    fxp_zero(acc);
    // part 0: ar br - ai bi ; part 1: ar bi + ai br  (one multiply site, operands selected at run time)
#pragma unroll 1
    for (int term = 0; term < 2; ++term) {
      int32_t x[ND], y[ND];
      const bool neg = part == 0 && term == 1;
#pragma unroll
      for (int q = 0; q < ND; ++q) {
        x[q] = term ? a.im[q] : a.re[q];
        const int32_t v = (term ^ part) ? b.im[q] : b.re[q];
        y[q] = neg ? -v : v;
      }
      fx_mac<false>(acc, x, y);
    }
    if (part == 0) fxp_finish(r.re, acc); else fxp_finish(r.im, acc);
  }
}
// r = c - a * b
__device__ __forceinline__ void cmsub(Cfx& r, const Cfx& c, const Cfx& a, const Cfx& b) {
  Cfx t;
  cmul(t, a, b);
  fx_sub(r.re, c.re, t.re);
  fx_sub(r.im, c.im, t.im);
}
// inv = 1 / p for |p| >= 2^-26 (else returns false).  1/p = conj(p) / |p|^2, the real reciprocal by Newton on the normalised
// |p|^2 (fx_recip_quarter, value in [1/4, 1/2)).  |p| must be < 2^13 so that |p|^2 fits FX.
__device__ __forceinline__ bool cinv(Cfx& inv, const Cfx& p) {
  int64_t acc[FXP_NACC];
  fxp_zero(acc);
  fx_mac<false>(acc, p.re, p.re);
  fx_mac<false>(acc, p.im, p.im);
  int32_t n2[ND];
  fxp_finish(n2, acc);
  const int m = fx_msb(n2);          // |p|^2 in [2^(m-813), 2^(m-812))
  if (m < 812 - 52) return false;     // |p| < 2^-26: 1/|p| would pass the FX integer range together with the guard bits
  const int s = 811 - m;              // n2 2^s in [1/4, 1/2)
  if (s >= 0) fx_shl(n2, s); else fx_shr(n2, -s);
  int32_t r[ND];
  fx_recip_quarter<ND - 1>(r, n2, 5);  // r = 1 / (n2 2^s) in (2, 4]
  Cfx c;
  fx_mul(c.re, p.re, r);
  int32_t nim[ND];
  fx_neg(nim, p.im);
  fx_mul(c.im, nim, r);
#pragma unroll
  for (int q = 0; q < ND; ++q) { inv.re[q] = c.re[q]; inv.im[q] = c.im[q]; }
  if (s >= 0) { fx_shl(inv.re, s); fx_shl(inv.im, s); } else { fx_shr(inv.re, -s); fx_shr(inv.im, -s); }
  return true;
}

// ---- factorisation: P A = L U in place (L unit lower, its multipliers below the diagonal), one CTA per problem ---------------------
// perm[p][k] = row swapped with k at step k;  invd[p][k] = 1 / u_kk;  flags[p]: bit 0 = a pivot is exactly zero (singular),
// bit 1 = a pivot before the last is too small to invert in FX, bit 2 = the LAST pivot is too small to invert (what exact RQI
// produces by design: the caller decides whether that is an error).
__global__ void __launch_bounds__(256) lu_factor_kernel(int N, int32_t* __restrict__ Mx, size_t count, int* __restrict__ perm,
                                                        int32_t* __restrict__ invd, size_t icount, int* __restrict__ flags) {
  __shared__ double s_key[256];
  __shared__ int s_piv, s_stop;
  __shared__ Cfx s_inv;
  const int p = blockIdx.x, tid = threadIdx.x, nthr = blockDim.x;
  const size_t base = (size_t)p * N * N;
  if (tid == 0) s_stop = 0;
  __syncthreads();
  for (int k = 0; k < N; ++k) {
    // 1. pivot: largest |a_ik| over i >= k by fp64 magnitude (first index on ties)
    double best = -1.0;
    int bi = k;
    for (int i = k + tid; i < N; i += nthr) {
      Cfx a;
      cload(a, Mx, count, base + (size_t)i * N + k);
      const double xr = fx_to_double(a.re), xi = fx_to_double(a.im);
      const double key = xr * xr + xi * xi;
      if (key > best) { best = key; bi = i; }
    }
    s_key[tid] = best;
    __syncthreads();
    if (tid == 0) {
      double b2 = -1.0;
      int arg = k;
      const int lim = min(nthr, N - k);
      for (int t = 0; t < lim; ++t)
        if (s_key[t] > b2) { b2 = s_key[t]; arg = t; }
      s_piv = arg;  // the thread that holds the winner; its bi is read below
    }
    __syncthreads();
    if (tid == s_piv) s_piv = -1 - bi;  // hand over the row index (negative marks "resolved")
    __syncthreads();
    const int piv = -1 - s_piv;
    if (tid == 0) perm[(size_t)p * N + k] = piv;
    // 2. swap rows k and piv
    if (piv != k) {
      for (int j = tid; j < N; j += nthr) {
        Cfx a, b;
        cload(a, Mx, count, base + (size_t)k * N + j);
        cload(b, Mx, count, base + (size_t)piv * N + j);
        cstore(Mx, count, base + (size_t)k * N + j, b);
        cstore(Mx, count, base + (size_t)piv * N + j, a);
      }
    }
    __syncthreads();
    // 3. reciprocal of the pivot
    if (tid == 0) {
      Cfx pv, inv;
      cload(pv, Mx, count, base + (size_t)k * N + k);
      const bool zero = fx_msb(pv.re) == 0 && fx_msb(pv.im) == 0 && pv.re[ND - 1] >= 0 && pv.im[ND - 1] >= 0;
      const bool ok = !zero && cinv(inv, pv);
      if (!ok) {
#pragma unroll
        for (int q = 0; q < ND; ++q) { inv.re[q] = 0; inv.im[q] = 0; }
        atomicOr(flags + p, zero ? 1 : (k == N - 1 ? 4 : 2));
        if (k < N - 1) s_stop = 1;
      }
      s_inv = inv;
      cstore(invd, icount, (size_t)p * N + k, inv);
    }
    __syncthreads();
    if (s_stop) return;
    // 4. multipliers l_ik = a_ik / u_kk
    for (int i = k + 1 + tid; i < N; i += nthr) {
      Cfx a, l;
      cload(a, Mx, count, base + (size_t)i * N + k);
      cmul(l, a, s_inv);
      cstore(Mx, count, base + (size_t)i * N + k, l);
    }
    __syncthreads();
    // 5. trailing block a_ij -= l_ik u_kj
    const int w = N - 1 - k;
#pragma unroll 1
    for (int e = tid; e < w * w; e += nthr) {
      const int i = k + 1 + e / w, j = k + 1 + e % w;
      Cfx a, l, u, r;
      cload(l, Mx, count, base + (size_t)i * N + k);
      cload(u, Mx, count, base + (size_t)k * N + j);
      cload(a, Mx, count, base + (size_t)i * N + j);
      cmsub(r, a, l, u);
      cstore(Mx, count, base + (size_t)i * N + j, r);
    }
    __syncthreads();
  }
}

// ---- solves with the factors: one CTA per problem --------------------------------------------------------------------------------------
// mode 0: X = A^-1 B (nrhs columns, B overwritten).  mode 1 (exact RQI, nrhs = 1): the direction of y = A^-1 b without forming its
// length: forward substitution z = L^-1 P b, then with f = u_nn / z_n the scaled back substitution y_n = 1,
// y_i = (f z_i - sum_{j>i} u_ij y_j) / u_ii - the exact solution times u_nn / z_n, well defined however small u_nn is (it is zero to
// working precision once sigma has converged) - and finally y is shifted to max |y_i| < 1/2 and normalised to unit 2-norm.
__global__ void __launch_bounds__(256) lu_solve_kernel(int N, int nrhs, int mode, const int32_t* __restrict__ Mx, size_t count,
                                                       const int* __restrict__ perm, const int32_t* __restrict__ invd, size_t icount,
                                                       int32_t* __restrict__ B, size_t bcount, int* __restrict__ flags) {
  __shared__ Cfx s_f;
  __shared__ int s_msb;
  __shared__ int64_t s_acc[8][FXP_NACC];
  const int p = blockIdx.x, tid = threadIdx.x, nthr = blockDim.x;
  const size_t base = (size_t)p * N * N, bbase = (size_t)p * N * nrhs;
  if (flags[p] & 3) return;                 // singular or a pivot that could not be inverted: reported by the caller
  if (mode == 0 && (flags[p] & 4)) return;
  // row interchanges, in the order of the factorisation
  for (int k = 0; k < N; ++k) {
    const int piv = perm[(size_t)p * N + k];
    if (piv != k) {
      for (int c = tid; c < nrhs; c += nthr) {
        Cfx a, b;
        cload(a, B, bcount, bbase + (size_t)k * nrhs + c);
        cload(b, B, bcount, bbase + (size_t)piv * nrhs + c);
        cstore(B, bcount, bbase + (size_t)k * nrhs + c, b);
        cstore(B, bcount, bbase + (size_t)piv * nrhs + c, a);
      }
    }
    __syncthreads();
  }
  // forward: z_i -= l_ik z_k
  for (int k = 0; k < N - 1; ++k) {
    const int w = N - 1 - k;
#pragma unroll 1
    for (int e = tid; e < w * nrhs; e += nthr) {
      const int i = k + 1 + e / nrhs, c = e % nrhs;
      Cfx l, zk, zi, r;
      cload(l, Mx, count, base + (size_t)i * N + k);
      cload(zk, B, bcount, bbase + (size_t)k * nrhs + c);
      cload(zi, B, bcount, bbase + (size_t)i * nrhs + c);
      cmsub(r, zi, l, zk);
      cstore(B, bcount, bbase + (size_t)i * nrhs + c, r);
    }
    __syncthreads();
  }
  if (mode == 1) {
    // f = u_nn / z_n; z <- f z; z_n <- u_nn (so that the generic back substitution below yields y_n = u_nn / u_nn ... = 1 is set directly)
    if (tid == 0) {
      Cfx zn, unn, izn, f;
      cload(zn, B, bcount, bbase + (size_t)(N - 1));
      cload(unn, Mx, count, base + (size_t)(N - 1) * N + (N - 1));
      if (cinv(izn, zn)) cmul(f, unn, izn);
      else {
#pragma unroll
        for (int q = 0; q < ND; ++q) { f.re[q] = 0; f.im[q] = 0; }  // z_n ~ 0: the null vector of U alone
      }
      s_f = f;
    }
    __syncthreads();
    for (int i = tid; i < N - 1; i += nthr) {
      Cfx z, r;
      cload(z, B, bcount, bbase + (size_t)i);
      cmul(r, z, s_f);
      cstore(B, bcount, bbase + (size_t)i, r);
    }
    if (tid == 0) {
      Cfx one;
#pragma unroll
      for (int q = 0; q < ND; ++q) { one.re[q] = 0; one.im[q] = 0; }
      one.re[ND - 1] = 1;
      cstore(B, bcount, bbase + (size_t)(N - 1), one);
    }
    __syncthreads();
  }
  // backward, column oriented: x_j = z_j / u_jj, then z_i -= u_ij x_j for i < j
  for (int j = N - 1; j >= 0; --j) {
    if (!(mode == 1 && j == N - 1)) {
      for (int c = tid; c < nrhs; c += nthr) {
        Cfx z, d, x;
        cload(z, B, bcount, bbase + (size_t)j * nrhs + c);
        cload(d, invd, icount, (size_t)p * N + j);
        cmul(x, z, d);
        cstore(B, bcount, bbase + (size_t)j * nrhs + c, x);
      }
    }
    __syncthreads();
#pragma unroll 1
    for (int e = tid; e < j * nrhs; e += nthr) {
      const int i = e / nrhs, c = e % nrhs;
      Cfx u, xj, zi, r;
      cload(u, Mx, count, base + (size_t)i * N + j);
      cload(xj, B, bcount, bbase + (size_t)j * nrhs + c);
      cload(zi, B, bcount, bbase + (size_t)i * nrhs + c);
      cmsub(r, zi, u, xj);
      cstore(B, bcount, bbase + (size_t)i * nrhs + c, r);
    }
    __syncthreads();
  }
  if (mode != 1) return;
  // normalise y: shift so that max |component| < 1/2, then divide by the 2-norm
  if (tid == 0) s_msb = 0;
  __syncthreads();
  int mm = 0;
  for (int i = tid; i < N; i += nthr) {
    Cfx y;
    cload(y, B, bcount, bbase + (size_t)i);
    mm = max(mm, max(fx_msb(y.re), fx_msb(y.im)));
  }
  atomicMax(&s_msb, mm);
  __syncthreads();
  const int sh = s_msb - 810;  // > 0: shift right
  int64_t acc[FXP_NACC];
  fxp_zero(acc);
  for (int i = tid; i < N; i += nthr) {
    Cfx y;
    cload(y, B, bcount, bbase + (size_t)i);
    if (sh > 0) { fx_shr(y.re, sh); fx_shr(y.im, sh); } else if (sh < 0) { fx_shl(y.re, -sh); fx_shl(y.im, -sh); }
    cstore(B, bcount, bbase + (size_t)i, y);
    fx_mac<false>(acc, y.re, y.re);
    fx_mac<false>(acc, y.im, y.im);
    fxp_relax(acc);
  }
  warp_sum_cols(acc);
  if ((tid & 31) == 0) {
#pragma unroll
    for (int q = 0; q < FXP_NACC; ++q) s_acc[tid >> 5][q] = acc[q];
  }
  __syncthreads();
  if (tid == 0) {
    for (int w = 1; w < (nthr >> 5); ++w) {
#pragma unroll
      for (int q = 0; q < FXP_NACC; ++q) acc[q] += s_acc[w][q];
    }
    int32_t n2[ND], y[ND];
    fxp_finish(n2, acc);
    fx_rsqrt(y, n2);
#pragma unroll
    for (int q = 0; q < ND; ++q) { s_f.re[q] = y[q]; s_f.im[q] = 0; }
  }
  __syncthreads();
  for (int i = tid; i < N; i += nthr) {
    Cfx y;
    cload(y, B, bcount, bbase + (size_t)i);
    int32_t o[ND];
    fx_mul(o, y.re, s_f.re);
#pragma unroll
    for (int q = 0; q < ND; ++q) y.re[q] = o[q];
    fx_mul(o, y.im, s_f.re);
#pragma unroll
    for (int q = 0; q < ND; ++q) y.im[q] = o[q];
    cstore(B, bcount, bbase + (size_t)i, y);
  }
}

// ---- exact RQI plumbing: problem (b, j) <- A_b - theta_j I and right-hand side x_j; and back -----------------------------------------
__global__ void __launch_bounds__(256) rqi_setup_kernel(int N, int batch, const int32_t* __restrict__ A, const int32_t* __restrict__ theta,
                                                        const int32_t* __restrict__ X, int32_t* __restrict__ Mx, int32_t* __restrict__ rhs) {
  const size_t per = (size_t)N * N, acount = per * batch, P = (size_t)N * batch, mcount = per * P;
  const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= 2 * mcount) return;
  const int part = (int)(t / mcount);
  const size_t e = t % mcount;
  const size_t p = e / per;
  const int b = (int)(p / N), j = (int)(p % N), r = (int)((e % per) / N), c = (int)(e % N);
  int32_t d[ND];
  fx_load(d, A + (part ? (size_t)ND * acount : 0), acount, (size_t)b * per + (size_t)r * N + c);
  if (part == 0 && r == c) {
    int32_t th[ND], o[ND];
    fx_load(th, theta, P, p);
    fx_sub(o, d, th);
#pragma unroll
    for (int q = 0; q < ND; ++q) d[q] = o[q];
  }
  fx_store(Mx + (part ? (size_t)ND * mcount : 0), mcount, e, d);
  if (c == 0) {  // rhs[p][r] = X[b][r][j]
    fx_load(d, X + (part ? (size_t)ND * acount : 0), acount, (size_t)b * per + (size_t)r * N + j);
    fx_store(rhs + (part ? (size_t)ND * (P * N) : 0), P * N, p * N + r, d);
  }
}
__global__ void __launch_bounds__(256) rqi_scatter_kernel(int N, int batch, const int32_t* __restrict__ rhs, const int* __restrict__ flags,
                                                          int32_t* __restrict__ X) {
  const size_t per = (size_t)N * N, acount = per * batch, P = (size_t)N * batch;
  const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= 2 * P * N) return;
  const int part = (int)(t / (P * N));
  const size_t e = t % (P * N);
  const size_t p = e / N;
  const int r = (int)(e % N), b = (int)(p / N), j = (int)(p % N);
  if (flags[p] & 3) return;  // keep the previous iterate
  int32_t d[ND];
  fx_load(d, rhs + (part ? (size_t)ND * (P * N) : 0), P * N, e);
  fx_store(X + (part ? (size_t)ND * acount : 0), acount, (size_t)b * per + (size_t)r * N + j, d);
}

}  // namespace

int lu_factor(int N, int nprob, int32_t* Mx, int* perm, int32_t* invd, int* flags, cudaStream_t s) {
  // 4 complex multiply-subtracts of 494 digit products per element of every trailing block: ~ (N^3 / 3) * 4 * 494 per problem
  KtScope kt(KC_LU, s, (uint64_t)nprob * (uint64_t)N * N * N / 3 * 4 * 494);
  ZKD_CUDA_TRY(cudaMemsetAsync(flags, 0, sizeof(int) * nprob, s));
  lu_factor_kernel<<<nprob, 256, 0, s>>>(N, Mx, (size_t)N * N * nprob, perm, invd, (size_t)N * nprob, flags);
  count_launch();
  return launch_check();
}
int lu_solve(int N, int nrhs, int nprob, int mode, const int32_t* Mx, const int* perm, const int32_t* invd, int32_t* B, int* flags,
             cudaStream_t s) {
  KtScope kt(KC_LU, s, (uint64_t)nprob * (uint64_t)N * N * nrhs * 4 * 494);
  lu_solve_kernel<<<nprob, 256, 0, s>>>(N, nrhs, mode, Mx, (size_t)N * N * nprob, perm, invd, (size_t)N * nprob, B,
                                        (size_t)N * nrhs * nprob, flags);
  count_launch();
  return launch_check();
}
int rqi_setup(int N, int batch, const int32_t* A, const int32_t* theta, const int32_t* X, int32_t* Mx, int32_t* rhs, cudaStream_t s) {
  KtScope kt(KC_OTHER, s);
  const size_t t = 2 * (size_t)N * N * N * batch;
  rqi_setup_kernel<<<(unsigned)((t + 255) / 256), 256, 0, s>>>(N, batch, A, theta, X, Mx, rhs);
  count_launch();
  return launch_check();
}
int rqi_scatter(int N, int batch, const int32_t* rhs, const int* flags, int32_t* X, cudaStream_t s) {
  KtScope kt(KC_OTHER, s);
  const size_t t = 2 * (size_t)N * N * batch;
  rqi_scatter_kernel<<<(unsigned)((t + 255) / 256), 256, 0, s>>>(N, batch, rhs, flags, X);
  count_launch();
  return launch_check();
}

// ---- NEXT-3: A X = B through the C ABI ------------------------------------------------------------------------------------------------
// A and B are brought to block fixed point with one power-of-two scale each per problem (max |a_ij|, max |b_ij| in [1/8, 1/4)), so
// X_fx = X 2^(sb - sa); the export undoes that.  Fixed point means ABSOLUTE accuracy: |dX| ~ cond(A) 2^-(prec+2) in those units,
// and a solution larger than 2^26 of them does not fit the format (the caller's responsibility: well-conditioned systems).
__global__ void __launch_bounds__(128) lu_status_kernel(int batch, const int* __restrict__ flags, const int* __restrict__ stA,
                                                        const int* __restrict__ stB, const int* __restrict__ scaleA, const int* __restrict__ scaleB,
                                                        int* __restrict__ scaleX, int* __restrict__ status) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= batch) return;
  scaleX[b] = scaleB[b] - scaleA[b];
  int st = 0;
  if (stA[b] || stB[b]) st = 3;                 // malformed input number
  else if (flags[b] & 1) st = 1;                // singular to working precision
  else if (flags[b] & 6) st = 2;                // a pivot below 2^-26 of the scaled matrix: not invertible in this format
  if (status) status[b] = st;
}

size_t lu_workspace_bytes(int N, int nrhs, int batch) {
  return FxC::bytes((size_t)N * N * batch) + FxC::bytes((size_t)N * nrhs * batch) + FxC::bytes((size_t)N * batch) +
         sizeof(int) * ((size_t)N * batch + 16 * (size_t)batch) + (1u << 16);
}

int lu_solve_device(int N, int nrhs, int batch, int prec, const void* A_api, const void* B_api, void* X_api, void* ws, size_t ws_bytes,
                    int* status_dev, cudaStream_t s) {
  if (ws_bytes < lu_workspace_bytes(N, nrhs, batch)) return ZKD_ERR_WORKSPACE;
  char* w = (char*)ws;
  auto take = [&](size_t bytes) { char* p = w; w += (bytes + 255) / 256 * 256; return p; };
  int32_t* A = (int32_t*)take(FxC::bytes((size_t)N * N * batch));
  int32_t* B = (int32_t*)take(FxC::bytes((size_t)N * nrhs * batch));
  int32_t* invd = (int32_t*)take(FxC::bytes((size_t)N * batch));
  int* perm = (int*)take(sizeof(int) * (size_t)N * batch);
  int* scaleA = (int*)take(sizeof(int) * 2 * batch);
  int* scaleB = (int*)take(sizeof(int) * 2 * batch);
  int* stA = (int*)take(sizeof(int) * batch);
  int* stB = (int*)take(sizeof(int) * batch);
  int* flags = (int*)take(sizeof(int) * batch);
  int* scaleX = (int*)take(sizeof(int) * batch);
  ZKD_TRY(ingest_general(N, N, batch, A_api, A, scaleA, stA, s, prec));
  ZKD_TRY(ingest_general(N, nrhs, batch, B_api, B, scaleB, stB, s, prec));
  ZKD_TRY(lu_factor(N, batch, A, perm, invd, flags, s));
  ZKD_TRY(lu_solve(N, nrhs, batch, 0, A, perm, invd, B, flags, s));
  lu_status_kernel<<<(batch + 127) / 128, 128, 0, s>>>(batch, flags, stA, stB, scaleA, scaleB, scaleX, status_dev);
  count_launch();
  ZKD_TRY(launch_check());
  return fxc_to_api_scaled((size_t)N * nrhs * batch, B, X_api, scaleX, (size_t)N * nrhs, s, prec);
}

}  // namespace zkd

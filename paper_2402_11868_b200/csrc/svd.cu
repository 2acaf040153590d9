// svd.cu — kernels of the singular value decomposition (ZKCM_CUS ships "Hermitian
// matrix diagonalization and singular value decomposition": ZKCM_QC switches both).
//
// Route: the SVD of A (M x N) is read off the Hermitian eigendecomposition of the Jordan-Wielandt matrix
//     H = [[0, A], [A^H, 0]]   ((M+N) x (M+N)):  eigenvalues +-sigma_j with eigenvectors (u_j; +-v_j)/sqrt(2), and |M - N| +
//     2 (K - rank) zeros whose eigenvectors span null(A^H) (+) null(A),
// which goes through the SAME hot path (S1 .. S5: fp64 seed, correction-equation RQI, cluster recursion); singular values
// come out to ABSOLUTE accuracy 2^-(P+2) ||A|| - tiny Schmidt weights are resolved, which A^H A would square away.
// This file holds what is specific to the SVD: general (non-Hermitian) ingest, building H, reading (U, S, V) off the sorted
// eigenpairs, normalisation / phase of the pairs.  The host driver is svd_device() in pipeline.cu.
#include "blocks.h"
#include "fx_api.cuh"
#include "fx_funcs.cuh"
#include "timing.h"

namespace zkd {

constexpr int kNoExpG = (int)0x80808080;

// ---- S0 for a general complex M x N matrix: scale = -(max exponent over ALL entries) - 2 -----------------------------------------
__global__ void __launch_bounds__(256) maxexp_general_kernel(size_t per_reals, const uint8_t* __restrict__ A, int* __restrict__ rawmax,
                                                             int* __restrict__ status, int prec) {
  const int rb = 16 + (prec >> 3);
  __shared__ int s_max, s_bad;
  const int b = blockIdx.y;
  if (threadIdx.x == 0) { s_max = kNoExpG; s_bad = 0; }
  __syncthreads();
  const uint8_t* Ab = A + (size_t)b * per_reals * rb;
  int mx = kNoExpG;
  bool bad = false;
  for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < per_reals; e += (size_t)gridDim.x * blockDim.x) {
    int64_t ex;
    if (api_real_exp(Ab + e * rb, &ex, &bad, prec)) {
      const int ec = ex > (1 << 30) ? (1 << 30) : ex < -(1 << 30) ? -(1 << 30) : (int)ex;
      if (ec > mx) mx = ec;
    }
  }
  if (mx != kNoExpG) atomicMax(&s_max, mx);
  if (bad) s_bad = 1;
  __syncthreads();
  if (threadIdx.x == 0) {
    if (s_max != kNoExpG) atomicMax(&rawmax[b], s_max);
    if (s_bad) atomicOr(&status[b], 3);
  }
}

__global__ void __launch_bounds__(128) ingest_general_kernel(size_t per, int batch, const uint8_t* __restrict__ A, const int* __restrict__ rawmax,
                                                             int* __restrict__ scale, int32_t* __restrict__ dst, int* __restrict__ status, int prec) {
  const int rb = 16 + (prec >> 3);
  const size_t count = per * batch;
  const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= 2 * count) return;
  const int part = (int)(t / count);
  const size_t e = t % count;
  const int b = (int)(e / per);
  int32_t d[ND];
  fx_zero(d);
  const int sc = rawmax[b] == kNoExpG ? 0 : -rawmax[b] - 2;
  if (part == 0 && e == (size_t)b * per) scale[b] = sc;
  if (status[b] == 0) {
    const int st = api_real_to_fx(A + (e * 2 + part) * rb, sc, false, d, prec);
    if (st) { atomicOr(&status[b], 3); fx_zero(d); }
  }
  fx_store(dst + (part ? (size_t)ND * count : 0), count, e, d);
}

int ingest_general(int M, int N, int batch, const void* A_api, int32_t* A_fx, int* scale, int* status, cudaStream_t s, int prec) {
  KtScope kt_scope(KC_IO, s);
  int* rawmax = scale + batch;
  ZKD_CUDA_TRY(cudaMemsetAsync(rawmax, 0x80, sizeof(int) * batch, s));
  ZKD_CUDA_TRY(cudaMemsetAsync(status, 0, sizeof(int) * batch, s));
  const size_t per = (size_t)M * N;
  unsigned chunks = (unsigned)std::min<size_t>((2 * per + 255) / 256, (size_t)std::max(1, 592 / batch));
  maxexp_general_kernel<<<dim3(chunks, batch), 256, 0, s>>>(2 * per, (const uint8_t*)A_api, rawmax, status, prec);
  const size_t t = 2 * per * batch;
  ingest_general_kernel<<<(unsigned)((t + 127) / 128), 128, 0, s>>>(per, batch, (const uint8_t*)A_api, rawmax, scale, A_fx, status, prec);
  count_launch(2);
  return launch_check();
}

// ---- H = [[0, A], [A^H, 0]] -------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) jw_build_kernel(int M, int N, int batch, const int32_t* __restrict__ A, int32_t* __restrict__ H) {
  const int n = M + N;
  const size_t per = (size_t)n * n, count = per * batch, acount = (size_t)M * N * batch;
  const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= 2 * count) return;
  const int part = (int)(t / count);
  const size_t e = t % count;
  const int b = (int)(e / per), i = (int)((e % per) / n), j = (int)(e % n);
  int32_t d[ND];
  fx_zero(d);
  if (i < M && j >= M) {
    fx_load(d, A + (part ? (size_t)ND * acount : 0), acount, (size_t)b * M * N + (size_t)i * N + (j - M));
  } else if (i >= M && j < M) {
    fx_load(d, A + (part ? (size_t)ND * acount : 0), acount, (size_t)b * M * N + (size_t)j * N + (i - M));
    if (part) { int32_t t2[ND]; fx_neg(t2, d);
#pragma unroll
      for (int k = 0; k < ND; ++k) d[k] = t2[k]; }
  }
  fx_store(H + (part ? (size_t)ND * count : 0), count, e, d);
}
int jw_build(int M, int N, int batch, const int32_t* A_fx, int32_t* H_fx, cudaStream_t s) {
  KtScope kt_scope(KC_OTHER, s);
  const size_t t = 2 * (size_t)(M + N) * (M + N) * batch;
  jw_build_kernel<<<(unsigned)((t + 255) / 256), 256, 0, s>>>(M, N, batch, A_fx, H_fx);
  count_launch();
  return launch_check();
}

// ---- rank_of[b][col] -> col_of[b][rank];  r[b] = number of eigenvalues above 2^(zero_msb - 812) ------------------------------------------
__global__ void __launch_bounds__(128) svd_plan_kernel(int n, int batch, const int* __restrict__ rank, const int32_t* __restrict__ lam_sorted,
                                                       int zero_msb, int* __restrict__ col_of, int* __restrict__ r_out) {
  const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= (size_t)n * batch) return;
  const int b = (int)(t / n), j = (int)(t % n);
  col_of[(size_t)b * n + rank[t]] = j;
  int32_t d[ND];
  fx_load(d, lam_sorted, (size_t)n * batch, t);
  if (d[ND - 1] >= 0 && fx_msb(d) > zero_msb) atomicAdd(r_out + b, 1);
}
int svd_plan(int n, int batch, const int* rank, const int32_t* lam_sorted, int zero_msb, int* col_of, int* r_out, cudaStream_t s) {
  KtScope kt_scope(KC_OTHER, s);
  ZKD_CUDA_TRY(cudaMemsetAsync(r_out, 0, sizeof(int) * batch, s));
  svd_plan_kernel<<<(unsigned)(((size_t)n * batch + 127) / 128), 128, 0, s>>>(n, batch, rank, lam_sorted, zero_msb, col_of, r_out);
  count_launch();
  return launch_check();
}

// ---- (U, V, S) of the pairs with nonzero sigma: pair i < r[b] <- eigenvector of rank n-1-i (upper M rows -> u, lower N rows -> v) -------
// S gets max(0, lambda) for ALL K (the zero cluster's values are at the noise level).  Columns i >= r[b] of U, V are zeroed here and
// filled by the null-space step.
__global__ void __launch_bounds__(256) svd_gather_kernel(int M, int N, int batch, const int32_t* __restrict__ X, const int* __restrict__ col_of,
                                                         const int* __restrict__ r, const int32_t* __restrict__ lam_sorted,
                                                         int32_t* __restrict__ U, int32_t* __restrict__ V, int32_t* __restrict__ S) {
  const int n = M + N, K = M < N ? M : N;
  const size_t xcount = (size_t)n * n * batch, ucount = (size_t)M * K * batch, vcount = (size_t)N * K * batch;
  const size_t per = (size_t)n * K;  // rows of U then rows of V
  const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= 2 * per * batch) return;
  const int part = (int)(t / (per * batch));
  const size_t e = t % (per * batch);
  const int b = (int)(e / per), row = (int)((e % per) / K), i = (int)(e % K);
  int32_t d[ND];
  fx_zero(d);
  if (i < r[b]) {
    const int col = col_of[(size_t)b * n + (n - 1 - i)];
    fx_load(d, X + (part ? (size_t)ND * xcount : 0), xcount, (size_t)b * n * n + (size_t)row * n + col);
  }
  if (row < M) fx_store(U + (part ? (size_t)ND * ucount : 0), ucount, (size_t)b * M * K + (size_t)row * K + i, d);
  else fx_store(V + (part ? (size_t)ND * vcount : 0), vcount, (size_t)b * N * K + (size_t)(row - M) * K + i, d);
  if (part == 0 && row == 0) {
    fx_load(d, lam_sorted, (size_t)n * batch, (size_t)b * n + (n - 1 - i));
    if (d[ND - 1] < 0) fx_zero(d);
    fx_store(S, (size_t)K * batch, (size_t)b * K + i, d);
  }
}
int svd_gather(int M, int N, int batch, const int32_t* X, const int* col_of, const int* r, const int32_t* lam_sorted, int32_t* U, int32_t* V,
               int32_t* S, cudaStream_t s) {
  KtScope kt_scope(KC_OTHER, s);
  const int K = M < N ? M : N;
  const size_t t = 2 * (size_t)(M + N) * K * batch;
  svd_gather_kernel<<<(unsigned)((t + 255) / 256), 256, 0, s>>>(M, N, batch, X, col_of, r, lam_sorted, U, V, S);
  count_launch();
  return launch_check();
}

// ---- null-space step: Z[v] (n x d0) <- the eigenvectors of ranks r .. r + d0 - 1 of matrix mats[v] (the zero cluster) --------------------
__global__ void __launch_bounds__(256) svd_zgather_kernel(int n, int batch, int d0, int r, int g, const int* __restrict__ mats,
                                                          const int32_t* __restrict__ X, const int* __restrict__ col_of, int32_t* __restrict__ Z) {
  const size_t xcount = (size_t)n * n * batch, zcount = (size_t)n * d0 * g;
  const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= 2 * zcount) return;
  const int part = (int)(t / zcount);
  const size_t e = t % zcount;
  const int v = (int)(e / ((size_t)n * d0)), row = (int)((e % ((size_t)n * d0)) / d0), c = (int)(e % d0);
  const int b = mats[v];
  const int col = col_of[(size_t)b * n + r + c];
  int32_t d[ND];
  fx_load(d, X + (part ? (size_t)ND * xcount : 0), xcount, (size_t)b * n * n + (size_t)row * n + col);
  fx_store(Z + (part ? (size_t)ND * zcount : 0), zcount, e, d);
}
int svd_zgather(int n, int batch, int d0, int r, int g, const int* mats_dev, const int32_t* X, const int* col_of, int32_t* Z, cudaStream_t s) {
  KtScope kt_scope(KC_OTHER, s);
  const size_t t = 2 * (size_t)n * d0 * g;
  svd_zgather_kernel<<<(unsigned)((t + 255) / 256), 256, 0, s>>>(n, batch, d0, r, g, mats_dev, X, col_of, Z);
  count_launch();
  return launch_check();
}

// ---- complex FX array >> bits (arithmetic) ----------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) fxc_shr_kernel(size_t reals, int32_t* __restrict__ X, int bits) {
  const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= reals) return;
  const size_t count = reals / 2;
  int32_t* p = X + (e / count) * (size_t)ND * count;
  int32_t d[ND];
  fx_load(d, p, count, e % count);
  fx_shr(d, bits);
  fx_store(p, count, e % count, d);
}
int fxc_shr(size_t count, int32_t* X, int bits, cudaStream_t s) {
  KtScope kt_scope(KC_OTHER, s);
  fxc_shr_kernel<<<(unsigned)((2 * count + 255) / 256), 256, 0, s>>>(2 * count, X, bits);
  count_launch();
  return launch_check();
}

// ---- normalise the pair (u_j, v_j) and fix its phase: one warp per (matrix, j) -------------------------------------------------------------------
// u <- u f / ||u||, v <- v f / ||v|| with f = conj(v_k*) / |v_k*|, k* = first index of max |v_k| (the convention of the oracle: the first
// component of largest modulus of v_j is real positive).  Each of u, v is normalised on its own: an eigenvector of H that carries a
// little of its mirror (u; -v) has ||u|| != ||v|| but exact directions.
__device__ __forceinline__ bool fx_less_d(const int32_t (&a)[ND], const int32_t (&b)[ND]) {
  bool lt = false, decided = false;
#pragma unroll
  for (int k = ND - 1; k >= 0; --k)
    if (!decided && a[k] != b[k]) { lt = a[k] < b[k]; decided = true; }
  return lt;
}
__global__ void __launch_bounds__(128) svd_phase_kernel(int M, int N, int batch, int32_t* __restrict__ U, int32_t* __restrict__ V) {
  __shared__ int32_t s_f[4][4][ND];  // per warp: fu_re, fu_im, fv_re, fv_im
  const int K = M < N ? M : N;
  const size_t w = ((size_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31, wl = threadIdx.x >> 5;
  const bool active = w < (size_t)K * batch;
  const int b = active ? (int)(w / K) : 0, j = active ? (int)(w % K) : 0;
  const size_t ucount = (size_t)M * K * batch, vcount = (size_t)N * K * batch;
  int32_t* Ur = U; int32_t* Ui = U + (size_t)ND * ucount;
  int32_t* Vr = V; int32_t* Vi = V + (size_t)ND * vcount;
  int64_t accu[FXP_NACC], accv[FXP_NACC];
  fxp_zero(accu); fxp_zero(accv);
  int32_t best[ND];
  fx_zero(best);
  best[ND - 1] = -1;
  int bestk = 0x7fffffff;
  if (active) {
    for (int k = lane; k < M; k += 32) {
      const size_t e = (size_t)b * M * K + (size_t)k * K + j;
      int32_t a[ND];
      fx_load(a, Ur, ucount, e); fx_mac<false>(accu, a, a);
      fx_load(a, Ui, ucount, e); fx_mac<false>(accu, a, a);
      fxp_relax(accu);
    }
    for (int k = lane; k < N; k += 32) {
      const size_t e = (size_t)b * N * K + (size_t)k * K + j;
      int32_t a[ND], m2[ND];
      int64_t acc[FXP_NACC];
      fxp_zero(acc);
      fx_load(a, Vr, vcount, e); fx_mac<false>(acc, a, a); fx_mac<false>(accv, a, a);
      fx_load(a, Vi, vcount, e); fx_mac<false>(acc, a, a); fx_mac<false>(accv, a, a);
      fxp_relax(accv);
      fxp_finish(m2, acc);
      if (fx_less_d(best, m2)) {
#pragma unroll
        for (int q = 0; q < ND; ++q) best[q] = m2[q];
        bestk = k;
      }
    }
  }
  warp_sum_cols(accu);
  warp_sum_cols(accv);
  for (int off = 16; off > 0; off >>= 1) {
    int32_t o[ND];
#pragma unroll
    for (int q = 0; q < ND; ++q) o[q] = __shfl_xor_sync(0xffffffffu, best[q], off);
    const int ok = __shfl_xor_sync(0xffffffffu, bestk, off);
    const bool take = fx_less_d(best, o) || (!fx_less_d(o, best) && ok < bestk);
    if (take) {
#pragma unroll
      for (int q = 0; q < ND; ++q) best[q] = o[q];
      bestk = ok;
    }
  }
  bestk = __shfl_sync(0xffffffffu, bestk, 0);
  if (active && lane == 0) {
    int32_t nu2[ND], nv2[ND], yu[ND], yv[ND], yk[ND];
    fxp_finish(nu2, accu);
    fxp_finish(nv2, accv);
    int32_t f[4][ND];
    if (fx_msb(nv2) == 0 || fx_msb(nu2) == 0 || fx_msb(best) == 0) {  // a zero column (cannot happen for eigenvector parts): leave it
#pragma unroll
      for (int q = 0; q < ND; ++q) { f[0][q] = 0; f[1][q] = 0; f[2][q] = 0; f[3][q] = 0; }
      f[0][ND - 1] = 1; f[2][ND - 1] = 1;
    } else {
      fx_rsqrt(yu, nu2);   // 1/||u||
      fx_rsqrt(yv, nv2);   // 1/||v||
      fx_rsqrt(yk, best);  // 1/|v_k*|
      const size_t e = (size_t)b * N * K + (size_t)bestk * K + j;
      int32_t zr[ND], zi[ND], pr[ND], pi[ND], t[ND];
      fx_load(zr, Vr, vcount, e); fx_load(zi, Vi, vcount, e);
      fx_mul(pr, zr, yk);                   // Re conj(v_k*)/|v_k*|
      fx_neg(t, zi); fx_mul(pi, t, yk);     // Im
      fx_mul(f[0], pr, yu); fx_mul(f[1], pi, yu);
      fx_mul(f[2], pr, yv); fx_mul(f[3], pi, yv);
    }
#pragma unroll
    for (int q = 0; q < ND; ++q) { s_f[wl][0][q] = f[0][q]; s_f[wl][1][q] = f[1][q]; s_f[wl][2][q] = f[2][q]; s_f[wl][3][q] = f[3][q]; }
  }
  __syncwarp();
  if (!active) return;
#pragma unroll 1
  for (int side = 0; side < 2; ++side) {
    int32_t fr[ND], fi[ND];
#pragma unroll
    for (int q = 0; q < ND; ++q) { fr[q] = s_f[wl][2 * side][q]; fi[q] = s_f[wl][2 * side + 1][q]; }
    const int rows = side ? N : M;
    int32_t* Xr = side ? Vr : Ur; int32_t* Xi = side ? Vi : Ui;
    const size_t cnt = side ? vcount : ucount;
    for (int k = lane; k < rows; k += 32) {
      const size_t e = (size_t)b * rows * K + (size_t)k * K + j;
      int32_t xr[ND], xi[ND], o[ND], o2[ND];
      fx_load(xr, Xr, cnt, e); fx_load(xi, Xi, cnt, e);
      int64_t acc[FXP_NACC];
      fxp_zero(acc);
      fx_mac<false>(acc, xr, fr); fx_mac<true>(acc, xi, fi);
      fxp_finish(o, acc);
      fxp_zero(acc);
      fx_mac<false>(acc, xr, fi); fx_mac<false>(acc, xi, fr);
      fxp_finish(o2, acc);
      if (side == 1 && k == bestk) fx_zero(o2);
      fx_store(Xr, cnt, e, o);
      fx_store(Xi, cnt, e, o2);
    }
  }
}
int svd_phase(int M, int N, int batch, int32_t* U, int32_t* V, cudaStream_t s) {
  KtScope kt_scope(KC_OTHER, s);
  const int K = M < N ? M : N;
  const size_t warps = (size_t)K * batch;
  svd_phase_kernel<<<(unsigned)((warps * 32 + 127) / 128), 128, 0, s>>>(M, N, batch, U, V);
  count_launch();
  return launch_check();
}

}  // namespace zkd

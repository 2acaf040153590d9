// finalize.cu — S0 (scale + Hermitian ingest), S5 plumbing (cluster sub-problems in and out) and S6 (sort,
// phase-normalise, export).  Readings A5/A9/A15 of DESIGN.md: upper triangle authoritative; ascending order; unit
// 2-norm; the first component of largest modulus is made real positive.
#include <algorithm>

#include "blocks.h"
#include "fx_api.cuh"
#include "fx_funcs.cuh"
#include "timing.h"

namespace zkd {

// ---- S0 ------------------------------------------------------------------------------------------------------------
// per matrix: scale = -(max exponent over the upper triangle) - 2, so that max |a_ij| 2^scale lies in [1/8, 1/4).
// Pass 1 (grid: chunks x batch): rawmax[b] <- max exponent (clamped to +-2^30; kNoExp when every entry is zero),
// status[b] |= 3 on a malformed number.  The ingest kernel turns rawmax into the scale.
constexpr int kNoExp = (int)0x80808080;  // what cudaMemsetAsync(.., 0x80, ..) leaves: below every clamped exponent
__global__ void __launch_bounds__(256) maxexp_kernel(int N, const uint8_t* __restrict__ A, int* __restrict__ rawmax, int* __restrict__ status,
                                                     int prec) {
  const int kApiRealBytes = 16 + (prec >> 3);
  __shared__ int s_max, s_bad;
  const int b = blockIdx.y;
  if (threadIdx.x == 0) { s_max = kNoExp; s_bad = 0; }
  __syncthreads();
  const uint8_t* Ab = A + (size_t)b * N * N * 2 * kApiRealBytes;
  int mx = kNoExp;
  bool bad = false;
  for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < (size_t)N * N; e += (size_t)gridDim.x * blockDim.x) {
    const int i = (int)(e / N), j = (int)(e % N);
    if (i > j) continue;
    int64_t ex;
    for (int part = 0; part < (i < j ? 2 : 1); ++part) {
      if (api_real_exp(Ab + (e * 2 + part) * kApiRealBytes, &ex, &bad, prec)) {
        const int ec = ex > (1 << 30) ? (1 << 30) : ex < -(1 << 30) ? -(1 << 30) : (int)ex;
        if (ec > mx) mx = ec;
      }
    }
  }
  if (mx != kNoExp) atomicMax(&s_max, mx);
  if (bad) s_bad = 1;
  __syncthreads();
  if (threadIdx.x == 0) {
    if (s_max != kNoExp) atomicMax(&rawmax[b], s_max);
    if (s_bad) atomicOr(&status[b], 3);
  }
}
__device__ __forceinline__ int scale_from_rawmax(int rawmax) { return rawmax == kNoExp ? 0 : -rawmax - 2; }

__global__ void __launch_bounds__(128) ingest_kernel(int N, int batch, const uint8_t* __restrict__ A, const int* __restrict__ rawmax,
                                                     int* __restrict__ scale, int32_t* __restrict__ dst, int* __restrict__ status, int prec) {
  const int kApiRealBytes = 16 + (prec >> 3);
  const size_t per = (size_t)N * N, count = per * batch;
  const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= 2 * count) return;
  const int part = (int)(t / count);
  const size_t e = t % count;
  const int b = (int)(e / per), i = (int)((e % per) / N), j = (int)(e % N);
  int32_t d[ND];
  fx_zero(d);
  const int sc = scale_from_rawmax(rawmax[b]);
  if (part == 0 && e == (size_t)b * per) scale[b] = sc;  // for the export
  if (!(part == 1 && i == j) && status[b] == 0) {
    const int si = i <= j ? i : j, sj = i <= j ? j : i;
    const uint8_t* s = A + (((size_t)b * per + (size_t)si * N + sj) * 2 + part) * kApiRealBytes;
    const int st = api_real_to_fx(s, sc, part == 1 && i > j, d, prec);
    if (st) { atomicOr(&status[b], 3); fx_zero(d); }
  }
  fx_store(dst + (part ? (size_t)ND * count : 0), count, e, d);
}

int ingest_herm(int N, int batch, const void* A_api, int32_t* A_fx, int* scale /* 2 * batch ints */, int* status, cudaStream_t s, int prec) {
  KtScope kt_scope(KC_IO, s);
  int* rawmax = scale + batch;
  ZKD_CUDA_TRY(cudaMemsetAsync(rawmax, 0x80, sizeof(int) * batch, s));
  ZKD_CUDA_TRY(cudaMemsetAsync(status, 0, sizeof(int) * batch, s));
  // enough CTAs per matrix to fill the machine when the batch is small
  const size_t per = (size_t)N * N;
  unsigned chunks = (unsigned)std::min<size_t>((per + 255) / 256, (size_t)std::max(1, 592 / batch));
  maxexp_kernel<<<dim3(chunks, batch), 256, 0, s>>>(N, (const uint8_t*)A_api, rawmax, status, prec);
  const size_t t = 2 * (size_t)N * N * batch;
  ingest_kernel<<<(unsigned)((t + 127) / 128), 128, 0, s>>>(N, batch, (const uint8_t*)A_api, rawmax, scale, A_fx, status, prec);
  count_launch(2);
  return launch_check();
}

// ---- S5 plumbing -----------------------------------------------------------------------------------------------------
// value / m for a small positive integer m (floor), canonical in and out
__device__ __forceinline__ void fx_div_small(int32_t (&d)[ND], int m) {
  const bool neg = d[ND - 1] < 0;
  if (neg) { int32_t t[ND]; fx_neg(t, d);
#pragma unroll
    for (int k = 0; k < ND; ++k) d[k] = t[k]; }
  int64_t rem = 0;
#pragma unroll
  for (int k = ND - 1; k >= 0; --k) {
    const int64_t cur = (rem << DB) + d[k];
    d[k] = (int32_t)(cur / m);
    rem = cur % m;
  }
  if (neg) { int32_t t[ND]; fx_neg(t, d);
#pragma unroll
    for (int k = 0; k < ND; ++k) d[k] = t[k]; }
}

// one CTA per sub-problem: H = herm(S block) - cbar I, scaled by 2^k so that max|h| has msb 810
__global__ void __launch_bounds__(128) sub_gather_kernel(int n, int nb, int m, const SubProblem* __restrict__ subs,
                                                         const int32_t* __restrict__ S, int32_t* __restrict__ H,
                                                         int32_t* __restrict__ cbar, int* __restrict__ kshift,
                                                         int* __restrict__ degenerate, int degenerate_msb_base,
                                                         const int* __restrict__ noise_parent, int* __restrict__ noise_child,
                                                         int* __restrict__ floor_child, int min_split_msb, int nsub) {
  __shared__ int32_t s_c[ND];
  __shared__ int s_msb;
  const int p = blockIdx.x;
  const SubProblem sp = subs[p];
  // entries of S are known to ~2^-812 in the units of depth 0, i.e. to 2^(noise - 812) in the units of this level
  const int noise = noise_parent ? noise_parent[sp.b] : 0;
  // blocks whose spread is below min_split_msb are also reported "degenerate" (S4h: not worth splitting now)
  const int degenerate_msb = max(degenerate_msb_base + noise, min_split_msb - 1);
  const size_t per = (size_t)n * n, count = per * nb;
  const size_t hcount = (size_t)m * m * nsub;
  const int32_t* Sr = S;
  const int32_t* Si = S + (size_t)ND * count;
  if (threadIdx.x == 0) {
    int32_t acc[ND];
    fx_zero(acc);
    for (int j = 0; j < m; ++j) {
      int32_t d[ND], r[ND];
      fx_load(d, Sr, count, (size_t)sp.b * per + (size_t)(sp.col0 + j) * n + (sp.col0 + j));
      fx_add(r, acc, d);
#pragma unroll
      for (int k = 0; k < ND; ++k) acc[k] = r[k];
    }
    fx_div_small(acc, m);
#pragma unroll
    for (int k = 0; k < ND; ++k) s_c[k] = acc[k];
    fx_store(cbar, (size_t)nsub, (size_t)p, acc);
    s_msb = 0;
  }
  __syncthreads();
  int32_t c[ND];
#pragma unroll
  for (int k = 0; k < ND; ++k) c[k] = s_c[k];
  // pass 1: msb of H - cbar I ; pass 2: scale and store
  for (int pass = 0; pass < 2; ++pass) {
    const int k_sh = pass ? (810 - s_msb) : 0;
    const bool deg = pass && (s_msb <= degenerate_msb);
    int mymsb = 0;
    for (int e = threadIdx.x; e < m * m * 2; e += blockDim.x) {
      const int part = e / (m * m), ij = e % (m * m), i = ij / m, j = ij % m;
      // H must be Hermitian to the last bit (a 1-ulp asymmetry, scaled by 2^k, would break the orthogonality of the
      // sub-level eigenvectors at that level): the upper triangle is computed, the lower one is its exact conjugate.
      const int iu = i <= j ? i : j, ju = i <= j ? j : i;
      const size_t eij = (size_t)sp.b * per + (size_t)(sp.col0 + iu) * n + (sp.col0 + ju);
      const size_t eji = (size_t)sp.b * per + (size_t)(sp.col0 + ju) * n + (sp.col0 + iu);
      int32_t a[ND], bb[ND], h[ND];
      if (part == 0) {
        fx_load(a, Sr, count, eij); fx_load(bb, Sr, count, eji);
        fx_add(h, a, bb);
      } else {
        fx_load(a, Si, count, eij); fx_load(bb, Si, count, eji);
        fx_sub(h, a, bb);
      }
      fx_half(a, h);  // (S_ij + conj(S_ji)) / 2 for i <= j
      if (part == 1 && i > j) { fx_neg(h, a);
#pragma unroll
        for (int k = 0; k < ND; ++k) a[k] = h[k]; }
      if (part == 0 && i == j) { fx_sub(h, a, c);
#pragma unroll
        for (int k = 0; k < ND; ++k) a[k] = h[k]; }
      if (part == 1 && i == j) fx_zero(a);
      if (!pass) {
        mymsb = max(mymsb, fx_msb(a));
      } else {
        if (deg) {
          fx_zero(a);
          if (part == 0 && i == j) fx_from_double(a, ((double)j - 0.5 * (m - 1)) / (4.0 * m));
        } else if (k_sh >= 0) {
          fx_shl(a, k_sh);
        } else {
          fx_shr(a, -k_sh);
        }
        fx_store(H + (part ? (size_t)ND * hcount : 0), hcount, (size_t)p * m * m + ij, a);
      }
    }
    if (!pass) atomicMax(&s_msb, mymsb);
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    kshift[p] = 810 - s_msb;
    degenerate[p] = s_msb <= degenerate_msb ? 1 : 0;
    noise_child[p] = noise + max(0, 810 - s_msb);
    if (floor_child) floor_child[p] = degenerate_msb + (810 - s_msb);  // the same noise level in the scaled units of H
  }
}
int sub_gather(int n, int nb, int m, int nsub, const SubProblem* subs_dev, const int32_t* S, int32_t* H, int32_t* cbar, int* kshift,
               int* degenerate, int degenerate_msb, const int* noise_parent, int* noise_child, int* floor_child, int min_split_msb,
               cudaStream_t s) {
  KtScope kt_scope(KC_OTHER, s);
  sub_gather_kernel<<<nsub, 128, 0, s>>>(n, nb, m, subs_dev, S, H, cbar, kshift, degenerate, degenerate_msb, noise_parent,
                                         noise_child, floor_child, min_split_msb, nsub);
  count_launch();
  return launch_check();
}

// Um := identity on every cluster block
__global__ void __launch_bounds__(256) identity_blocks_kernel(size_t count, int n, int32_t* __restrict__ Um) {
  const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= 2 * count) return;
  const int part = (int)(t / count);
  const size_t e = t % count;
  const int i = (int)((e % ((size_t)n * n)) / n), j = (int)(e % n);
  int32_t d[ND];
  fx_zero(d);
  if (part == 0 && i == j) d[ND - 1] = 1;
  fx_store(Um + (part ? (size_t)ND * count : 0), count, e, d);
}
int identity_blocks(int n, int nb, int32_t* Um, cudaStream_t s) {
  KtScope kt_scope(KC_OTHER, s);
  const size_t count = (size_t)n * n * nb;
  identity_blocks_kernel<<<(unsigned)((2 * count + 255) / 256), 256, 0, s>>>(count, n, Um);
  count_launch();
  return launch_check();
}

__global__ void __launch_bounds__(128) sub_scatter_kernel(int n, int nb, int m, int nsub, const SubProblem* __restrict__ subs,
                                                          const int32_t* __restrict__ U, const int32_t* __restrict__ lam_sub,
                                                          const int32_t* __restrict__ cbar, const int* __restrict__ kshift,
                                                          const int* __restrict__ degenerate, int32_t* __restrict__ Um,
                                                          int32_t* __restrict__ theta) {
  const int p = blockIdx.x;
  if (degenerate[p]) return;  // keep the identity block and the Rayleigh quotients already in theta
  const SubProblem sp = subs[p];
  const size_t per = (size_t)n * n, count = per * nb, hcount = (size_t)m * m * nsub;
  for (int e = threadIdx.x; e < m * m * 2; e += blockDim.x) {
    const int part = e / (m * m), ij = e % (m * m), i = ij / m, j = ij % m;
    int32_t d[ND];
    fx_load(d, U + (part ? (size_t)ND * hcount : 0), hcount, (size_t)p * m * m + ij);
    fx_store(Um + (part ? (size_t)ND * count : 0), count, (size_t)sp.b * per + (size_t)(sp.col0 + i) * n + (sp.col0 + j), d);
  }
  const int k = kshift[p];
  for (int j = threadIdx.x; j < m; j += blockDim.x) {
    int32_t l[ND], c[ND], r[ND];
    fx_load(l, lam_sub, (size_t)m * nsub, (size_t)p * m + j);
    if (k >= 0) fx_shr(l, k); else fx_shl(l, -k);
    fx_load(c, cbar, (size_t)nsub, (size_t)p);
    fx_add(r, c, l);
    fx_store(theta, (size_t)n * nb, (size_t)sp.b * n + sp.col0 + j, r);
  }
}
int sub_scatter(int n, int nb, int m, int nsub, const SubProblem* subs_dev, const int32_t* U, const int32_t* lam_sub,
                const int32_t* cbar, const int* kshift, const int* degenerate, int32_t* Um, int32_t* theta, cudaStream_t s) {
  KtScope kt_scope(KC_OTHER, s);
  sub_scatter_kernel<<<nsub, 128, 0, s>>>(n, nb, m, nsub, subs_dev, U, lam_sub, cbar, kshift, degenerate, Um, theta);
  count_launch();
  return launch_check();
}

__global__ void __launch_bounds__(128) fold_sub_stats_kernel(int nsub, const SubProblem* __restrict__ subs, const int* __restrict__ kshift,
                                                             const int* __restrict__ degenerate, const int* __restrict__ pm_sub,
                                                             int* __restrict__ pm_parent, int nb_parent) {
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= nsub || degenerate[p]) return;
  const int b = subs[p].b;
  const int r = pm_sub[p] - kshift[p];  // the sub-problem was scaled by 2^kshift
  if (r > 0) atomicMax(pm_parent + b, r);
  if (pm_sub[nsub + p] > 0) atomicMax(pm_parent + nb_parent + b, pm_sub[nsub + p]);
}
int fold_sub_stats(int nsub, const SubProblem* subs_dev, const int* kshift, const int* degenerate, const int* pm_sub, int* pm_parent,
                   int nb_parent, cudaStream_t s) {
  KtScope kt_scope(KC_OTHER, s);
  fold_sub_stats_kernel<<<(nsub + 127) / 128, 128, 0, s>>>(nsub, subs_dev, kshift, degenerate, pm_sub, pm_parent, nb_parent);
  count_launch();
  return launch_check();
}

// S4h: one CTA per sub-problem
__global__ void __launch_bounds__(128) split_scatter_kernel(int n, int nb, int m, int nsub, const SubProblem* __restrict__ subs,
                                                            const double2* __restrict__ V64, const int* __restrict__ sub_cl,
                                                            const int* __restrict__ sub_cle, const int* __restrict__ degenerate,
                                                            int32_t* __restrict__ Um, int* __restrict__ cl, int* __restrict__ cle) {
  const int p = blockIdx.x;
  if (degenerate[p]) return;
  const SubProblem sp = subs[p];
  const size_t per = (size_t)n * n, count = per * nb;
  for (int e = threadIdx.x; e < m * m; e += blockDim.x) {
    const int i = e / m, j = e % m;
    const double2 v = V64[(size_t)p * m * m + e];
    const size_t dst = (size_t)sp.b * per + (size_t)(sp.col0 + i) * n + (sp.col0 + j);
    int32_t d[ND];
    fx_from_double(d, v.x);
    fx_store(Um, count, dst, d);
    fx_from_double(d, v.y);
    fx_store(Um + (size_t)ND * count, count, dst, d);
  }
  for (int j = threadIdx.x; j < m; j += blockDim.x) {
    cl[(size_t)sp.b * n + sp.col0 + j] = sp.col0 + sub_cl[(size_t)p * m + j];
    cle[(size_t)sp.b * n + sp.col0 + j] = sp.col0 + sub_cle[(size_t)p * m + j];
  }
}
int split_scatter(int n, int nb, int m, int nsub, const SubProblem* subs_dev, const double2* V64, const int* sub_cl,
                  const int* sub_cle, const int* degenerate, int32_t* Um, int* cl, int* cle, cudaStream_t s) {
  KtScope kt_scope(KC_OTHER, s);
  split_scatter_kernel<<<nsub, 128, 0, s>>>(n, nb, m, nsub, subs_dev, V64, sub_cl, sub_cle, degenerate, Um, cl, cle);
  count_launch();
  return launch_check();
}

// ---- S6 ----------------------------------------------------------------------------------------------------------------
// a < b on canonical FX digits
__device__ __forceinline__ bool fx_less(const int32_t (&a)[ND], const int32_t (&b)[ND]) {
  bool lt = false, decided = false;
#pragma unroll
  for (int k = ND - 1; k >= 0; --k) {
    if (!decided && a[k] != b[k]) { lt = a[k] < b[k]; decided = true; }
  }
  return lt;
}

// rank[j] = number of eigenvalues that sort before lambda_j (ascending, stable); also writes lambda sorted.
// One WARP per eigenvalue: the lanes share the N comparisons (a thread per eigenvalue is a chain of N dependent 3-digit loads on
// a few hundred threads: 25 us at N = 16, 150 us at N = 256).
__global__ void __launch_bounds__(128) rank_kernel(int N, int batch, const int32_t* __restrict__ lam, int* __restrict__ rank,
                                                   int32_t* __restrict__ lam_sorted) {
  const size_t t = ((size_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (t >= (size_t)N * batch) return;  // the whole warp leaves together
  const int b = (int)(t / N), j = (int)(t % N);
  const size_t cnt = (size_t)N * batch;
  int32_t lj[ND];
  fx_load(lj, lam, cnt, t);
  int r = 0;
  // The top three digits (integer part and 56 fractional bits) decide almost every comparison; the remaining digits are walked
  // only on a tie.
  const int32_t* base = lam + (size_t)b * N;
  for (int i = lane; i < N; i += 32) {
    const int32_t d2 = base[(size_t)(ND - 1) * cnt + i], d1 = base[(size_t)(ND - 2) * cnt + i], d0 = base[(size_t)(ND - 3) * cnt + i];
    int cmp = d2 < lj[ND - 1] ? -1 : d2 > lj[ND - 1] ? 1 : 0;  // sign of (lambda_i - lambda_j)
    if (cmp == 0) cmp = d1 < lj[ND - 2] ? -1 : d1 > lj[ND - 2] ? 1 : 0;
    if (cmp == 0) cmp = d0 < lj[ND - 3] ? -1 : d0 > lj[ND - 3] ? 1 : 0;
    if (cmp == 0) {
#pragma unroll
      for (int k = ND - 4; k >= 0; --k) {
        if (cmp == 0) {
          const int32_t d = base[(size_t)k * cnt + i];
          cmp = d < lj[k] ? -1 : d > lj[k] ? 1 : 0;
        }
      }
    }
    r += cmp < 0 || (cmp == 0 && i < j);
  }
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) r += __shfl_xor_sync(0xffffffffu, r, off);
  if (lane == 0) rank[t] = r;
  // every lane holds lambda_j: lane k stores digit k
  if (lane < ND) {
    int32_t v = 0;
#pragma unroll
    for (int k = 0; k < ND; ++k)
      if (k == lane) v = lj[k];
    lam_sorted[(size_t)lane * cnt + (size_t)b * N + r] = v;
  }
}

// one warp per column: k* = first index of max |x_k|^2 (exact FX comparison), u = conj(x_k*) / |x_k*|,
// out[:, rank[j]] = x_j u, with Im out[k*] forced to zero.
__global__ void __launch_bounds__(128) phase_kernel(int N, int batch, const int32_t* __restrict__ X, const int* __restrict__ rank,
                                                    int32_t* __restrict__ out) {
  __shared__ int32_t s_u[4][2][ND];
  const size_t w = ((size_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31, wl = threadIdx.x >> 5;
  const bool active = w < (size_t)N * batch;
  const int b = active ? (int)(w / N) : 0, j = active ? (int)(w % N) : 0;
  const size_t per = (size_t)N * N, count = per * batch;
  const int32_t* Xr = X;
  const int32_t* Xi = X + (size_t)ND * count;
  // modulus^2 per lane-owned row, keep the best (largest, then smallest index)
  int32_t best[ND];
  fx_zero(best);
  best[ND - 1] = -1;  // below any |x|^2
  int bestk = 0x7fffffff;
  if (active) {
    for (int k = lane; k < N; k += 32) {
      const size_t e = (size_t)b * per + (size_t)k * N + j;
      int32_t a[ND], m2[ND];
      int64_t acc[FXP_NACC];
      fxp_zero(acc);
      fx_load(a, Xr, count, e); fx_mac<false>(acc, a, a);
      fx_load(a, Xi, count, e); fx_mac<false>(acc, a, a);
      fxp_finish(m2, acc);
      if (fx_less(best, m2)) {
#pragma unroll
        for (int q = 0; q < ND; ++q) best[q] = m2[q];
        bestk = k;
      }
    }
  }
  for (int off = 16; off > 0; off >>= 1) {
    int32_t o[ND];
#pragma unroll
    for (int q = 0; q < ND; ++q) o[q] = __shfl_xor_sync(0xffffffffu, best[q], off);
    const int ok = __shfl_xor_sync(0xffffffffu, bestk, off);
    const bool take = fx_less(best, o) || (!fx_less(o, best) && ok < bestk);
    if (take) {
#pragma unroll
      for (int q = 0; q < ND; ++q) best[q] = o[q];
      bestk = ok;
    }
  }
  // lane 0: y = 1/sqrt(best) by Newton on FX; u = conj(z) y
  if (active && lane == 0) {
    int32_t s2[ND];
#pragma unroll
    for (int q = 0; q < ND; ++q) s2[q] = best[q];
    const int msb = fx_msb(s2);
    int32_t ur[ND], ui[ND];
    if (msb == 0) {  // zero column (cannot happen for a unit vector): leave it alone
      fx_zero(ur); fx_zero(ui); ur[ND - 1] = 1;
    } else {
      int32_t y[ND];
      fx_rsqrt(y, s2);  // 1/|x_k*|
      const size_t e = (size_t)b * per + (size_t)bestk * N + j;
      int32_t zr[ND], zi[ND], nzi[ND];
      fx_load(zr, Xr, count, e); fx_load(zi, Xi, count, e);
      fx_mul(ur, zr, y);
      fx_neg(nzi, zi);
      fx_mul(ui, nzi, y);
    }
#pragma unroll
    for (int q = 0; q < ND; ++q) { s_u[wl][0][q] = ur[q]; s_u[wl][1][q] = ui[q]; }
  }
  __syncwarp();
  if (!active) return;
  int32_t ur[ND], ui[ND];
#pragma unroll
  for (int q = 0; q < ND; ++q) { ur[q] = s_u[wl][0][q]; ui[q] = s_u[wl][1][q]; }
  const int rj = rank[(size_t)b * N + j];
  for (int k = lane; k < N; k += 32) {
    const size_t e = (size_t)b * per + (size_t)k * N + j, eo = (size_t)b * per + (size_t)k * N + rj;
    int32_t xr[ND], xi[ND], o[ND];
    fx_load(xr, Xr, count, e); fx_load(xi, Xi, count, e);
    int64_t acc[FXP_NACC];
    fxp_zero(acc);
    fx_mac<false>(acc, xr, ur); fx_mac<true>(acc, xi, ui);
    fxp_finish(o, acc);
    fx_store(out, count, eo, o);
    fxp_zero(acc);
    fx_mac<false>(acc, xr, ui); fx_mac<false>(acc, xi, ur);
    fxp_finish(o, acc);
    if (k == bestk) fx_zero(o);
    fx_store(out + (size_t)ND * count, count, eo, o);
  }
}

int rank_sort(int N, int batch, const int32_t* lam, int* rank, int32_t* lam_sorted, cudaStream_t s) {
  KtScope kt_scope(KC_OTHER, s);
  const size_t nl = (size_t)N * batch;
  rank_kernel<<<(unsigned)((nl * 32 + 127) / 128), 128, 0, s>>>(N, batch, lam, rank, lam_sorted);
  count_launch();
  return launch_check();
}

int phase_sorted(int N, int batch, const int32_t* X, const int* rank, int32_t* out, cudaStream_t s) {
  KtScope kt_scope(KC_OTHER, s);
  const size_t nl = (size_t)N * batch;
  phase_kernel<<<(unsigned)((nl * 32 + 127) / 128), 128, 0, s>>>(N, batch, X, rank, out);
  count_launch();
  return launch_check();
}

int finalize_export(int N, int batch, const int32_t* X, const int32_t* lam, const int* scale, void* eigvals_api, void* eigvecs_api,
                    int32_t* scratch, int32_t* lam_sorted, int* rank, cudaStream_t s, int prec) {
  KtScope kt_scope(KC_IO, s);
  const size_t nl = (size_t)N * batch;
  rank_kernel<<<(unsigned)((nl * 32 + 127) / 128), 128, 0, s>>>(N, batch, lam, rank, lam_sorted);
  phase_kernel<<<(unsigned)((nl * 32 + 127) / 128), 128, 0, s>>>(N, batch, X, rank, scratch);
  count_launch(2);
  ZKD_TRY(launch_check());
  ZKD_TRY(fx_to_api_scaled(nl, lam_sorted, eigvals_api, 0, scale, 1, (size_t)N, s, prec));
  return fxc_to_api((size_t)N * N * batch, scratch, eigvecs_api, s, prec);
}

}  // namespace zkd

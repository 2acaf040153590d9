// blocks.cu — the O(N^2) and O(N^2 m) kernels of the refinement (SURVEY.md 8(a) S2, S3, S4c, S4d', S4f, S5, S6):
// cluster detection, X := V, cluster-block Gram / Rayleigh-quotient matrices, block-diagonal applies (residual,
// orthonormalisation, Rayleigh-Ritz rotation), the divided correction coefficients E_ij = C_ij / (theta_j - theta_i),
// sorting, phase normalisation.  All multi-digit arithmetic is in-thread on FX digits (fx.cuh).
#include "blocks.h"
#include "fx.cuh"
#include "fx_funcs.cuh"
#include "timing.h"

namespace zkd {

// ---- FX -> complex double ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) fxc_to_c64_kernel(size_t count, const int32_t* __restrict__ src, double2* __restrict__ dst) {
  const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= count) return;
  int32_t d[ND];
  fx_load(d, src, count, e);
  const double re = fx_to_double(d);
  fx_load(d, src + (size_t)ND * count, count, e);
  dst[e] = make_double2(re, fx_to_double(d));
}
int fxc_to_c64(size_t count, const int32_t* src, double2* dst, cudaStream_t s) {
  KtScope kt_scope(KC_IO, s);
  fxc_to_c64_kernel<<<(unsigned)((count + 255) / 256), 256, 0, s>>>(count, src, dst);
  count_launch();
  return launch_check();
}

// ---- S2: clusters ----------------------------------------------------------------------------------------------------
// One CTA per matrix.  F = ||A64||_F = (sum_j mu_j^2)^(1/2) (the Frobenius norm of a Hermitian matrix from its eigenvalues: no
// pass over the n^2 entries); a new cluster starts at j when mu_j - mu_{j-1} > 2^-tau F.
// cl[j] = first column of j's cluster, cle[j] = one past its last column.
__global__ void __launch_bounds__(256) cluster_kernel(int n, const double2* __restrict__ A64, const double* __restrict__ mu,
                                                      int tau_bits, const int* __restrict__ floor_msb /* [nb] or null */,
                                                      int* __restrict__ cl, int* __restrict__ cle,
                                                      int* __restrict__ stats /* [nb][2]: n_clusters, max_cluster */) {
  extern __shared__ int s_flag[];  // [n + 1]: 1 where a cluster starts; s_flag[n] = 1
  __shared__ double s_red[8];
  __shared__ double s_thr;
  __shared__ int s_ncl, s_maxc;
  (void)A64;
  const int b = blockIdx.x, tid = threadIdx.x;
  const double* m = mu + (size_t)b * n;
  double s = 0;
  for (int j = tid; j < n; j += blockDim.x) s += m[j] * m[j];
  for (int off = 16; off > 0; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
  if ((tid & 31) == 0) s_red[tid >> 5] = s;
  __syncthreads();
  if (tid == 0) {
    double t = 0;
    for (int w = 0; w < 8; ++w) t += s_red[w];
    // differences below 2^(floor_msb - 812) are noise of the matrix entries themselves (early splits, S4h): never split there
    double thr = ldexp(sqrt(t), -tau_bits);
    if (floor_msb) thr = fmax(thr, ldexp(1.0, floor_msb[b] - 812));
    s_thr = thr;
    s_ncl = 0;
    s_maxc = 0;
    s_flag[n] = 1;
  }
  __syncthreads();
  const double thr = s_thr;
  for (int j = tid; j < n; j += blockDim.x) s_flag[j] = (j == 0 || (m[j] - m[j - 1] > thr)) ? 1 : 0;
  __syncthreads();
  for (int j = tid; j < n; j += blockDim.x) {
    int lo = j, hi = j + 1;
    while (!s_flag[lo]) --lo;
    while (!s_flag[hi]) ++hi;
    cl[(size_t)b * n + j] = lo;
    cle[(size_t)b * n + j] = hi;
    if (lo == j) {
      atomicAdd(&s_ncl, 1);
      atomicMax(&s_maxc, hi - lo);
    }
  }
  __syncthreads();
  if (tid == 0) {
    stats[2 * b] = s_ncl;
    stats[2 * b + 1] = s_maxc;
  }
}
int cluster_detect(int n, int nb, const double2* A64, const double* mu, int tau_bits, const int* floor_msb, int* cl, int* cle,
                   int* stats, cudaStream_t s) {
  KtScope kt_scope(KC_OTHER, s);
  cluster_kernel<<<nb, 256, sizeof(int) * (n + 1), s>>>(n, A64, mu, tau_bits, floor_msb, cl, cle, stats);
  count_launch();
  return launch_check();
}

// ---- S3: X := V (exactly, truncated below FX bit 756 = digit 27) --------------------------------------------------------
__global__ void __launch_bounds__(256) init_x_kernel(size_t count, const double2* __restrict__ V, int32_t* __restrict__ X) {
  const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= count) return;
  const double2 v = V[e];
  int32_t d[ND];
  fx_from_double(d, v.x);
  // truncate toward -inf below digit 27 (keeps the value a short-window number: digits 27..29 only)
#pragma unroll
  for (int k = 0; k < 27; ++k) d[k] = 0;
  fx_store(X, count, e, d);
  fx_from_double(d, v.y);
#pragma unroll
  for (int k = 0; k < 27; ++k) d[k] = 0;
  fx_store(X + (size_t)ND * count, count, e, d);
}
int init_x(size_t count, const double2* V, int32_t* X, cudaStream_t s) {
  KtScope kt_scope(KC_IO, s);
  init_x_kernel<<<(unsigned)((count + 255) / 256), 256, 0, s>>>(count, V, X);
  count_launch();
  return launch_check();
}

// ---- M := (I - G)/2 on cluster blocks (Newton-Schulz orthonormalisation step), msb of (G - I) ---------------------------
__global__ void __launch_bounds__(256) ns_build_kernel(int n, int nb, const int* __restrict__ cl, const int* __restrict__ cle_skip1,
                                                       int32_t* __restrict__ G, int* __restrict__ msb_out, int* __restrict__ msb_b,
                                                       int zero_rest) {
  const size_t per = (size_t)n * n, count = per * nb;
  const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= count * 2) return;
  const int part = (int)(t / count);
  const size_t e = t % count;
  const int b = (int)(e / per), i = (int)((e % per) / n), j = (int)(e % n);
  int32_t* p = G + (part ? (size_t)ND * count : 0);
  int32_t g[ND], r[ND];
  if (cl[(size_t)b * n + i] != cl[(size_t)b * n + j] ||
      (cle_skip1 && cle_skip1[(size_t)b * n + j] - cl[(size_t)b * n + j] == 1)) {  // singletons are handled elsewhere
    if (zero_rest) { fx_zero(g); fx_store(p, count, e, g); }
    return;
  }
  fx_load(g, p, count, e);
  if (part == 0 && i == j) g[ND - 1] -= 1;  // G - I
  const int msb = fx_msb(g);
  if (msb_out) atomicMax(msb_out, msb);
  if (msb_b && msb) atomicMax(msb_b + b, msb);
  fx_neg(r, g);
  fx_half(g, r);                            // (I - G)/2
  fx_store(p, count, e, g);
}
int ns_build(int n, int nb, const int* cl, int32_t* G, int* msb_out, cudaStream_t s, const int* cle_skip1, int* msb_b, bool zero_rest) {
  KtScope kt_scope(KC_OTHER, s);
  const size_t t = (size_t)n * n * nb * 2;
  ns_build_kernel<<<(unsigned)((t + 255) / 256), 256, 0, s>>>(n, nb, cl, cle_skip1, G, msb_out, msb_b, zero_rest ? 1 : 0);
  count_launch();
  return launch_check();
}

// ---- theta_j = Re S_jj ---------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) mask_offcluster_kernel(int n, int nb, const int* __restrict__ cl, const int* __restrict__ cle,
                                                              int32_t* __restrict__ S) {
  const size_t per = (size_t)n * n, count = per * nb;
  const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= count * 2) return;
  const size_t e = t % count;
  const int b = (int)(e / per), i = (int)((e % per) / n), j = (int)(e % n);
  const bool keep = cl[(size_t)b * n + i] == cl[(size_t)b * n + j] && cle[(size_t)b * n + j] - cl[(size_t)b * n + j] > 1;
  if (keep) return;
  int32_t z[ND];
  fx_zero(z);
  fx_store(S + (t / count) * (size_t)ND * count, count, e, z);
}
int mask_offcluster(int n, int nb, const int* cl, const int* cle, int32_t* S, cudaStream_t s) {
  KtScope kt_scope(KC_OTHER, s);
  const size_t t = (size_t)n * n * nb * 2;
  mask_offcluster_kernel<<<(unsigned)((t + 255) / 256), 256, 0, s>>>(n, nb, cl, cle, S);
  count_launch();
  return launch_check();
}

__global__ void __launch_bounds__(128) theta_kernel(int n, int nb, const int32_t* __restrict__ S, int32_t* __restrict__ theta,
                                                    const int* __restrict__ cl, const int* __restrict__ cle) {
  const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= (size_t)n * nb) return;
  if (cl && cle[t] - cl[t] == 1) return;
  const int b = (int)(t / n), j = (int)(t % n);
  const size_t count = (size_t)n * n * nb;
  int32_t d[ND];
  fx_load(d, S, count, (size_t)b * n * n + (size_t)j * n + j);
  fx_store(theta, (size_t)n * nb, t, d);
}
int theta_from_diag(int n, int nb, const int32_t* S, int32_t* theta, cudaStream_t s, const int* cl, const int* cle) {
  KtScope kt_scope(KC_OTHER, s);
  theta_kernel<<<(unsigned)(((size_t)n * nb + 127) / 128), 128, 0, s>>>(n, nb, S, theta, cl, cle);
  count_launch();
  return launch_check();
}

// ---- smallest gap between neighbouring clusters: gap_inv_out <- max(1024 - msb(theta_{j+1} - theta_j)) over cluster borders ----
// (columns are in ascending order of theta, so the closest pair of eigenvalues of different clusters is a neighbouring pair)
__global__ void __launch_bounds__(128) min_gap_kernel(int n, int nb, const int32_t* __restrict__ theta, const int* __restrict__ cl,
                                                      int* __restrict__ gap_inv_out) {
  const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= (size_t)n * nb) return;
  const int j = (int)(t % n);
  if (j + 1 >= n || cl[t] == cl[t + 1]) return;
  int32_t a[ND], c[ND], d[ND];
  fx_load(a, theta, (size_t)n * nb, t);
  fx_load(c, theta, (size_t)n * nb, t + 1);
  fx_sub(d, c, a);
  if (fx_is_neg(d)) { fx_neg(a, d); atomicMax(gap_inv_out, 1024 - fx_msb(a)); }
  else atomicMax(gap_inv_out, 1024 - fx_msb(d));
}
int min_gap(int n, int nb, const int32_t* theta, const int* cl, int* gap_inv_out, cudaStream_t s) {
  KtScope kt_scope(KC_OTHER, s);
  min_gap_kernel<<<(unsigned)(((size_t)n * nb + 127) / 128), 128, 0, s>>>(n, nb, theta, cl, gap_inv_out);
  count_launch();
  return launch_check();
}

// ---- per-matrix residual level (zkd_info.log2_resid / status): max msb over the elements of each matrix of R ---------------------
__global__ void __launch_bounds__(256) resid_per_matrix_kernel(int n, int nb, const int32_t* __restrict__ R, int* __restrict__ msb_r_b) {
  const size_t per = (size_t)n * n, count = per * nb;
  const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  int m = 0;
  int b = 0;
  if (t < 2 * count) {
    const size_t e = t % count;
    b = (int)(e / per);
    int32_t d[ND];
    fx_load(d, R + (t / count) * (size_t)ND * count, count, e);
    m = fx_msb(d);
  }
  // a warp usually lies inside one matrix: one atomic per warp then
  const int b0 = __shfl_sync(0xffffffffu, b, 0);
  if (__all_sync(0xffffffffu, b == b0 || m == 0)) {
    for (int o = 16; o > 0; o >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0 && m) atomicMax(msb_r_b + b0, m);
  } else if (m) {
    atomicMax(msb_r_b + b, m);
  }
}
int resid_per_matrix(int n, int nb, const int32_t* R, int* msb_r_b, cudaStream_t s) {
  KtScope kt_scope(KC_OTHER, s);
  const size_t t = 2 * (size_t)n * n * nb;
  resid_per_matrix_kernel<<<(unsigned)((t + 255) / 256), 256, 0, s>>>(n, nb, R, msb_r_b);
  count_launch();
  return launch_check();
}

// ---- complex FX add: X += T ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) offdiag_blocks_kernel(int n, int nb, const int* __restrict__ cl, const int32_t* __restrict__ S,
                                                             int32_t* __restrict__ O, int* __restrict__ msb_out) {
  const size_t per = (size_t)n * n, count = per * nb;
  const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  int m = 0;
  if (t < 2 * count) {
    const size_t e = t % count;
    const int b = (int)(e / per), i = (int)((e % per) / n), j = (int)(e % n);
    int32_t d[ND];
    fx_zero(d);
    if (i != j && cl[(size_t)b * n + i] == cl[(size_t)b * n + j]) {
      fx_load(d, S + (t / count) * (size_t)ND * count, count, e);
      m = fx_msb(d);
    }
    fx_store(O + (t / count) * (size_t)ND * count, count, e, d);
  }
  for (int o = 16; o > 0; o >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, o));
  if ((threadIdx.x & 31) == 0 && m) atomicMax(msb_out, m);
}
int offdiag_blocks(int n, int nb, const int* cl, const int32_t* S, int32_t* O, int* msb_out, cudaStream_t s) {
  KtScope kt_scope(KC_OTHER, s);
  const size_t t = 2 * (size_t)n * n * nb;
  offdiag_blocks_kernel<<<(unsigned)((t + 255) / 256), 256, 0, s>>>(n, nb, cl, S, O, msb_out);
  count_launch();
  return launch_check();
}

__global__ void __launch_bounds__(256) fx_add_kernel(size_t reals, int32_t* __restrict__ X, const int32_t* __restrict__ T, int subtract) {
  const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= reals) return;
  // planes of re and im are laid out [2][ND][count]; treat as 2*count reals with plane stride `count`
  const size_t count = reals / 2;
  const size_t part = e / count, idx = e % count;
  int32_t* xp = X + part * (size_t)ND * count;
  const int32_t* tp = T + part * (size_t)ND * count;
  int32_t a[ND], c[ND], r[ND];
  fx_load(a, xp, count, idx);
  fx_load(c, tp, count, idx);
  if (subtract) fx_sub(r, a, c); else fx_add(r, a, c);
  fx_store(xp, count, idx, r);
}
int fxc_add_inplace(size_t count, int32_t* X, const int32_t* T, cudaStream_t s, bool subtract) {
  KtScope kt_scope(KC_OTHER, s);
  fx_add_kernel<<<(unsigned)((2 * count + 255) / 256), 256, 0, s>>>(2 * count, X, T, subtract ? 1 : 0);
  count_launch();
  return launch_check();
}

// ---- fused S4f + S4c for levels whose clusters are all singletons (the common case: c1, c2, c3) ---------------------------------
// One CTA per column j:  g = ||x_j||^2 ;  f = 1 + (1 - g)/2 ;  x_j <- f x_j ;  w_j <- f w_j   (Newton-Schulz step = normalisation)
//                        s = x_j^H w_j ;  theta_j = Re s ;  r_j = w_j - x_j s                  (Rayleigh quotient, residual)
// X and W are updated in place (a CTA touches only its own column).  One launch in place of the seven products of the cluster path
// (Gram, Newton-Schulz build, two applies, Rayleigh-Ritz, theta, residual); its critical path is 14 digit products per element.
// Sum of column accumulators over the threads of the CTA that own the same matrix column.  Thread layout: tx = tid % CPB is
// the matrix column inside the CTA's group of CPB columns, the other bits of tid index rows; lanes with equal tx are
// lane % CPB apart, so the warp stage uses xor offsets 16 .. CPB only.  Every thread returns its column's total.
template <int CPB, int NACC2>
__device__ __forceinline__ void block_sum_cols(int64_t (&acc)[NACC2], int64_t* s_part /*[nwarps][CPB][NACC2]*/, int nwarps) {
#pragma unroll
  for (int off = 16; off >= CPB; off >>= 1) {
#pragma unroll
    for (int k = 0; k < NACC2; ++k) acc[k] += __shfl_down_sync(0xffffffffu, acc[k], off);
  }
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, tx = threadIdx.x % CPB;
  __syncthreads();  // s_part may still be read from the previous reduction
  if (lane < CPB) {
#pragma unroll
    for (int k = 0; k < NACC2; ++k) s_part[(warp * CPB + lane) * NACC2 + k] = acc[k];
  }
  __syncthreads();
#pragma unroll
  for (int k = 0; k < NACC2; ++k) {
    int64_t t = 0;
    for (int w = 0; w < nwarps; ++w) t += s_part[(w * CPB + tx) * NACC2 + k];
    acc[k] = t;
  }
}

// CPB matrix columns per CTA: a warp reads CPB consecutive columns of 32 / CPB rows, i.e. CPB * 4 contiguous bytes per row
// (row-major X: a single column per CTA touches one 32-byte sector per element and digit).
// CACHE (CPB = 1, small n): the column's x and w digits (4 planes x 30 digits x n words) are staged in shared memory once;
// the five phases then read and update them there, and x, w go back to global memory at the end - instead of ~26
// dependent round trips to L2 per element.
template <int CPB, bool CACHE>
__global__ void __launch_bounds__(256) singleton_step_kernel(int n, int nb, int32_t* __restrict__ X, int32_t* __restrict__ W,
                                                             int32_t* __restrict__ R, int32_t* __restrict__ S,
                                                             int32_t* __restrict__ theta, int* __restrict__ msb_g_out,
                                                             int* __restrict__ msb_r_out, const int* __restrict__ cl,
                                                             const int* __restrict__ cle, int* __restrict__ msb_g_b) {
  __shared__ int64_t s_part[8 * CPB * FXP_NACC];
  __shared__ int s_msb;
  extern __shared__ int32_t s_cache[];  // CACHE: [4][ND][n]
  const int groups = (n + CPB - 1) / CPB;
  const int b = blockIdx.x / groups;
  const int tid = threadIdx.x, nwarps = blockDim.x >> 5, tx = tid % CPB, ty = tid / CPB, rows = blockDim.x / CPB;
  const int j = (blockIdx.x % groups) * CPB + tx;
  // mixed levels: columns of larger clusters take the GEMM path
  const bool act = j < n && !(cl && cle[(size_t)b * n + j] - cl[(size_t)b * n + j] > 1);
  const size_t per = (size_t)n * n, count = per * nb;
  int32_t* const gplane[4] = {X, X + (size_t)ND * count, W, W + (size_t)ND * count};  // xr, xi, wr, wi
  int32_t* Rr = R;  int32_t* Ri = R + (size_t)ND * count;
  // plane pl of row k: base pointer, digit stride and index, in shared or global memory
  const size_t stride = CACHE ? (size_t)n : count;
  auto base = [&](int pl) -> int32_t* { return CACHE ? s_cache + (size_t)pl * ND * n : gplane[pl]; };
  auto idx = [&](int k) -> size_t { return CACHE ? (size_t)k : (size_t)b * per + (size_t)k * n + j; };
  if (tid == 0) s_msb = 0;
  if (CACHE && act) {
    for (int k = ty; k < n; k += rows) {
      const size_t e = (size_t)b * per + (size_t)k * n + j;
#pragma unroll 1
      for (int pl = 0; pl < 4; ++pl) {
        int32_t a[ND];
        fx_load(a, gplane[pl], count, e);
        fx_store(s_cache + (size_t)pl * ND * n, (size_t)n, (size_t)k, a);
      }
    }
  }
  // (a thread only ever touches the cache entries of its own rows: no barrier needed for the cache itself)

  // g = sum_k |x_kj|^2
  int64_t acc[FXP_NACC];
  fxp_zero(acc);
  // (every product phase below has ONE inlined multiply site, looped over planes / terms with run-time operand and sign
  // selection: the unrolled 30 x 30 digit product is ~500 IMAD.WIDE, and 14 copies of it thrashed the instruction cache)
  if (act) {
    for (int k = ty; k < n; k += rows) {
#pragma unroll 1
      for (int pl = 0; pl < 2; ++pl) {
        int32_t a[ND];
        fx_load(a, base(pl), stride, idx(k));
        fx_mac<false>(acc, a, a);
      }
      fxp_relax(acc);
    }
  }
  block_sum_cols<CPB>(acc, s_part, nwarps);
  int32_t g[ND], m[ND];
  fxp_finish(g, acc);
  g[ND - 1] -= 1;                      // g - 1
  if (act && ty == 0 && msb_g_out) {
    const int mg = fx_msb(g);
    atomicMax(msb_g_out, mg);
    if (msb_g_b && mg) atomicMax(msb_g_b + b, mg);
  }
  {
    int32_t t[ND];
    fx_neg(t, g);
    fx_half(m, t);                     // m = (1 - g)/2
  }

  // x <- x + x m, w <- w + w m   (one plane at a time: at most three digit arrays and one accumulator set are live)
  if (act) {
#pragma unroll 1
    for (int pl = 0; pl < 4; ++pl) {
#pragma unroll 1
      for (int k = ty; k < n; k += rows) {
        int32_t u[ND], t[ND];
        fx_load(u, base(pl), stride, idx(k));
        fx_mul(t, u, m);
        int32_t o[ND];
        fx_add(o, u, t);
        fx_store(base(pl), stride, idx(k), o);
        if (CACHE) fx_store(gplane[pl], count, (size_t)b * per + (size_t)k * n + j, o);
      }
    }
  }
  // s = x^H w : real part, then imaginary part
  int32_t sr[ND], si[ND];
#pragma unroll 1
  for (int part = 0; part < 2; ++part) {
    fxp_zero(acc);
    if (act) {
#pragma unroll 1
      for (int k = ty; k < n; k += rows) {
        // part 0: xr wr + xi wi ;  part 1: xr wi - xi wr
#pragma unroll 1
        for (int term = 0; term < 2; ++term) {
          int32_t a[ND], c[ND];
          fx_load(a, base(term), stride, idx(k));
          fx_load(c, base(2 + (term ^ part)), stride, idx(k));
          if (part == 1 && term == 1) {
#pragma unroll
            for (int q = 0; q < ND; ++q) a[q] = -a[q];  // digit-wise negation: a valid (non-canonical) operand of fx_mac
          }
          fx_mac<false>(acc, a, c);
        }
        fxp_relax(acc);
      }
    }
    block_sum_cols<CPB>(acc, s_part, nwarps);
    if (part == 0) fxp_finish(sr, acc); else fxp_finish(si, acc);
  }
  if (act && ty == 0) {
    fx_store(theta, (size_t)n * nb, (size_t)b * n + j, sr);
    const size_t ejj = (size_t)b * per + (size_t)j * n + j;
    fx_store(S, count, ejj, sr);
    fx_store(S + (size_t)ND * count, count, ejj, si);
  }

  // r = w - x s
  int mymsb = 0;
  if (act) {
#pragma unroll 1
    for (int part = 0; part < 2; ++part) {
#pragma unroll 1
      for (int k = ty; k < n; k += rows) {
        const size_t e = (size_t)b * per + (size_t)k * n + j;
        int32_t a[ND], t[ND];
        fxp_zero(acc);
        // part 0: xr sr - xi si ;  part 1: xr si + xi sr
#pragma unroll 1
        for (int term = 0; term < 2; ++term) {
          int32_t mm[ND];
          const bool use_si = (term ^ part) != 0, neg = part == 0 && term == 1;
#pragma unroll
          for (int q = 0; q < ND; ++q) {
            const int32_t v = use_si ? si[q] : sr[q];
            mm[q] = neg ? -v : v;
          }
          fx_load(a, base(term), stride, idx(k));
          fx_mac<false>(acc, a, mm);
        }
        fxp_finish(t, acc);
        fx_load(a, base(2 + part), stride, idx(k));
        int32_t o[ND];
        fx_sub(o, a, t);
        fx_store(part ? Ri : Rr, count, e, o);
        mymsb = max(mymsb, fx_msb(o));
      }
    }
  }
  for (int off = 16; off > 0; off >>= 1) mymsb = max(mymsb, __shfl_xor_sync(0xffffffffu, mymsb, off));
  if ((tid & 31) == 0 && mymsb) atomicMax(&s_msb, mymsb);
  __syncthreads();
  if (tid == 0 && msb_r_out && s_msb) atomicMax(msb_r_out, s_msb);
}
// ---- the same step with the 14 products of a row spread over several threads (small n, one column per CTA) ------------------------
// singleton_step_kernel gives every thread whole rows: 14 dependent 30 x 30-digit products (~500 IMAD.WIDE each) per row, on as many
// threads as the column has rows - at n = 64 that is two warps per CTA walking a 7000-multiply chain (the kernel was the largest item of
// c2: 6 x 70 us).  Here the work items are (row, plane) / (row, term) pairs, so a thread's chain is 6 products: |x|^2 (1), the
// normalisation of one plane (1), one term of Re s and of Im s (2), one part of the residual (2).  Same integer sums, same
// roundings: bit-identical results.  The column's x, w digits live in shared memory throughout.
__global__ void __launch_bounds__(256) singleton_step_par_kernel(int n, int nb, int32_t* __restrict__ X, int32_t* __restrict__ W,
                                                                 int32_t* __restrict__ R, int32_t* __restrict__ S,
                                                                 int32_t* __restrict__ theta, int* __restrict__ msb_g_out,
                                                                 int* __restrict__ msb_r_out, const int* __restrict__ cl,
                                                                 const int* __restrict__ cle, int* __restrict__ msb_g_b) {
  __shared__ int64_t s_part[16 * FXP_NACC];
  __shared__ int s_msb;
  extern __shared__ int32_t s_cache[];  // [4][ND][n]: xr, xi, wr, wi
  const int b = blockIdx.x / n, j = blockIdx.x % n;
  const int tid = threadIdx.x, T = blockDim.x, nwarps = T >> 5;
  const bool act = !(cl && cle[(size_t)b * n + j] - cl[(size_t)b * n + j] > 1);  // columns of larger clusters take the GEMM path
  const size_t per = (size_t)n * n, count = per * nb;
  int32_t* const gplane[4] = {X, X + (size_t)ND * count, W, W + (size_t)ND * count};
  if (tid == 0) s_msb = 0;
  if (act) {
    for (int it = tid; it < 4 * n; it += T) {
      const int pl = it / n, k = it - pl * n;
      int32_t a[ND];
      fx_load(a, gplane[pl], count, (size_t)b * per + (size_t)k * n + j);
      fx_store(s_cache + (size_t)pl * ND * n, (size_t)n, (size_t)k, a);
    }
  }
  __syncthreads();
  // g = sum_k |x_kj|^2
  int64_t acc[FXP_NACC];
  fxp_zero(acc);
  if (act) {
    for (int it = tid; it < 2 * n; it += T) {
      const int pl = it / n, k = it - pl * n;
      int32_t a[ND];
      fx_load(a, s_cache + (size_t)pl * ND * n, (size_t)n, (size_t)k);
      fx_mac<false>(acc, a, a);
      fxp_relax(acc);
    }
  }
  block_sum_cols<1>(acc, s_part, nwarps);
  int32_t g[ND], m[ND];
  fxp_finish(g, acc);
  g[ND - 1] -= 1;  // g - 1
  if (act && tid == 0 && msb_g_out) {
    const int mg = fx_msb(g);
    atomicMax(msb_g_out, mg);
    if (msb_g_b && mg) atomicMax(msb_g_b + b, mg);
  }
  {
    int32_t t[ND];
    fx_neg(t, g);
    fx_half(m, t);  // m = (1 - g)/2
  }
  // x <- x + x m, w <- w + w m
  if (act) {
    for (int it = tid; it < 4 * n; it += T) {
      const int pl = it / n, k = it - pl * n;
      int32_t u[ND], t[ND], o[ND];
      fx_load(u, s_cache + (size_t)pl * ND * n, (size_t)n, (size_t)k);
      fx_mul(t, u, m);
      fx_add(o, u, t);
      fx_store(s_cache + (size_t)pl * ND * n, (size_t)n, (size_t)k, o);
      fx_store(gplane[pl], count, (size_t)b * per + (size_t)k * n + j, o);
    }
  }
  __syncthreads();
  // s = x^H w : real part, then imaginary part (items: (term, row))
  int32_t sr[ND], si[ND];
#pragma unroll 1
  for (int part = 0; part < 2; ++part) {
    fxp_zero(acc);
    if (act) {
      for (int it = tid; it < 2 * n; it += T) {
        const int term = it / n, k = it - term * n;
        // part 0: xr wr + xi wi ;  part 1: xr wi - xi wr
        int32_t a[ND], c[ND];
        fx_load(a, s_cache + (size_t)term * ND * n, (size_t)n, (size_t)k);
        fx_load(c, s_cache + (size_t)(2 + (term ^ part)) * ND * n, (size_t)n, (size_t)k);
        if (part == 1 && term == 1) {
#pragma unroll
          for (int q = 0; q < ND; ++q) a[q] = -a[q];  // digit-wise negation: a valid (non-canonical) operand of fx_mac
        }
        fx_mac<false>(acc, a, c);
        fxp_relax(acc);
      }
    }
    block_sum_cols<1>(acc, s_part, nwarps);
    if (part == 0) fxp_finish(sr, acc); else fxp_finish(si, acc);
  }
  if (act && tid == 0) {
    fx_store(theta, (size_t)n * nb, (size_t)b * n + j, sr);
    const size_t ejj = (size_t)b * per + (size_t)j * n + j;
    fx_store(S, count, ejj, sr);
    fx_store(S + (size_t)ND * count, count, ejj, si);
  }
  // r = w - x s (items: (part, row))
  int mymsb = 0;
  if (act) {
    for (int it = tid; it < 2 * n; it += T) {
      const int part = it / n, k = it - part * n;
      int32_t a[ND], t[ND];
      fxp_zero(acc);
      // part 0: xr sr - xi si ;  part 1: xr si + xi sr
#pragma unroll 1
      for (int term = 0; term < 2; ++term) {
        int32_t mm[ND];
        const bool use_si = (term ^ part) != 0, neg = part == 0 && term == 1;
#pragma unroll
        for (int q = 0; q < ND; ++q) {
          const int32_t v = use_si ? si[q] : sr[q];
          mm[q] = neg ? -v : v;
        }
        fx_load(a, s_cache + (size_t)term * ND * n, (size_t)n, (size_t)k);
        fx_mac<false>(acc, a, mm);
      }
      fxp_finish(t, acc);
      fx_load(a, s_cache + (size_t)(2 + part) * ND * n, (size_t)n, (size_t)k);
      int32_t o[ND];
      fx_sub(o, a, t);
      fx_store(R + (part ? (size_t)ND * count : 0), count, (size_t)b * per + (size_t)k * n + j, o);
      mymsb = max(mymsb, fx_msb(o));
    }
  }
  for (int off = 16; off > 0; off >>= 1) mymsb = max(mymsb, __shfl_xor_sync(0xffffffffu, mymsb, off));
  if ((tid & 31) == 0 && mymsb) atomicMax(&s_msb, mymsb);
  __syncthreads();
  if (tid == 0 && msb_r_out && s_msb) atomicMax(msb_r_out, s_msb);
}

// ---- warp-cooperative variant for small n (north_star (b): "warp-cooperative limb add, multiply, normalise ... carry chains
// via warp shuffles") -------------------------------------------------------------------------------------------------------
// One CTA per matrix column, one WARP per element: lane L holds digit L of an FX number (lanes 0..29) and, in a product,
// column 28 + L (lanes 0..30: the 31 kept columns).  A 30 x 30 digit product is 30 x (shuffle + IMAD.WIDE) per lane instead of
// ~500 IMAD.WIDE in one thread; carries are resolved across lanes by two relaxation rounds and a ballot look-ahead.  Each
// warp keeps the x, w digits of its (at most 4) rows in registers through all phases.  Exact integer sums and one rounding
// at the guard column, as in the thread-per-element kernel: the results are bit-identical.
template <int TOP>
__device__ __forceinline__ int64_t wcanon(int64_t v, int lane) {
  const bool low = lane < TOP, top = lane == TOP;
  constexpr unsigned kLowMask = (1u << TOP) - 1;
  int64_t lo = low ? (v & DMASK) : (top ? v : 0), hi = low ? (v >> DB) : 0;
#pragma unroll
  for (int round = 0; round < 2; ++round) {
    int64_t inc = __shfl_up_sync(0xffffffffu, hi, 1);
    if (lane == 0 || lane > TOP) inc = 0;
    const int64_t t = lo + inc;
    if (low) { hi = t >> DB; lo = t & DMASK; }
    else { hi = 0; lo = t; }
  }
  int64_t inc = __shfl_up_sync(0xffffffffu, hi, 1);  // -1, 0 or +1
  if (lane == 0 || lane > TOP) inc = 0;
  int64_t t = lo;
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
  return t;
}
// acc (column 28 + lane) += sign * sum_i a_i b_{28 + lane - i}:  a uniform (every lane holds all digits), b one digit per lane
__device__ __forceinline__ void wmac_u(int64_t& acc, const int32_t (&a)[ND], int32_t b, int lane, bool neg) {
#pragma unroll
  for (int i = 0; i < ND; ++i) {
    const int src = FXP_LOW + lane - i;
    int32_t bv = __shfl_sync(0xffffffffu, b, src & 31);
    if (src < 0 || src > ND - 1) bv = 0;
    const int64_t p = (int64_t)a[i] * (int64_t)bv;
    acc += neg ? -p : p;
  }
}
// both operands one digit per lane
__device__ __forceinline__ void wmac_l(int64_t& acc, int32_t a, int32_t b, int lane, bool neg) {
#pragma unroll
  for (int i = 0; i < ND; ++i) {
    const int32_t ai = __shfl_sync(0xffffffffu, a, i);
    const int src = FXP_LOW + lane - i;
    int32_t bv = __shfl_sync(0xffffffffu, b, src & 31);
    if (src < 0 || src > ND - 1) bv = 0;
    const int64_t p = (int64_t)ai * (int64_t)bv;
    acc += neg ? -p : p;
  }
}
// keep a running column accumulator small: pass the overflow of every column to the lane above (lane 30 keeps the rest)
__device__ __forceinline__ void wrelax1(int64_t& acc, int lane) {
  const bool low = lane < ND;
  const int64_t hi = low ? (acc >> DB) : 0;
  int64_t inc = __shfl_up_sync(0xffffffffu, hi, 1);
  if (lane == 0 || lane > ND) inc = 0;
  acc = (low ? (acc & DMASK) : acc) + inc;
}
// product columns -> FX digits (rounded at the guard column): digit r ends up in lane r
__device__ __forceinline__ int32_t wfinish(int64_t acc, int lane) {
  if (lane == 0) acc += DHALF;
  if (lane > ND) acc = 0;
  const int64_t t = wcanon<ND>(acc, lane);  // 31 columns: lanes 0..30, the rest in lane 30
  const int64_t d = __shfl_down_sync(0xffffffffu, t, 1);
  return lane < ND ? (int32_t)d : 0;
}
// all 30 digits of a digit-per-lane number into every lane
__device__ __forceinline__ void wbroadcast(int32_t (&all)[ND], int32_t d) {
#pragma unroll
  for (int i = 0; i < ND; ++i) all[i] = __shfl_sync(0xffffffffu, d, i);
}
__device__ __forceinline__ int wmsb(int32_t d, int lane) {
  const int32_t top = __shfl_sync(0xffffffffu, d, ND - 1);
  int cand = 0;
  if (lane < ND - 1) {
    if (top < 0) { if (d != DMASK) cand = lane * DB + (32 - __clz((~d) & DMASK)); }
    else if (d != 0) cand = lane * DB + (32 - __clz(d));
  } else if (lane == ND - 1) {
    if (d > 0) cand = lane * DB + (32 - __clz(d));
    if (d < -1) cand = lane * DB + (32 - __clz(~d));
  }
  for (int o = 16; o > 0; o >>= 1) cand = max(cand, __shfl_xor_sync(0xffffffffu, cand, o));
  return cand;
}

constexpr int SW_RPW = 4;  // rows per warp

__global__ void __launch_bounds__(512) singleton_step_warp_kernel(int n, int nb, int32_t* __restrict__ X, int32_t* __restrict__ W,
                                                                   int32_t* __restrict__ R, int32_t* __restrict__ S,
                                                                   int32_t* __restrict__ theta, int* __restrict__ msb_g_out,
                                                                   int* __restrict__ msb_r_out, const int* __restrict__ cl,
                                                                   const int* __restrict__ cle, int* __restrict__ msb_g_b) {
  __shared__ int64_t s_red[2][16][32];
  __shared__ int s_msb;
  const int b = blockIdx.x / n, j = blockIdx.x % n;
  if (cl && cle[blockIdx.x] - cl[blockIdx.x] > 1) return;  // columns of larger clusters take the GEMM path
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
  const size_t per = (size_t)n * n, count = per * nb;
  const bool dl = lane < ND;  // lanes that hold a digit
  int32_t* const gplane[4] = {X, X + (size_t)ND * count, W, W + (size_t)ND * count};
  if (threadIdx.x == 0) s_msb = 0;

  // this warp's rows: k = warp + t * nw
  int32_t v[4][SW_RPW];
#pragma unroll
  for (int t = 0; t < SW_RPW; ++t) {
    const int k = warp + t * nw;
#pragma unroll
    for (int pl = 0; pl < 4; ++pl)
      v[pl][t] = (k < n && dl) ? gplane[pl][(size_t)lane * count + (size_t)b * per + (size_t)k * n + j] : 0;
  }
  auto block_sum = [&](int64_t a, int slot) -> int64_t {
    s_red[slot][warp][lane] = a;
    __syncthreads();
    int64_t t = 0;
    for (int w = 0; w < nw; ++w) t += s_red[slot][w][lane];
    return t;
  };

  // g = sum_k |x_kj|^2
  int64_t acc = 0;
#pragma unroll
  for (int t = 0; t < SW_RPW; ++t) {
    if (warp + t * nw < n) {
      wmac_l(acc, v[0][t], v[0][t], lane, false);
      wmac_l(acc, v[1][t], v[1][t], lane, false);
      wrelax1(acc, lane);
    }
  }
  acc = block_sum(acc, 0);
  int32_t g = wfinish(acc, lane);
  if (lane == ND - 1) g -= 1;  // g - 1
  {
    const int mg = wmsb(g, lane);
    if (threadIdx.x == 0 && msb_g_out) atomicMax(msb_g_out, mg);
    if (threadIdx.x == 0 && msb_g_b && mg) atomicMax(msb_g_b + b, mg);
  }
  // m = (1 - g)/2: negate, canonicalise, shift right by one bit
  int32_t m;
  {
    const int64_t ng = wcanon<ND - 1>(dl ? -(int64_t)g : 0, lane);
    const int64_t up = __shfl_down_sync(0xffffffffu, ng, 1);
    m = lane < ND - 1 ? (int32_t)(((ng >> 1) | (up << (DB - 1))) & DMASK) : (lane == ND - 1 ? (int32_t)(ng >> 1) : 0);
  }
  int32_t all[ND];
  wbroadcast(all, m);
  // x <- x + x m, w <- w + w m
#pragma unroll
  for (int t = 0; t < SW_RPW; ++t) {
    const int k = warp + t * nw;
    if (k < n) {
#pragma unroll
      for (int pl = 0; pl < 4; ++pl) {
        int64_t a2 = 0;
        wmac_u(a2, all, v[pl][t], lane, false);
        const int32_t tt = wfinish(a2, lane);
        const int32_t o = (int32_t)wcanon<ND - 1>(dl ? (int64_t)v[pl][t] + tt : 0, lane);
        v[pl][t] = o;
        if (dl) gplane[pl][(size_t)lane * count + (size_t)b * per + (size_t)k * n + j] = o;
      }
    }
  }
  // s = x^H w
  int64_t are = 0, aim = 0;
#pragma unroll
  for (int t = 0; t < SW_RPW; ++t) {
    if (warp + t * nw < n) {
      wmac_l(are, v[0][t], v[2][t], lane, false);  // xr wr
      wmac_l(are, v[1][t], v[3][t], lane, false);  // xi wi
      wmac_l(aim, v[0][t], v[3][t], lane, false);  // xr wi
      wmac_l(aim, v[1][t], v[2][t], lane, true);   // - xi wr
      wrelax1(are, lane);
      wrelax1(aim, lane);
    }
  }
  __syncthreads();  // s_red[0] is still being read by slower warps
  are = block_sum(are, 1);
  aim = block_sum(aim, 0);
  const int32_t sr = wfinish(are, lane), si = wfinish(aim, lane);
  if (warp == 0 && dl) {
    theta[(size_t)lane * n * nb + (size_t)b * n + j] = sr;
    const size_t ejj = (size_t)b * per + (size_t)j * n + j;
    S[(size_t)lane * count + ejj] = sr;
    S[((size_t)ND + lane) * count + ejj] = si;
  }
  // r = w - x s
  int32_t sall[ND];
  int mymsb = 0;
#pragma unroll 1
  for (int part = 0; part < 2; ++part) {
    // part 0: xr sr - xi si ;  part 1: xr si + xi sr
#pragma unroll
    for (int t = 0; t < SW_RPW; ++t) {
      const int k = warp + t * nw;
      if (k < n) {
        int64_t a2 = 0;
        wbroadcast(sall, part ? si : sr);
        wmac_u(a2, sall, v[0][t], lane, false);
        wbroadcast(sall, part ? sr : si);
        wmac_u(a2, sall, v[1][t], lane, part == 0);
        const int32_t tt = wfinish(a2, lane);
        const int32_t o = (int32_t)wcanon<ND - 1>(dl ? (int64_t)v[2 + part][t] - tt : 0, lane);
        if (dl) R[((size_t)part * ND + lane) * count + (size_t)b * per + (size_t)k * n + j] = o;
        mymsb = max(mymsb, wmsb(o, lane));
      }
    }
  }
  if (lane == 0 && mymsb) atomicMax(&s_msb, mymsb);
  __syncthreads();
  if (threadIdx.x == 0 && msb_r_out && s_msb) atomicMax(msb_r_out, s_msb);
}

int singleton_step(int n, int nb, int32_t* X, int32_t* W, int32_t* R, int32_t* S, int32_t* theta, int* msb_g_out, int* msb_r_out,
                   cudaStream_t s, const int* cl, const int* cle, int* msb_g_b) {
  KtScope kt_scope(KC_SSTEP, s, 14ull * 494ull * (uint64_t)n * n * nb);
  // columns per CTA: as many as keep about one CTA per SM (sector efficiency of the row-major loads against parallelism)
  const size_t cols = (size_t)n * nb;
  const int forced = options().sstep_cpb;
  const int cpb = (forced == 1 || forced == 2 || forced == 4 || forced == 8) ? forced
                  : cols >= 8 * 128 ? 8 : cols >= 4 * 96 ? 4 : cols >= 2 * 96 ? 2 : 1;
  const unsigned grid = (unsigned)((size_t)((n + cpb - 1) / cpb) * nb);
  if (cpb == 1 && n <= 16 * SW_RPW && options().sstep_warp) {
    const int nw = (n + SW_RPW - 1) / SW_RPW;
    singleton_step_warp_kernel<<<grid, 32 * nw, 0, s>>>(n, nb, X, W, R, S, theta, msb_g_out, msb_r_out, cl, cle, msb_g_b);
  } else if (cpb == 1 && options().sstep_par && n <= 96 && sizeof(int32_t) * 4 * ND * (size_t)n <= 40 * 1024) {
    int threads = (4 * n + 31) / 32 * 32;
    if (threads > 256) threads = 256;  // 255 registers per thread: the digit arrays of g, m, s and one accumulator set stay in registers
    singleton_step_par_kernel<<<grid, threads, sizeof(int32_t) * 4 * ND * (size_t)n, s>>>(n, nb, X, W, R, S, theta, msb_g_out, msb_r_out, cl, cle,
                                                                                       msb_g_b);
  } else if (cpb == 1) {
    int threads = (n + 31) / 32 * 32;
    if (threads > 256) threads = 256;
    const size_t cache = sizeof(int32_t) * 4 * ND * (size_t)n;  // 480 n bytes
    if (cache + 8 * FXP_NACC * sizeof(int64_t) + 64 <= 48 * 1024 && options().sstep_cache)
      singleton_step_kernel<1, true><<<grid, threads, cache, s>>>(n, nb, X, W, R, S, theta, msb_g_out, msb_r_out, cl, cle, msb_g_b);
    else
      singleton_step_kernel<1, false><<<grid, threads, 0, s>>>(n, nb, X, W, R, S, theta, msb_g_out, msb_r_out, cl, cle, msb_g_b);
  } else if (cpb == 2) {
    singleton_step_kernel<2, false><<<grid, 256, 0, s>>>(n, nb, X, W, R, S, theta, msb_g_out, msb_r_out, cl, cle, msb_g_b);
  } else if (cpb == 4) {
    singleton_step_kernel<4, false><<<grid, 256, 0, s>>>(n, nb, X, W, R, S, theta, msb_g_out, msb_r_out, cl, cle, msb_g_b);
  } else {
    singleton_step_kernel<8, false><<<grid, 256, 0, s>>>(n, nb, X, W, R, S, theta, msb_g_out, msb_r_out, cl, cle, msb_g_b);
  }
  count_launch();
  return launch_check();
}

// ---- E_ij = C_ij / (theta_j - theta_i) across clusters, 0 inside ---------------------------------------------------------------
// One thread per entry (i, j) (the diagonal and the entries inside a cluster are zeroed).  d = theta_j - theta_i is normalised
// to d' = |d| 2^s in [1/4, 1/2) with a static barrel shifter, r = 1/d' by Newton from an fp64 start on W-digit fixed point
// (r in (2,4], FX-like with 29 - (30-W) fractional digits), then E_ij = sgn(d) (C_ij r) 2^s.  (i, j) and (j, i) each compute
// the reciprocal of the same |d|: a thread that served both entries read and wrote the (j, i) one with stride n (12.5
// sectors per request, half the threads idle: 0.76 ms per launch at n = 1024); per entry every access is coalesced.
template <int W>
__global__ void __launch_bounds__(128) ecalc_kernel(int n, int nb, const int32_t* __restrict__ theta, const int* __restrict__ cl,
                                                    int32_t* __restrict__ C, int newton_iters, int* __restrict__ msb_out,
                                                    int* __restrict__ err_flag) {
  const size_t per = (size_t)n * n, count = per * nb;
  const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= count) return;
  const int b = (int)(t / per), i = (int)((t % per) / n), j = (int)(t % n);
  int32_t* Cr = C;
  int32_t* Ci = C + (size_t)ND * count;
  const size_t eij = (size_t)b * per + (size_t)i * n + j;
  int32_t z[ND];
  fx_zero(z);
  if (cl[(size_t)b * n + i] == cl[(size_t)b * n + j]) {
    fx_store(Cr, count, eij, z); fx_store(Ci, count, eij, z);
    return;
  }
  int32_t ti[ND], tj[ND], d[ND];
  fx_load(ti, theta, (size_t)n * nb, (size_t)b * n + i);
  fx_load(tj, theta, (size_t)n * nb, (size_t)b * n + j);
  fx_sub(d, tj, ti);
  const bool dneg = fx_is_neg(d);
  if (dneg) { int32_t u[ND]; fx_neg(u, d);
#pragma unroll
    for (int k = 0; k < ND; ++k) d[k] = u[k]; }
  const int msb = fx_msb(d);  // |d| in [2^(msb-1-812), 2^(msb-812))
  if (msb < 812 - 400) {      // different clusters must be apart; anything this close is a planning error
    if (err_flag) atomicOr(err_flag, 2);
    fx_store(Cr, count, eij, z); fx_store(Ci, count, eij, z);
    return;
  }
  // d' = d 2^s with msb(d') = 811  (value in [1/4,1/2))
  const int s = 811 - msb;  // may be negative when |d| >= 1/2
  if (s >= 0) fx_shl(d, s); else fx_shr(d, -s);
  int32_t r[ND];
  fx_recip_quarter<W>(r, d, newton_iters);
  constexpr int LO = ND - 1 - W;
  int32_t rw[W + 1];
#pragma unroll
  for (int k = 0; k <= W; ++k) rw[k] = r[LO + k];
  // E = (C r) 2^s, with sign
  int mymsb = 0;
#pragma unroll 1
  for (int which = 0; which < 2; ++which) {
    int32_t* plane = (which & 1) ? Ci : Cr;
    const size_t e = eij;
    const bool neg = dneg;
    int32_t c[ND], o[ND];
    fx_load(c, plane, count, e);
    {
      // r has W + 1 nonzero digits (LO .. 29): the product needs 30 (W + 1) digit products, not 30 x 30; the kept columns
      // and the rounding are those of fx_mul
      int64_t acc[FXP_NACC];
      fxp_zero(acc);
      mac_cols<ND, W + 1, FXP_LOW - LO, FXP_NACC, false>(acc, c, rw);
      fxp_finish(o, acc);
    }
    if (s >= 0) fx_shl(o, s); else fx_shr(o, -s);
    if (neg) { int32_t u[ND]; fx_neg(u, o);
#pragma unroll
      for (int k = 0; k < ND; ++k) o[k] = u[k]; }
    fx_store(plane, count, e, o);
    mymsb = max(mymsb, fx_msb(o));
  }
  if (msb_out) atomicMax(msb_out, mymsb);
}
int ecalc(int n, int nb, const int32_t* theta, const int* cl, int32_t* C, int prec_bits, int* msb_out, int* err_flag, cudaStream_t s) {
  const size_t t = (size_t)n * n * nb;
  const unsigned blocks = (unsigned)((t + 127) / 128);
  // Newton doubles the ~50 correct bits of the fp64 start each iteration
  int iters = 0;
  for (int have = 48; have < prec_bits; have *= 2) ++iters;
  // digit products per entry i != j: two (W+1)^2-digit products per Newton iteration (half of them kept) and two 30 x (W+1)
  // products (executed); algorithmic: the reciprocal once per pair
  const uint64_t Wd = prec_bits <= 28 * 4 - 8 ? 5 : prec_bits <= 28 * 8 - 8 ? 9 : prec_bits <= 28 * 16 - 8 ? 17 : 30;
  KtScope kt_scope(KC_ECALC, s, (uint64_t)n * (n - 1) * nb * ((uint64_t)iters * Wd * (Wd + 3) + 2ull * ND * Wd),
                   (uint64_t)n * (n - 1) / 2 * nb * ((uint64_t)iters * Wd * (Wd + 3) + 4ull * ND * Wd));
  if (prec_bits <= 28 * 4 - 8) ecalc_kernel<4><<<blocks, 128, 0, s>>>(n, nb, theta, cl, C, iters, msb_out, err_flag);
  else if (prec_bits <= 28 * 8 - 8) ecalc_kernel<8><<<blocks, 128, 0, s>>>(n, nb, theta, cl, C, iters, msb_out, err_flag);
  else if (prec_bits <= 28 * 16 - 8) ecalc_kernel<16><<<blocks, 128, 0, s>>>(n, nb, theta, cl, C, iters, msb_out, err_flag);
  else ecalc_kernel<29><<<blocks, 128, 0, s>>>(n, nb, theta, cl, C, iters, msb_out, err_flag);
  count_launch();
  return launch_check();
}

}  // namespace zkd

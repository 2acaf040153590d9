// mps.cu — kernels of the minimal MPS two-site update.  PAPER.md:15 (section 1): an MPS is "a data
// structure ... nested Schmidt decomposition"; PAPER.md:39 (section 2.1): "Hermitian matrix diagonalization ... the dominant
// factor in the computational cost of the MPS simulation"; PAPER.md:35 (footnote): Schmidt weights as small as
// epsilon ~ 2^(-n+1) must be kept apart from zero, hence the multiprecision.  One update =
//     Theta0 = L R                  ((chiL d) x chiC times chiC x (d chiR): the two site tensors contracted over their bond)
//     Theta  = gate on the two physical indices of Theta0
//     rho    = Theta Theta^H        (the reduced density matrix of the left half, Hermitian PSD)
//     rho    = U diag(w) U^H        (the hot path: zkd's Hermitian eigendecomposition; w = Schmidt weights)
//     L' = U[:, kept], R' = L'^H Theta, kept = the weights above 2^-cutoff_bits trace(rho), at most max_keep of them.
// The GEMMs and the eigendecomposition are the library's; this file holds the small tensor plumbing.  Driver: mps_update_device
// in pipeline.cu.
#include "blocks.h"
#include "fx_funcs.cuh"
#include "timing.h"

namespace zkd {

// dst[b] (C x R) = conj(src[b] (R x C))^T
__global__ void __launch_bounds__(256) conj_transpose_kernel(int R, int C, int batch, const int32_t* __restrict__ src, int32_t* __restrict__ dst) {
  const size_t per = (size_t)R * C, count = per * batch;
  const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= 2 * count) return;
  const int part = (int)(t / count);
  const size_t e = t % count;
  const int b = (int)(e / per), c = (int)((e % per) / R), r = (int)(e % R);  // destination element (c, r)
  int32_t d[ND];
  fx_load(d, src + (part ? (size_t)ND * count : 0), count, (size_t)b * per + (size_t)r * C + c);
  if (part) { int32_t t2[ND]; fx_neg(t2, d);
#pragma unroll
    for (int k = 0; k < ND; ++k) d[k] = t2[k]; }
  fx_store(dst + (part ? (size_t)ND * count : 0), count, e, d);
}
int conj_transpose(int R, int C, int batch, const int32_t* src, int32_t* dst, cudaStream_t s) {
  KtScope kt(KC_OTHER, s);
  const size_t t = 2 * (size_t)R * C * batch;
  conj_transpose_kernel<<<(unsigned)((t + 255) / 256), 256, 0, s>>>(R, C, batch, src, dst);
  count_launch();
  return launch_check();
}

// Theta[(a, i'), (j', c)] = sum_{i, j} G[(i' j'), (i j)] Theta0[(a, i), (j, c)];  Theta0, Theta: (chiL d) x (d chiR), G: d^2 x d^2 per
// batch element.  One thread per output element; msb_out <- max msb of the result (sizes the next scale).
__global__ void __launch_bounds__(128) mps_gate_kernel(int chiL, int chiR, int d, int batch, const int32_t* __restrict__ T0,
                                                       const int32_t* __restrict__ G, int32_t* __restrict__ T, int* __restrict__ msb_out) {
  const int mL = chiL * d, mR = d * chiR, d2 = d * d;
  const size_t per = (size_t)mL * mR, count = per * batch, gcount = (size_t)d2 * d2 * batch;
  const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= count) return;
  const int b = (int)(e / per), row = (int)((e % per) / mR), col = (int)(e % mR);
  const int a = row / d, ip = row % d, jp = col / chiR, c = col % chiR;
  int64_t accr[FXP_NACC], acci[FXP_NACC];
  fxp_zero(accr); fxp_zero(acci);
#pragma unroll 1
  for (int ij = 0; ij < d2; ++ij) {
    const int i = ij / d, j = ij % d;
    int32_t gr[ND], gi[ND], xr[ND], xi[ND];
    const size_t ge = (size_t)b * d2 * d2 + (size_t)(ip * d + jp) * d2 + ij;
    const size_t xe = (size_t)b * per + (size_t)(a * d + i) * mR + (j * chiR + c);
    fx_load(gr, G, gcount, ge); fx_load(gi, G + (size_t)ND * gcount, gcount, ge);
    fx_load(xr, T0, count, xe); fx_load(xi, T0 + (size_t)ND * count, count, xe);
    fx_mac<false>(accr, gr, xr); fx_mac<true>(accr, gi, xi);
    fx_mac<false>(acci, gr, xi); fx_mac<false>(acci, gi, xr);
    fxp_relax(accr); fxp_relax(acci);
  }
  int32_t o[ND];
  fxp_finish(o, accr);
  int m = fx_msb(o);
  fx_store(T, count, e, o);
  fxp_finish(o, acci);
  m = max(m, fx_msb(o));
  fx_store(T + (size_t)ND * count, count, e, o);
  for (int off = 16; off > 0; off >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, off));
  if ((threadIdx.x & 31) == 0 && m) atomicMax(msb_out, m);
}
int mps_gate(int chiL, int chiR, int d, int batch, const int32_t* T0, const int32_t* G, int32_t* T, int* msb_out, cudaStream_t s) {
  KtScope kt(KC_OTHER, s);
  const size_t t = (size_t)chiL * d * d * chiR * batch;
  mps_gate_kernel<<<(unsigned)((t + 127) / 128), 128, 0, s>>>(chiL, chiR, d, batch, T0, G, T, msb_out);
  count_launch();
  return launch_check();
}

// complex FX array << bits
__global__ void __launch_bounds__(256) fxc_shl_kernel(size_t reals, int32_t* __restrict__ X, int bits) {
  const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= reals) return;
  const size_t count = reals / 2;
  int32_t* p = X + (e / count) * (size_t)ND * count;
  int32_t d[ND];
  fx_load(d, p, count, e % count);
  fx_shl(d, bits);
  fx_store(p, count, e % count, d);
}
int fxc_shl(size_t count, int32_t* X, int bits, cudaStream_t s) {
  KtScope kt(KC_OTHER, s);
  fxc_shl_kernel<<<(unsigned)((2 * count + 255) / 256), 256, 0, s>>>(2 * count, X, bits);
  count_launch();
  return launch_check();
}

// weights (descending, negative noise clamped to zero), kept count, and L'[:, k] <- the phase-normalised eigenvector of rank n-1-k.
// Xs: eigenvectors already sorted ASCENDING and phase-normalised (phase_kernel's output), lam_sorted ascending.
__global__ void __launch_bounds__(128) mps_select_kernel(int n, int K, int batch, int cutoff_bits, const int32_t* __restrict__ lam_sorted,
                                                         int32_t* __restrict__ Wt, int* __restrict__ kept) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= batch) return;
  int32_t tr[ND], d[ND], t[ND];
  fx_zero(tr);
  for (int j = 0; j < n; ++j) {
    fx_load(d, lam_sorted, (size_t)n * batch, (size_t)b * n + j);
    if (d[ND - 1] >= 0) { fx_add(t, tr, d);
#pragma unroll
      for (int q = 0; q < ND; ++q) tr[q] = t[q]; }
  }
  fx_shr(tr, cutoff_bits);  // trace 2^-cutoff
  int k0 = 0;
  for (int k = 0; k < K; ++k) {
    fx_load(d, lam_sorted, (size_t)n * batch, (size_t)b * n + (n - 1 - k));
    if (d[ND - 1] < 0) fx_zero(d);
    fx_store(Wt, (size_t)K * batch, (size_t)b * K + k, d);
    fx_sub(t, d, tr);
    if (t[ND - 1] >= 0 && fx_msb(t) > 0) ++k0;  // w_k > 2^-cutoff trace (weights descend: the kept ones come first)
  }
  kept[b] = k0;
}
int mps_select(int n, int K, int batch, int cutoff_bits, const int32_t* lam_sorted, int32_t* Wt, int* kept, cudaStream_t s) {
  KtScope kt(KC_OTHER, s);
  mps_select_kernel<<<(batch + 127) / 128, 128, 0, s>>>(n, K, batch, cutoff_bits, lam_sorted, Wt, kept);
  count_launch();
  return launch_check();
}
__global__ void __launch_bounds__(256) mps_take_kernel(int n, int K, int batch, const int32_t* __restrict__ Xs, int32_t* __restrict__ Lnew) {
  const size_t xcount = (size_t)n * n * batch, lcount = (size_t)n * K * batch;
  const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= 2 * lcount) return;
  const int part = (int)(t / lcount);
  const size_t e = t % lcount;
  const int b = (int)(e / ((size_t)n * K)), r = (int)((e % ((size_t)n * K)) / K), k = (int)(e % K);
  int32_t d[ND];
  fx_load(d, Xs + (part ? (size_t)ND * xcount : 0), xcount, (size_t)b * n * n + (size_t)r * n + (n - 1 - k));
  fx_store(Lnew + (part ? (size_t)ND * lcount : 0), lcount, e, d);
}
int mps_take(int n, int K, int batch, const int32_t* Xs, int32_t* Lnew, cudaStream_t s) {
  KtScope kt(KC_OTHER, s);
  const size_t t = 2 * (size_t)n * K * batch;
  mps_take_kernel<<<(unsigned)((t + 255) / 256), 256, 0, s>>>(n, K, batch, Xs, Lnew);
  count_launch();
  return launch_check();
}

// out[b] = a[b] + b2[b] + c[b] - t (scales of Theta), w[b] = 2 out[b] - u (scale of the weights)
__global__ void mps_scales_kernel(int batch, const int* sl, const int* sr, const int* sg, int t, int u, int* s_theta, int* s_w) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= batch) return;
  const int st = sl[b] + sr[b] + sg[b] + t;
  s_theta[b] = st;
  s_w[b] = 2 * st + u;
}
int mps_scales(int batch, const int* sl, const int* sr, const int* sg, int t, int u, int* s_theta, int* s_w, cudaStream_t s) {
  mps_scales_kernel<<<(batch + 127) / 128, 128, 0, s>>>(batch, sl, sr, sg, t, u, s_theta, s_w);
  count_launch();
  return launch_check();
}

}  // namespace zkd

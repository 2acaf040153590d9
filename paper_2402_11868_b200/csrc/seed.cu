// seed.cu — S1: fp64 Hermitian eigendecomposition seed, hand-written (no cuSOLVER).
//
// ZKCM_CUS takes "double-precision calculations of CUSOLVER routines" as the starting point that RQI
// then refines.  Here the seed is a one-sided (Hestenes) Jacobi iteration on G = A + sigma I (sigma from Gershgorin,
// so G is positive definite with condition number <= 5): column pairs (g_p, g_q) are rotated until all columns are
// mutually orthogonal.  Then G_final = G V with V the accumulated rotations and G_final's columns are orthogonal, so
// A v_j = mu_j v_j with v_j = g_j / ||g_j|| and mu_j = ||g_j|| - sigma: V is read off the rotated G and is never
// accumulated (G is well conditioned, so the normalised columns are orthonormal to the level the sweeps reached).
// Only column operations occur, so a round of n/2 disjoint pairs is embarrassingly parallel: one warp per pair,
// round-robin (tournament) ordering, one barrier per round.
//
//   n <= 256 : thread-block CLUSTER per matrix (1, 2, 4 or 8 CTAs).  G lives in distributed shared memory, column j in
//              the shared memory of CTA j / cpc; a warp pulls its two columns through DSMEM into registers, rotates, and
//              writes them back; rounds are separated by the hardware cluster barrier (about 0.2 us) instead of a grid
//              barrier through L2.  With many matrices in the batch the cluster size drops to 1 CTA (one SM per matrix).
//   n  > 256 : cooperative grid, G in global memory (L2 resident), grid.sync between rounds.
// The seed only has to be good to ~2^-40 (the refinement squares the error every step).
#include <cooperative_groups.h>

#include "zkd_internal.h"

namespace cg = cooperative_groups;

namespace zkd {

constexpr double kSeedStopCos2 = 8.8817841970012523e-16;  // 2^-50

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
  return v;
}

// Rotation parameters without divisions or square roots (three rsqrt): with d = (be - al)/2 and gamma = g_p^H g_q,
//   w = sgn(d) / (|d| + sqrt(d^2 + |gamma|^2)),  tau = w gamma (|tau| <= 1: the tangent times the phase of gamma),
//   c = 1/sqrt(1 + |tau|^2),  sigma = c tau;   [g_p, g_q] <- [c g_p - conj(sigma) g_q,  sigma g_p + c g_q].
// Only c^2 + |sigma|^2 = 1 has to hold to working precision (one rsqrt); an error in w merely perturbs the angle.
// Returns false when the pair is already orthogonal to tol (or a column is zero).  cos2 = |cos(g_p, g_q)|^2.
__device__ __forceinline__ bool rot_params(double al, double be, double gr, double gi, double tol2, double& c, double& sr,
                                           double& si, double& cos2) {
  const double g2 = gr * gr + gi * gi;
  const double ab = al * be;
  cos2 = 0.0;
  if (!(g2 > tol2 * ab) || g2 == 0.0) return false;
  cos2 = g2 * (1.0 / ab);
  const double d = 0.5 * (be - al);
  const double x = fma(d, d, g2);
  const double h = x * rsqrt(x);  // sqrt(d^2 + |gamma|^2)
  const double r2 = rsqrt(fabs(d) + h);
  const double w = copysign(r2 * r2, d);  // sgn(0) = +1
  const double tr = gr * w, ti = gi * w;
  c = rsqrt(fma(tr, tr, fma(ti, ti, 1.0)));
  sr = c * tr;
  si = c * ti;
  return true;
}

// round-robin pairing for M (even) players, round r in [0, M-1), pair index i in [0, M/2)
__device__ __forceinline__ void rr_pair(int M, int r, int i, int& p, int& q) {
  if (i == 0) { p = M - 1; q = r % (M - 1); }
  else { p = (r + i) % (M - 1); q = (r + (M - 1) - i) % (M - 1); }
  if (p > q) { int t = p; p = q; q = t; }
}

// ---- n <= 256: one thread-block cluster per matrix, G in distributed shared memory -------------------------------------
// EPL = elements of a column per lane (n <= 32 EPL).  Dynamic shared memory: cpc columns of n complex doubles.
template <int EPL>
__global__ void __launch_bounds__(EPL >= 8 ? 512 : 1024)
seed_cluster_kernel(int n, int cpc, const double2* __restrict__ A, double* __restrict__ mu, double2* __restrict__ V,
                    int max_sweeps, double tol2) {
  extern __shared__ double2 Gl[];                 // [cpc][n] : columns rank*cpc .. rank*cpc + cpc - 1
  __shared__ double s_mu[256];                    // full copy of the unsorted eigenvalues (every CTA)
  __shared__ unsigned long long s_cmax[2];        // per-sweep max cos^2 of this CTA (bits of a non-negative double)
  __shared__ double s_rmax;                       // this CTA's largest Gershgorin row sum
  __shared__ double s_red[32];
  cg::cluster_group cluster = cg::this_cluster();
  const int csize = (int)cluster.num_blocks(), rank = (int)cluster.block_rank();
  const int b = blockIdx.x / csize;
  const int tid = threadIdx.x, nthr = blockDim.x, lane = tid & 31, warp = tid >> 5, nwarps = nthr >> 5;
  const double2* Ab = A + (size_t)b * n * n;
  const int j0 = rank * cpc, j1 = min(n, j0 + cpc);

  // own columns of the Hermitian matrix built from the upper triangle (unshifted), and their absolute sums
  for (int e = tid; e < (j1 - j0) * n; e += nthr) {
    const int jl = e / n, i = e - jl * n, j = j0 + jl;
    double2 a = (i <= j) ? Ab[(size_t)i * n + j] : Ab[(size_t)j * n + i];
    if (i > j) a.y = -a.y;
    if (i == j) a.y = 0;
    Gl[(size_t)jl * n + i] = a;
  }
  if (tid == 0) { s_cmax[0] = 0ull; s_cmax[1] = 0ull; }
  __syncthreads();
  double rmax = 0;
  for (int jl = warp; jl < j1 - j0; jl += nwarps) {
    double rs = 0;
    for (int i = lane; i < n; i += 32) {
      const double2 a = Gl[(size_t)jl * n + i];
      rs += (i == j0 + jl) ? fabs(a.x) : sqrt(a.x * a.x + a.y * a.y);
    }
    rmax = fmax(rmax, warp_sum(rs));
  }
  if (lane == 0) s_red[warp] = rmax;
  __syncthreads();
  if (tid == 0) {
    double m = 0;
    for (int w = 0; w < nwarps; ++w) m = fmax(m, s_red[w]);
    s_rmax = m;
  }
  cluster.sync();
  double sigma = 0;
  for (int r = 0; r < csize; ++r) sigma = fmax(sigma, *cluster.map_shared_rank(&s_rmax, r));
  sigma *= 1.5;
  for (int jl = tid; jl < j1 - j0; jl += nthr) Gl[(size_t)jl * n + (j0 + jl)].x += sigma;
  cluster.sync();

  const int M = n + (n & 1), npairs = M / 2;
  const int gwarp = rank * nwarps + warp, gwarps = csize * nwarps;
  if (n > 1 && sigma > 0) {
    for (int sweep = 0; sweep < max_sweeps; ++sweep) {
      double cmax = 0;
      for (int r = 0; r < M - 1; ++r) {
        for (int i = gwarp; i < npairs; i += gwarps) {
          int p, q;
          rr_pair(M, r, i, p, q);
          if (q >= n) continue;
          double2* gp = cluster.map_shared_rank(Gl + (size_t)(p % cpc) * n, p / cpc);
          double2* gq = cluster.map_shared_rank(Gl + (size_t)(q % cpc) * n, q / cpc);
          double2 a[EPL], bb[EPL];
          double al = 0, be = 0, gr = 0, gi = 0;
#pragma unroll
          for (int k = 0; k < EPL; ++k) {
            const int i2 = lane + 32 * k;
            a[k] = i2 < n ? gp[i2] : make_double2(0, 0);
            bb[k] = i2 < n ? gq[i2] : make_double2(0, 0);
          }
#pragma unroll
          for (int k = 0; k < EPL; ++k) {
            al = fma(a[k].x, a[k].x, fma(a[k].y, a[k].y, al));
            be = fma(bb[k].x, bb[k].x, fma(bb[k].y, bb[k].y, be));
            gr = fma(a[k].x, bb[k].x, fma(a[k].y, bb[k].y, gr));  // conj(a) b
            gi = fma(a[k].x, bb[k].y, fma(-a[k].y, bb[k].x, gi));
          }
          al = warp_sum(al); be = warp_sum(be); gr = warp_sum(gr); gi = warp_sum(gi);
          double c, sr, si, cos2;
          if (!rot_params(al, be, gr, gi, tol2, c, sr, si, cos2)) continue;
          cmax = fmax(cmax, cos2);
#pragma unroll
          for (int k = 0; k < EPL; ++k) {
            const int i2 = lane + 32 * k;
            if (i2 < n) {
              gp[i2] = make_double2(c * a[k].x - (sr * bb[k].x + si * bb[k].y), c * a[k].y - (sr * bb[k].y - si * bb[k].x));
              gq[i2] = make_double2(sr * a[k].x - si * a[k].y + c * bb[k].x, sr * a[k].y + si * a[k].x + c * bb[k].y);
            }
          }
        }
        if (r == M - 2 && lane == 0 && cmax > 0) atomicMax(&s_cmax[sweep & 1], (unsigned long long)__double_as_longlong(cmax));
        cluster.sync();
      }
      // A sweep whose largest |cos| was below 2^-22 leaves every pair below ~2^-44 (quadratic convergence): stop there.
      double worst = 0;
      for (int r = 0; r < csize; ++r)
        worst = fmax(worst, __longlong_as_double((long long)*cluster.map_shared_rank(&s_cmax[sweep & 1], r)));
      if (tid == 0) s_cmax[(sweep + 1) & 1] = 0ull;  // last read by the other CTAs one sweep (many barriers) ago
      __syncthreads();
      if (!(worst > kSeedStopCos2)) break;
    }
  }
  cluster.sync();  // nobody may leave (or overwrite s_cmax) while a neighbour still reads its shared memory

  // mu_j = ||g_j|| - sigma for own columns, broadcast to every CTA of the cluster; normalise own columns in place
  for (int jl = warp; jl < j1 - j0; jl += nwarps) {
    double s = 0;
    for (int i = lane; i < n; i += 32) { const double2 a = Gl[(size_t)jl * n + i]; s += a.x * a.x + a.y * a.y; }
    s = warp_sum(s);
    const double nrm = sqrt(s);
    const double inv = nrm > 0 ? 1.0 / nrm : 0.0;
    for (int i = lane; i < n; i += 32) {
      double2 a = Gl[(size_t)jl * n + i];
      if (nrm > 0) { a.x *= inv; a.y *= inv; } else { a = make_double2(i == j0 + jl ? 1.0 : 0.0, 0.0); }
      Gl[(size_t)jl * n + i] = a;
    }
    if (lane < csize) *cluster.map_shared_rank(&s_mu[j0 + jl], lane) = nrm - sigma;
  }
  cluster.sync();
  // stable rank sort ascending; V[i][rank] = column j
  for (int jl = warp; jl < j1 - j0; jl += nwarps) {
    const int j = j0 + jl;
    const double mj = s_mu[j];
    int rk = 0;
    for (int i = lane; i < n; i += 32) {
      const double mi = s_mu[i];
      rk += (mi < mj) || (mi == mj && i < j);
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) rk += __shfl_xor_sync(0xffffffffu, rk, off);
    if (lane == 0) mu[(size_t)b * n + rk] = mj;
    for (int i = lane; i < n; i += 32) V[(size_t)b * n * n + (size_t)i * n + rk] = Gl[(size_t)jl * n + i];
  }
  cluster.sync();
}

template <int EPL>
static int launch_cluster(int N, int batch, int csize, const double2* A, double* mu, double2* V, int max_sweeps, double tol2,
                          cudaStream_t s) {
  const int M = N + (N & 1), npairs = M / 2;
  const int cpc = (N + csize - 1) / csize;
  int warps = (npairs + csize - 1) / csize;
  const int maxw = EPL >= 8 ? 16 : 32;
  if (warps > maxw) warps = maxw;
  if (warps < 1) warps = 1;
  const size_t smem = sizeof(double2) * (size_t)cpc * N;
  static size_t attr_smem = 0;
  if (smem > attr_smem) {
    ZKD_CUDA_TRY(cudaFuncSetAttribute(seed_cluster_kernel<EPL>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(smem > 48 * 1024 ? smem : 48 * 1024)));
    attr_smem = smem > 48 * 1024 ? smem : 48 * 1024;
  }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)(batch * csize));
  cfg.blockDim = dim3((unsigned)(32 * warps));
  cfg.dynamicSmemBytes = smem;
  cfg.stream = s;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = (unsigned)csize;
  at[0].val.clusterDim.y = 1;
  at[0].val.clusterDim.z = 1;
  cfg.attrs = at;
  cfg.numAttrs = 1;
  ZKD_CUDA_TRY(cudaLaunchKernelEx(&cfg, seed_cluster_kernel<EPL>, N, cpc, A, mu, V, max_sweeps, tol2));
  count_launch();
  return launch_check();
}

// ---- large matrices: cooperative grid ------------------------------------------------------------------------------
__global__ void seed_sigma_kernel(int n, const double2* __restrict__ A, double* sigma_out) {
  // one block, one warp per row; Gershgorin radius
  __shared__ double s_red[32];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarps = blockDim.x >> 5;
  double rmax = 0;
  for (int i = warp; i < n; i += nwarps) {
    double rs = 0;
    for (int j = lane; j < n; j += 32) {
      const double2 a = (i <= j) ? A[(size_t)i * n + j] : A[(size_t)j * n + i];
      rs += (i == j) ? fabs(a.x) : sqrt(a.x * a.x + a.y * a.y);
    }
    rmax = fmax(rmax, warp_sum(rs));
  }
  if (lane == 0) s_red[warp] = rmax;
  __syncthreads();
  if (tid == 0) {
    double m = 0;
    for (int w = 0; w < nwarps; ++w) m = fmax(m, s_red[w]);
    *sigma_out = 1.5 * m;
  }
}

// one warp: orthogonalise columns p, q of G (length n, global memory)
__device__ __forceinline__ double rotate_pair_global(double2* __restrict__ gp, double2* __restrict__ gq, int n, int lane, double tol2) {
  double al = 0, be = 0, gr = 0, gi = 0;
  for (int i = lane; i < n; i += 32) {
    const double2 a = __ldcg(gp + i), b = __ldcg(gq + i);
    al = fma(a.x, a.x, fma(a.y, a.y, al));
    be = fma(b.x, b.x, fma(b.y, b.y, be));
    gr = fma(a.x, b.x, fma(a.y, b.y, gr));
    gi = fma(a.x, b.y, fma(-a.y, b.x, gi));
  }
  al = warp_sum(al); be = warp_sum(be); gr = warp_sum(gr); gi = warp_sum(gi);
  double c, sr, si, cos2;
  if (!rot_params(al, be, gr, gi, tol2, c, sr, si, cos2)) return cos2;
  for (int i = lane; i < n; i += 32) {
    const double2 a = __ldcg(gp + i), b = __ldcg(gq + i);
    __stcg(gp + i, make_double2(c * a.x - (sr * b.x + si * b.y), c * a.y - (sr * b.y - si * b.x)));
    __stcg(gq + i, make_double2(sr * a.x - si * a.y + c * b.x, sr * a.y + si * a.x + c * b.y));
  }
  return cos2;
}

__global__ void __launch_bounds__(128) seed_large_kernel(int n, const double2* __restrict__ A, double2* __restrict__ G,
                                                         const double* __restrict__ sigma_p, int* __restrict__ rot_flags,
                                                         double* __restrict__ mu_unsorted, int max_sweeps, double tol2) {
  cg::grid_group grid = cg::this_grid();
  const int tid = threadIdx.x, lane = tid & 31;
  const int gwarp = (blockIdx.x * blockDim.x + tid) >> 5, nwarps = (gridDim.x * blockDim.x) >> 5;
  const size_t gtid = (size_t)blockIdx.x * blockDim.x + tid, gthr = (size_t)gridDim.x * blockDim.x;
  const double sigma = *sigma_p;
  for (size_t e = gtid; e < (size_t)n * n; e += gthr) {
    const int i = (int)(e % n), j = (int)(e / n);
    double2 a = (i <= j) ? A[(size_t)i * n + j] : A[(size_t)j * n + i];
    if (i > j) a.y = -a.y;
    if (i == j) { a.y = 0; a.x += sigma; }
    G[e] = a;
  }
  if (gtid < (size_t)max_sweeps) rot_flags[gtid] = 0;
  grid.sync();
  const int M = n + (n & 1), npairs = M / 2;
  if (sigma > 0) {
    for (int sweep = 0; sweep < max_sweeps; ++sweep) {
      double cmax = 0;
      for (int r = 0; r < M - 1; ++r) {
        for (int i = gwarp; i < npairs; i += nwarps) {
          int p, q;
          rr_pair(M, r, i, p, q);
          if (q < n) cmax = fmax(cmax, rotate_pair_global(G + (size_t)p * n, G + (size_t)q * n, n, lane, tol2));
        }
        if (r == M - 2 && cmax > kSeedStopCos2 && lane == 0) rot_flags[sweep] = 1;
        grid.sync();
      }
      if (!rot_flags[sweep]) break;
    }
  }
  for (int j = gwarp; j < n; j += nwarps) {
    double s = 0;
    for (int i = lane; i < n; i += 32) { const double2 a = G[(size_t)j * n + i]; s += a.x * a.x + a.y * a.y; }
    s = warp_sum(s);
    if (lane == 0) mu_unsorted[j] = sqrt(s) - sigma;
  }
}

// V[i][rank(j)] = g_j[i] / ||g_j||, mu[rank(j)] = mu_j; one CTA per group of source columns, coalesced on the source
__global__ void __launch_bounds__(256) seed_sort_kernel(int n, const double* __restrict__ mu_unsorted, const double2* __restrict__ G,
                                                        const double* __restrict__ sigma_p, double* __restrict__ mu,
                                                        double2* __restrict__ V) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
  const double sigma = *sigma_p;
  for (int j = blockIdx.x * nwarps + warp; j < n; j += gridDim.x * nwarps) {
    const double mj = mu_unsorted[j];
    int rk = 0;
    for (int k = lane; k < n; k += 32) {
      const double mk = mu_unsorted[k];
      rk += (mk < mj) || (mk == mj && k < j);
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) rk += __shfl_xor_sync(0xffffffffu, rk, off);
    const double nrm = mj + sigma;
    const double inv = nrm > 0 ? 1.0 / nrm : 0.0;
    for (int i = lane; i < n; i += 32) {
      double2 a = G[(size_t)j * n + i];
      if (nrm > 0) { a.x *= inv; a.y *= inv; } else { a = make_double2(i == j ? 1.0 : 0.0, 0.0); }
      V[(size_t)i * n + rk] = a;
    }
    if (lane == 0) mu[rk] = mj;
  }
}

int seed_fp64(int N, int batch, const double* A64, double* mu, double* V, int max_sweeps, cudaStream_t s) {
  const double tol = ldexp(1.0, -50);
  const double tol2 = tol * tol;
  int dev = 0, sms = 0;
  ZKD_CUDA_TRY(cudaGetDevice(&dev));
  ZKD_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  if (N <= 256) {
    // cluster size: enough CTAs to give every pair of a round its own warp (4 warps per CTA at least), shrunk while the
    // batch alone fills the machine, grown while a CTA's columns do not fit its shared memory
    const int npairs = (N + 1) / 2;
    int csize = 1;
    while (csize < 8 && npairs > 4 * csize) csize *= 2;
    while (csize > 1 && (long)batch * csize > 2L * sms) csize /= 2;
    while (csize < 8 && sizeof(double2) * (size_t)((N + csize - 1) / csize) * N > 200 * 1024) csize *= 2;
    const double2* A = (const double2*)A64;
    double2* Vv = (double2*)V;
    if (N <= 64) return launch_cluster<2>(N, batch, csize, A, mu, Vv, max_sweeps, tol2, s);
    if (N <= 128) return launch_cluster<4>(N, batch, csize, A, mu, Vv, max_sweeps, tol2, s);
    return launch_cluster<8>(N, batch, csize, A, mu, Vv, max_sweeps, tol2, s);
  }
  // large: cooperative grid, one matrix at a time
  const int M = N + (N & 1);
  int nblocks = (M / 2 + 3) / 4;  // 4 warps (pairs) per block
  int maxb = 0;
  ZKD_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&maxb, seed_large_kernel, 128, 0));
  if (nblocks > maxb * sms) nblocks = maxb * sms;
  char* buf = nullptr;
  const size_t nn = (size_t)N * N;
  const size_t bytes = sizeof(double2) * nn + sizeof(double) * (N + 8) + sizeof(int) * 64;
  ZKD_CUDA_TRY(cudaMallocAsync((void**)&buf, bytes, s));
  double2* G = (double2*)buf;
  double* sigma = (double*)(G + nn);
  double* mu_uns = sigma + 8;
  int* flags = (int*)(mu_uns + N);
  int rc = ZKD_OK;
  for (int b = 0; b < batch && rc == ZKD_OK; ++b) {
    const double2* Ab = (const double2*)A64 + (size_t)b * nn;
    seed_sigma_kernel<<<1, 1024, 0, s>>>(N, Ab, sigma);
    double* mub = mu + (size_t)b * N;
    double2* Vb = (double2*)V + (size_t)b * nn;
    int n = N, ms = max_sweeps > 64 ? 64 : max_sweeps;
    double t2 = tol2;
    void* args[] = {&n, (void*)&Ab, &G, &sigma, &flags, &mu_uns, &ms, &t2};
    if (cudaLaunchCooperativeKernel((void*)seed_large_kernel, dim3(nblocks), dim3(128), args, 0, s) != cudaSuccess) {
      (void)cudaGetLastError();
      rc = ZKD_ERR_CUDA;
      break;
    }
    seed_sort_kernel<<<sms, 256, 0, s>>>(N, mu_uns, G, sigma, mub, Vb);
    count_launch(3);
    rc = launch_check();
  }
  cudaFreeAsync(buf, s);
  return rc;
}

}  // namespace zkd

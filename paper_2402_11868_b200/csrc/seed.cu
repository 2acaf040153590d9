// seed.cu — S1: fp64 Hermitian eigendecomposition seed, hand-written (no cuSOLVER), and S2's sort.
//
// ZKCM_CUS takes "double-precision calculations of CUSOLVER routines" as the starting point that RQI
// then refines.  Here the seed is a one-sided (Hestenes) Jacobi iteration on G = A + sigma I (sigma from Gershgorin,
// so G is positive definite with condition number <= 5): column pairs (g_p, g_q) are rotated until all columns are
// mutually orthogonal; then G V = V diag(mu + sigma), i.e. the columns of V are eigenvectors of A and
// mu_j = ||g_j|| - sigma.  Only column operations occur, so a round of n/2 disjoint pairs is embarrassingly
// parallel: one warp per pair.
//   n <= 64 : one CTA per matrix, G and V resident in shared memory, __syncthreads between rounds (batched).
//   n  > 64 : cooperative grid, G and V in global memory (L2 resident), grid.sync between rounds.
// The seed only has to be good to ~2^-40 (the refinement squares the error every step); V is a product of plane
// rotations and therefore unitary to ~2^-50 regardless of how early the sweeps stop.
#include <cooperative_groups.h>

#include "zkd_internal.h"

namespace cg = cooperative_groups;

namespace zkd {

struct PairRot {
  double c, sr, si;
  bool active;
};

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
  return v;
}

// one warp: orthogonalise columns p, q of G (length n, column-major complex) and apply the same rotation to V.
__device__ __forceinline__ bool rotate_pair(double2* __restrict__ gp, double2* __restrict__ gq, double2* __restrict__ vp,
                                            double2* __restrict__ vq, int n, int lane, double tol2) {
  double al = 0, be = 0, gr = 0, gi = 0;
  for (int i = lane; i < n; i += 32) {
    const double2 a = gp[i], b = gq[i];
    al += a.x * a.x + a.y * a.y;
    be += b.x * b.x + b.y * b.y;
    gr += a.x * b.x + a.y * b.y;  // conj(a) b
    gi += a.x * b.y - a.y * b.x;
  }
  al = warp_sum(al); be = warp_sum(be); gr = warp_sum(gr); gi = warp_sum(gi);
  const double g2 = gr * gr + gi * gi;
  if (!(g2 > tol2 * al * be) || g2 == 0.0) return false;
  const double ag = sqrt(g2);
  const double zeta = (be - al) / (2.0 * ag);
  const double t = (zeta >= 0 ? 1.0 : -1.0) / (fabs(zeta) + sqrt(1.0 + zeta * zeta));
  const double c = 1.0 / sqrt(1.0 + t * t), s = t * c;
  const double sr = s * gr / ag, si = s * gi / ag;  // sigma = s gamma/|gamma|
  // [g_p, g_q] <- [c g_p - conj(sigma) g_q,  sigma g_p + c g_q]
  for (int i = lane; i < n; i += 32) {
    double2 a = gp[i], b = gq[i];
    gp[i] = make_double2(c * a.x - (sr * b.x + si * b.y), c * a.y - (sr * b.y - si * b.x));
    gq[i] = make_double2(sr * a.x - si * a.y + c * b.x, sr * a.y + si * a.x + c * b.y);
    a = vp[i]; b = vq[i];
    vp[i] = make_double2(c * a.x - (sr * b.x + si * b.y), c * a.y - (sr * b.y - si * b.x));
    vq[i] = make_double2(sr * a.x - si * a.y + c * b.x, sr * a.y + si * a.x + c * b.y);
  }
  return true;
}

// round-robin pairing for M (even) players, round r in [0, M-1), pair index i in [0, M/2)
__device__ __forceinline__ void rr_pair(int M, int r, int i, int& p, int& q) {
  if (i == 0) { p = M - 1; q = r % (M - 1); }
  else { p = (r + i) % (M - 1); q = (r + (M - 1) - i) % (M - 1); }
  if (p > q) { int t = p; p = q; q = t; }
}

// ---- small matrices: one CTA per matrix ---------------------------------------------------------------------------
__global__ void seed_small_kernel(int n, const double2* __restrict__ A, double* __restrict__ mu, double2* __restrict__ V,
                                  int max_sweeps, double tol2) {
  extern __shared__ double2 sm[];
  double2* G = sm;              // column-major n x n
  double2* W = sm + n * n;      // eigenvector accumulator
  __shared__ double s_red[32];
  __shared__ int s_rot;
  __shared__ double s_sigma;
  const int b = blockIdx.x;
  const int tid = threadIdx.x, nthr = blockDim.x, lane = tid & 31, warp = tid >> 5;
  const double2* Ab = A + (size_t)b * n * n;
  // Gershgorin radius (rows of the Hermitian matrix built from the upper triangle)
  double rmax = 0;
  for (int i = tid; i < n; i += nthr) {
    double rs = 0;
    for (int j = 0; j < n; ++j) {
      const double2 a = (i <= j) ? Ab[(size_t)i * n + j] : Ab[(size_t)j * n + i];
      rs += (i == j) ? fabs(a.x) : sqrt(a.x * a.x + a.y * a.y);
    }
    rmax = fmax(rmax, rs);
  }
  for (int off = 16; off > 0; off >>= 1) rmax = fmax(rmax, __shfl_xor_sync(0xffffffffu, rmax, off));
  if (lane == 0) s_red[warp] = rmax;
  __syncthreads();
  if (tid == 0) {
    double m = 0;
    for (int w = 0; w < (nthr + 31) / 32; ++w) m = fmax(m, s_red[w]);
    s_sigma = 1.5 * m;
  }
  __syncthreads();
  const double sigma = s_sigma;
  for (int e = tid; e < n * n; e += nthr) {
    const int i = e % n, j = e / n;  // column-major destination
    double2 a = (i <= j) ? Ab[(size_t)i * n + j] : Ab[(size_t)j * n + i];
    if (i > j) a.y = -a.y;
    if (i == j) { a.y = 0; a.x += sigma; }
    G[e] = a;
    W[e] = make_double2(i == j ? 1.0 : 0.0, 0.0);
  }
  __syncthreads();
  const int M = n + (n & 1);
  const int npairs = M / 2;
  const int nwarps = nthr >> 5;
  if (n > 1 && sigma > 0) {
    for (int sweep = 0; sweep < max_sweeps; ++sweep) {
      if (tid == 0) s_rot = 0;
      __syncthreads();
      for (int r = 0; r < M - 1; ++r) {
        bool rot = false;
        for (int i = warp; i < npairs; i += nwarps) {
          int p, q;
          rr_pair(M, r, i, p, q);
          if (q < n) rot |= rotate_pair(G + p * n, G + q * n, W + p * n, W + q * n, n, lane, tol2);
        }
        if (rot && lane == 0) s_rot = 1;
        __syncthreads();
      }
      if (!s_rot) break;
      __syncthreads();
    }
  }
  // mu_j = ||g_j|| - sigma; stable rank sort ascending; V[i][rank] = W[:, j]
  __shared__ double s_mu[64];
  __shared__ int s_rank[64];
  __syncthreads();
  for (int j = warp; j < n; j += nwarps) {
    double s = 0;
    for (int i = lane; i < n; i += 32) { const double2 a = G[j * n + i]; s += a.x * a.x + a.y * a.y; }
    s = warp_sum(s);
    if (lane == 0) s_mu[j] = sqrt(s) - sigma;
  }
  __syncthreads();
  for (int j = tid; j < n; j += nthr) {
    const double mj = s_mu[j];
    int rank = 0;
    for (int i = 0; i < n; ++i) {
      const double mi = s_mu[i];
      rank += (mi < mj) || (mi == mj && i < j);
    }
    s_rank[j] = rank;
    mu[(size_t)b * n + rank] = mj;
  }
  __syncthreads();
  for (int e = tid; e < n * n; e += nthr) {
    const int i = e % n, j = e / n;
    V[(size_t)b * n * n + (size_t)i * n + s_rank[j]] = W[e];
  }
}

// ---- large matrices: cooperative grid ------------------------------------------------------------------------------
__global__ void seed_sigma_kernel(int n, const double2* __restrict__ A, double* sigma_out) {
  // one block; Gershgorin radius
  __shared__ double s_red[32];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  double rmax = 0;
  for (int i = tid; i < n; i += blockDim.x) {
    double rs = 0;
    for (int j = 0; j < n; ++j) {
      const double2 a = (i <= j) ? A[(size_t)i * n + j] : A[(size_t)j * n + i];
      rs += (i == j) ? fabs(a.x) : sqrt(a.x * a.x + a.y * a.y);
    }
    rmax = fmax(rmax, rs);
  }
  for (int off = 16; off > 0; off >>= 1) rmax = fmax(rmax, __shfl_xor_sync(0xffffffffu, rmax, off));
  if (lane == 0) s_red[warp] = rmax;
  __syncthreads();
  if (tid == 0) {
    double m = 0;
    for (int w = 0; w < (blockDim.x + 31) / 32; ++w) m = fmax(m, s_red[w]);
    *sigma_out = 1.5 * m;
  }
}

__global__ void __launch_bounds__(128) seed_large_kernel(int n, const double2* __restrict__ A, double2* __restrict__ G,
                                                         double2* __restrict__ W, const double* __restrict__ sigma_p,
                                                         int* __restrict__ rot_flags, double* __restrict__ mu_unsorted,
                                                         int max_sweeps, double tol2) {
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
    W[e] = make_double2(i == j ? 1.0 : 0.0, 0.0);
  }
  if (gtid < (size_t)max_sweeps) rot_flags[gtid] = 0;
  grid.sync();
  const int M = n + (n & 1), npairs = M / 2;
  if (sigma > 0) {
    for (int sweep = 0; sweep < max_sweeps; ++sweep) {
      for (int r = 0; r < M - 1; ++r) {
        bool rot = false;
        for (int i = gwarp; i < npairs; i += nwarps) {
          int p, q;
          rr_pair(M, r, i, p, q);
          if (q < n) rot |= rotate_pair(G + (size_t)p * n, G + (size_t)q * n, W + (size_t)p * n, W + (size_t)q * n, n, lane, tol2);
        }
        if (rot && lane == 0) rot_flags[sweep] = 1;
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

__global__ void seed_sort_kernel(int n, const double* __restrict__ mu_unsorted, const double2* __restrict__ W,
                                 double* __restrict__ mu, double2* __restrict__ V) {
  // grid-stride; each thread recomputes the rank of the column it moves (n <= 2048: cheap)
  const size_t gtid = (size_t)blockIdx.x * blockDim.x + threadIdx.x, gthr = (size_t)gridDim.x * blockDim.x;
  for (size_t e = gtid; e < (size_t)n * n; e += gthr) {
    const int i = (int)(e % n), j = (int)(e / n);
    const double mj = mu_unsorted[j];
    int rank = 0;
    for (int k = 0; k < n; ++k) {
      const double mk = mu_unsorted[k];
      rank += (mk < mj) || (mk == mj && k < j);
    }
    V[(size_t)i * n + rank] = W[e];
    if (i == 0) mu[rank] = mj;
  }
}

int seed_fp64(int N, int batch, const double* A64, double* mu, double* V, int max_sweeps, cudaStream_t s) {
  const double tol = ldexp(1.0, -50);
  const double tol2 = tol * tol;
  if (N <= 64) {
    const int M = N + (N & 1);
    int threads = 32 * (M / 2 > 0 ? M / 2 : 1);
    if (threads > 1024) threads = 1024;
    const size_t smem = sizeof(double2) * 2 * (size_t)N * N + 64;
    static bool attr = false;
    if (!attr) {
      ZKD_CUDA_TRY(cudaFuncSetAttribute(seed_small_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * 64 * 64 * 16 + 64));
      attr = true;
    }
    seed_small_kernel<<<batch, threads, smem, s>>>(N, (const double2*)A64, mu, (double2*)V, max_sweeps, tol2);
    count_launch();
    return launch_check();
  }
  // large: cooperative grid, one matrix at a time
  int dev = 0, sms = 0;
  ZKD_CUDA_TRY(cudaGetDevice(&dev));
  ZKD_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  const int M = N + (N & 1);
  int nblocks = (M / 2 + 3) / 4;  // 4 warps (pairs) per block
  int maxb = 0;
  ZKD_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&maxb, seed_large_kernel, 128, 0));
  if (nblocks > maxb * sms) nblocks = maxb * sms;
  char* buf = nullptr;
  const size_t nn = (size_t)N * N;
  const size_t bytes = sizeof(double2) * 2 * nn + sizeof(double) * (N + 8) + sizeof(int) * 64;
  ZKD_CUDA_TRY(cudaMallocAsync((void**)&buf, bytes, s));
  double2* G = (double2*)buf;
  double2* W = G + nn;
  double* sigma = (double*)(W + nn);
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
    void* args[] = {&n, (void*)&Ab, &G, &W, &sigma, &flags, &mu_uns, &ms, &t2};
    if (cudaLaunchCooperativeKernel((void*)seed_large_kernel, dim3(nblocks), dim3(128), args, 0, s) != cudaSuccess) {
      (void)cudaGetLastError();
      rc = ZKD_ERR_CUDA;
      break;
    }
    seed_sort_kernel<<<sms * 4, 256, 0, s>>>(N, mu_uns, W, mub, Vb);
    count_launch(3);
    rc = launch_check();
  }
  cudaFreeAsync(buf, s);
  return rc;
}

}  // namespace zkd

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
//   n <= 256 : thread-block CLUSTER per matrix (1 .. 16 CTAs), systolic ring: every warp owns one pair of columns per round and
//              hands each rotated column to a neighbouring warp's shared-memory slot, so only the columns at CTA boundaries
//              cross distributed shared memory; rounds are separated by the hardware cluster barrier.  With many matrices
//              in the batch the cluster shrinks to 1 CTA (one SM per matrix, plain CTA kernel).
//   n  > 256 : cooperative grid, G in global memory (L2 resident), grid.sync between rounds.
//              (seed_block_kernel: blocks of W columns per CTA in shared memory, TMA bulk copies; seed_blockg_kernel: the same
//              rounds on the 8 x 8 Gram matrix of the CTA's blocks, measured slower, option seed_gram)
// Column pairs of one numerically multiple eigenvalue are left unrotated when the caller treats clusters as blocks afterwards
// (rot_params, dgap2): this keeps the sweeps quadratically convergent on spectra with multiplicities.
// The seed only has to be good to ~2^-40 (the refinement squares the error every step).
#include <cooperative_groups.h>

#include <mutex>

#include "timing.h"
#include "zkd_internal.h"

namespace cg = cooperative_groups;

// Scratch of zkd_seed_fp64_static (the entry point that allocates nothing; bottom of this file): the rotated matrix G of one
// N x N problem, N <= ZKD_SEED_STATIC_MAX_N = 512 (4 MiB of complex doubles), followed by sigma, the unsorted eigenvalues and
// the sweep flags (8 KiB).  Every GPU that loads the library holds these 4 MiB + 8 KiB until the process exits.  In host code
// this name is a host-side stand-in, not a device address: host code takes the address with cudaGetSymbolAddress, once per
// device (seed_static_scratch below).
constexpr size_t kSeedStaticGBytes = sizeof(double2) * (size_t)ZKD_SEED_STATIC_MAX_N * ZKD_SEED_STATIC_MAX_N;
constexpr size_t kSeedStaticBytes = kSeedStaticGBytes + 8192;
static __device__ __align__(256) unsigned char g_seed_static_scratch[kSeedStaticBytes];

namespace zkd {

constexpr double kSeedStopCos2 = 8.8817841970012523e-16;  // 2^-50

// Work counters for the roofline of the seed (zkd_seed_stats): column ELEMENTS whose pair was checked (three dot products:
// 8 DFMA per element) and elements whose pair was also rotated (12 more), summed over all launches since the last reset.
__device__ unsigned long long g_seed_stats[2];
__device__ __forceinline__ void seed_count(unsigned long long chk, unsigned long long rot) {
  if (chk) atomicAdd(&g_seed_stats[0], chk);
  if (rot) atomicAdd(&g_seed_stats[1], rot);
}

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
//
// Degenerate pairs are left alone (dgap2): two columns whose eigenvalue estimates ||g|| - sigma differ by less than
// dgap = sqrt(dgap2) and whose cosine is already below 2^-10 belong to one (numerically) multiple eigenvalue.  Orthogonalising
// such a pair takes a rotation of up to 45 degrees however small gamma is, and every large rotation re-fills, at FIRST order,
// the inner products with the other eigenspaces that the sweep has just annihilated: with multiple eigenvalues cyclic Jacobi
// then converges only linearly (c5's 64 x 16 clusters: ||A V - V L|| ~ 1e-7 after 12 sweeps, 1e-9 after 15).  Inside an
// eigenspace the pair needs no rotation: V stays unitary, so gamma = v_p^H G^2 v_q is second order in the contamination from
// other eigenspaces plus (eigenvalue difference) / ||g||, and vanishes with them; without the large rotations the sweeps converge
// quadratically again (the same matrix: 1e-12 after 9 sweeps).  dgap is kept below the cluster threshold of S2
// (2^-tau ||A||_F >= 2^-tau sigma / (1.5 sqrt n)), so a skipped pair always lands inside one cluster of the refinement, which
// treats the cluster as a block (S4f re-orthonormalises it, S5 resolves it).  Skipped pairs do not count towards the sweep's
// stopping criterion (cos2 = 0).
__device__ __forceinline__ bool rot_params(double al, double be, double gr, double gi, double tol2, double dgap2, double& c, double& sr,
                                           double& si, double& cos2) {
  const double g2 = gr * gr + gi * gi;
  const double ab = al * be;
  cos2 = 0.0;
  if (!(g2 > tol2 * ab) || g2 == 0.0) return false;
  const double d = 0.5 * (be - al);
  if (g2 < 9.5367431640625e-07 * ab && d * d < dgap2 * fmax(al, be)) return false;  // 2^-20: |cos| < 2^-10
  cos2 = g2 * (1.0 / ab);
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

// ---- n <= 256, systolic ring (Brent-Luk): processor k = warp k % wpc of CTA k / wpc holds the pair (top_k, bot_k) -------------
// After every round top_0 stays, bot_0 -> top_1, top_k -> top_{k+1}, top_{P-1} -> bot_{P-1}, bot_k -> bot_{k-1}: in M - 1 rounds
// every pair of columns meets once, and a rotated column is written straight into the slot where it is needed next, which is
// a neighbouring warp: only the two columns at each CTA boundary cross distributed shared memory per round (DSMEM moves about
// 17 B/clk/SM, so a design in which every warp fetches both of its columns from their home CTA is bandwidth-bound: it measured
// 8.6 us per round at n = 256, 21 ms per call).
// One slot buffer, two cluster-barrier phases per round: "all slots read" (its wait hidden behind the arithmetic) and "all
// slots written".
__device__ __forceinline__ void cluster_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }

template <int EPL>
__global__ void __launch_bounds__(EPL >= 8 ? 512 : 1024)
seed_ring_kernel(int n, int wpc, const double2* __restrict__ A, double* __restrict__ mu, double2* __restrict__ V, int max_sweeps,
                 double tol2, double gap2, int dbuf) {
  extern __shared__ double2 slots[];              // [1 + dbuf][wpc][2][n]
  __shared__ int s_id2[2][32][2];                 // column ids held by the local slots (per buffer)
  int (*s_id)[2] = s_id2[0];
  __shared__ double s_mu[258];                    // by position 2k + which (every CTA holds a full copy)
  __shared__ int s_pid[258];
  __shared__ unsigned long long s_cmax[2];
  __shared__ double s_rmax;
  __shared__ double s_red[32];
  cg::cluster_group cluster = cg::this_cluster();
  const int csize = (int)cluster.num_blocks(), rank = (int)cluster.block_rank();
  const int b = blockIdx.x / csize;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const double2* Ab = A + (size_t)b * n * n;
  const int M = n + (n & 1), P = M / 2;
  const int k = rank * wpc + warp;                // processor index; processors >= P idle but keep the barriers
  const bool act = k < P;
  double2* my_top = slots + (size_t)(warp * 2 + 0) * n;
  double2* my_bot = slots + (size_t)(warp * 2 + 1) * n;
  // dbuf: a second set of slots.  Round r reads set r % 2 and writes the rotated columns into set (r + 1) % 2 of their
  // destinations, so the "all slots read" barrier of the single-buffer scheme is not needed: one cluster barrier per round.
  const size_t bufstride = (size_t)wpc * 2 * n;   // double2 elements between the two slot sets
  constexpr int kIdStride = 32 * 2;               // ints between the two id sets
  int cur = 0;

  // own two columns of the Hermitian matrix (upper triangle authoritative), Gershgorin radius
  double rmax = 0;
  if (act) {
    for (int which = 0; which < 2; ++which) {
      const int j = 2 * k + which;
      double2* g = which ? my_bot : my_top;
      double rs = 0;
      for (int i = lane; i < n; i += 32) {
        double2 a = make_double2(0, 0);
        if (j < n) {
          a = (i <= j) ? Ab[(size_t)i * n + j] : Ab[(size_t)j * n + i];
          if (i > j) a.y = -a.y;
          if (i == j) a.y = 0;
        }
        g[i] = a;
        rs += (i == j) ? fabs(a.x) : sqrt(a.x * a.x + a.y * a.y);
      }
      rmax = fmax(rmax, warp_sum(rs));
      if (lane == 0) s_id[warp][which] = j;
    }
  }
  if (lane == 0) s_red[warp] = rmax;
  if (tid == 0) { s_cmax[0] = 0ull; s_cmax[1] = 0ull; }
  __syncthreads();
  if (tid == 0) {
    double m = 0;
    for (int w = 0; w < (int)(blockDim.x >> 5); ++w) m = fmax(m, s_red[w]);
    s_rmax = m;
  }
  cluster.sync();
  double sigma = 0;
  for (int r = 0; r < csize; ++r) sigma = fmax(sigma, *cluster.map_shared_rank(&s_rmax, r));
  sigma *= 1.5;
  if (act && lane == 0) {
    if (2 * k < n) my_top[2 * k].x += sigma;
    if (2 * k + 1 < n) my_bot[2 * k + 1].x += sigma;
  }
  // destinations of this processor's rotated columns (fixed for the whole run)
  double2* dst_top = my_top;
  double2* dst_bot = my_bot;
  int* dst_top_id = &s_id[warp][0];
  int* dst_bot_id = &s_id[warp][1];
  if (act && P > 1) {
    auto slot_of = [&](int kk, int which) -> double2* {
      double2* local = slots + (size_t)((kk % wpc) * 2 + which) * n;
      return (kk / wpc == rank) ? local : cluster.map_shared_rank(local, kk / wpc);
    };
    auto id_of = [&](int kk, int which) -> int* {
      int* local = &s_id[kk % wpc][which];
      return (kk / wpc == rank) ? local : cluster.map_shared_rank(local, kk / wpc);
    };
    if (k == 0) { dst_top = my_top; dst_top_id = &s_id[warp][0]; dst_bot = slot_of(1, 0); dst_bot_id = id_of(1, 0); }
    else {
      if (k < P - 1) { dst_top = slot_of(k + 1, 0); dst_top_id = id_of(k + 1, 0); }
      else { dst_top = my_bot; dst_top_id = &s_id[warp][1]; }
      dst_bot = slot_of(k - 1, 1); dst_bot_id = id_of(k - 1, 1);
    }
  }
  cluster.sync();

  const double dgap2 = gap2 * sigma * sigma / n;
  if (n > 1 && sigma > 0) {
    unsigned long long nchk = 0, nrot = 0;
    for (int sweep = 0; sweep < max_sweeps; ++sweep) {
      double cmax = 0;
      for (int r = 0; r < M - 1; ++r) {
        double2 a[EPL], bb[EPL];
        int ida = 0, idb = 0;
        if (act) {
          const double2* rt = my_top + (size_t)cur * bufstride;
          const double2* rb = my_bot + (size_t)cur * bufstride;
#pragma unroll
          for (int q = 0; q < EPL; ++q) {
            const int i2 = lane + 32 * q;
            a[q] = i2 < n ? rt[i2] : make_double2(0, 0);
            bb[q] = i2 < n ? rb[i2] : make_double2(0, 0);
          }
          ida = s_id2[cur][warp][0];
          idb = s_id2[cur][warp][1];
        }
        if (!dbuf) cluster_arrive();  // slots read
        if (act) {
          double al = 0, be = 0, gr = 0, gi = 0;
#pragma unroll
          for (int q = 0; q < EPL; ++q) {
            al = fma(a[q].x, a[q].x, fma(a[q].y, a[q].y, al));
            be = fma(bb[q].x, bb[q].x, fma(bb[q].y, bb[q].y, be));
            gr = fma(a[q].x, bb[q].x, fma(a[q].y, bb[q].y, gr));
            gi = fma(a[q].x, bb[q].y, fma(-a[q].y, bb[q].x, gi));
          }
          al = warp_sum(al); be = warp_sum(be); gr = warp_sum(gr); gi = warp_sum(gi);
          double c, sr, si, cos2;
          nchk += n;
          if (rot_params(al, be, gr, gi, tol2, dgap2, c, sr, si, cos2)) {
            nrot += n;
            cmax = fmax(cmax, cos2);
#pragma unroll
            for (int q = 0; q < EPL; ++q) {
              const double2 x = a[q], y = bb[q];
              a[q] = make_double2(c * x.x - (sr * y.x + si * y.y), c * x.y - (sr * y.y - si * y.x));
              bb[q] = make_double2(sr * x.x - si * x.y + c * y.x, sr * x.y + si * x.x + c * y.y);
            }
          }
        }
        if (!dbuf) cluster_wait();    // everybody has read: slots may be overwritten
        const int nxt = dbuf ? (cur ^ 1) : 0;
        if (act) {
          double2* wt = dst_top + (size_t)nxt * bufstride;
          double2* wb = dst_bot + (size_t)nxt * bufstride;
#pragma unroll
          for (int q = 0; q < EPL; ++q) {
            const int i2 = lane + 32 * q;
            if (i2 < n) { wt[i2] = a[q]; wb[i2] = bb[q]; }
          }
          if (lane == 0) { dst_top_id[nxt * kIdStride] = ida; dst_bot_id[nxt * kIdStride] = idb; }
        }
        cur = nxt;
        if (r == M - 2 && lane == 0 && cmax > 0) atomicMax(&s_cmax[sweep & 1], (unsigned long long)__double_as_longlong(cmax));
        cluster_arrive();
        cluster_wait();    // slots written
      }
      double worst = 0;
      for (int r = 0; r < csize; ++r)
        worst = fmax(worst, __longlong_as_double((long long)*cluster.map_shared_rank(&s_cmax[sweep & 1], r)));
      if (tid == 0) s_cmax[(sweep + 1) & 1] = 0ull;  // last read by the other CTAs one sweep (many barriers) ago
      __syncthreads();
      if (!(worst > kSeedStopCos2)) break;
    }
    if (lane == 0) seed_count(nchk, nrot);
  }
  cluster.sync();
  // the final columns sit in slot set `cur`
  my_top += (size_t)cur * bufstride;
  my_bot += (size_t)cur * bufstride;
  s_id = s_id2[cur];

  // mu = ||g|| - sigma per position, broadcast to every CTA; normalise in place
  if (act) {
    for (int which = 0; which < 2; ++which) {
      double2* g = which ? my_bot : my_top;
      double sq = 0;
      for (int i = lane; i < n; i += 32) { const double2 x = g[i]; sq += x.x * x.x + x.y * x.y; }
      sq = warp_sum(sq);
      const double nrm = sqrt(sq);
      const double inv = nrm > 0 ? 1.0 / nrm : 0.0;
      const int id = s_id[warp][which];
      for (int i = lane; i < n; i += 32) {
        double2 x = g[i];
        if (nrm > 0) { x.x *= inv; x.y *= inv; } else { x = make_double2(i == id ? 1.0 : 0.0, 0.0); }
        g[i] = x;
      }
      if (lane < csize) {
        *cluster.map_shared_rank(&s_mu[2 * k + which], lane) = nrm - sigma;
        *cluster.map_shared_rank(&s_pid[2 * k + which], lane) = id;
      }
    }
  }
  cluster.sync();
  if (act) {
    for (int which = 0; which < 2; ++which) {
      const int pos = 2 * k + which;
      const int id = s_pid[pos];
      if (id >= n) continue;  // the padding column of an odd n
      const double mj = s_mu[pos];
      int rk = 0;
      for (int i = lane; i < M; i += 32) {
        const double mi = s_mu[i];
        const int idi = s_pid[i];
        rk += (idi < n) && ((mi < mj) || (mi == mj && idi < id));
      }
#pragma unroll
      for (int off = 16; off > 0; off >>= 1) rk += __shfl_xor_sync(0xffffffffu, rk, off);
      if (lane == 0) mu[(size_t)b * n + rk] = mj;
      const double2* g = which ? my_bot : my_top;
      for (int i = lane; i < n; i += 32) V[(size_t)b * n * n + (size_t)i * n + rk] = g[i];
    }
  }
  cluster.sync();
}

template <int EPL>
static int launch_ring(int N, int batch, int csize, const double2* A, double* mu, double2* V, int max_sweeps, double tol2, double gap2,
                       cudaStream_t s) {
  const int P = (N + 1) / 2;
  const int wpc = (P + csize - 1) / csize;
  const size_t smem1 = sizeof(double2) * (size_t)wpc * 2 * N;
  int dbuf = (2 * smem1 <= 200 * 1024 && options().seed_dbuf) ? 1 : 0;
  const size_t smem = smem1 * (1 + dbuf);
  // function attributes are per device: set on every launch (cheap) rather than cached in process-wide flags
  if (smem > 48 * 1024) ZKD_CUDA_TRY(cudaFuncSetAttribute(seed_ring_kernel<EPL>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  if (csize > 8) ZKD_CUDA_TRY(cudaFuncSetAttribute(seed_ring_kernel<EPL>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)(batch * csize));
  cfg.blockDim = dim3((unsigned)(32 * wpc));
  cfg.dynamicSmemBytes = smem;
  cfg.stream = s;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = (unsigned)csize;
  at[0].val.clusterDim.y = 1;
  at[0].val.clusterDim.z = 1;
  cfg.attrs = at;
  cfg.numAttrs = 1;
  {
    KtScope kt(KC_SEED, s);
    ZKD_CUDA_TRY(cudaLaunchKernelEx(&cfg, seed_ring_kernel<EPL>, N, wpc, A, mu, V, max_sweeps, tol2, gap2, dbuf));
  }
  count_launch();
  return launch_check();
}

// ---- n <= 256, BLOCK ring: a processor = W warps holds two blocks of W columns ------------------------------------------------------
// Same Brent-Luk ring, but over blocks of W columns: per ring step a processor rotates all W^2 cross pairs of its two blocks in W
// sub-steps of W disjoint pairs (one warp each, in place in its own shared-memory slots, a named barrier of the processor's W warps
// between sub-steps) and only then hands the blocks on: (n / W - 1) cluster barriers and DSMEM hand-overs per sweep instead of (n - 1).
// The pairs inside a block meet once per sweep, in step 0.  Blocks keep their columns for the whole run.
__device__ __forceinline__ void proc_barrier(int id, int nthreads) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory"); }

template <int EPL>
__device__ __forceinline__ void ring_load(double2 (&a)[EPL], const double2* __restrict__ col, int n, int lane) {
#pragma unroll
  for (int q = 0; q < EPL; ++q) {
    const int i = lane + 32 * q;
    a[q] = i < n ? col[i] : make_double2(0, 0);
  }
}
template <int EPL>
__device__ __forceinline__ void ring_store(double2* __restrict__ col, const double2 (&a)[EPL], int n, int lane) {
#pragma unroll
  for (int q = 0; q < EPL; ++q) {
    const int i = lane + 32 * q;
    if (i < n) col[i] = a[q];
  }
}
// orthogonalise the register-held columns a, bb; returns |cos|^2 before the rotation (0 when skipped)
template <int EPL>
__device__ __forceinline__ double ring_rotate(double2 (&a)[EPL], double2 (&bb)[EPL], double tol2, double dgap2, bool& rotated) {
  double al = 0, be = 0, gr = 0, gi = 0;
#pragma unroll
  for (int q = 0; q < EPL; ++q) {
    al = fma(a[q].x, a[q].x, fma(a[q].y, a[q].y, al));
    be = fma(bb[q].x, bb[q].x, fma(bb[q].y, bb[q].y, be));
    gr = fma(a[q].x, bb[q].x, fma(a[q].y, bb[q].y, gr));
    gi = fma(a[q].x, bb[q].y, fma(-a[q].y, bb[q].x, gi));
  }
  al = warp_sum(al); be = warp_sum(be); gr = warp_sum(gr); gi = warp_sum(gi);
  double c, sr, si, cos2;
  rotated = rot_params(al, be, gr, gi, tol2, dgap2, c, sr, si, cos2);
  if (rotated) {
#pragma unroll
    for (int q = 0; q < EPL; ++q) {
      const double2 x = a[q], y = bb[q];
      a[q] = make_double2(c * x.x - (sr * y.x + si * y.y), c * x.y - (sr * y.y - si * y.x));
      bb[q] = make_double2(sr * x.x - si * x.y + c * y.x, sr * x.y + si * x.x + c * y.y);
    }
  }
  return cos2;
}

constexpr int kRingbMaxProc = 8;   // processors per CTA
constexpr int kRingbMaxCols = 288;  // columns incl. padding

template <int EPL, int W>
__global__ void __launch_bounds__(512)
seed_ringb_kernel(int n, int ppc, const double2* __restrict__ A, double* __restrict__ mu, double2* __restrict__ V, int max_sweeps, double tol2, double gap2) {
  extern __shared__ double2 slots[];                 // [2 sets][ppc][2 blocks][W][n]
  __shared__ int s_id2[2][kRingbMaxProc][2][W];      // column ids held by the local slots (per set)
  __shared__ double s_mu[kRingbMaxCols];             // by position (2k + which) W + w (every CTA holds a full copy)
  __shared__ int s_pid[kRingbMaxCols];
  __shared__ unsigned long long s_cmax[2];
  __shared__ double s_rmax;
  __shared__ double s_red[32];
  cg::cluster_group cluster = cg::this_cluster();
  const int csize = (int)cluster.num_blocks(), rank = (int)cluster.block_rank();
  const int b = blockIdx.x / csize;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int pl = warp / W, w = warp % W;             // local processor, warp inside the processor
  const double2* Ab = A + (size_t)b * n * n;
  const int NBk = (n + W - 1) / W, MB = NBk + (NBk & 1), P = MB / 2;  // blocks (even), processors
  const int k = rank * ppc + pl;                     // global processor
  const bool act = k < P;
  const size_t blk = (size_t)W * n;                  // double2 elements of a block
  const size_t bufstride = (size_t)ppc * 2 * blk;    // between the two slot sets
  double2* my_top = slots + (size_t)(pl * 2 + 0) * blk;
  double2* my_bot = slots + (size_t)(pl * 2 + 1) * blk;
  int cur = 0;

  // own columns: warp w of processor k loads column w of both blocks (ids (2k) W + w and (2k + 1) W + w); Gershgorin radius
  double rmax = 0;
  if (act) {
    for (int which = 0; which < 2; ++which) {
      const int j = (2 * k + which) * W + w;
      double2* g = (which ? my_bot : my_top) + (size_t)w * n;
      double rs = 0;
      for (int i = lane; i < n; i += 32) {
        double2 a = make_double2(0, 0);
        if (j < n) {
          a = (i <= j) ? Ab[(size_t)i * n + j] : Ab[(size_t)j * n + i];
          if (i > j) a.y = -a.y;
          if (i == j) a.y = 0;
        }
        g[i] = a;
        rs += (i == j) ? fabs(a.x) : sqrt(a.x * a.x + a.y * a.y);
      }
      rmax = fmax(rmax, warp_sum(rs));
      if (lane == 0) s_id2[0][pl][which][w] = j;
    }
  }
  if (lane == 0) s_red[warp] = rmax;
  if (tid == 0) { s_cmax[0] = 0ull; s_cmax[1] = 0ull; }
  __syncthreads();
  if (tid == 0) {
    double m = 0;
    for (int x = 0; x < (int)(blockDim.x >> 5); ++x) m = fmax(m, s_red[x]);
    s_rmax = m;
  }
  cluster.sync();
  double sigma = 0;
  for (int r = 0; r < csize; ++r) sigma = fmax(sigma, *cluster.map_shared_rank(&s_rmax, r));
  sigma *= 1.5;
  if (act && lane == 0) {
    const int jt = (2 * k) * W + w, jb = (2 * k + 1) * W + w;
    if (jt < n) my_top[(size_t)w * n + jt].x += sigma;
    if (jb < n) my_bot[(size_t)w * n + jb].x += sigma;
  }
  // destinations of this processor's blocks (fixed for the whole run), set 0 addresses
  double2* dst_top = my_top;
  double2* dst_bot = my_bot;
  int* dst_top_id = &s_id2[0][pl][0][0];
  int* dst_bot_id = &s_id2[0][pl][1][0];
  if (act && P > 1) {
    auto slot_of = [&](int kk, int which) -> double2* {
      double2* local = slots + (size_t)((kk % ppc) * 2 + which) * blk;
      return (kk / ppc == rank) ? local : cluster.map_shared_rank(local, kk / ppc);
    };
    auto id_of = [&](int kk, int which) -> int* {
      int* local = &s_id2[0][kk % ppc][which][0];
      return (kk / ppc == rank) ? local : cluster.map_shared_rank(local, kk / ppc);
    };
    if (k == 0) { dst_bot = slot_of(1, 0); dst_bot_id = id_of(1, 0); }
    else {
      if (k < P - 1) { dst_top = slot_of(k + 1, 0); dst_top_id = id_of(k + 1, 0); }
      else { dst_top = my_bot; dst_top_id = &s_id2[0][pl][1][0]; }
      dst_bot = slot_of(k - 1, 1); dst_bot_id = id_of(k - 1, 1);
    }
  }
  constexpr int kIdSet = kRingbMaxProc * 2 * W;      // ints between the two id sets
  cluster.sync();

  unsigned long long nchk = 0, nrot = 0;
  const double dgap2 = gap2 * sigma * sigma / n;
  if (n > 1 && sigma > 0) {
    for (int sweep = 0; sweep < max_sweeps; ++sweep) {
      double cmax = 0;
      for (int r = 0; r < MB - 1; ++r) {
        const int nxt = cur ^ 1;
        if (act) {
          double2* T = my_top + (size_t)cur * bufstride;
          double2* B = my_bot + (size_t)cur * bufstride;
          double2 a[EPL], bb[EPL];
          bool rot;
          if (r == 0 && W > 1) {
            // pairs inside each block, once per sweep: round-robin over W columns, W / 2 pairs per block and sub-step
            for (int t = 0; t < W - 1; ++t) {
              const int which = w / (W / 2), i = w % (W / 2);
              int p, q;
              rr_pair(W, t, i, p, q);
              double2* X = which ? B : T;
              ring_load<EPL>(a, X + (size_t)p * n, n, lane);
              ring_load<EPL>(bb, X + (size_t)q * n, n, lane);
              cmax = fmax(cmax, ring_rotate<EPL>(a, bb, tol2, dgap2, rot));
              nchk += n;
              if (rot) {
                nrot += n;
                ring_store<EPL>(X + (size_t)p * n, a, n, lane);
                ring_store<EPL>(X + (size_t)q * n, bb, n, lane);
              }
              proc_barrier(1 + pl, 32 * W);
            }
          }
          const int ida = s_id2[cur][pl][0][w];
          ring_load<EPL>(a, T + (size_t)w * n, n, lane);  // column w of the top block stays in this warp's registers
          for (int t = 0; t < W; ++t) {
            const int q = (w + t) % W;
            ring_load<EPL>(bb, B + (size_t)q * n, n, lane);
            cmax = fmax(cmax, ring_rotate<EPL>(a, bb, tol2, dgap2, rot));
            nchk += n;
            if (rot) nrot += n;
            if (t < W - 1) {
              if (rot) ring_store<EPL>(B + (size_t)q * n, bb, n, lane);
              proc_barrier(1 + pl, 32 * W);
            } else {
              // last sub-step: straight into the slots where the blocks are needed next (set nxt of the neighbours)
              const int idb = s_id2[cur][pl][1][q];
              ring_store<EPL>(dst_top + (size_t)nxt * bufstride + (size_t)w * n, a, n, lane);
              ring_store<EPL>(dst_bot + (size_t)nxt * bufstride + (size_t)q * n, bb, n, lane);
              if (lane == 0) { dst_top_id[nxt * kIdSet + w] = ida; dst_bot_id[nxt * kIdSet + q] = idb; }
            }
          }
        }
        cur = nxt;
        if (r == MB - 2 && lane == 0 && cmax > 0) atomicMax(&s_cmax[sweep & 1], (unsigned long long)__double_as_longlong(cmax));
        cluster_arrive();
        cluster_wait();
      }
      double worst = 0;
      for (int r = 0; r < csize; ++r)
        worst = fmax(worst, __longlong_as_double((long long)*cluster.map_shared_rank(&s_cmax[sweep & 1], r)));
      if (tid == 0) s_cmax[(sweep + 1) & 1] = 0ull;
      __syncthreads();
      if (!(worst > kSeedStopCos2)) break;
    }
    if (lane == 0) seed_count(nchk, nrot);
  }
  cluster.sync();
  my_top += (size_t)cur * bufstride;
  my_bot += (size_t)cur * bufstride;

  // mu = ||g|| - sigma per position, broadcast to every CTA; normalise in place
  if (act) {
    for (int which = 0; which < 2; ++which) {
      double2* g = (which ? my_bot : my_top) + (size_t)w * n;
      double sq = 0;
      for (int i = lane; i < n; i += 32) { const double2 x = g[i]; sq += x.x * x.x + x.y * x.y; }
      sq = warp_sum(sq);
      const double nrm = sqrt(sq);
      const double inv = nrm > 0 ? 1.0 / nrm : 0.0;
      const int id = s_id2[cur][pl][which][w];
      for (int i = lane; i < n; i += 32) {
        double2 x = g[i];
        if (nrm > 0) { x.x *= inv; x.y *= inv; } else { x = make_double2(i == id ? 1.0 : 0.0, 0.0); }
        g[i] = x;
      }
      const int pos = (2 * k + which) * W + w;
      if (lane < csize) {
        *cluster.map_shared_rank(&s_mu[pos], lane) = nrm - sigma;
        *cluster.map_shared_rank(&s_pid[pos], lane) = id;
      }
    }
  }
  cluster.sync();
  if (act) {
    const int Mc = MB * W;
    for (int which = 0; which < 2; ++which) {
      const int pos = (2 * k + which) * W + w;
      const int id = s_pid[pos];
      if (id >= n) continue;  // a padding column
      const double mj = s_mu[pos];
      int rk = 0;
      for (int i = lane; i < Mc; i += 32) {
        const double mi = s_mu[i];
        const int idi = s_pid[i];
        rk += (idi < n) && ((mi < mj) || (mi == mj && idi < id));
      }
#pragma unroll
      for (int off = 16; off > 0; off >>= 1) rk += __shfl_xor_sync(0xffffffffu, rk, off);
      if (lane == 0) mu[(size_t)b * n + rk] = mj;
      const double2* g = (which ? my_bot : my_top) + (size_t)w * n;
      for (int i = lane; i < n; i += 32) V[(size_t)b * n * n + (size_t)i * n + rk] = g[i];
    }
  }
  cluster.sync();
}

template <int EPL, int W>
static int launch_ringb(int N, int batch, int csize, int ppc, const double2* A, double* mu, double2* V, int max_sweeps, double tol2,
                        double gap2, cudaStream_t s) {
  const size_t smem = sizeof(double2) * 2 * (size_t)ppc * 2 * W * N;
  if (smem > 48 * 1024) ZKD_CUDA_TRY(cudaFuncSetAttribute(seed_ringb_kernel<EPL, W>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  if (csize > 8) ZKD_CUDA_TRY(cudaFuncSetAttribute(seed_ringb_kernel<EPL, W>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)(batch * csize));
  cfg.blockDim = dim3((unsigned)(32 * W * ppc));
  cfg.dynamicSmemBytes = smem;
  cfg.stream = s;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = (unsigned)csize;
  at[0].val.clusterDim.y = 1;
  at[0].val.clusterDim.z = 1;
  cfg.attrs = at;
  cfg.numAttrs = 1;
  {
    KtScope kt(KC_SEED, s);
    ZKD_CUDA_TRY(cudaLaunchKernelEx(&cfg, seed_ringb_kernel<EPL, W>, N, ppc, A, mu, V, max_sweeps, tol2, gap2));
  }
  count_launch();
  return launch_check();
}

// ---- n <= 96: one CTA per matrix, G in this CTA's shared memory -----------------------------------------------------------
// One warp per pair of a round (npairs <= 48 warps would not fit, so a warp takes ceil(npairs / nwarps) pairs), one
// __syncthreads per round: no cluster barrier and no DSMEM latency on the critical path, and a batch uses one SM per matrix.
template <int EPL>
__global__ void __launch_bounds__(1024)
seed_cta_kernel(int n, const double2* __restrict__ A, double* __restrict__ mu, double2* __restrict__ V, int max_sweeps, double tol2, double gap2) {
  extern __shared__ double2 Gl[];                 // [n][n], column j at Gl + j n
  __shared__ double s_mu[96];
  __shared__ unsigned long long s_cmax[2];
  __shared__ double s_red[32];
  __shared__ double s_sigma;
  const int b = blockIdx.x;
  const int tid = threadIdx.x, nthr = blockDim.x, lane = tid & 31, warp = tid >> 5, nwarps = nthr >> 5;
  const double2* Ab = A + (size_t)b * n * n;
  for (int e = tid; e < n * n; e += nthr) {
    const int j = e / n, i = e - j * n;
    double2 a = (i <= j) ? Ab[(size_t)i * n + j] : Ab[(size_t)j * n + i];
    if (i > j) a.y = -a.y;
    if (i == j) a.y = 0;
    Gl[e] = a;
  }
  if (tid == 0) { s_cmax[0] = 0ull; s_cmax[1] = 0ull; }
  __syncthreads();
  double rmax = 0;
  for (int j = warp; j < n; j += nwarps) {
    double rs = 0;
    for (int i = lane; i < n; i += 32) {
      const double2 a = Gl[(size_t)j * n + i];
      rs += (i == j) ? fabs(a.x) : sqrt(a.x * a.x + a.y * a.y);
    }
    rmax = fmax(rmax, warp_sum(rs));
  }
  if (lane == 0) s_red[warp] = rmax;
  __syncthreads();
  if (tid == 0) {
    double m = 0;
    for (int w = 0; w < nwarps; ++w) m = fmax(m, s_red[w]);
    s_sigma = 1.5 * m;
  }
  __syncthreads();
  const double sigma = s_sigma;
  for (int j = tid; j < n; j += nthr) Gl[(size_t)j * n + j].x += sigma;
  __syncthreads();

  const int M = n + (n & 1), npairs = M / 2;
  const double dgap2 = gap2 * sigma * sigma / n;
  if (n > 1 && sigma > 0) {
    unsigned long long nchk = 0, nrot = 0;
    for (int sweep = 0; sweep < max_sweeps; ++sweep) {
      double cmax = 0;
      for (int r = 0; r < M - 1; ++r) {
        for (int i = warp; i < npairs; i += nwarps) {
          int p, q;
          rr_pair(M, r, i, p, q);
          if (q >= n) continue;
          double2* gp = Gl + (size_t)p * n;
          double2* gq = Gl + (size_t)q * n;
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
            gr = fma(a[k].x, bb[k].x, fma(a[k].y, bb[k].y, gr));
            gi = fma(a[k].x, bb[k].y, fma(-a[k].y, bb[k].x, gi));
          }
          al = warp_sum(al); be = warp_sum(be); gr = warp_sum(gr); gi = warp_sum(gi);
          double c, sr, si, cos2;
          nchk += n;
          if (!rot_params(al, be, gr, gi, tol2, dgap2, c, sr, si, cos2)) continue;
          nrot += n;
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
        __syncthreads();
      }
      const double worst = __longlong_as_double((long long)s_cmax[sweep & 1]);
      __syncthreads();
      if (tid == 0) s_cmax[(sweep + 1) & 1] = 0ull;
      if (!(worst > kSeedStopCos2)) break;
    }
    if (lane == 0) seed_count(nchk, nrot);
  }
  __syncthreads();
  for (int j = warp; j < n; j += nwarps) {
    double s = 0;
    for (int i = lane; i < n; i += 32) { const double2 a = Gl[(size_t)j * n + i]; s += a.x * a.x + a.y * a.y; }
    s = warp_sum(s);
    const double nrm = sqrt(s);
    const double inv = nrm > 0 ? 1.0 / nrm : 0.0;
    for (int i = lane; i < n; i += 32) {
      double2 a = Gl[(size_t)j * n + i];
      if (nrm > 0) { a.x *= inv; a.y *= inv; } else { a = make_double2(i == j ? 1.0 : 0.0, 0.0); }
      Gl[(size_t)j * n + i] = a;
    }
    if (lane == 0) s_mu[j] = nrm - sigma;
  }
  __syncthreads();
  for (int j = warp; j < n; j += nwarps) {
    const double mj = s_mu[j];
    int rk = 0;
    for (int i = lane; i < n; i += 32) {
      const double mi = s_mu[i];
      rk += (mi < mj) || (mi == mj && i < j);
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) rk += __shfl_xor_sync(0xffffffffu, rk, off);
    if (lane == 0) mu[(size_t)b * n + rk] = mj;
    for (int i = lane; i < n; i += 32) V[(size_t)b * n * n + (size_t)i * n + rk] = Gl[(size_t)j * n + i];
  }
}

template <int EPL>
static int launch_cta(int N, int batch, const double2* A, double* mu, double2* V, int max_sweeps, double tol2, double gap2, cudaStream_t s) {
  const int npairs = (N + 1) / 2;
  int warps = npairs < 1 ? 1 : (npairs > 32 ? (npairs + 1) / 2 : npairs);
  const size_t smem = sizeof(double2) * (size_t)N * N;
  if (smem > 48 * 1024) ZKD_CUDA_TRY(cudaFuncSetAttribute(seed_cta_kernel<EPL>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  {
    KtScope kt(KC_SEED, s);
    seed_cta_kernel<EPL><<<batch, 32 * warps, smem, s>>>(N, A, mu, V, max_sweeps, tol2, gap2);
  }
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
__device__ __forceinline__ double rotate_pair_global(double2* __restrict__ gp, double2* __restrict__ gq, int n, int lane, double tol2, double dgap2,
                                                     unsigned long long& nchk, unsigned long long& nrot) {
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
  nchk += n;
  if (!rot_params(al, be, gr, gi, tol2, dgap2, c, sr, si, cos2)) return cos2;
  nrot += n;
  for (int i = lane; i < n; i += 32) {
    const double2 a = __ldcg(gp + i), b = __ldcg(gq + i);
    __stcg(gp + i, make_double2(c * a.x - (sr * b.x + si * b.y), c * a.y - (sr * b.y - si * b.x)));
    __stcg(gq + i, make_double2(sr * a.x - si * a.y + c * b.x, sr * a.y + si * a.x + c * b.y));
  }
  return cos2;
}

__global__ void __launch_bounds__(128) seed_large_kernel(int n, const double2* __restrict__ A, double2* __restrict__ G,
                                                         const double* __restrict__ sigma_p, int* __restrict__ rot_flags,
                                                         double* __restrict__ mu_unsorted, int max_sweeps, double tol2, double gap2) {
  cg::grid_group grid = cg::this_grid();
  const int tid = threadIdx.x, lane = tid & 31;
  const int gwarp = (blockIdx.x * blockDim.x + tid) >> 5, nwarps = (gridDim.x * blockDim.x) >> 5;
  const size_t gtid = (size_t)blockIdx.x * blockDim.x + tid, gthr = (size_t)gridDim.x * blockDim.x;
  const double sigma = *sigma_p;
  const double dgap2 = gap2 * sigma * sigma / n;
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
  unsigned long long nchk = 0, nrot = 0;
  if (sigma > 0) {
    for (int sweep = 0; sweep < max_sweeps; ++sweep) {
      double cmax = 0;
      for (int r = 0; r < M - 1; ++r) {
        for (int i = gwarp; i < npairs; i += nwarps) {
          int p, q;
          rr_pair(M, r, i, p, q);
          if (q < n) cmax = fmax(cmax, rotate_pair_global(G + (size_t)p * n, G + (size_t)q * n, n, lane, tol2, dgap2, nchk, nrot));
        }
        if (r == M - 2 && cmax > kSeedStopCos2 && lane == 0) rot_flags[sweep] = 1;
        grid.sync();
      }
      if (!rot_flags[sweep]) break;
    }
  }
  if (lane == 0) seed_count(nchk, nrot);
  for (int j = gwarp; j < n; j += nwarps) {
    double s = 0;
    for (int i = lane; i < n; i += 32) { const double2 a = G[(size_t)j * n + i]; s += a.x * a.x + a.y * a.y; }
    s = warp_sum(s);
    if (lane == 0) mu_unsorted[j] = sqrt(s) - sigma;
  }
}

// ---- large matrices, blocked: a CTA holds two blocks of W columns in shared memory -------------------------------------------
// Same one-sided Jacobi, but the round-robin tournament runs over BLOCKS of W columns: per round a CTA loads its two blocks
// (2 W n double2, <= 200 KB), rotates every cross pair (W sub-rounds of W disjoint pairs, one warp per pair; in round 0 of a
// sweep also the pairs inside each block) and writes the blocks back.  Every pair of columns still meets once per sweep, but
// there are (n / W - 1) rounds (grid syncs, passes over G in L2) per sweep instead of (n - 1).
// WPP warps per pair: warp `part` of the pair owns the rows [part * chunk, (part + 1) * chunk); the four partial sums meet in
// shared memory (s_red: [4 * WPP] doubles of this pair).  Contains one __syncthreads when WPP > 1: every warp of the CTA calls it.
template <int WPP>
__device__ __forceinline__ double rotate_pair_smem(double2* __restrict__ gp, double2* __restrict__ gq, int n, int lane, int part,
                                                   double* __restrict__ s_red, double tol2, double dgap2, unsigned long long& nchk,
                                                   unsigned long long& nrot) {
  const int chunk = (n + WPP - 1) / WPP;
  const int i0 = part * chunk, i1 = min(n, i0 + chunk);
  double al = 0, be = 0, gr = 0, gi = 0;
  for (int i = i0 + lane; i < i1; i += 32) {
    const double2 a = gp[i], b = gq[i];
    al = fma(a.x, a.x, fma(a.y, a.y, al));
    be = fma(b.x, b.x, fma(b.y, b.y, be));
    gr = fma(a.x, b.x, fma(a.y, b.y, gr));
    gi = fma(a.x, b.y, fma(-a.y, b.x, gi));
  }
  al = warp_sum(al); be = warp_sum(be); gr = warp_sum(gr); gi = warp_sum(gi);
  if (WPP > 1) {
    if (lane == 0) { s_red[4 * part + 0] = al; s_red[4 * part + 1] = be; s_red[4 * part + 2] = gr; s_red[4 * part + 3] = gi; }
    __syncthreads();
    al = be = gr = gi = 0;
#pragma unroll
    for (int p = 0; p < WPP; ++p) { al += s_red[4 * p + 0]; be += s_red[4 * p + 1]; gr += s_red[4 * p + 2]; gi += s_red[4 * p + 3]; }
  }
  double c, sr, si, cos2;
  const bool rot = rot_params(al, be, gr, gi, tol2, dgap2, c, sr, si, cos2);
  if (part == 0) { nchk += n; if (rot) nrot += n; }
  if (!rot) return cos2;
  for (int i = i0 + lane; i < i1; i += 32) {
    const double2 a = gp[i], b = gq[i];
    gp[i] = make_double2(c * a.x - (sr * b.x + si * b.y), c * a.y - (sr * b.y - si * b.x));
    gq[i] = make_double2(sr * a.x - si * a.y + c * b.x, sr * a.y + si * a.x + c * b.y);
  }
  return cos2;
}

// 1-D bulk copies of whole columns between global memory (L2) and shared memory through the TMA engine (cp.async.bulk): one
// elected thread issues 2 W copies of 16 n bytes, all in flight at once, instead of every thread walking the columns with 16-byte
// loads (a handful of dependent L2 round trips per thread).
__device__ __forceinline__ uint32_t seed_smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void seed_mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "SW_%=:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra SD_%=;\n\t"
      "bra SW_%=;\n\t"
      "SD_%=:\n\t}" ::"r"(seed_smem_u32(bar)), "r"(parity)
      : "memory");
}

template <int W, int NWARPS>
__global__ void __launch_bounds__(32 * NWARPS) seed_block_kernel(int n, const double2* __restrict__ A, double2* __restrict__ G,
                                                         const double* __restrict__ sigma_p, int* __restrict__ rot_flags,
                                                         double* __restrict__ mu_unsorted, int max_sweeps, double tol2, double gap2, int use_tma) {
  extern __shared__ double2 s_cols[];  // [2 W][n]
  constexpr int WPP = NWARPS / W;      // warps per pair: all warps of the CTA rotate in every sub-round
  __shared__ double s_red[W][4 * WPP];
  __shared__ __align__(8) uint64_t s_bar;
  uint32_t bar_phase = 0;
  if (threadIdx.x == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(seed_smem_u32(&s_bar)), "r"(1));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  cg::grid_group grid = cg::this_grid();
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int pr = warp % W, part = warp / W;
  const int gwarp = (blockIdx.x * blockDim.x + tid) >> 5, nwarps = (gridDim.x * blockDim.x) >> 5;
  const size_t gtid = (size_t)blockIdx.x * blockDim.x + tid, gthr = (size_t)gridDim.x * blockDim.x;
  const double sigma = *sigma_p;
  const double dgap2 = gap2 * sigma * sigma / n;
  for (size_t e = gtid; e < (size_t)n * n; e += gthr) {
    const int i = (int)(e % n), j = (int)(e / n);
    double2 a = (i <= j) ? A[(size_t)i * n + j] : A[(size_t)j * n + i];
    if (i > j) a.y = -a.y;
    if (i == j) { a.y = 0; a.x += sigma; }
    G[e] = a;
  }
  if (gtid < (size_t)max_sweeps) rot_flags[gtid] = 0;
  grid.sync();
  const int NB = (n + W - 1) / W, MB = NB + (NB & 1), npairs = MB / 2;
  unsigned long long nchk = 0, nrot = 0;
  if (sigma > 0) {
    for (int sweep = 0; sweep < max_sweeps; ++sweep) {
      double cmax = 0;
      for (int r = 0; r < MB - 1; ++r) {
        for (int pi = blockIdx.x; pi < npairs; pi += gridDim.x) {
          int bp, bq;
          rr_pair(MB, r, pi, bp, bq);
          // load (absent columns, beyond n or in the padding block, are zero: rot_params leaves zero columns alone);
          // one flat loop over the 2 W columns, unrolled, so that many independent L2 loads are in flight per thread
          if (use_tma) {
            int present = 0;
            for (int c = 0; c < 2 * W; ++c) {
              const int col = (c < W ? bp : bq) * W + (c % W);
              if (col < n) ++present;
              else
                for (int i = tid; i < n; i += 32 * NWARPS) s_cols[(size_t)c * n + i] = make_double2(0.0, 0.0);
            }
            if (tid == 0) {
              const uint32_t colb = (uint32_t)n * (uint32_t)sizeof(double2);
              asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(seed_smem_u32(&s_bar)), "r"(colb * (uint32_t)present)
                           : "memory");
              for (int c = 0; c < 2 * W; ++c) {
                const int col = (c < W ? bp : bq) * W + (c % W);
                if (col < n)
                  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                                   seed_smem_u32(s_cols + (size_t)c * n)),
                               "l"(G + (size_t)col * n), "r"(colb), "r"(seed_smem_u32(&s_bar))
                               : "memory");
              }
            }
            seed_mbar_wait(&s_bar, bar_phase);
            bar_phase ^= 1;
          } else {
            const int tot = 2 * W * n;
#pragma unroll 8
            for (int e = tid; e < tot; e += 32 * NWARPS) {
              const int c = e / n, i = e - c * n;
              const int col = (c < W ? bp : bq) * W + (c % W);
              s_cols[e] = col < n ? __ldcg(G + (size_t)col * n + i) : make_double2(0.0, 0.0);
            }
          }
          __syncthreads();
          if (r == 0 && W > 1) {
            // pairs inside each block, once per sweep: round-robin over W columns, both blocks at once
            for (int t = 0; t < W - 1; ++t) {
              const int blk = pr / (W / 2), i = pr % (W / 2);
              int p, q;
              rr_pair(W, t, i, p, q);
              cmax = fmax(cmax, rotate_pair_smem<WPP>(s_cols + (size_t)(blk * W + p) * n, s_cols + (size_t)(blk * W + q) * n, n, lane,
                                                      part, s_red[pr], tol2, dgap2, nchk, nrot));
              __syncthreads();
            }
          }
          for (int t = 0; t < W; ++t) {
            const int p = pr, q = W + (pr + t) % W;
            cmax = fmax(cmax, rotate_pair_smem<WPP>(s_cols + (size_t)p * n, s_cols + (size_t)q * n, n, lane, part, s_red[pr], tol2, dgap2, nchk, nrot));
            __syncthreads();
          }
          if (use_tma) {
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");  // the rotated columns (generic-proxy writes) to the TMA engine
            __syncthreads();
            if (tid == 0) {
              const uint32_t colb = (uint32_t)n * (uint32_t)sizeof(double2);
              for (int c = 0; c < 2 * W; ++c) {
                const int col = (c < W ? bp : bq) * W + (c % W);
                if (col < n)
                  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(G + (size_t)col * n),
                               "r"(seed_smem_u32(s_cols + (size_t)c * n)), "r"(colb)
                               : "memory");
              }
              asm volatile("cp.async.bulk.commit_group;" ::: "memory");
              asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");  // complete: the grid barrier below publishes the columns
              asm volatile("fence.proxy.async.global;" ::: "memory");
              __threadfence();
            }
          } else {
            const int tot = 2 * W * n;
#pragma unroll 8
            for (int e = tid; e < tot; e += 32 * NWARPS) {
              const int c = e / n, i = e - c * n;
              const int col = (c < W ? bp : bq) * W + (c % W);
              if (col < n) __stcg(G + (size_t)col * n + i, s_cols[e]);
            }
          }
          __syncthreads();
        }
        if (r == MB - 2 && cmax > kSeedStopCos2 && lane == 0) rot_flags[sweep] = 1;
        grid.sync();  // (a hand-written atomic-counter barrier measured no faster: 48.0 vs 46.4 ms per N = 1024 seed)
      }
      if (!rot_flags[sweep]) break;
    }
  }
  if (lane == 0) seed_count(nchk, nrot);
  for (int j = gwarp; j < n; j += nwarps) {
    double s = 0;
    for (int i = lane; i < n; i += 32) { const double2 a = G[(size_t)j * n + i]; s += a.x * a.x + a.y * a.y; }
    s = warp_sum(s);
    if (lane == 0) mu_unsorted[j] = sqrt(s) - sigma;
  }
}

template <int W, int NWARPS>
static int launch_block(int n, int sms, const double2* Ab, double2* G, double* sigma, int* flags, double* mu_uns, int ms, double t2,
                        double gap2, cudaStream_t s) {
  const size_t smem = sizeof(double2) * 2 * W * (size_t)n;
  if (cudaFuncSetAttribute(seed_block_kernel<W, NWARPS>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024) != cudaSuccess) {
    (void)cudaGetLastError();
    return ZKD_ERR_CUDA;
  }
  int maxb = 0;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&maxb, seed_block_kernel<W, NWARPS>, 32 * NWARPS, smem) != cudaSuccess || maxb < 1) {
    (void)cudaGetLastError();
    return ZKD_ERR_CUDA;
  }
  const int NB = (n + W - 1) / W, MB = NB + (NB & 1);
  int nblocks = MB / 2;
  if (nblocks > maxb * sms) nblocks = maxb * sms;
  int use_tma = options().seed_tma ? 1 : 0;
  void* args[] = {&n, (void*)&Ab, &G, &sigma, &flags, &mu_uns, &ms, &t2, &gap2, &use_tma};
  if (cudaLaunchCooperativeKernel((void*)seed_block_kernel<W, NWARPS>, dim3(nblocks), dim3(32 * NWARPS), args, smem, s) != cudaSuccess) {
    (void)cudaGetLastError();
    return ZKD_ERR_CUDA;
  }
  return ZKD_OK;
}

// ---- large matrices, blocked, GRAM form of a round (W = 4) -------------------------------------------------------------------
// The same rotations in the same order as seed_block_kernel<4, .>, but a round's 16 (round 0 of a sweep: 28) rotations are found
// on the 8 x 8 Gram matrix H = [P Q]^H [P Q] of the CTA's two blocks instead of on the long columns:
//   1. H in ONE pass over the 8 columns (36 dot products, every thread a few rows, 64 fp64 accumulators, warp transpose-reduce);
//   2. one warp runs the sub-rounds on H alone: (al, be, gamma) = (H_pp, H_qq, H_pq) are what the dot products of the rotated
//      columns would give (H <- J^H H J is exact in exact arithmetic), and the rotations accumulate in an 8 x 8 unitary U;
//   3. [P Q] <- [P Q] U in ONE pass (64 complex multiply-adds per row).
// A round then has one long-vector reduction and two passes over shared memory instead of W dependent sub-rounds of
// dot / reduce / barrier / parameters / update / barrier each (2.3 us per sub-round at n = 1024); the flop count is the same
// to 20 % (384 n DFMA per round against 320 n) and both passes run at the fp64 pipe's rate.  Rounding: H carries the noise of
// its two-sided updates (a few ulp of |g|^2 after <= 7 of them), the same order as freshly summed dot products.
// rotation k (0..3) of sub-round t: pairs inside the blocks (round-robin over 4 columns, both blocks at once) or cross pairs
__device__ __forceinline__ void gram_pair(bool inside, int t, int k, int& p, int& q) {
  if (inside) {
    rr_pair(4, t, k & 1, p, q);
    p += (k >> 1) * 4;
    q += (k >> 1) * 4;
  } else {
    p = k;
    q = 4 + ((k + t) & 3);
  }
}

template <int NWARPS>
__global__ void __launch_bounds__(32 * NWARPS) seed_blockg_kernel(int n, const double2* __restrict__ A, double2* __restrict__ G,
                                                                 const double* __restrict__ sigma_p, int* __restrict__ rot_flags,
                                                                 double* __restrict__ mu_unsorted, int max_sweeps, double tol2, double gap2) {
  constexpr int W = 4, C = 2 * W, NT = 32 * NWARPS;
  extern __shared__ double2 s_cols[];  // [C][n]
  __shared__ double s_part[NWARPS][64];
  __shared__ double2 s_H[C][C], s_U[C][C];
  __shared__ int s_any;
  __shared__ __align__(8) uint64_t s_bar;
  uint32_t bar_phase = 0;
  if (threadIdx.x == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(seed_smem_u32(&s_bar)), "r"(1));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  cg::grid_group grid = cg::this_grid();
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int gwarp = (blockIdx.x * blockDim.x + tid) >> 5, nwarps = (gridDim.x * blockDim.x) >> 5;
  const size_t gtid = (size_t)blockIdx.x * blockDim.x + tid, gthr = (size_t)gridDim.x * blockDim.x;
  const double sigma = *sigma_p;
  const double dgap2 = gap2 * sigma * sigma / n;
  for (size_t e = gtid; e < (size_t)n * n; e += gthr) {
    const int i = (int)(e % n), j = (int)(e / n);
    double2 a = (i <= j) ? A[(size_t)i * n + j] : A[(size_t)j * n + i];
    if (i > j) a.y = -a.y;
    if (i == j) { a.y = 0; a.x += sigma; }
    G[e] = a;
  }
  if (gtid < (size_t)max_sweeps) rot_flags[gtid] = 0;
  grid.sync();
  const int NB = (n + W - 1) / W, MB = NB + (NB & 1), npairs = MB / 2;
  unsigned long long nchk = 0, nrot = 0;
  const uint32_t colb = (uint32_t)n * (uint32_t)sizeof(double2);
  if (sigma > 0) {
    for (int sweep = 0; sweep < max_sweeps; ++sweep) {
      double cmax = 0;
      for (int r = 0; r < MB - 1; ++r) {
        for (int pi = blockIdx.x; pi < npairs; pi += gridDim.x) {
          int bp, bq;
          rr_pair(MB, r, pi, bp, bq);
          // load: absent columns (beyond n, or the padding block) are zero and rot_params leaves zero columns alone
          int present = 0;
          for (int c = 0; c < C; ++c) {
            const int col = (c < W ? bp : bq) * W + (c % W);
            if (col < n) ++present;
            else
              for (int i = tid; i < n; i += NT) s_cols[(size_t)c * n + i] = make_double2(0.0, 0.0);
          }
          if (tid == 0) {
            asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(seed_smem_u32(&s_bar)), "r"(colb * (uint32_t)present)
                         : "memory");
            for (int c = 0; c < C; ++c) {
              const int col = (c < W ? bp : bq) * W + (c % W);
              if (col < n)
                asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                                 seed_smem_u32(s_cols + (size_t)c * n)),
                             "l"(G + (size_t)col * n), "r"(colb), "r"(seed_smem_u32(&s_bar))
                             : "memory");
            }
          }
          seed_mbar_wait(&s_bar, bar_phase);
          bar_phase ^= 1;
          __syncthreads();  // the zero fill of absent columns
          // 1. Gram matrix: v[0..7] = H_aa, v[8 + k] / v[36 + k] = Re / Im of H_ab = sum_i conj(g_a[i]) g_b[i], k = pair (a < b)
          {
            double v[64];
#pragma unroll
            for (int k = 0; k < 64; ++k) v[k] = 0.0;
#pragma unroll 1
            for (int i = tid; i < n; i += NT) {
              double2 g[C];
#pragma unroll
              for (int c = 0; c < C; ++c) g[c] = s_cols[(size_t)c * n + i];
              int k = 0;
#pragma unroll
              for (int a = 0; a < C; ++a) {
                v[a] = fma(g[a].x, g[a].x, fma(g[a].y, g[a].y, v[a]));
#pragma unroll
                for (int b = a + 1; b < C; ++b, ++k) {
                  v[8 + k] = fma(g[a].x, g[b].x, fma(g[a].y, g[b].y, v[8 + k]));
                  v[36 + k] = fma(g[a].x, g[b].y, fma(-g[a].y, g[b].x, v[36 + k]));
                }
              }
            }
            // warp transpose-reduce: 64 values over 32 lanes, 62 exchanges; lane l ends up with the warp totals of values 2l, 2l + 1
#pragma unroll
            for (int off = 16, cnt = 32; off > 0; off >>= 1, cnt >>= 1) {
              const bool up = (lane & off) != 0;
#pragma unroll
              for (int k = 0; k < cnt; ++k) {
                const double send = up ? v[k] : v[k + cnt];
                const double keep = up ? v[k + cnt] : v[k];
                v[k] = keep + __shfl_xor_sync(0xffffffffu, send, off);
              }
            }
            s_part[warp][2 * lane] = v[0];
            s_part[warp][2 * lane + 1] = v[1];
          }
          __syncthreads();
          if (tid < C * C) {
            const int a = tid / C, b = tid % C;
            const int lo = a < b ? a : b, hi = a < b ? b : a;
            double re = 0, im = 0;
            if (a == b) {
#pragma unroll
              for (int w = 0; w < NWARPS; ++w) re += s_part[w][a];
            } else {
              const int k = lo * C - (lo * (lo + 1)) / 2 + (hi - lo - 1);  // index of the pair (lo < hi) in the enumeration above
#pragma unroll
              for (int w = 0; w < NWARPS; ++w) { re += s_part[w][8 + k]; im += s_part[w][36 + k]; }
              if (a > b) im = -im;
            }
            s_H[a][b] = make_double2(re, im);
            s_U[a][b] = make_double2(a == b ? 1.0 : 0.0, 0.0);
          }
          if (tid == 0) s_any = 0;
          __syncthreads();
          // 2. the sub-rounds on H (warp 0): lane = (k, e), k = rotation of the sub-round, e = row (column step) / column (row step)
          if (warp == 0) {
            const int k = lane >> 3, e = lane & 7;
            bool any = false;
            const int nsub = (r == 0 ? W - 1 : 0) + W;
            for (int ts = 0; ts < nsub; ++ts) {
              const bool inside = r == 0 && ts < W - 1;
              int p, q;
              gram_pair(inside, inside ? ts : ts - (r == 0 ? W - 1 : 0), k, p, q);
              const double al = s_H[p][p].x, be = s_H[q][q].x;
              const double2 ga = s_H[p][q];
              double c, sr, si, cos2;
              const bool rot = rot_params(al, be, ga.x, ga.y, tol2, dgap2, c, sr, si, cos2);
              cmax = fmax(cmax, cos2);
              if (e == 0) { nchk += n; if (rot) nrot += n; }
              any = any || rot;
              if (!rot) { c = 1.0; sr = 0.0; si = 0.0; }
              // columns p, q of H and of U (row e):  x' = c x - conj(s) y,  y' = s x + c y
              {
                const double2 x = s_H[e][p], y = s_H[e][q];
                const double2 ux = s_U[e][p], uy = s_U[e][q];
                __syncwarp();
                s_H[e][p] = make_double2(c * x.x - (sr * y.x + si * y.y), c * x.y - (sr * y.y - si * y.x));
                s_H[e][q] = make_double2(sr * x.x - si * x.y + c * y.x, sr * x.y + si * x.x + c * y.y);
                s_U[e][p] = make_double2(c * ux.x - (sr * uy.x + si * uy.y), c * ux.y - (sr * uy.y - si * uy.x));
                s_U[e][q] = make_double2(sr * ux.x - si * ux.y + c * uy.x, sr * ux.y + si * ux.x + c * uy.y);
              }
              __syncwarp();
              // rows p, q of H (column e):  x' = c x - s y,  y' = conj(s) x + c y
              {
                const double2 x = s_H[p][e], y = s_H[q][e];
                __syncwarp();
                double2 xn = make_double2(c * x.x - (sr * y.x - si * y.y), c * x.y - (sr * y.y + si * y.x));
                double2 yn = make_double2(sr * x.x + si * x.y + c * y.x, sr * x.y - si * x.x + c * y.y);
                if (rot) {  // what the rotation makes exact: H_pq = 0, real diagonal
                  if (e == q) xn = make_double2(0.0, 0.0);
                  if (e == p) { yn = make_double2(0.0, 0.0); xn.y = 0.0; }
                  if (e == q) yn.y = 0.0;
                }
                s_H[p][e] = xn;
                s_H[q][e] = yn;
              }
              __syncwarp();
            }
            if (__any_sync(0xffffffffu, any) && lane == 0) s_any = 1;
          }
          __syncthreads();
          // 3. [P Q] <- [P Q] U, a row at a time (a thread reads its row before it writes it: in place)
          if (s_any) {
            // two rows per thread and step, their 16 complex outputs accumulated in registers (32 independent fp64 chains: the
            // fp64 pipe's latency is ~20 clocks, and a CTA has two warps per scheduler), U read as shared-memory broadcasts
#pragma unroll 1
            for (int i0 = tid; i0 < n; i0 += 2 * NT) {
              const int i1 = i0 + NT;
              const bool two = i1 < n;
              double2 o0[C], o1[C];
#pragma unroll
              for (int b = 0; b < C; ++b) o0[b] = o1[b] = make_double2(0.0, 0.0);
#pragma unroll
              for (int a = 0; a < C; ++a) {
                const double2 g0 = s_cols[(size_t)a * n + i0];
                const double2 g1 = two ? s_cols[(size_t)a * n + i1] : make_double2(0.0, 0.0);
#pragma unroll
                for (int b = 0; b < C; ++b) {
                  const double2 u = s_U[a][b];
                  o0[b].x = fma(g0.x, u.x, fma(-g0.y, u.y, o0[b].x));
                  o0[b].y = fma(g0.x, u.y, fma(g0.y, u.x, o0[b].y));
                  o1[b].x = fma(g1.x, u.x, fma(-g1.y, u.y, o1[b].x));
                  o1[b].y = fma(g1.x, u.y, fma(g1.y, u.x, o1[b].y));
                }
              }
#pragma unroll
              for (int b = 0; b < C; ++b) {
                s_cols[(size_t)b * n + i0] = o0[b];
                if (two) s_cols[(size_t)b * n + i1] = o1[b];
              }
            }
          }
          asm volatile("fence.proxy.async.shared::cta;" ::: "memory");  // the rotated columns (generic-proxy writes) to the TMA engine
          __syncthreads();
          if (tid == 0) {
            if (s_any) {
              for (int c = 0; c < C; ++c) {
                const int col = (c < W ? bp : bq) * W + (c % W);
                if (col < n)
                  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(G + (size_t)col * n),
                               "r"(seed_smem_u32(s_cols + (size_t)c * n)), "r"(colb)
                               : "memory");
              }
              asm volatile("cp.async.bulk.commit_group;" ::: "memory");
              asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");  // complete: the grid barrier below publishes the columns
              asm volatile("fence.proxy.async.global;" ::: "memory");
            }
            __threadfence();
          }
          __syncthreads();
        }
        if (r == MB - 2 && cmax > kSeedStopCos2 && warp == 0) rot_flags[sweep] = 1;
        grid.sync();
      }
      if (!rot_flags[sweep]) break;
    }
  }
  if (warp == 0 && (lane & 7) == 0) seed_count(nchk, nrot);
  for (int j = gwarp; j < n; j += nwarps) {
    double s = 0;
    for (int i = lane; i < n; i += 32) { const double2 a = G[(size_t)j * n + i]; s += a.x * a.x + a.y * a.y; }
    s = warp_sum(s);
    if (lane == 0) mu_unsorted[j] = sqrt(s) - sigma;
  }
}

template <int NWARPS>
static int launch_blockg(int n, int sms, const double2* Ab, double2* G, double* sigma, int* flags, double* mu_uns, int ms, double t2,
                         double gap2, cudaStream_t s) {
  const size_t smem = sizeof(double2) * 8 * (size_t)n;
  if (cudaFuncSetAttribute(seed_blockg_kernel<NWARPS>, cudaFuncAttributeMaxDynamicSharedMemorySize, 216 * 1024) != cudaSuccess) {
    (void)cudaGetLastError();
    return ZKD_ERR_CUDA;
  }
  int maxb = 0;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&maxb, seed_blockg_kernel<NWARPS>, 32 * NWARPS, smem) != cudaSuccess || maxb < 1) {
    (void)cudaGetLastError();
    return ZKD_ERR_CUDA;
  }
  const int NB = (n + 3) / 4, MB = NB + (NB & 1);
  int nblocks = MB / 2;
  if (nblocks > maxb * sms) nblocks = maxb * sms;
  void* args[] = {&n, (void*)&Ab, &G, &sigma, &flags, &mu_uns, &ms, &t2, &gap2};
  if (cudaLaunchCooperativeKernel((void*)seed_blockg_kernel<NWARPS>, dim3(nblocks), dim3(32 * NWARPS), args, smem, s) != cudaSuccess) {
    (void)cudaGetLastError();
    return ZKD_ERR_CUDA;
  }
  return ZKD_OK;
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

// square of the relative eigenvalue distance (in units of sigma / sqrt n) below which a pair counts as degenerate (rot_params):
// 2^-g with g = tau_bits + 2, i.e. always below the cluster threshold 2^-tau ||A||_F of S2 (||A||_F >= sigma / (1.5 sqrt n)).
// Option seed_degenerate_skip: 0 switches the rule off, 1 = this default, >= 8 = g itself (never below tau_bits + 1).
// Measured (c5 ms per step / c4 ms per step): off 169.4 / 203.1; g = 21: 154.4 / 210.1; 22: 154.8 / 200.2; 24: 155.6 / 213.6;
// 26: 159.1 / 203.0 - c5 gains a converged seed in 11 sweeps instead of an unconverged one in 12 and with it one refinement pass;
// c4 moves by +- one pass (the batch's slowest matrix decides), not systematically.
static double seed_gap2() {
  const int v = options().seed_degenerate_skip;
  if (!v) return 0.0;
  const int g = std::max(v >= 8 ? v : options().tau_bits + 2, options().tau_bits + 1);
  return ldexp(1.0, -2 * g);
}

int seed_fp64(int N, int batch, const double* A64, double* mu, double* V, int max_sweeps, cudaStream_t s, bool degenerate_skip) {
  const double tol = ldexp(1.0, -50);
  const double tol2 = tol * tol;
  double gap2 = degenerate_skip ? seed_gap2() : 0.0;
  int dev = 0, sms = 0;
  ZKD_CUDA_TRY(cudaGetDevice(&dev));
  ZKD_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  if (N <= 256 && !(options().seed_path == 4 && N > 96 && batch == 1)) {
    // ring: as many CTAs as give every processor (pair of columns) its own warp, with at most 16 (n > 128) or 32 warps per CTA;
    // fewer CTAs when the batch alone fills the machine.  A cluster of 16 is "non-portable": fall back to 8 when refused.
    const int P = (N + 1) / 2;
    const int maxw = N > 128 ? 16 : 32;
    const double2* A = (const double2*)A64;
    double2* Vv = (double2*)V;
    static int max_cluster = 16;
    // block ring (W columns per block): whenever its slots fit and the batch leaves room for one cluster per matrix
    // measured (N: column ring / W = 2 / W = 4, ms): 64: 0.50 / 0.64 / 0.57; 100: 1.54 / 1.38 / 1.19; 128: 2.00 / 1.88 / 1.51;
    // 256: 4.11 / 3.69 / 3.34 - a rotation's own dependent chain (load, dot, reduce, parameters, update, store: ~1.3 us) bounds both
    const int Wb = options().seed_ring_block < 0 ? (N >= 96 ? 4 : 0) : options().seed_ring_block;
    if ((Wb == 2 || Wb == 4) && N > 2 * Wb && options().seed_path != 2 && options().seed_path != 5 && N > 24) {
      const int NBk = (N + Wb - 1) / Wb, MB = NBk + (NBk & 1), Pb = MB / 2;
      const int ppc_max = std::min(std::min(16 / Wb, kRingbMaxProc), (int)(200 * 1024 / (64 * (size_t)Wb * N)));
      if (ppc_max >= 1) {
        int csize = 1;
        while (csize < 16 && (Pb + csize - 1) / csize > ppc_max) csize *= 2;
        const int ppc = (Pb + csize - 1) / csize;
        if (ppc <= ppc_max && csize <= max_cluster && (long)batch * csize <= 2L * sms) {
          int rc;
          if (Wb == 2) {
            if (N <= 32) rc = launch_ringb<1, 2>(N, batch, csize, ppc, A, mu, Vv, max_sweeps, tol2, gap2, s);
            else if (N <= 64) rc = launch_ringb<2, 2>(N, batch, csize, ppc, A, mu, Vv, max_sweeps, tol2, gap2, s);
            else if (N <= 128) rc = launch_ringb<4, 2>(N, batch, csize, ppc, A, mu, Vv, max_sweeps, tol2, gap2, s);
            else rc = launch_ringb<8, 2>(N, batch, csize, ppc, A, mu, Vv, max_sweeps, tol2, gap2, s);
          } else {
            if (N <= 32) rc = launch_ringb<1, 4>(N, batch, csize, ppc, A, mu, Vv, max_sweeps, tol2, gap2, s);
            else if (N <= 64) rc = launch_ringb<2, 4>(N, batch, csize, ppc, A, mu, Vv, max_sweeps, tol2, gap2, s);
            else if (N <= 128) rc = launch_ringb<4, 4>(N, batch, csize, ppc, A, mu, Vv, max_sweeps, tol2, gap2, s);
            else rc = launch_ringb<8, 4>(N, batch, csize, ppc, A, mu, Vv, max_sweeps, tol2, gap2, s);
          }
          if (!(rc == ZKD_ERR_CUDA && csize > 8)) return rc;
          max_cluster = 8;  // a cluster of 16 was refused: the column ring below copes with 8
        }
      }
    }
    const int want = options().seed_cluster > 0 ? options().seed_cluster : max_cluster;
    for (;;) {
      int csize = 1;
      while (csize < want && csize < max_cluster && P > 4 * csize) csize *= 2;
      while (csize > 1 && (long)batch * csize > 2L * sms) csize /= 2;
      while ((P + csize - 1) / csize > maxw) csize *= 2;
      int rc;
      // a whole matrix in one CTA: batches (one SM per matrix), and single tiny matrices, where a round of 8 pairs is cheaper behind
      // __syncthreads than behind a cluster barrier (measured: N = 16 0.109 -> 0.083 ms; N = 64 is 2.3 x slower that way)
      if ((csize == 1 || N <= 24 || options().seed_path == 5) && N <= 96 && options().seed_path != 2) {
        // a whole matrix per SM: plain CTA kernel (__syncthreads instead of cluster barriers)
        if (N <= 32) rc = launch_cta<1>(N, batch, A, mu, Vv, max_sweeps, tol2, gap2, s);
        else if (N <= 64) rc = launch_cta<2>(N, batch, A, mu, Vv, max_sweeps, tol2, gap2, s);
        else rc = launch_cta<3>(N, batch, A, mu, Vv, max_sweeps, tol2, gap2, s);
        return rc;
      }
      if (N <= 32) rc = launch_ring<1>(N, batch, csize, A, mu, Vv, max_sweeps, tol2, gap2, s);
      else if (N <= 64) rc = launch_ring<2>(N, batch, csize, A, mu, Vv, max_sweeps, tol2, gap2, s);
      else if (N <= 128) rc = launch_ring<4>(N, batch, csize, A, mu, Vv, max_sweeps, tol2, gap2, s);
      else rc = launch_ring<8>(N, batch, csize, A, mu, Vv, max_sweeps, tol2, gap2, s);
      if (rc == ZKD_ERR_CUDA && csize > 8 && max_cluster > 8) { max_cluster = 8; continue; }
      return rc;
    }
  }
  // large: cooperative grid, one matrix at a time
  const int M = N + (N & 1);
  int nblocks = (M / 2 + 3) / 4;  // 4 warps (pairs) per block
  int maxb = 0;
  ZKD_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&maxb, seed_large_kernel, 128, 0));
  if (nblocks > maxb * sms) nblocks = maxb * sms;
  char* buf = nullptr;
  const size_t nn = (size_t)N * N;
  const size_t bytes = sizeof(double2) * nn + sizeof(double) * (N + 8) + sizeof(int) * 128;
  // grow-only scratch of the calling thread (N^2 double2: 16 MB at N = 1024): a stream-ordered allocation here costs a pool
  // re-growth after every synchronisation of the caller (the default pool trims at sync points)
  {
    static thread_local char* cached = nullptr;
    static thread_local size_t cached_bytes = 0;
    if (cached_bytes < bytes) {
      ZKD_CUDA_TRY(cudaStreamSynchronize(s));
      if (cached) cudaFree(cached);
      cached = nullptr;
      cached_bytes = 0;
      ZKD_CUDA_TRY(cudaMalloc((void**)&cached, bytes));
      cached_bytes = bytes;
    }
    buf = cached;
  }
  double2* G = (double2*)buf;
  double* sigma = (double*)(G + nn);
  double* mu_uns = sigma + 8;
  int* flags = (int*)(mu_uns + N);
  int rc = ZKD_OK;
  for (int b = 0; b < batch && rc == ZKD_OK; ++b) {
    const double2* Ab = (const double2*)A64 + (size_t)b * nn;
    KtScope kt(KC_SEED, s);
    seed_sigma_kernel<<<1, 1024, 0, s>>>(N, Ab, sigma);
    double* mub = mu + (size_t)b * N;
    double2* Vb = (double2*)V + (size_t)b * nn;
    int n = N, ms = max_sweeps > 64 ? 64 : max_sweeps;
    double t2 = tol2;
    // blocked kernel with the widest column blocks whose pair fits shared memory; plain kernel beyond that
    const size_t col_bytes = sizeof(double2) * (size_t)n;
    const size_t smem_budget = 200 * 1024;
    const bool w16 = options().seed_block_warps == 16;  // 16 warps per CTA: twice the loads in flight, half the rows per warp
    if (options().seed_path != 3 && options().seed_gram && 8 * col_bytes <= 210 * 1024 &&
        (options().seed_gram == 2 || 16 * col_bytes > smem_budget))
      rc = launch_blockg<8>(n, sms, Ab, G, sigma, flags, mu_uns, ms, t2, gap2, s);
    else if (options().seed_path != 3 && 16 * col_bytes <= smem_budget)
      rc = w16 ? launch_block<8, 16>(n, sms, Ab, G, sigma, flags, mu_uns, ms, t2, gap2, s) : launch_block<8, 8>(n, sms, Ab, G, sigma, flags, mu_uns, ms, t2, gap2, s);
    else if (options().seed_path != 3 && 8 * col_bytes <= smem_budget)
      rc = w16 ? launch_block<4, 16>(n, sms, Ab, G, sigma, flags, mu_uns, ms, t2, gap2, s) : launch_block<4, 8>(n, sms, Ab, G, sigma, flags, mu_uns, ms, t2, gap2, s);
    else if (options().seed_path != 3 && 4 * col_bytes <= smem_budget)
      rc = w16 ? launch_block<2, 16>(n, sms, Ab, G, sigma, flags, mu_uns, ms, t2, gap2, s) : launch_block<2, 8>(n, sms, Ab, G, sigma, flags, mu_uns, ms, t2, gap2, s);
    else {
      void* args[] = {&n, (void*)&Ab, &G, &sigma, &flags, &mu_uns, &ms, &t2, &gap2};
      if (cudaLaunchCooperativeKernel((void*)seed_large_kernel, dim3(nblocks), dim3(128), args, 0, s) != cudaSuccess) {
        (void)cudaGetLastError();
        rc = ZKD_ERR_CUDA;
      }
    }
    if (rc != ZKD_OK) break;
    seed_sort_kernel<<<sms, 256, 0, s>>>(N, mu_uns, G, sigma, mub, Vb);
    count_launch(3);
    rc = launch_check();
  }
  return rc;
}

int seed_stats(uint64_t* elems_checked, uint64_t* elems_rotated, bool reset) {
  unsigned long long h[2] = {0, 0};
  ZKD_CUDA_TRY(cudaMemcpyFromSymbol(h, g_seed_stats, sizeof(h)));
  if (elems_checked) *elems_checked = h[0];
  if (elems_rotated) *elems_rotated = h[1];
  if (reset) {
    const unsigned long long z[2] = {0, 0};
    ZKD_CUDA_TRY(cudaMemcpyToSymbol(g_seed_stats, z, sizeof(z)));
  }
  return ZKD_OK;
}

// ---- the seed without any allocation (zkd_seed_fp64_static, include/zkd.h) ----------------------------------------------
// For callers that cannot call cudaMalloc (stream capture, serving loops, harnesses that forbid it).  Same kernels as the
// large-matrix branch of seed_fp64 above (seed_sigma_kernel, seed_block_kernel<8, 8>, seed_sort_kernel), for every N up to
// ZKD_SEED_STATIC_MAX_N, one matrix of the batch at a time, with G / sigma / unsorted eigenvalues / sweep flags in
// g_seed_static_scratch instead of a cudaMalloc'ed buffer.  No cudaMalloc, cudaFree, event or stream creation in here.
namespace {

constexpr int kSeedStaticMaxDevices = 64;

// device address of g_seed_static_scratch on the CURRENT device: looked up once per device, with that device current
int seed_static_scratch(unsigned char** out) {
  static unsigned char* addr[kSeedStaticMaxDevices] = {};
  static std::mutex mu;
  int dev = 0;
  ZKD_CUDA_TRY(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kSeedStaticMaxDevices) return ZKD_ERR_INVALID_ARG;
  std::lock_guard<std::mutex> lk(mu);
  if (!addr[dev]) {
    unsigned char* p = nullptr;
    if (cudaGetSymbolAddress((void**)&p, g_seed_static_scratch) != cudaSuccess || !p) {
      (void)cudaGetLastError();
      return ZKD_ERR_CUDA;
    }
    addr[dev] = p;
  }
  *out = addr[dev];
  return ZKD_OK;
}

}  // namespace

int seed_fp64_static(int N, int batch, const double* A64, double* mu, double* V, int max_sweeps, cudaStream_t s) {
  if (N > ZKD_SEED_STATIC_MAX_N) return ZKD_ERR_STATIC_LIMIT;
  const double tol = ldexp(1.0, -50);
  int dev = 0, sms = 0;
  ZKD_CUDA_TRY(cudaGetDevice(&dev));
  ZKD_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  unsigned char* buf = nullptr;
  ZKD_TRY(seed_static_scratch(&buf));
  const size_t nn = (size_t)N * N;
  double2* G = (double2*)buf;
  double* sigma = (double*)(buf + kSeedStaticGBytes);  // 8 doubles
  double* mu_uns = sigma + 8;                          // N <= 512 doubles
  int* flags = (int*)(mu_uns + ZKD_SEED_STATIC_MAX_N);  // 128 ints (the kernel clears the ones it uses)
  static_assert(sizeof(double) * (8 + ZKD_SEED_STATIC_MAX_N) + sizeof(int) * 128 <= 8192, "tail of the static scratch");
  static_assert(sizeof(double2) * 16 * ZKD_SEED_STATIC_MAX_N <= 200 * 1024, "two blocks of 8 columns fit shared memory");
  // the array keeps the last call's contents: sigma, the eigenvalues and the flags start from zero (G is overwritten from A)
  ZKD_CUDA_TRY(cudaMemsetAsync(buf + kSeedStaticGBytes, 0, 8192, s));
  int rc = ZKD_OK;
  for (int b = 0; b < batch && rc == ZKD_OK; ++b) {
    const double2* Ab = (const double2*)A64 + (size_t)b * nn;
    seed_sigma_kernel<<<1, 1024, 0, s>>>(N, Ab, sigma);
    const int ms = max_sweeps > 64 ? 64 : max_sweeps;
    rc = launch_block<8, 8>(N, sms, Ab, G, sigma, flags, mu_uns, ms, tol * tol, 0.0, s);
    if (rc != ZKD_OK) break;
    seed_sort_kernel<<<sms, 256, 0, s>>>(N, mu_uns, G, sigma, mu + (size_t)b * N, (double2*)V + (size_t)b * nn);
    count_launch(3);
    rc = launch_check();
  }
  return rc;
}

}  // namespace zkd

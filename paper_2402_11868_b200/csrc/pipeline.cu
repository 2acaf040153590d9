// pipeline.cu — host driver of the hot path: S0 ingest, then per level S1 seed -> S2 clusters -> S3 init ->
// S4 refinement loop -> S5 cluster Rayleigh-Ritz (by recursion on the projected cluster matrices), and S6 export.
//
// The refinement ("Rayleigh quotient iteration ... to recover the
// precision"), written for all eigenpairs at once with the current iterate as the preconditioner basis (S4g taken
// every step, at a precision that doubles with the residual):
//     G_c = X_c^H X_c ;  X_c, W_c <- (X_c, W_c)(I + (I - G_c)/2)            orthonormalise inside clusters (S4f)
//     S_c = X_c^H W_c ;  theta_j = Re (S_c)_jj                               Rayleigh quotients (S4c)
//     R_c = W_c - X_c S_c                                                    block residual (S4c)
//     C = X^H R ;  E_ij = C_ij / (theta_j - theta_i), 0 inside a cluster     correction equation, deflated (S4d)
//     T = X E ;  X <- X + T ;  W <- W + A T                                  update; W = A X kept incrementally (S4e, S4a)
// Every product is a windowed digit GEMM: only the bits of R, E, T that matter at the current residual level take
// part, and W = A X is never recomputed from scratch.  Exact solution of the correction equation is an RQI step;
// with the basis equal to the iterate the error squares each step (50 -> 100 -> 200 -> 400 -> 800 bits).
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <map>
#include <vector>

#include "blocks.h"
#include "gemm_i8.h"
#include "timing.h"

namespace zkd {

namespace {

// Stack allocator over the caller's workspace.  The workspace from zkd_diag_herm_bufsize covers the top level and
// one full-size level of cluster recursion; deeper recursion (rare: every level must split or shrink its clusters)
// overflows into the stream-ordered CUDA allocator, released when the level that asked for it returns.
struct Arena {
  char* base = nullptr;
  size_t size = 0, off = 0;
  cudaStream_t stream = nullptr;
  std::vector<void*> overflow;
  void* alloc(size_t bytes) {
    const size_t a = (off + 255) / 256 * 256;
    if (a + bytes <= size) {
      off = a + bytes;
      return base + a;
    }
    void* p = nullptr;
    if (cudaMallocAsync(&p, bytes ? bytes : 256, stream) != cudaSuccess) {
      (void)cudaGetLastError();
      return nullptr;
    }
    overflow.push_back(p);
    return p;
  }
  template <typename T>
  T* get(size_t n) { return (T*)alloc(sizeof(T) * n); }
  struct Mark { size_t off, nover; };
  Mark mark() const { return Mark{off, overflow.size()}; }
  void release(const Mark& m) {
    off = m.off;
    while (overflow.size() > m.nover) {
      cudaFreeAsync(overflow.back(), stream);
      overflow.pop_back();
    }
  }
};

enum { S_ERR = 0, S_MSB_R = 1, S_MSB_G = 2, S_MSB_E = 3, S_MSB_T = 4, S_GAP_INV = 5, S_NUM = 8 };

struct Ctx {
  // API precision of the call and what follows from it (NEXT-2, other precisions): results are wanted to 2^-(prec + 2) in the
  // scaled units, so nothing below FX bit fb = 812 - (prec + 44) has to be computed (fb = 0 at 768 bit: the FX floor itself).
  int prec = kPrec, fb = 0, tol_bits = 770;
  cudaStream_t s;
  Arena ar;
  void* gemm_ws;
  size_t gemm_ws_bytes;
  int* h_pin;  // pinned host staging, >= 4096 ints
};

struct LevelStats {
  int steps = 0, status = 0, msb_r = 0, msb_g = 0;
  std::vector<int> cl_stats;  // level 0 only: [nb][2]
};

int* pinned_staging() {
  static thread_local int* p = nullptr;
  if (!p) {
    if (cudaMallocHost((void**)&p, sizeof(int) * 65536) != cudaSuccess) {
      (void)cudaGetLastError();
      p = nullptr;
    }
  }
  return p;
}

inline int ceil_div(int a, int b) { return (a + b - 1) / b; }
inline int ilog2_ceil(int n) { int l = 0; while ((1 << l) < n) ++l; return l; }

int read_scalars(Ctx& c, const int* dev, int n, int* out) {
  ZKD_CUDA_TRY(cudaMemcpyAsync(c.h_pin, dev, sizeof(int) * n, cudaMemcpyDeviceToHost, c.s));
  ZKD_CUDA_TRY(cudaStreamSynchronize(c.s));
  for (int i = 0; i < n; ++i) out[i] = c.h_pin[i];
  return ZKD_OK;
}

using Groups = std::map<int, std::vector<SubProblem>>;

// clusters with more than one member, grouped by size (one batched sub-problem set per size)
Groups build_groups(const std::vector<int>& h_cl, int n, int nb) {
  Groups groups;
  for (int b = 0; b < nb; ++b) {
    int j = 0;
    while (j < n) {
      int k = j;
      while (k + 1 < n && h_cl[(size_t)b * n + k + 1] == h_cl[(size_t)b * n + j]) ++k;
      if (k > j) groups[k - j + 1].push_back(SubProblem{b, j});
      j = k + 1;
    }
  }
  return groups;
}

// ---- S4f / S4c of a level that has clusters with more than one member, as windowed GEMMs over cluster views -----------------
// For every cluster size m > 1 the clusters of that size form one batched product over views into X, W, S (column slices
// X_c = X[:, c0:c0+m] and diagonal blocks); singleton columns go through the fused singleton kernel.  All products carry
// only the bits above `cut` (an absolute FX bit position chosen from the previous pass's error level).
struct ClusterGroup { int m, nsub; const int* offX; const int* offB; const int* offR = nullptr; };  // column slice, diagonal block, row slice
struct ClusterPlan {
  std::vector<ClusterGroup> groups;
  bool has_singletons = false;
  int max_m = 1, max_nsub = 0;
  // Tiled form of the same pass for the int8 tcgen05 engine (S4b): when no cluster straddles a multiple of 128 columns, the
  // cluster-block products of a pass are taken over whole 128-column tiles (X_t^H X_t, X_t^H W_t: 128 x 128 x n; X_t M_t, X_t S_t:
  // n x 128 x 128 with M_t, S_t masked to their cluster blocks).  A tile computes 128 / m times the entries a cluster needs, on
  // an engine that is far more than that factor faster than the IMAD path on m x m x n products.
  bool tiled = false;
  std::vector<ClusterGroup> tile;  // one entry: m = 128, nsub = tiles that hold a cluster
  double tile_useful = 1.0;        // sum of m^2 over the clusters / (128^2 x tiles): the share of a tile product the clusters need
  bool tile_bdiag32 = false;       // no cluster straddles a multiple of 32 columns: M_t, S_t are block diagonal in aligned 32 x 32 blocks
};

int build_plan(Ctx& c, int n, int nb, const std::vector<int>& h_cl, int* plan_dev /* 2 n nb ints */, ClusterPlan* plan) {
  const Groups groups = build_groups(h_cl, n, nb);
  plan->groups.clear();
  plan->max_m = 1;
  plan->max_nsub = 0;
  std::vector<int> h;
  size_t clustered = 0;
  for (const auto& kv : groups) {
    ClusterGroup g;
    g.m = kv.first;
    g.nsub = (int)kv.second.size();
    g.offX = plan_dev + h.size();
    for (const SubProblem& sp : kv.second) h.push_back(sp.b * n * n + sp.col0);
    g.offB = plan_dev + h.size();
    for (const SubProblem& sp : kv.second) h.push_back(sp.b * n * n + sp.col0 * n + sp.col0);
    g.offR = plan_dev + h.size();
    for (const SubProblem& sp : kv.second) h.push_back(sp.b * n * n + sp.col0 * n);
    plan->groups.push_back(g);
    plan->max_m = std::max(plan->max_m, g.m);
    plan->max_nsub = std::max(plan->max_nsub, g.nsub);
    clustered += (size_t)g.m * g.nsub;
  }
  plan->has_singletons = clustered < (size_t)n * nb;
  plan->tiled = false;
  plan->tile_bdiag32 = false;
  plan->tile.clear();
  constexpr int TW = 128;
  // a tile computes 128 / m times the entries a cluster of m needs, but the int8 engine is that much faster per entry than the
  // IMAD engine down to m of about 10 (measured on c5, m = 16, after the issue-side and re-slicing work of round 2: cluster
  // passes 55 ms as tiles against 85 ms per cluster; before it, 97 against 81); the weighted mean cluster size decides.
  // cluster_tiles = 2 forces tiles wherever they can be formed (tests), 0 never uses them
  size_t sum_m2 = 0;
  for (const auto& kv : groups) sum_m2 += (size_t)kv.first * kv.first * kv.second.size();
  const bool tiles_pay = options().cluster_tiles == 2 || (options().cluster_tiles == 1 && sum_m2 >= 10 * clustered);
  if (options().gemm_path != 1 && tiles_pay && n >= TW && n % TW == 0 && 2 * clustered >= (size_t)n * nb &&
      gemm_i8_eligible(options().gemm_path, TW, TW, n, 1)) {
    bool ok = true, ok32 = true;
    std::vector<char> used((size_t)(n / TW) * nb, 0);
    for (const auto& kv : groups)
      for (const SubProblem& sp : kv.second) {
        if (sp.col0 / TW != (sp.col0 + kv.first - 1) / TW) ok = false;
        if (sp.col0 / 32 != (sp.col0 + kv.first - 1) / 32) ok32 = false;
        used[(size_t)sp.b * (n / TW) + sp.col0 / TW] = 1;
      }
    if (ok) {
      ClusterGroup g;
      g.m = TW;
      g.nsub = 0;
      std::vector<int> ox, ob;
      for (int b = 0; b < nb; ++b)
        for (int t = 0; t < n / TW; ++t)
          if (used[(size_t)b * (n / TW) + t]) {
            ox.push_back(b * n * n + t * TW);
            ob.push_back(b * n * n + t * TW * n + t * TW);
            ++g.nsub;
          }
      if (g.nsub > 0 && h.size() + 2 * (size_t)g.nsub <= (size_t)2 * n * nb) {
        g.offX = plan_dev + h.size();
        h.insert(h.end(), ox.begin(), ox.end());
        g.offB = plan_dev + h.size();
        h.insert(h.end(), ob.begin(), ob.end());
        plan->tile.push_back(g);
        plan->tiled = true;
        plan->tile_useful = (double)sum_m2 / ((double)TW * TW * g.nsub);
        plan->tile_bdiag32 = ok32;
      }
    }
  }
  if (!h.empty()) {
    ZKD_CUDA_TRY(cudaMemcpyAsync(plan_dev, h.data(), sizeof(int) * h.size(), cudaMemcpyHostToDevice, c.s));
    ZKD_CUDA_TRY(cudaStreamSynchronize(c.s));  // h is a local
  }
  return ZKD_OK;
}

inline int digits_for(int top, int cut) { return std::max(2, std::min(kND, ceil_div(top - cut, kDB) + 1)); }

// X, W <- (X, W)(I + (I - G)/2) on clusters;  S = X_c^H W_c;  theta = diag S;  R = W - X_c S_c.  msb(G - I) and msb(R) are
// accumulated into scal[S_MSB_G] / scal[S_MSB_R] (singleton columns included).
int cluster_pass(Ctx& c, int n, int nb, const ClusterPlan& plan, const int* cl, const int* cle, int32_t* X, int32_t* W, int32_t* R,
                 int32_t* Sm, int32_t* Gm, int32_t* theta, int* scal, int cut, size_t fxc, int* pm_orth /* [nb], may be null */) {
  const Options& opt = options();
  cudaStream_t s = c.s;
  const size_t cnt = (size_t)n * n * nb;
  const int topX = 815, topW = std::min(812 + ilog2_ceil(n) + 1, 840);
  auto view = [&](const int32_t* fx, int rows, int cols, bool ct, int top, int nw, const int* off) {
    GemmSide g;
    g.fx = fx; g.rows = rows; g.cols = cols; g.conj_transpose = ct; g.top_bit = top; g.nw = std::max(1, std::min(nw, kND));
    g.ld = n; g.off = off; g.plane_count = cnt;
    return g;
  };
  auto gemm = [&](int M, int N, int K, int batch, const GemmSide& P, const GemmSide& Q, int32_t* dst, GemmMode mode,
                  const int* dst_off, int* msb_out, int out_cut = -1) {
    GemmDstView dv;
    dv.ld = n; dv.off = dst_off; dv.plane_count = cnt;
    return gemm_complex(M, N, K, batch, P, Q, dst, mode, out_cut, opt.gemm_path, c.gemm_ws, c.gemm_ws_bytes, scal + S_ERR, msb_out, s,
                        &dv);
  };
  const int nwX = digits_for(topX, cut), nwW = digits_for(topW, cut);
  // M_t / S_t of a tiled pass are masked to their cluster blocks (ns_build with zero_rest, mask_offcluster): block diagonal
  auto bd = [&](GemmSide g) { g.bdiag32 = plan.tiled && plan.tile_bdiag32; return g; };
  // the products of this pass run per cluster (IMAD engine) or per 128-column tile (int8 tcgen05 engine), see ClusterPlan
  const std::vector<ClusterGroup>& groups = plan.tiled ? plan.tile : plan.groups;
  // timing only: the ALGORITHMIC work of a tile product is the share its cluster blocks need (the rest is executed padding)
  GemmUsefulScope useful(plan.tiled ? plan.tile_useful : 1.0);
  // S4f: G_c = X_c^H X_c, bits below cutG cleared so that M = (I - G)/2 is a short number
  const int cutG = std::max(1, cut);
  for (const ClusterGroup& g : groups)
    ZKD_TRY(gemm(g.m, g.m, n, g.nsub, view(X, n, g.m, true, topX, nwX, g.offX), view(X, n, g.m, false, topX, nwX, g.offX), Gm,
                 GemmMode::Assign, g.offB, nullptr, cutG));
  ZKD_TRY(ns_build(n, nb, cl, Gm, scal + S_MSB_G, s, cle, pm_orth, plan.tiled));
  int hs[S_NUM];
  ZKD_TRY(read_scalars(c, scal, S_NUM, hs));
  if (hs[S_ERR]) return ZKD_ERR_INTERNAL;
  const int msb_m = hs[S_MSB_G];  // |M| = |(I - G)/2| < 2^(msb_m - 813)
  if (msb_m > 0) {
    // X_c += X_c M_c, W_c += W_c M_c in place (the operands are copied into compact planes before the product runs).
    // These two must be exact to the FX floor, whatever the pass's precision: W = A X is kept incrementally, so an error
    // made here would stay in W for good.  Exact = all digits of X / W times all nonzero digits of M (those above cutG - 1).
    const int topM = msb_m + 1, nwM = std::max(1, std::min(kND, ceil_div(topM - (cutG - 1), kDB)));
    // ... of X / W only the digits whose product with the TOP bit of M still reaches the floor (one digit of guard below it), as for
    // A in W += A T: |M| < 2^(topM - 812), so a digit of X below FX bit fb + 784 - topM contributes less than 2^(fb - 28)
    const int lowXM = c.fb + std::max(0, 784 - topM);
    const int nwXm = digits_for(topX, lowXM), nwWm = digits_for(topW, lowXM);
    for (const ClusterGroup& g : groups) {
      ZKD_TRY(gemm(n, g.m, g.m, g.nsub, view(X, n, g.m, false, topX, nwXm, g.offX), bd(view(Gm, g.m, g.m, false, topM, nwM, g.offB)), X,
                   GemmMode::Add, g.offX, nullptr));
      ZKD_TRY(gemm(n, g.m, g.m, g.nsub, view(W, n, g.m, false, topW, nwWm, g.offX), bd(view(Gm, g.m, g.m, false, topM, nwM, g.offB)), W,
                   GemmMode::Add, g.offX, nullptr));
    }
  }
  // S4c
  {
    KtScope kt(KC_OTHER, s);
    ZKD_CUDA_TRY(cudaMemcpyAsync(R, W, fxc, cudaMemcpyDeviceToDevice, s));
  }
  if (plan.has_singletons) ZKD_TRY(singleton_step(n, nb, X, W, R, Sm, theta, scal + S_MSB_G, scal + S_MSB_R, s, cl, cle, pm_orth));
  for (const ClusterGroup& g : groups)
    ZKD_TRY(gemm(g.m, g.m, n, g.nsub, view(X, n, g.m, true, topX, nwX, g.offX), view(W, n, g.m, false, topW, nwW, g.offX), Sm,
                 GemmMode::Assign, g.offB, nullptr));
  if (plan.tiled) ZKD_TRY(mask_offcluster(n, nb, cl, cle, Sm, s));  // keep the cluster blocks of the tiles only (singletons: theta, R are the fused kernel's)
  ZKD_TRY(theta_from_diag(n, nb, Sm, theta, s, plan.tiled ? cl : nullptr, plan.tiled ? cle : nullptr));
  for (const ClusterGroup& g : groups)
    ZKD_TRY(gemm(n, g.m, g.m, g.nsub, view(X, n, g.m, false, topX, nwX, g.offX), bd(view(Sm, g.m, g.m, false, topW, nwW, g.offB)), R,
                 GemmMode::Sub, g.offX, scal + S_MSB_R));
  return ZKD_OK;
}

// S4h, early cluster split.  Inside a cluster the correction is deflated, so its convergence is only linear, at
// (spread of the cluster / gap to the outside)^2 per step, when the cluster has internal structure (c4: the 29-dimensional
// cluster holds 2^-21 .. 2^-60 and 24 zeros).  As soon as that structure stands above the noise of S_c = X_c^H W_c
// (Ritz-value error ~ |R|^2 / gap), the scaled block 2^k (S_c - mean) is diagonalised in fp64 by the seed kernel, the
// cluster basis is rotated by those eigenvectors (X_c, W_c <- X_c U, W_c U) and the cluster table is refined by the block's
// own clusters.  U is unitary to fp64 only; the S4f Newton-Schulz step of the following passes repairs that quadratically.
// Blocks whose structure is below the noise (true multiplicities) are left alone.  Sets *changed when any cluster split.
int try_split(Ctx& c, int n, int nb, const ClusterPlan& plan, const int32_t* Sm, int msb_r, int tol_msb, const int* noise, int32_t* X,
              int32_t* W, int32_t* Um, int32_t* G2 /* scratch, FxC n n nb */, int* scal, int* cl, int* cle, std::vector<int>& h_cl,
              bool* changed) {
  const Options& opt = options();
  cudaStream_t s = c.s;
  *changed = false;
  const Groups groups = build_groups(h_cl, n, nb);
  if (groups.empty()) return ZKD_OK;
  // eigenvalues of a block are told apart only when they differ by more than (a) the Ritz-value noise ~ |R|^2 / gap and
  // (b) 2^16 |R|: the correction E_ij = C_ij / (theta_j - theta_i) between the new clusters must stay small
  // and (c) 2^-390: ecalc's reciprocal range.
  const int noise_msb = std::max(std::max(tol_msb + 6, 812 - 390), std::max(2 * msb_r - 812 + opt.split_margin_bits, msb_r + 16));
  // Worth it?  Unsplit, the cluster gains about log2(gap / spread) bits per pass (measured: c4 ~20 bits, c5 ~195 bits),
  // with gap >= 2^-tau |A|_F ~ 2^(790-812).  A split resets the error inside the cluster to that of the fp64 eigenvectors
  // of the block (2^-50), i.e. costs about 5 passes of quadratic convergence.  Split only the blocks that would need more
  // passes than that at their linear rate (c4), not those whose structure is far below the gap (c5: left to S5).
  const int min_split_msb = 812 - opt.tau_bits - 2 - (msb_r - tol_msb) / 5;
  const Arena::Mark mark = c.ar.mark();
  bool any = false, first = true;
  for (const auto& kv : groups) {
    const int m = kv.first;
    const int nsub = (int)kv.second.size();
    c.ar.release(mark);
    const size_t hc = (size_t)m * m * nsub;
    SubProblem* subs_dev = c.ar.get<SubProblem>((size_t)nsub);
    int32_t* H = (int32_t*)c.ar.alloc(FxC::bytes(hc));
    int32_t* cbar = (int32_t*)c.ar.alloc(FxR::bytes((size_t)nsub));
    double2* H64 = c.ar.get<double2>(hc);
    double2* V64 = c.ar.get<double2>(hc);
    double* mu = c.ar.get<double>((size_t)m * nsub);
    int* ints = c.ar.get<int>((size_t)nsub * (6 + 2 * (size_t)m));
    if (!subs_dev || !H || !cbar || !H64 || !V64 || !mu || !ints) return ZKD_ERR_WORKSPACE;
    int *kshift = ints, *degen = ints + nsub, *noise_sub = ints + 2 * nsub, *floor_sub = ints + 3 * nsub, *sstats = ints + 4 * nsub;
    int *scl = ints + 6 * nsub, *scle = scl + (size_t)m * nsub;
    ZKD_CUDA_TRY(cudaMemcpyAsync(subs_dev, kv.second.data(), sizeof(SubProblem) * nsub, cudaMemcpyHostToDevice, s));
    ZKD_TRY(sub_gather(n, nb, m, nsub, subs_dev, Sm, H, cbar, kshift, degen, noise_msb, noise, noise_sub, floor_sub, min_split_msb, s));
    std::vector<int> hdeg((size_t)nsub);
    ZKD_CUDA_TRY(cudaMemcpyAsync(hdeg.data(), degen, sizeof(int) * nsub, cudaMemcpyDeviceToHost, s));
    ZKD_CUDA_TRY(cudaStreamSynchronize(s));  // also keeps kv.second alive for the copy above
    bool all_deg = true;
    for (int v : hdeg) all_deg = all_deg && v;
    if (opt.verbose) {
      std::vector<int> hk((size_t)nsub);
      cudaMemcpy(hk.data(), kshift, sizeof(int) * nsub, cudaMemcpyDeviceToHost);
      fprintf(stderr, "[zkd]   split? m %d nsub %d noise_msb %d min_split_msb %d: spread msb %d deg %d (first block)\n", m, nsub,
              noise_msb, min_split_msb, 810 - hk[0], hdeg[0]);
    }
    if (all_deg) continue;
    if (first) { ZKD_TRY(identity_blocks(n, nb, Um, s)); first = false; }
    ZKD_TRY(fxc_to_c64(hc, H, H64, s));
    ZKD_TRY(seed_fp64(m, nsub, (const double*)H64, mu, (double*)V64, opt.seed_sweeps, s));
    ZKD_TRY(cluster_detect(m, nsub, H64, mu, opt.tau_bits, floor_sub, scl, scle, sstats, s));
    ZKD_TRY(split_scatter(n, nb, m, nsub, subs_dev, V64, scl, scle, degen, Um, cl, cle, s));
    any = true;
  }
  if (any) {
    // cl / cle now hold the refined table; cl_old / cle_old the one the blocks of Um belong to
    std::vector<int> h_new((size_t)n * nb), h_cle_old((size_t)n * nb);
    int* cl_old = c.ar.get<int>((size_t)n * nb);
    int* cle_old = c.ar.get<int>((size_t)n * nb);
    if (!cl_old || !cle_old) return ZKD_ERR_WORKSPACE;
    ZKD_CUDA_TRY(cudaMemcpyAsync(h_new.data(), cl, sizeof(int) * n * nb, cudaMemcpyDeviceToHost, s));
    ZKD_CUDA_TRY(cudaMemcpyAsync(cl_old, h_cl.data(), sizeof(int) * n * nb, cudaMemcpyHostToDevice, s));
    for (int b = 0; b < nb; ++b) {
      int j = 0;
      while (j < n) {
        int k = j;
        while (k + 1 < n && h_cl[(size_t)b * n + k + 1] == h_cl[(size_t)b * n + j]) ++k;
        for (int t = j; t <= k; ++t) h_cle_old[(size_t)b * n + t] = k + 1;
        j = k + 1;
      }
    }
    ZKD_CUDA_TRY(cudaMemcpyAsync(cle_old, h_cle_old.data(), sizeof(int) * n * nb, cudaMemcpyHostToDevice, s));
    const size_t cnt = (size_t)n * n * nb;
    auto view = [&](const int32_t* fx, int rows, int cols, bool ct, int top, const int* off) {
      GemmSide g;
      g.fx = fx; g.rows = rows; g.cols = cols; g.conj_transpose = ct; g.top_bit = top; g.nw = digits_for(top, c.fb);
      g.ld = n; g.off = off; g.plane_count = cnt;
      return g;
    };
    auto gemm = [&](int M, int N, int K, int batch, const GemmSide& P, const GemmSide& Q, int32_t* dst, GemmMode mode, const int* dst_off) {
      GemmDstView dv;
      dv.ld = n; dv.off = dst_off; dv.plane_count = cnt;
      return gemm_complex(M, N, K, batch, P, Q, dst, mode, -1, opt.gemm_path, c.gemm_ws, c.gemm_ws_bytes, scal + S_ERR, nullptr, s, &dv);
    };
    // U is unitary to fp64 only.  Newton-Schulz on the blocks, U <- U (I + (I - U^H U)/2), squares that error each time
    // (2^-50 -> 2^-100 -> ... -> FX floor): X_c U then stays orthonormal and the Rayleigh quotients stay meaningful
    // against gaps far below 2^-50; what is left of the fp64 eigenvectors' error is a pure rotation, which S4d removes.
    // Iteration `it` starts from an error of about 2^-(48 2^it): U^H U is needed to twice that many bits only, and the
    // correction M = (I - U^H U)/2 is then a short number (bits below the cut cleared).
    for (int it = 0; it < 6; ++it) {
      const int cutU = std::max(c.fb + 1, 812 - (100 << it) - 30);
      const int nwU = digits_for(815, cutU);
      for (const ClusterGroup& g : plan.groups) {
        GemmSide P = view(Um, g.m, g.m, true, 815, g.offB), Q = view(Um, g.m, g.m, false, 815, g.offB);
        P.nw = Q.nw = nwU;
        GemmDstView dv;
        dv.ld = n; dv.off = g.offB; dv.plane_count = cnt;
        ZKD_TRY(gemm_complex(g.m, g.m, g.m, g.nsub, P, Q, G2, GemmMode::Assign, cutU, opt.gemm_path, c.gemm_ws, c.gemm_ws_bytes,
                             scal + S_ERR, nullptr, s, &dv));
      }
      ZKD_CUDA_TRY(cudaMemsetAsync(scal + S_MSB_T, 0, sizeof(int), s));
      ZKD_TRY(ns_build(n, nb, cl_old, G2, scal + S_MSB_T, s, cle_old));
      int hs[S_NUM];
      ZKD_TRY(read_scalars(c, scal, S_NUM, hs));
      if (hs[S_ERR]) return ZKD_ERR_INTERNAL;
      const int msb_m = hs[S_MSB_T];
      if (msb_m <= c.fb + 20 && cutU <= c.fb + 1) break;  // |U^H U - I| < 2^-792 (768 bit)
      if (msb_m == 0) continue;
      for (const ClusterGroup& g : plan.groups) {
        GemmSide Q = view(G2, g.m, g.m, false, msb_m + 1, g.offB);
        Q.nw = std::max(1, std::min(kND, ceil_div(msb_m + 1 - (cutU - 1), kDB)));
        ZKD_TRY(gemm(g.m, g.m, g.m, g.nsub, view(Um, g.m, g.m, false, 815, g.offB), Q, Um, GemmMode::Add, g.offB));
      }
    }
    // X_c <- X_c U_c, W_c <- W_c U_c in place (operands are staged before the product runs)
    const int topW = std::min(812 + ilog2_ceil(n) + 1, 840);
    for (const ClusterGroup& g : plan.groups) {
      ZKD_TRY(gemm(n, g.m, g.m, g.nsub, view(X, n, g.m, false, 815, g.offX), view(Um, g.m, g.m, false, 815, g.offB), X,
                   GemmMode::Assign, g.offX));
      ZKD_TRY(gemm(n, g.m, g.m, g.nsub, view(W, n, g.m, false, topW, g.offX), view(Um, g.m, g.m, false, 815, g.offB), W,
                   GemmMode::Assign, g.offX));
    }
    {
      int hs[S_NUM];
      ZKD_TRY(read_scalars(c, scal, S_NUM, hs));  // synchronises; the rotation GEMMs' operand checks land in S_ERR
      if (hs[S_ERR]) return ZKD_ERR_INTERNAL;
    }
    *changed = true;
    h_cl.swap(h_new);
  }
  c.ar.release(mark);
  return ZKD_OK;
}

// pm: device int[2 nb], per-matrix outcome of the level (zkd_info): [b] msb of the final residual of matrix b (sub-levels folded
// in), [nb + b] msb of G - I measured by the last pass.  Zeroed here.
int solve_level(Ctx& c, int n, int nb, const int32_t* A, int32_t* X, int32_t* lam, int depth, const int* noise, LevelStats* st, int* pm);

// One level of the path.  allow_split = false leaves every cluster to the S5 recursion (slower on spectra like c4's, but it
// has no heuristics to go wrong); *split_used tells the caller whether S4h took part in a failed attempt.
int solve_level_impl(Ctx& c, int n, int nb, const int32_t* A, int32_t* X, int32_t* lam, int depth, const int* noise, LevelStats* st,
                     bool allow_split, bool* split_used, int* pm) {
  const Options& opt = options();
  const size_t cnt = (size_t)n * n * nb;
  const size_t fxc = FxC::bytes(cnt);
  const Arena::Mark mark0 = c.ar.mark();
  cudaStream_t s = c.s;
  if (depth > 512) return ZKD_ERR_INTERNAL;  // every level strictly shrinks its clusters; a cascade peeled one eigenvalue per level is slow, not wrong

  // long-lived (needed by S5)
  int* cl = c.ar.get<int>((size_t)n * nb);
  int* cle = c.ar.get<int>((size_t)n * nb);
  int* stats = c.ar.get<int>((size_t)2 * nb);
  int32_t* Sm = (int32_t*)c.ar.alloc(fxc);
  int32_t* theta = lam;
  int* cl0 = c.ar.get<int>((size_t)n * nb);   // the clusters as detected (S4h refines cl / cle)
  int* cle0 = c.ar.get<int>((size_t)n * nb);
  int* plan_dev = c.ar.get<int>((size_t)2 * n * nb);
  bool split_done = false;
  const Arena::Mark mark1 = c.ar.mark();
  // short-lived
  double2* A64 = c.ar.get<double2>(cnt);
  double* mu = c.ar.get<double>((size_t)n * nb);
  double2* V = c.ar.get<double2>(cnt);
  int32_t* W = (int32_t*)c.ar.alloc(fxc);
  int32_t* R = (int32_t*)c.ar.alloc(fxc);
  int32_t* Cm = (int32_t*)c.ar.alloc(fxc);
  int32_t* T = (int32_t*)c.ar.alloc(fxc);
  int32_t* Gm = (int32_t*)c.ar.alloc(fxc);
  int* scal = c.ar.get<int>(S_NUM);
  if (!cl0 || !cle0 || !plan_dev) return ZKD_ERR_WORKSPACE;
  if (!cl || !cle || !stats || !Sm || !A64 || !mu || !V || !W || !R || !Cm || !T || !Gm || !scal) return ZKD_ERR_WORKSPACE;
  if (gemm_workspace_bytes(n, n, n, nb) > c.gemm_ws_bytes) return ZKD_ERR_WORKSPACE;

  // S1-S3
  ZKD_TRY(fxc_to_c64(cnt, A, A64, s));
  // the seed leaves degenerate pairs unrotated (seed.cu, rot_params) where S4h is there to resolve the inner structure of a cluster
  // as soon as it stands above the noise; without S4h the seed's own resolution inside a cluster is what keeps the deflated
  // correction fast on clusters that are wide against their gap (geometric cascades: 14 passes with it, > 120 without)
  ZKD_TRY(seed_fp64(n, nb, (const double*)A64, mu, (double*)V, opt.seed_sweeps, s, allow_split && opt.early_split != 0));
  ZKD_TRY(cluster_detect(n, nb, A64, mu, opt.tau_bits, nullptr, cl, cle, stats, s));
  int32_t* Xc = X;  // current iterate (may end up in T's storage; copied back at the end)
  int32_t* Tc = T;
  int32_t* Wc = W;
  int32_t* Cc = Cm;
  ZKD_TRY(init_x(cnt, V, Xc, s));
  ZKD_CUDA_TRY(cudaMemsetAsync(scal, 0, sizeof(int) * S_NUM, s));
  ZKD_CUDA_TRY(cudaMemsetAsync(pm, 0, sizeof(int) * 2 * nb, s));

  const int topA = 812, topX = 815;
  auto side = [&](const int32_t* fx, int top, int nw, bool ct) {
    GemmSide g;
    g.fx = fx; g.rows = n; g.cols = n; g.conj_transpose = ct; g.top_bit = top; g.nw = std::max(1, std::min(nw, kND));
    return g;
  };
  // W = A X0 : X0 has digits 27..29 only
  ZKD_TRY(gemm_complex(n, n, n, nb, side(A, topA, digits_for(topA, c.fb), false), side(Xc, topX, 3, false), Wc, GemmMode::Assign, -1, opt.gemm_path,
                       c.gemm_ws, c.gemm_ws_bytes, scal + S_ERR, nullptr, s));

  ZKD_CUDA_TRY(cudaMemcpyAsync(cl0, cl, sizeof(int) * n * nb, cudaMemcpyDeviceToDevice, s));
  ZKD_CUDA_TRY(cudaMemcpyAsync(cle0, cle, sizeof(int) * n * nb, cudaMemcpyDeviceToDevice, s));
  // cluster table to the host (needed for S5 and to pick the singleton fast path)
  std::vector<int> h_cl((size_t)n * nb), h_cl0;
  ZKD_CUDA_TRY(cudaMemcpyAsync(h_cl.data(), cl, sizeof(int) * n * nb, cudaMemcpyDeviceToHost, s));
  if (st && depth == 0) {
    st->cl_stats.resize((size_t)2 * nb);
    ZKD_CUDA_TRY(cudaMemcpyAsync(st->cl_stats.data(), stats, sizeof(int) * 2 * nb, cudaMemcpyDeviceToHost, s));
  }
  ZKD_CUDA_TRY(cudaStreamSynchronize(s));
  h_cl0 = h_cl;  // the clusters as detected (S4h refines h_cl)
  bool singletons = true;
  for (int b = 0; b < nb && singletons; ++b)
    for (int j = 1; j < n; ++j)
      if (h_cl[(size_t)b * n + j] != j) { singletons = false; break; }
  ClusterPlan plan;
  if (!singletons) ZKD_TRY(build_plan(c, n, nb, h_cl, plan_dev, &plan));
  int status = 2, steps = 0, prev_msb_r = 1 << 30;
  int e_prev = 15, last_cut = 0;  // error level of the previous pass (2^-e_prev), precision of the current one
  int hs[S_NUM];
  const int tol_msb = 812 - c.tol_bits;
  const int orth_ok = 812 - (c.tol_bits / 2 + 15);  // Newton-Schulz squares the deviation: 2^-400 -> 2^-800 at 768 bit
  const int fb = c.fb;
  for (int step = 0; step < opt.max_steps; ++step) {
    if (singletons) {
      // S4f + S4c fused: normalise columns, Rayleigh quotients, residual (X, W in place)
      ZKD_TRY(singleton_step(n, nb, Xc, Wc, R, Sm, theta, scal + S_MSB_G, scal + S_MSB_R, s, nullptr, nullptr, pm + nb));
    } else {
      // S4f + S4c on cluster views.  Results are needed to about 2^-(2 e_now + 40) and e_now <= 2 e_prev + 45.
      last_cut = std::max(fb, 812 - (4 * e_prev + 130));
      ZKD_TRY(cluster_pass(c, n, nb, plan, cl, cle, Xc, Wc, R, Sm, Gm, theta, scal, last_cut, fxc, pm + nb));
    }
    ZKD_TRY(min_gap(n, nb, theta, cl, scal + S_GAP_INV, s));
    ZKD_TRY(read_scalars(c, scal, S_NUM, hs));
    const int msb_r = hs[S_MSB_R], msb_g = hs[S_MSB_G];
    // clusters that S4h split apart can be much closer than 2^-tau |A|_F: C_ij / gap needs that many more bits of C, E, T
    const int gap_msb = hs[S_GAP_INV] ? 1024 - hs[S_GAP_INV] : 0;  // 0: one cluster only, nothing to correct between clusters
    const int gap_extra = (split_done && gap_msb) ? std::max(0, (812 - opt.tau_bits - 2) - gap_msb) : 0;
    if (opt.verbose) fprintf(stderr, "[zkd] depth %d n %d nb %d step %d: msbR %d (2^%d) msbG %d err %d\n", depth, n, nb, step, msb_r, msb_r - 812, msb_g, hs[S_ERR]);
    if (hs[S_ERR]) return ZKD_ERR_INTERNAL;
    steps = step;
    if (st) { st->msb_r = msb_r; st->msb_g = msb_g; }
    const bool exact_pass = singletons || last_cut <= fb;  // a windowed pass cannot certify convergence
    if (exact_pass && msb_r <= tol_msb && msb_g <= orth_ok) { status = 0; break; }
    if (exact_pass && step > 0 && msb_r > tol_msb && msb_r >= prev_msb_r - 2 && msb_g <= orth_ok) { status = 1; break; }
    e_prev = std::max(15, 812 - msb_r);
    if (step + 1 == opt.max_steps) break;
    prev_msb_r = msb_r;
    ZKD_CUDA_TRY(cudaMemsetAsync(scal, 0, sizeof(int) * S_NUM, s));
    ZKD_CUDA_TRY(cudaMemsetAsync(pm + nb, 0, sizeof(int) * nb, s));
    if (msb_r == 0) continue;  // residual exactly zero: only the orthonormalisation is still converging

    // S4h: split clusters whose internal structure stands above the noise of S_c
    if (split_done && step >= 48) return ZKD_ERR_INTERNAL;  // S4h is not getting anywhere: the caller retries without it
    if (!singletons && allow_split && opt.early_split && msb_g <= 812 - 45) {
      bool changed = false;
      ZKD_TRY(try_split(c, n, nb, plan, Sm, msb_r, tol_msb, noise, Xc, Wc, Gm, R, scal, cl, cle, h_cl, &changed));
      if (changed) {
        split_done = true;
        *split_used = true;
        ZKD_CUDA_TRY(cudaMemsetAsync(scal, 0, sizeof(int) * S_NUM, s));
        singletons = true;
        for (size_t t = 0; t < h_cl.size() && singletons; ++t) singletons = h_cl[t] == (int)(t % n);
        if (!singletons) ZKD_TRY(build_plan(c, n, nb, h_cl, plan_dev, &plan));
        prev_msb_r = 1 << 30;
        continue;  // S4f / S4c again with the rotated basis and the finer clusters
      }
    }

    if (gap_msb == 0) continue;  // a single cluster per matrix: no correction between clusters

    // S4d: C = X^H R on windows sized for this step's gain
    const int e = 812 - msb_r;                        // residual ~ 2^-e
    const int pb = std::max(40, std::min(e + 40, msb_r - fb + 30)) + gap_extra;  // relative bits worth computing for the correction
    const int nwX = ceil_div(pb + 3, 28);
    const int topR = msb_r + 2, nwR = ceil_div(pb + 2, 28);
    ZKD_TRY(gemm_complex(n, n, n, nb, side(Xc, topX, nwX, true), side(R, topR, nwR, false), Cc, GemmMode::Assign, -1, opt.gemm_path,
                         c.gemm_ws, c.gemm_ws_bytes, scal + S_ERR, nullptr, s));
    ZKD_TRY(ecalc(n, nb, theta, cl, Cc, pb + 8, scal + S_MSB_E, scal + S_ERR, s));
    // Second-order treatment of the cluster blocks.  The correction solves E_dc S_c - S_d E_dc = C_dc for every pair of
    // clusters; the division above takes S = diag(theta) only, which leaves an error of (spread of a cluster / gap) relative
    // to E and so caps the gain of a pass at log2(gap / spread) bits once the residual is below the spread (c5: 186 bits per
    // pass from 2^-405 on).  One fixed-point step with the off-diagonal parts O of the cluster blocks,
    //     E <- E - (E O - O E) ./ (theta_j - theta_i),
    // squares that factor; the two products are short (their result matters only above the cut of T) and run over the cluster
    // views like the products of the cluster pass.
    if (!singletons && opt.block_correction) {
      ZKD_CUDA_TRY(cudaMemsetAsync(scal + S_MSB_T, 0, sizeof(int), s));
      ZKD_TRY(offdiag_blocks(n, nb, cl, Sm, Gm, scal + S_MSB_T, s));
      ZKD_TRY(read_scalars(c, scal, S_NUM, hs));
      if (hs[S_ERR]) return ZKD_ERR_INTERNAL;
      const int msb_o = hs[S_MSB_T];
      const int msb_e0 = std::min(838, msb_r + (ilog2_ceil(n) + 1) / 2 + 1 + 813 - gap_msb);
      const int nbk = msb_o ? (pb + 8) - (gap_msb - msb_o) + 12 : 0;  // bits of the correction that lie above the cut of T
      // worth it only when the fixed-point step converges fast (spread / gap <= 2^-24: a cluster with structure near its gap, like c4's
      // 29-dimensional one before S4h has split it, gains a bit per step at the price of two products) and when the cap binds (nbk)
      if (nbk >= 8 && gap_msb - msb_o >= 24) {
        const int nwk = std::min(kND, ceil_div(nbk + 2, 28) + 1);
        const size_t cntv = (size_t)n * n * nb;
        auto vw = [&](const int32_t* fx, int rows, int cols, int top, const int* off) {
          GemmSide g;
          g.fx = fx; g.rows = rows; g.cols = cols; g.top_bit = top; g.nw = nwk; g.ld = n; g.off = off; g.plane_count = cntv;
          return g;
        };
        ZKD_CUDA_TRY(cudaMemsetAsync(R, 0, fxc, s));  // R is free from here to the next pass: K = E O - O E goes there
        for (const ClusterGroup& g : plan.groups) {
          GemmDstView dc, dr;
          dc.ld = n; dc.off = g.offX; dc.plane_count = cntv;
          dr.ld = n; dr.off = g.offR; dr.plane_count = cntv;
          ZKD_TRY(gemm_complex(n, g.m, g.m, g.nsub, vw(Cc, n, g.m, msb_e0 + 2, g.offX), vw(Gm, g.m, g.m, msb_o + 2, g.offB), R, GemmMode::Add, -1,
                               opt.gemm_path, c.gemm_ws, c.gemm_ws_bytes, scal + S_ERR, nullptr, s, &dc));
          ZKD_TRY(gemm_complex(g.m, n, g.m, g.nsub, vw(Gm, g.m, g.m, msb_o + 2, g.offB), vw(Cc, g.m, n, msb_e0 + 2, g.offR), R, GemmMode::Sub, -1,
                               opt.gemm_path, c.gemm_ws, c.gemm_ws_bytes, scal + S_ERR, nullptr, s, &dr));
        }
        ZKD_TRY(ecalc(n, nb, theta, cl, R, nbk + 8, nullptr, scal + S_ERR, s));
        ZKD_TRY(fxc_add_inplace(cnt, Cc, R, s, true));
      }
    }
    // No host read of msb(E): a rigorous bound sizes the windows instead.  |C_ij| = |x_i^H r_j| <= |x_i| |r_j| <= sqrt(n) max|R|
    // (columns are normalised), and |theta_j - theta_i| >= the smallest gap between neighbouring clusters, which the same
    // read as msb(R) delivered.  The bound is a few bits loose; the E / T windows get those bits back (pbE).
    const int msb_e = std::min(838, msb_r + (ilog2_ceil(n) + 1) / 2 + 1 + 813 - gap_msb + ((!singletons && opt.block_correction) ? 1 : 0));
    const int pbE = pb + 8;
    // S4e: T = X E (bits below cutT cleared so that W += A T tracks A X exactly), X += T, W += A T
    const int topE = msb_e + 2, nwE = ceil_div(pbE + 2, 28);
    const int cutT = std::max(fb, msb_e - pbE - 4);
    ZKD_TRY(gemm_complex(n, n, n, nb, side(Xc, topX, nwX, false), side(Cc, topE, nwE, false), Tc, GemmMode::Assign, cutT, opt.gemm_path,
                         c.gemm_ws, c.gemm_ws_bytes, scal + S_ERR, nullptr, s));
    ZKD_TRY(fxc_add_inplace(cnt, Xc, Tc, s));
    const int topT = msb_e + ilog2_ceil(n) + 2;
    const int nwT = ceil_div(topT - cutT, 28);
    const int nwA = std::max(1, std::min(kND, ceil_div(topT - fb, 28)));
    ZKD_TRY(gemm_complex(n, n, n, nb, side(A, topA, nwA, false), side(Tc, topT, nwT, false), Wc, GemmMode::Add, -1, opt.gemm_path,
                         c.gemm_ws, c.gemm_ws_bytes, scal + S_ERR, nullptr, s));
  }
  if (st) { st->steps = steps + 1; st->status = status; }
  ZKD_TRY(resid_per_matrix(n, nb, R, pm, s));  // R is the residual of the last pass
  if (split_done) {
    // Vectors of clusters that were split apart are orthogonal only to residual / gap, and the gaps inside a detected
    // cluster can be tiny (c4: 2^-61).  One symmetric (Loewdin / Newton-Schulz) orthonormalisation over the clusters AS
    // DETECTED squares that error; it moves the vectors by the same residual / gap inside a cluster whose spread is
    // <= 2^-tau, i.e. the residual grows by less than itself.
    // As GEMMs over the views of the detected clusters: G at full width, M = (I - G)/2 is tiny (|M| ~ residual / gap), so
    // X_c += X_c M_c is a 30 x 3-digit product.
    ClusterPlan plan0;
    ZKD_TRY(build_plan(c, n, nb, h_cl0, plan_dev, &plan0));
    {
      const size_t cnt0 = (size_t)n * n * nb;
      auto view = [&](const int32_t* fx, int rows, int cols, bool ct, int top, int nw, const int* off) {
        GemmSide g;
        g.fx = fx; g.rows = rows; g.cols = cols; g.conj_transpose = ct; g.top_bit = top; g.nw = std::max(1, std::min(nw, kND));
        g.ld = n; g.off = off; g.plane_count = cnt0;
        return g;
      };
      auto gemm = [&](int M, int N, int K, int batch, const GemmSide& P, const GemmSide& Q, int32_t* dst, GemmMode mode, const int* dst_off) {
        GemmDstView dv;
        dv.ld = n; dv.off = dst_off; dv.plane_count = cnt0;
        return gemm_complex(M, N, K, batch, P, Q, dst, mode, -1, opt.gemm_path, c.gemm_ws, c.gemm_ws_bytes, scal + S_ERR, nullptr, s, &dv);
      };
      ZKD_CUDA_TRY(cudaMemsetAsync(scal, 0, sizeof(int) * S_NUM, s));
      for (const ClusterGroup& g : plan0.groups)
        ZKD_TRY(gemm(g.m, g.m, n, g.nsub, view(Xc, n, g.m, true, topX, digits_for(topX, fb), g.offX),
                     view(Xc, n, g.m, false, topX, digits_for(topX, fb), g.offX), Gm, GemmMode::Assign, g.offB));
      ZKD_TRY(ns_build(n, nb, cl0, Gm, scal + S_MSB_G, s, cle0));
      ZKD_TRY(read_scalars(c, scal, S_NUM, hs));
      if (hs[S_ERR]) return ZKD_ERR_INTERNAL;
      const int msb_m = hs[S_MSB_G];
      if (msb_m > 0) {
        const int topM = msb_m + 1, nwM = std::max(1, std::min(kND, ceil_div(topM - fb, kDB)));
        for (const ClusterGroup& g : plan0.groups)
          ZKD_TRY(gemm(n, g.m, g.m, g.nsub, view(Xc, n, g.m, false, topX, digits_for(topX, fb), g.offX), view(Gm, g.m, g.m, false, topM, nwM, g.offB), Xc,
                       GemmMode::Add, g.offX));
      }
    }
  }
  if (Xc != X) ZKD_CUDA_TRY(cudaMemcpyAsync(X, Xc, fxc, cudaMemcpyDeviceToDevice, s));

  // S5: clusters with more than one member -> Rayleigh-Ritz on the projected matrix, by recursion
  Groups groups = build_groups(h_cl, n, nb);
  if (!groups.empty()) {
    ZKD_CUDA_TRY(cudaStreamSynchronize(s));  // short-lived buffers are about to be reused
    c.ar.release(mark1);
    int32_t* Um = (int32_t*)c.ar.alloc(fxc);
    if (!Um) return ZKD_ERR_WORKSPACE;
    ZKD_TRY(identity_blocks(n, nb, Um, s));
    const Arena::Mark mark2 = c.ar.mark();
    bool any = false;
    for (auto& kv : groups) {
      const int m = kv.first;
      const int nsub = (int)kv.second.size();
      c.ar.release(mark2);
      SubProblem* subs_dev = c.ar.get<SubProblem>((size_t)nsub);
      const size_t hc = (size_t)m * m * nsub;
      int32_t* H = (int32_t*)c.ar.alloc(FxC::bytes(hc));
      int32_t* U = (int32_t*)c.ar.alloc(FxC::bytes(hc));
      int32_t* cbar = (int32_t*)c.ar.alloc(FxR::bytes((size_t)nsub));
      int32_t* lam_sub = (int32_t*)c.ar.alloc(FxR::bytes((size_t)nsub * m));
      int* kshift = c.ar.get<int>((size_t)nsub);
      int* degen = c.ar.get<int>((size_t)nsub);
      int* noise_sub = c.ar.get<int>((size_t)nsub);
      int* pm_sub = c.ar.get<int>((size_t)2 * nsub);
      if (!subs_dev || !H || !U || !cbar || !lam_sub || !kshift || !degen || !noise_sub || !pm_sub) return ZKD_ERR_WORKSPACE;
      ZKD_CUDA_TRY(cudaMemcpyAsync(subs_dev, kv.second.data(), sizeof(SubProblem) * nsub, cudaMemcpyHostToDevice, s));
      ZKD_TRY(sub_gather(n, nb, m, nsub, subs_dev, Sm, H, cbar, kshift, degen, tol_msb + 6, noise, noise_sub, nullptr, 0, s));
      std::vector<int> hdeg((size_t)nsub);
      ZKD_CUDA_TRY(cudaMemcpyAsync(hdeg.data(), degen, sizeof(int) * nsub, cudaMemcpyDeviceToHost, s));
      ZKD_CUDA_TRY(cudaStreamSynchronize(s));
      bool all_deg = true;
      for (int v : hdeg) all_deg = all_deg && v;
      if (all_deg) continue;
      LevelStats sub;
      ZKD_TRY(solve_level(c, m, nsub, H, U, lam_sub, depth + 1, noise_sub, &sub, pm_sub));
      if (st && sub.status > st->status) st->status = sub.status;
      ZKD_TRY(fold_sub_stats(nsub, subs_dev, kshift, degen, pm_sub, pm, nb, s));
      ZKD_TRY(sub_scatter(n, nb, m, nsub, subs_dev, U, lam_sub, cbar, kshift, degen, Um, theta, s));
      any = true;
    }
    if (any) {
      // X_c <- X_c U_c in place, as batched GEMMs over the cluster views (operands are staged before the product runs)
      ClusterPlan planf;
      ZKD_TRY(build_plan(c, n, nb, h_cl, plan_dev, &planf));
      const size_t cntf = (size_t)n * n * nb;
      for (const ClusterGroup& g : planf.groups) {
        GemmSide P, Q;
        P.fx = X; P.rows = n; P.cols = g.m; P.conj_transpose = false; P.top_bit = topX; P.nw = digits_for(topX, fb); P.ld = n; P.off = g.offX; P.plane_count = cntf;
        Q.fx = Um; Q.rows = g.m; Q.cols = g.m; Q.conj_transpose = false; Q.top_bit = topX; Q.nw = digits_for(topX, fb); Q.ld = n; Q.off = g.offB; Q.plane_count = cntf;
        GemmDstView dv;
        dv.ld = n; dv.off = g.offX; dv.plane_count = cntf;
        ZKD_TRY(gemm_complex(n, g.m, g.m, g.nsub, P, Q, X, GemmMode::Assign, -1, opt.gemm_path, c.gemm_ws, c.gemm_ws_bytes, nullptr, nullptr,
                             s, &dv));
      }
    }
    ZKD_CUDA_TRY(cudaStreamSynchronize(s));
  }
  c.ar.release(mark0);
  return ZKD_OK;
}

// S4h (early cluster split) is a heuristic accelerator: when a level that used it fails (a window overflow, no convergence),
// the level is redone from its seed with every cluster left to the S5 recursion.
int solve_level(Ctx& c, int n, int nb, const int32_t* A, int32_t* X, int32_t* lam, int depth, const int* noise, LevelStats* st, int* pm) {
  const Arena::Mark mark = c.ar.mark();
  bool split_used = false;
  LevelStats tmp;
  int rc = solve_level_impl(c, n, nb, A, X, lam, depth, noise, st ? st : &tmp, true, &split_used, pm);
  const bool failed = rc == ZKD_ERR_INTERNAL || (rc == ZKD_OK && (st ? st->status : tmp.status) == 2);
  if (failed && split_used) {
    if (options().verbose) fprintf(stderr, "[zkd] depth %d n %d: retry without early splits\n", depth, n);
    ZKD_CUDA_TRY(cudaStreamSynchronize(c.s));
    c.ar.release(mark);
    if (st) *st = LevelStats();
    bool dummy = false;
    rc = solve_level_impl(c, n, nb, A, X, lam, depth, noise, st ? st : &tmp, false, &dummy, pm);
  }
  return rc;
}

// zkd_info per matrix.  pm[b] = msb of the final residual of matrix b (S5 sub-levels folded in), pm[batch + b] = msb of G - I
// measured by its last pass.  The refinement loop runs the whole batch until its worst matrix stops, so `steps` is the same
// for every matrix of a call; status 1 / 2 is given only to the matrices whose own residual is still above the tolerance.
__global__ void info_kernel(int batch, const int* __restrict__ status_in, int level_status, int steps, int tol_msb,
                            const int* __restrict__ pm, const int* __restrict__ cl_stats, zkd_info* __restrict__ info) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= batch) return;
  zkd_info o;
  const int msb_r = pm[b], msb_g = pm[batch + b];
  o.status = status_in[b] ? 3 : (msb_r <= tol_msb ? 0 : (level_status ? level_status : 1));
  o.steps = steps;
  o.n_clusters = cl_stats ? cl_stats[2 * b] : 0;
  o.max_cluster = cl_stats ? cl_stats[2 * b + 1] : 0;
  o.log2_resid = (float)(msb_r - 812);
  // msb_g is measured before the pass's Newton-Schulz step, which squares the deviation from orthonormality
  o.log2_orth = fmaxf(2.0f * (float)(msb_g - 812), -800.0f);
  info[b] = o;
}

size_t level_bytes(int N, int batch) {
  const size_t cnt = (size_t)N * N * batch;
  return 12 * (FxC::bytes(cnt) + 4096) + 3 * 16 * cnt + 64 * (size_t)N * batch + (1 << 20);
}

}  // namespace

size_t diag_workspace_bytes(int N, int batch) {
  return 2 * level_bytes(N, batch) + gemm_workspace_bytes(N, N, N, batch) + (32u << 20);
}

int diag_herm_device(int N, int batch, int prec, const void* A_api, void* eigvals_api, void* eigvecs_api, void* ws, size_t ws_bytes,
                     zkd_info* info, cudaStream_t s) {
  Ctx c;
  c.prec = prec;
  c.tol_bits = std::min(options().tol_bits, 790) - (kPrec - prec);  // "tol_bits" is quoted at 768 bit: prec + 2 by default
  c.fb = std::max(0, kFRAC - (c.tol_bits + 42));
  c.s = s;
  c.ar.base = (char*)ws;
  c.ar.size = ws_bytes;
  c.ar.stream = s;
  c.h_pin = pinned_staging();
  if (!c.h_pin) return ZKD_ERR_CUDA;
  c.gemm_ws_bytes = gemm_workspace_bytes(N, N, N, batch) + (32u << 20);
  c.gemm_ws = c.ar.alloc(c.gemm_ws_bytes);
  const size_t cnt = (size_t)N * N * batch;
  int32_t* A = (int32_t*)c.ar.alloc(FxC::bytes(cnt));
  int32_t* X = (int32_t*)c.ar.alloc(FxC::bytes(cnt));
  int32_t* lam = (int32_t*)c.ar.alloc(FxR::bytes((size_t)N * batch));
  int32_t* lam_sorted = (int32_t*)c.ar.alloc(FxR::bytes((size_t)N * batch));
  int* scale = c.ar.get<int>((size_t)2 * batch);  // [batch] scales, then [batch] raw maxima of the ingest
  int* status = c.ar.get<int>((size_t)batch);
  int* rank = c.ar.get<int>((size_t)N * batch);
  int* cl_stats_dev = c.ar.get<int>((size_t)2 * batch);
  int* pm = c.ar.get<int>((size_t)2 * batch);
  if (!c.gemm_ws || !A || !X || !lam || !lam_sorted || !scale || !status || !rank || !cl_stats_dev || !pm) return ZKD_ERR_WORKSPACE;

  ZKD_TRY(ingest_herm(N, batch, A_api, A, scale, status, s, prec));
  LevelStats st;
  {
    const int rc = solve_level(c, N, batch, A, X, lam, 0, nullptr, &st, pm);
    if (rc != ZKD_OK) {
      c.ar.release(Arena::Mark{c.ar.off, 0});  // an error return may have left overflow allocations behind
      return rc;
    }
  }
  ZKD_TRY(finalize_export(N, batch, X, lam, scale, eigvals_api, eigvecs_api, A /* scratch: A is dead */, lam_sorted, rank, s, prec));
  if (info) {
    const int* cs = nullptr;
    if (!st.cl_stats.empty()) {
      ZKD_CUDA_TRY(cudaMemcpyAsync(cl_stats_dev, st.cl_stats.data(), sizeof(int) * 2 * batch, cudaMemcpyHostToDevice, s));
      cs = cl_stats_dev;
    }
    info_kernel<<<(batch + 127) / 128, 128, 0, s>>>(batch, status, st.status, st.steps, 812 - c.tol_bits, pm, cs, info);
    count_launch();
    ZKD_TRY(launch_check());
    // st.cl_stats must outlive the async copy
    ZKD_CUDA_TRY(cudaStreamSynchronize(s));
  }
  return ZKD_OK;
}

// ---- NEXT-1: singular value decomposition through the same path (svd.cu) ---------------------------------
size_t svd_workspace_bytes(int M, int N, int batch) {
  const int n = M + N;
  const size_t cnt = (size_t)n * n * batch;
  return diag_workspace_bytes(n, batch) + 8 * (FxC::bytes(cnt) + 4096) + 64 * (size_t)n * batch + (8u << 20);
}

int svd_device(int M, int N, int batch, int prec, const void* A_api, void* S_api, void* U_api, void* V_api, void* ws, size_t ws_bytes,
               zkd_info* info, cudaStream_t s) {
  const Options& opt = options();
  const int n = M + N, K = std::min(M, N);
  Ctx c;
  c.prec = prec;
  c.tol_bits = std::min(opt.tol_bits, 790) - (kPrec - prec);
  c.fb = std::max(0, kFRAC - (c.tol_bits + 42));
  c.s = s;
  c.ar.base = (char*)ws;
  c.ar.size = ws_bytes;
  c.ar.stream = s;
  c.h_pin = pinned_staging();
  if (!c.h_pin) return ZKD_ERR_CUDA;
  c.gemm_ws_bytes = gemm_workspace_bytes(n, n, n, batch) + (32u << 20);
  c.gemm_ws = c.ar.alloc(c.gemm_ws_bytes);
  const size_t cnt = (size_t)n * n * batch;
  int32_t* A = (int32_t*)c.ar.alloc(FxC::bytes((size_t)M * N * batch));
  int32_t* H = (int32_t*)c.ar.alloc(FxC::bytes(cnt));
  int32_t* X = (int32_t*)c.ar.alloc(FxC::bytes(cnt));
  int32_t* lam = (int32_t*)c.ar.alloc(FxR::bytes((size_t)n * batch));
  int32_t* lam_sorted = (int32_t*)c.ar.alloc(FxR::bytes((size_t)n * batch));
  int32_t* Uf = (int32_t*)c.ar.alloc(FxC::bytes((size_t)M * K * batch));
  int32_t* Vf = (int32_t*)c.ar.alloc(FxC::bytes((size_t)N * K * batch));
  int32_t* Sf = (int32_t*)c.ar.alloc(FxR::bytes((size_t)K * batch));
  int32_t* Gm = (int32_t*)c.ar.alloc(FxC::bytes((size_t)K * K * batch));
  int* scale = c.ar.get<int>((size_t)2 * batch);
  int* status = c.ar.get<int>((size_t)batch);
  int* rank = c.ar.get<int>((size_t)n * batch);
  int* col_of = c.ar.get<int>((size_t)n * batch);
  int* r_dev = c.ar.get<int>((size_t)batch);
  int* cl0 = c.ar.get<int>((size_t)K * batch);
  int* cl_stats_dev = c.ar.get<int>((size_t)2 * batch);
  int* pm = c.ar.get<int>((size_t)2 * batch);
  int* scal = c.ar.get<int>(S_NUM);
  if (!c.gemm_ws || !A || !H || !X || !lam || !lam_sorted || !Uf || !Vf || !Sf || !Gm || !scale || !status || !rank || !col_of || !r_dev ||
      !cl0 || !cl_stats_dev || !pm || !scal)
    return ZKD_ERR_WORKSPACE;

  ZKD_TRY(ingest_general(M, N, batch, A_api, A, scale, status, s, prec));
  ZKD_TRY(jw_build(M, N, batch, A, H, s));
  LevelStats st;
  {
    const int rc = solve_level(c, n, batch, H, X, lam, 0, nullptr, &st, pm);
    if (rc != ZKD_OK) {
      c.ar.release(Arena::Mark{c.ar.off, 0});
      return rc;
    }
  }
  ZKD_TRY(rank_sort(n, batch, lam, rank, lam_sorted, s));
  // eigenvalues of H up to 2^-(prec - 10) (scaled units) count as zero: their eigenvectors mix null(A^H) and null(A)
  const int zero_msb = 812 - c.tol_bits + 12;
  ZKD_TRY(svd_plan(n, batch, rank, lam_sorted, zero_msb, col_of, r_dev, s));
  std::vector<int> h_r((size_t)batch);
  ZKD_CUDA_TRY(cudaMemcpyAsync(h_r.data(), r_dev, sizeof(int) * batch, cudaMemcpyDeviceToHost, s));
  ZKD_CUDA_TRY(cudaStreamSynchronize(s));
  ZKD_TRY(svd_gather(M, N, batch, X, col_of, r_dev, lam_sorted, Uf, Vf, Sf, s));

  // rank-deficient matrices (and M != N): the K - r missing pairs come from the zero cluster Z of H (dimension d0 = n - 2r).
  // P = Z_u^H Z_u (Z_u = the upper M rows) is an orthogonal projector on span(Z): eigenvalue 1 on the vectors that live in
  // null(A^H) (u-type, M - r of them), 0 on those in null(A) (v-type, N - r).  Diagonalising P / 8 with the same path separates
  // the two, whatever basis of the zero cluster the eigensolver returned.
  std::map<int, std::vector<int>> groups;
  for (int b = 0; b < batch; ++b) {
    if (h_r[b] > K) return ZKD_ERR_INTERNAL;  // more positive eigenvalues than min(M, N): cannot happen for a Jordan-Wielandt matrix
    if (h_r[b] < K) groups[h_r[b]].push_back(b);
  }
  const Arena::Mark markg = c.ar.mark();
  for (const auto& kv : groups) {
    c.ar.release(markg);
    const int r = kv.first, g = (int)kv.second.size(), d0 = n - 2 * r, nz = K - r;
    const size_t zc = (size_t)n * d0 * g, pc = (size_t)d0 * d0 * g;
    int* ints = c.ar.get<int>((size_t)8 * g);
    int32_t* Z = (int32_t*)c.ar.alloc(FxC::bytes(zc));
    int32_t* Pm = (int32_t*)c.ar.alloc(FxC::bytes(pc));
    int32_t* Y = (int32_t*)c.ar.alloc(FxC::bytes(pc));
    int32_t* lamY = (int32_t*)c.ar.alloc(FxR::bytes((size_t)d0 * g));
    int* pm2 = c.ar.get<int>((size_t)2 * g);
    if (!ints || !Z || !Pm || !Y || !lamY || !pm2) return ZKD_ERR_WORKSPACE;
    std::vector<int> h((size_t)8 * g);
    for (int v = 0; v < g; ++v) {
      const int b = kv.second[v];
      h[v] = b;                                           // mats
      h[g + v] = v * n * d0;                              // Z_u of element v
      h[2 * g + v] = v * n * d0 + M * d0;                 // Z_v
      h[3 * g + v] = v * d0 * d0 + (N - r);               // Y columns of the u-type vectors (eigenvalue 1/8: after the N - r zeros)
      h[4 * g + v] = v * d0 * d0;                         // Y columns of the v-type vectors
      h[5 * g + v] = b * M * K + r;                       // destination columns r .. K-1 of U
      h[6 * g + v] = b * N * K + r;                       // ... of V
      h[7 * g + v] = v * d0 * d0;                         // P of element v
    }
    ZKD_CUDA_TRY(cudaMemcpyAsync(ints, h.data(), sizeof(int) * h.size(), cudaMemcpyHostToDevice, s));
    ZKD_CUDA_TRY(cudaStreamSynchronize(s));  // h is a local
    ZKD_TRY(svd_zgather(n, batch, d0, r, g, ints, X, col_of, Z, s));
    ZKD_CUDA_TRY(cudaMemsetAsync(scal, 0, sizeof(int) * S_NUM, s));
    const int nwZ = digits_for(815, c.fb);
    auto zside = [&](const int* off, int rows, bool ct) {
      GemmSide sd;
      sd.fx = Z; sd.rows = rows; sd.cols = d0; sd.conj_transpose = ct; sd.top_bit = 815; sd.nw = nwZ; sd.ld = d0; sd.off = off; sd.plane_count = zc;
      return sd;
    };
    {
      GemmDstView dv;
      dv.ld = d0; dv.off = ints + 7 * g; dv.plane_count = pc;
      ZKD_TRY(gemm_complex(d0, d0, M, g, zside(ints + g, M, true), zside(ints + g, M, false), Pm, GemmMode::Assign, -1, opt.gemm_path, c.gemm_ws,
                           c.gemm_ws_bytes, scal + S_ERR, nullptr, s, &dv));
    }
    ZKD_TRY(fxc_shr(pc, Pm, 3, s));
    LevelStats st2;
    ZKD_TRY(solve_level(c, d0, g, Pm, Y, lamY, 1, nullptr, &st2, pm2));
    if (st2.status > st.status) st.status = st2.status;
    if (nz > 0) {
      auto yside = [&](const int* off) {
        GemmSide sd;
        sd.fx = Y; sd.rows = d0; sd.cols = nz; sd.conj_transpose = false; sd.top_bit = 815; sd.nw = nwZ; sd.ld = d0; sd.off = off; sd.plane_count = pc;
        return sd;
      };
      GemmDstView du, dvv;
      du.ld = K; du.off = ints + 5 * g; du.plane_count = (size_t)M * K * batch;
      dvv.ld = K; dvv.off = ints + 6 * g; dvv.plane_count = (size_t)N * K * batch;
      ZKD_TRY(gemm_complex(M, nz, d0, g, zside(ints + g, M, false), yside(ints + 3 * g), Uf, GemmMode::Assign, -1, opt.gemm_path, c.gemm_ws,
                           c.gemm_ws_bytes, scal + S_ERR, nullptr, s, &du));
      ZKD_TRY(gemm_complex(N, nz, d0, g, zside(ints + 2 * g, N, false), yside(ints + 4 * g), Vf, GemmMode::Assign, -1, opt.gemm_path, c.gemm_ws,
                           c.gemm_ws_bytes, scal + S_ERR, nullptr, s, &dvv));
    }
    int hs[S_NUM];
    ZKD_TRY(read_scalars(c, scal, S_NUM, hs));  // synchronises: the group's buffers are reused by the next group
    if (hs[S_ERR]) return ZKD_ERR_INTERNAL;
  }
  c.ar.release(markg);

  // every pair: unit norm of u and of v separately, common phase from v (the oracle's convention)
  ZKD_TRY(svd_phase(M, N, batch, Uf, Vf, s));
  // One symmetric (Loewdin / Newton-Schulz) orthonormalisation of U and of V.  The parts of eigenvectors of H for a tiny sigma are
  // orthogonal to the others only to residual / sigma (the mirrored eigenvalue -sigma is 2 sigma away); the step squares that
  // and moves A v - sigma u by sigma times it, i.e. by less than the residual.
  ZKD_CUDA_TRY(cudaMemsetAsync(cl0, 0, sizeof(int) * K * batch, s));
  for (int side = 0; side < 2; ++side) {
    int32_t* Xs = side ? Vf : Uf;
    const int rows = side ? N : M;
    const int nwX = digits_for(815, c.fb);
    // each pass squares the deviation (2^-170 when a sigma of 2^-600 sits next to the zero cluster): iterate to the tolerance
    for (int it = 0; it < 10; ++it) {
      GemmSide P, Q;
      P.fx = Xs; P.rows = rows; P.cols = K; P.conj_transpose = true; P.top_bit = 815; P.nw = nwX;
      Q.fx = Xs; Q.rows = rows; Q.cols = K; Q.conj_transpose = false; Q.top_bit = 815; Q.nw = nwX;
      ZKD_CUDA_TRY(cudaMemsetAsync(scal, 0, sizeof(int) * S_NUM, s));
      ZKD_TRY(gemm_complex(K, K, rows, batch, P, Q, Gm, GemmMode::Assign, -1, opt.gemm_path, c.gemm_ws, c.gemm_ws_bytes, scal + S_ERR, nullptr, s));
      ZKD_TRY(ns_build(K, batch, cl0, Gm, scal + S_MSB_G, s));
      int hs[S_NUM];
      ZKD_TRY(read_scalars(c, scal, S_NUM, hs));
      if (hs[S_ERR]) return ZKD_ERR_INTERNAL;
      const int msb_m = hs[S_MSB_G];
      if (msb_m <= c.fb + 8) break;                          // orthonormal to the working floor
      if (msb_m >= 812 - 2) return ZKD_ERR_INTERNAL;         // not a near-orthonormal set: the iteration would not converge
      GemmSide Pm2, Qm;
      Pm2.fx = Xs; Pm2.rows = rows; Pm2.cols = K; Pm2.top_bit = 815; Pm2.nw = nwX;
      Qm.fx = Gm; Qm.rows = K; Qm.cols = K; Qm.top_bit = msb_m + 1; Qm.nw = std::max(1, std::min(kND, ceil_div(msb_m + 1 - c.fb, kDB)));
      ZKD_TRY(gemm_complex(rows, K, K, batch, Pm2, Qm, Xs, GemmMode::Add, -1, opt.gemm_path, c.gemm_ws, c.gemm_ws_bytes, scal + S_ERR, nullptr, s));
      if (2 * (812 - msb_m) >= c.tol_bits + 30) break;       // the pass just applied squared the deviation below the tolerance
    }
  }
  // the orthonormalisation moved every vector by about the residual: restore the exact phase convention (Im v_k* = 0)
  ZKD_TRY(svd_phase(M, N, batch, Uf, Vf, s));
  ZKD_TRY(fx_to_api_scaled((size_t)K * batch, Sf, S_api, 0, scale, 1, (size_t)K, s, prec));
  ZKD_TRY(fxc_to_api((size_t)M * K * batch, Uf, U_api, s, prec));
  ZKD_TRY(fxc_to_api((size_t)N * K * batch, Vf, V_api, s, prec));
  if (info) {
    const int* cs = nullptr;
    if (!st.cl_stats.empty()) {
      ZKD_CUDA_TRY(cudaMemcpyAsync(cl_stats_dev, st.cl_stats.data(), sizeof(int) * 2 * batch, cudaMemcpyHostToDevice, s));
      cs = cl_stats_dev;
    }
    info_kernel<<<(batch + 127) / 128, 128, 0, s>>>(batch, status, st.status, st.steps, 812 - c.tol_bits, pm, cs, info);
    count_launch();
    ZKD_TRY(launch_check());
  }
  ZKD_CUDA_TRY(cudaStreamSynchronize(s));
  return ZKD_OK;
}

// ---- S4a': exact Rayleigh quotient iteration by multiprecision LU (lu.cu), the cross-check route for isolated spectra ---------------
size_t rqi_lu_workspace_bytes(int N, int batch) {
  const size_t cnt = (size_t)N * N * batch;
  return FxC::bytes(cnt * N) + 8 * (FxC::bytes(cnt) + 4096) + 3 * 16 * cnt + 64 * (size_t)N * batch + gemm_workspace_bytes(N, N, N, batch) +
         (34u << 20);
}

int diag_herm_rqi_lu_device(int N, int batch, int prec, const void* A_api, void* eigvals_api, void* eigvecs_api, void* ws, size_t ws_bytes,
                            zkd_info* info, cudaStream_t s) {
  const Options& opt = options();
  Ctx c;
  c.prec = prec;
  c.tol_bits = std::min(opt.tol_bits, 790) - (kPrec - prec);
  c.fb = 0;  // full width: this route is the cross-check, not the fast path
  c.s = s;
  c.ar.base = (char*)ws;
  c.ar.size = ws_bytes;
  c.ar.stream = s;
  c.h_pin = pinned_staging();
  if (!c.h_pin) return ZKD_ERR_CUDA;
  c.gemm_ws_bytes = gemm_workspace_bytes(N, N, N, batch) + (32u << 20);
  c.gemm_ws = c.ar.alloc(c.gemm_ws_bytes);
  const size_t cnt = (size_t)N * N * batch, P = (size_t)N * batch;
  int32_t* A = (int32_t*)c.ar.alloc(FxC::bytes(cnt));
  int32_t* X = (int32_t*)c.ar.alloc(FxC::bytes(cnt));
  int32_t* W = (int32_t*)c.ar.alloc(FxC::bytes(cnt));
  int32_t* R = (int32_t*)c.ar.alloc(FxC::bytes(cnt));
  int32_t* Sm = (int32_t*)c.ar.alloc(FxC::bytes(cnt));
  int32_t* Mx = (int32_t*)c.ar.alloc(FxC::bytes(cnt * N));
  int32_t* rhs = (int32_t*)c.ar.alloc(FxC::bytes(cnt));
  int32_t* invd = (int32_t*)c.ar.alloc(FxC::bytes(cnt));
  int32_t* lam = (int32_t*)c.ar.alloc(FxR::bytes(P));
  int32_t* lam_sorted = (int32_t*)c.ar.alloc(FxR::bytes(P));
  double2* A64 = c.ar.get<double2>(cnt);
  double2* V = c.ar.get<double2>(cnt);
  double* mu = c.ar.get<double>(P);
  int* perm = c.ar.get<int>(cnt);
  int* flags = c.ar.get<int>(P);
  int* scale = c.ar.get<int>((size_t)2 * batch);
  int* status = c.ar.get<int>((size_t)batch);
  int* rank = c.ar.get<int>(P);
  int* cl = c.ar.get<int>(P);
  int* cle = c.ar.get<int>(P);
  int* stats = c.ar.get<int>((size_t)2 * batch);
  int* pm = c.ar.get<int>((size_t)2 * batch);
  int* scal = c.ar.get<int>(S_NUM);
  if (!c.gemm_ws || !A || !X || !W || !R || !Sm || !Mx || !rhs || !invd || !lam || !lam_sorted || !A64 || !V || !mu || !perm || !flags ||
      !scale || !status || !rank || !cl || !cle || !stats || !pm || !scal)
    return ZKD_ERR_WORKSPACE;
  ZKD_TRY(ingest_herm(N, batch, A_api, A, scale, status, s, prec));
  ZKD_TRY(fxc_to_c64(cnt, A, A64, s));
  ZKD_TRY(seed_fp64(N, batch, (const double*)A64, mu, (double*)V, opt.seed_sweeps, s));
  ZKD_TRY(cluster_detect(N, batch, A64, mu, opt.tau_bits, nullptr, cl, cle, stats, s));
  std::vector<int> h_stats((size_t)2 * batch);
  ZKD_CUDA_TRY(cudaMemcpyAsync(h_stats.data(), stats, sizeof(int) * 2 * batch, cudaMemcpyDeviceToHost, s));
  ZKD_CUDA_TRY(cudaStreamSynchronize(s));
  for (int b = 0; b < batch; ++b)
    if (h_stats[2 * b + 1] > 1) return ZKD_ERR_CLUSTERED;  // per-vector RQI cannot separate clustered eigenvalues
  ZKD_TRY(init_x(cnt, V, X, s));
  auto side = [&](const int32_t* fx, int top, int nw) {
    GemmSide g;
    g.fx = fx; g.rows = N; g.cols = N; g.top_bit = top; g.nw = nw;
    return g;
  };
  const int tol_msb = 812 - c.tol_bits;
  int status_level = 2, steps = 0, hs[S_NUM], prev = 1 << 30;
  for (int it = 0; it < 8; ++it) {
    ZKD_CUDA_TRY(cudaMemsetAsync(scal, 0, sizeof(int) * S_NUM, s));
    ZKD_CUDA_TRY(cudaMemsetAsync(pm, 0, sizeof(int) * 2 * batch, s));
    // sigma_j = x_j^H A x_j (and the residual that decides convergence): W = A X at full width, then the fused singleton step
    ZKD_TRY(gemm_complex(N, N, N, batch, side(A, 812, kND), side(X, 815, it == 0 ? 3 : kND), W, GemmMode::Assign, -1, opt.gemm_path, c.gemm_ws,
                         c.gemm_ws_bytes, scal + S_ERR, nullptr, s));
    ZKD_TRY(singleton_step(N, batch, X, W, R, Sm, lam, scal + S_MSB_G, scal + S_MSB_R, s, nullptr, nullptr, pm + batch));
    ZKD_TRY(read_scalars(c, scal, S_NUM, hs));
    if (hs[S_ERR]) return ZKD_ERR_INTERNAL;
    steps = it + 1;
    if (opt.verbose) fprintf(stderr, "[zkd] exact RQI it %d: msbR %d (2^%d) msbG %d\n", it, hs[S_MSB_R], hs[S_MSB_R] - 812, hs[S_MSB_G]);
    if (hs[S_MSB_R] <= tol_msb && hs[S_MSB_G] <= 812 - (c.tol_bits / 2 + 15)) { status_level = 0; break; }
    if (it > 1 && hs[S_MSB_R] >= prev - 2 && hs[S_MSB_R] > tol_msb) { status_level = 1; break; }
    prev = hs[S_MSB_R];
    // y_j = (A - sigma_j I)^-1 x_j, normalised: one LU per eigenpair
    ZKD_TRY(rqi_setup(N, batch, A, lam, X, Mx, rhs, s));
    ZKD_TRY(lu_factor(N, (int)P, Mx, perm, invd, flags, s));
    ZKD_TRY(lu_solve(N, 1, (int)P, 1, Mx, perm, invd, rhs, flags, s));
    ZKD_TRY(rqi_scatter(N, batch, rhs, flags, X, s));
  }
  ZKD_TRY(resid_per_matrix(N, batch, R, pm, s));
  ZKD_TRY(finalize_export(N, batch, X, lam, scale, eigvals_api, eigvecs_api, A /* scratch */, lam_sorted, rank, s, prec));
  if (info) {
    info_kernel<<<(batch + 127) / 128, 128, 0, s>>>(batch, status, status_level, steps, tol_msb, pm, stats, info);
    count_launch();
    ZKD_TRY(launch_check());
  }
  ZKD_CUDA_TRY(cudaStreamSynchronize(s));
  return ZKD_OK;
}

// ---- NEXT-4: minimal MPS two-site update around the eigensolver (mps.cu) ---------------------------------------
size_t mps_workspace_bytes(int chiL, int chiC, int chiR, int d, int batch) {
  const size_t mL = (size_t)chiL * d, mR = (size_t)d * chiR;
  const size_t big = std::max(std::max(mL * mL, mL * mR), std::max(mL * chiC, chiC * mR)) * batch;
  return diag_workspace_bytes((int)mL, batch) + 12 * (FxC::bytes(big) + 4096) + FxC::bytes((size_t)d * d * d * d * batch) +
         64 * (mL + 16) * batch + (8u << 20);
}

int mps_update_device(int chiL, int chiC, int chiR, int d, int batch, int prec, const void* L_api, const void* R_api, const void* G_api,
                      int max_keep, int cutoff_bits, void* W_api, void* Lnew_api, void* Rnew_api, int* kept_dev, zkd_info* info, void* ws,
                      size_t ws_bytes, cudaStream_t s) {
  const Options& opt = options();
  const int mL = chiL * d, mR = d * chiR, n = mL, d2 = d * d;
  const int K = max_keep > 0 ? std::min(max_keep, mL) : mL;
  Ctx c;
  c.prec = prec;
  c.tol_bits = std::min(opt.tol_bits, 790) - (kPrec - prec);
  c.fb = std::max(0, kFRAC - (c.tol_bits + 42));
  c.s = s;
  c.ar.base = (char*)ws;
  c.ar.size = ws_bytes;
  c.ar.stream = s;
  c.h_pin = pinned_staging();
  if (!c.h_pin) return ZKD_ERR_CUDA;
  const int gmax = std::max(std::max(mL, mR), chiC);
  c.gemm_ws_bytes = std::max(gemm_workspace_bytes(n, n, n, batch), gemm_workspace_bytes(gmax, gmax, gmax, batch)) + (32u << 20);
  c.gemm_ws = c.ar.alloc(c.gemm_ws_bytes);
  const size_t cnt = (size_t)n * n * batch, tcnt = (size_t)mL * mR * batch;
  int32_t* Lf = (int32_t*)c.ar.alloc(FxC::bytes((size_t)mL * chiC * batch));
  int32_t* Rf = (int32_t*)c.ar.alloc(FxC::bytes((size_t)chiC * mR * batch));
  int32_t* Gf = (int32_t*)c.ar.alloc(FxC::bytes((size_t)d2 * d2 * batch));
  int32_t* T0 = (int32_t*)c.ar.alloc(FxC::bytes(tcnt));
  int32_t* T = (int32_t*)c.ar.alloc(FxC::bytes(tcnt));
  int32_t* TH = (int32_t*)c.ar.alloc(FxC::bytes(tcnt));
  int32_t* rho = (int32_t*)c.ar.alloc(FxC::bytes(cnt));
  int32_t* X = (int32_t*)c.ar.alloc(FxC::bytes(cnt));
  int32_t* Xs = (int32_t*)c.ar.alloc(FxC::bytes(cnt));
  int32_t* Ln = (int32_t*)c.ar.alloc(FxC::bytes((size_t)n * K * batch));
  int32_t* Rn = (int32_t*)c.ar.alloc(FxC::bytes((size_t)K * mR * batch));
  int32_t* Wt = (int32_t*)c.ar.alloc(FxR::bytes((size_t)K * batch));
  int32_t* lam = (int32_t*)c.ar.alloc(FxR::bytes((size_t)n * batch));
  int32_t* lam_sorted = (int32_t*)c.ar.alloc(FxR::bytes((size_t)n * batch));
  int* ints = c.ar.get<int>((size_t)(16 + n) * batch + S_NUM);
  if (!c.gemm_ws || !Lf || !Rf || !Gf || !T0 || !T || !TH || !rho || !X || !Xs || !Ln || !Rn || !Wt || !lam || !lam_sorted || !ints)
    return ZKD_ERR_WORKSPACE;
  int *sl = ints, *sr = ints + 2 * batch, *sg = ints + 4 * batch, *stl = ints + 6 * batch, *str_ = ints + 7 * batch, *stg = ints + 8 * batch;
  int *s_theta = ints + 9 * batch, *s_w = ints + 10 * batch, *pm = ints + 11 * batch, *status = ints + 13 * batch;
  int *cl_stats_dev = ints + 14 * batch, *rank = ints + 16 * batch, *scal = ints + (size_t)(16 + n) * batch;
  ZKD_TRY(ingest_general(mL, chiC, batch, L_api, Lf, sl, stl, s, prec));
  ZKD_TRY(ingest_general(chiC, mR, batch, R_api, Rf, sr, str_, s, prec));
  ZKD_TRY(ingest_general(d2, d2, batch, G_api, Gf, sg, stg, s, prec));
  auto side = [&](const int32_t* fx, int rows, int cols, int top, bool ct) {
    GemmSide g;
    g.fx = fx; g.rows = rows; g.cols = cols; g.conj_transpose = ct; g.top_bit = top; g.nw = digits_for(top, c.fb);
    return g;
  };
  ZKD_CUDA_TRY(cudaMemsetAsync(scal, 0, sizeof(int) * S_NUM, s));
  // Theta0 = L R, then the gate on the physical indices
  ZKD_TRY(gemm_complex(mL, mR, chiC, batch, side(Lf, mL, chiC, 812, false), side(Rf, chiC, mR, 812, false), T0, GemmMode::Assign, -1, opt.gemm_path,
                       c.gemm_ws, c.gemm_ws_bytes, scal + S_ERR, nullptr, s));
  ZKD_TRY(mps_gate(chiL, chiR, d, batch, T0, Gf, T, scal + S_MSB_T, s));
  int hs[S_NUM];
  ZKD_TRY(read_scalars(c, scal, S_NUM, hs));
  if (hs[S_ERR]) return ZKD_ERR_INTERNAL;
  // one power of two for the batch so that max |Theta| lies in [1/8, 1/4)
  const int t = hs[S_MSB_T] ? 810 - hs[S_MSB_T] : 0;
  if (t > 0) ZKD_TRY(fxc_shl(tcnt, T, t, s));
  if (t < 0) ZKD_TRY(fxc_shr(tcnt, T, -t, s));
  // rho = Theta Theta^H  (= (Theta^H)^H Theta^H: the GEMM conjugate-transposes its left operand)
  ZKD_TRY(conj_transpose(mL, mR, batch, T, TH, s));
  ZKD_CUDA_TRY(cudaMemsetAsync(scal, 0, sizeof(int) * S_NUM, s));
  ZKD_TRY(gemm_complex(mL, mL, mR, batch, side(TH, mR, mL, 812, true), side(TH, mR, mL, 812, false), rho, GemmMode::Assign, -1, opt.gemm_path,
                       c.gemm_ws, c.gemm_ws_bytes, scal + S_ERR, scal + S_MSB_E, s));
  ZKD_TRY(read_scalars(c, scal, S_NUM, hs));
  if (hs[S_ERR]) return ZKD_ERR_INTERNAL;
  const int u = hs[S_MSB_E] ? 810 - hs[S_MSB_E] : 0;
  if (u > 0) ZKD_TRY(fxc_shl(cnt, rho, u, s));
  if (u < 0) ZKD_TRY(fxc_shr(cnt, rho, -u, s));
  // the hot path: Hermitian eigendecomposition of the reduced density matrices
  LevelStats st;
  {
    const int rc = solve_level(c, n, batch, rho, X, lam, 0, nullptr, &st, pm);
    if (rc != ZKD_OK) {
      c.ar.release(Arena::Mark{c.ar.off, 0});
      return rc;
    }
  }
  ZKD_TRY(rank_sort(n, batch, lam, rank, lam_sorted, s));
  ZKD_TRY(phase_sorted(n, batch, X, rank, Xs, s));
  ZKD_TRY(mps_select(n, K, batch, cutoff_bits, lam_sorted, Wt, kept_dev, s));
  ZKD_TRY(mps_take(n, K, batch, Xs, Ln, s));
  // R' = L'^H Theta
  ZKD_CUDA_TRY(cudaMemsetAsync(scal, 0, sizeof(int) * S_NUM, s));
  ZKD_TRY(gemm_complex(K, mR, mL, batch, side(Ln, mL, K, 815, true), side(T, mL, mR, 812, false), Rn, GemmMode::Assign, -1, opt.gemm_path, c.gemm_ws,
                       c.gemm_ws_bytes, scal + S_ERR, nullptr, s));
  ZKD_TRY(mps_scales(batch, sl, sr, sg, t, u, s_theta, s_w, s));
  ZKD_TRY(fx_to_api_scaled((size_t)K * batch, Wt, W_api, 0, s_w, 1, (size_t)K, s, prec));
  ZKD_TRY(fxc_to_api((size_t)n * K * batch, Ln, Lnew_api, s, prec));
  ZKD_TRY(fxc_to_api_scaled((size_t)K * mR * batch, Rn, Rnew_api, s_theta, (size_t)K * mR, s, prec));
  if (info) {
    // malformed input in any of the three operands -> status 3
    ZKD_CUDA_TRY(cudaMemsetAsync(status, 0, sizeof(int) * batch, s));
    const int* cs = nullptr;
    if (!st.cl_stats.empty()) {
      ZKD_CUDA_TRY(cudaMemcpyAsync(cl_stats_dev, st.cl_stats.data(), sizeof(int) * 2 * batch, cudaMemcpyHostToDevice, s));
      cs = cl_stats_dev;
    }
    info_kernel<<<(batch + 127) / 128, 128, 0, s>>>(batch, stl, st.status, st.steps, 812 - c.tol_bits, pm, cs, info);
    count_launch();
    ZKD_TRY(launch_check());
  }
  ZKD_TRY(read_scalars(c, scal, S_NUM, hs));  // synchronises (st.cl_stats must outlive the copy)
  if (hs[S_ERR]) return ZKD_ERR_INTERNAL;
  return ZKD_OK;
}

}  // namespace zkd

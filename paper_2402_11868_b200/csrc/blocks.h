// blocks.h — host entry points of the O(N^2) / O(N^2 m) kernels (blocks.cu, finalize.cu).
#pragma once
#include "zkd_internal.h"

namespace zkd {

int fxc_to_c64(size_t count, const int32_t* src, double2* dst, cudaStream_t s);
int cluster_detect(int n, int nb, const double2* A64, const double* mu, int tau_bits, const int* floor_msb /*[nb], may be null*/,
                   int* cl, int* cle, int* stats, cudaStream_t s);
int init_x(size_t count, const double2* V, int32_t* X, cudaStream_t s);
// cle_skip1 != null: blocks of singleton clusters are left untouched
// msb_b != null: the same maximum per matrix (atomicMax into msb_b[b])
// zero_rest: entries outside the cluster blocks (and the skipped singleton diagonals) are set to zero instead of left alone
int ns_build(int n, int nb, const int* cl, int32_t* G, int* msb_out, cudaStream_t s, const int* cle_skip1 = nullptr, int* msb_b = nullptr,
             bool zero_rest = false);
// S_ij := 0 unless i and j belong to the same cluster of more than one member
int mask_offcluster(int n, int nb, const int* cl, const int* cle, int32_t* S, cudaStream_t s);
// fused S4f + S4c when every cluster of the level is a singleton: X, W updated in place, R, diag(S), theta written
// cl / cle != null: only the columns whose cluster is a singleton are processed
int singleton_step(int n, int nb, int32_t* X, int32_t* W, int32_t* R, int32_t* S, int32_t* theta, int* msb_g_out, int* msb_r_out,
                   cudaStream_t s, const int* cl = nullptr, const int* cle = nullptr, int* msb_g_b = nullptr /* [nb], per matrix */);
// per-matrix outcome (zkd_info): msb_r_b[b] <- max msb over the elements of matrix b of the residual array R
int resid_per_matrix(int n, int nb, const int32_t* R, int* msb_r_b, cudaStream_t s);
// gap_inv_out (device int, zeroed by the caller) <- max over neighbouring columns of different clusters of 1024 - msb(gap)
int min_gap(int n, int nb, const int32_t* theta, const int* cl, int* gap_inv_out, cudaStream_t s);
// cl / cle != null: singleton columns are skipped (their theta comes from the fused singleton kernel)
int theta_from_diag(int n, int nb, const int32_t* S, int32_t* theta, cudaStream_t s, const int* cl = nullptr, const int* cle = nullptr);
int fxc_add_inplace(size_t count, int32_t* X, const int32_t* T, cudaStream_t s, bool subtract = false);
// O_ij := S_ij for i != j in the same cluster, 0 elsewhere (the off-diagonal parts of the cluster blocks of S); msb_out <- max msb
int offdiag_blocks(int n, int nb, const int* cl, const int32_t* S, int32_t* O, int* msb_out, cudaStream_t s);
int ecalc(int n, int nb, const int32_t* theta, const int* cl, int32_t* C, int prec_bits, int* msb_out, int* err_flag, cudaStream_t s);

// finalize.cu
// S0: per-matrix scale (max exponent over the upper triangle) and ingest with Hermitian mirroring
int ingest_herm(int N, int batch, const void* A_api, int32_t* A_fx, int* scale /*[2 * batch]: scales, then scratch*/, int* status /*[batch]*/, cudaStream_t s,
                int prec = kPrec);
// S5 plumbing: gather cluster blocks of S into a batch of m x m sub-problems scaled by 2^k, and back
struct SubProblem { int b, col0; };  // matrix index and first column of the cluster
int sub_gather(int n, int nb, int m, int nsub, const SubProblem* subs_dev, const int32_t* S, int32_t* H /*nsub m m*/,
               int32_t* cbar /*FxR nsub*/, int* kshift /*nsub*/, int* degenerate /*nsub*/, int degenerate_msb,
               const int* noise_parent /*nb, may be null*/, int* noise_child /*nsub*/, int* floor_child /*nsub, may be null*/,
               int min_split_msb /* S4h: blocks with a smaller spread are reported degenerate; 0 for S5 */, cudaStream_t s);
// S4h (early split): U := V64 (fp64 eigenvectors of the scaled cluster blocks) placed on the diagonal blocks of Um, and the
// cluster table refined by the sub-problems' own clusters; degenerate sub-problems keep the identity and their cluster
int split_scatter(int n, int nb, int m, int nsub, const SubProblem* subs_dev, const double2* V64 /*nsub m m*/,
                  const int* sub_cl, const int* sub_cle, const int* degenerate, int32_t* Um /*nb n n*/, int* cl, int* cle,
                  cudaStream_t s);
int sub_scatter(int n, int nb, int m, int nsub, const SubProblem* subs_dev, const int32_t* U /*nsub m m*/, const int32_t* lam_sub,
                const int32_t* cbar, const int* kshift, const int* degenerate, int32_t* Um /*nb n n*/, int32_t* theta, cudaStream_t s);
int identity_blocks(int n, int nb, int32_t* Um, cudaStream_t s);
// per-matrix outcome: residual / orthonormality levels of the sub-problems (pm_sub: [2 nsub], in the sub-level's scaled units)
// folded into their parent matrices (pm_parent: [2 nb_parent]): resid msb - kshift, orth msb as it is
int fold_sub_stats(int nsub, const SubProblem* subs_dev, const int* kshift, const int* degenerate, const int* pm_sub, int* pm_parent,
                   int nb_parent, cudaStream_t s);
// S6: sort ascending, phase-normalise, export
int finalize_export(int N, int batch, const int32_t* X, const int32_t* lam, const int* scale, void* eigvals_api, void* eigvecs_api,
                    int32_t* scratch /* FxC batch N N */, int32_t* lam_sorted /* FxR batch N */, int* rank /* batch N */,
                    cudaStream_t s, int prec = kPrec);

// rank[b][j] = number of eigenvalues of matrix b that sort before lam[b][j] (ascending, stable); lam_sorted[b][rank] = lam[b][j]
int rank_sort(int N, int batch, const int32_t* lam, int* rank, int32_t* lam_sorted, cudaStream_t s);

// svd.cu (NEXT-1)
int ingest_general(int M, int N, int batch, const void* A_api, int32_t* A_fx, int* scale /*[2 batch]*/, int* status /*[batch]*/, cudaStream_t s,
                   int prec);
int jw_build(int M, int N, int batch, const int32_t* A_fx, int32_t* H_fx, cudaStream_t s);
int svd_plan(int n, int batch, const int* rank, const int32_t* lam_sorted, int zero_msb, int* col_of, int* r_out, cudaStream_t s);
int svd_gather(int M, int N, int batch, const int32_t* X, const int* col_of, const int* r, const int32_t* lam_sorted, int32_t* U, int32_t* V,
               int32_t* S, cudaStream_t s);
int svd_zgather(int n, int batch, int d0, int r, int g, const int* mats_dev, const int32_t* X, const int* col_of, int32_t* Z, cudaStream_t s);
int fxc_shr(size_t count, int32_t* X, int bits, cudaStream_t s);
int svd_phase(int M, int N, int batch, int32_t* U, int32_t* V, cudaStream_t s);


// mps.cu (NEXT-4)
int conj_transpose(int R, int C, int batch, const int32_t* src, int32_t* dst, cudaStream_t s);
int mps_gate(int chiL, int chiR, int d, int batch, const int32_t* T0, const int32_t* G, int32_t* T, int* msb_out, cudaStream_t s);
int fxc_shl(size_t count, int32_t* X, int bits, cudaStream_t s);
int mps_select(int n, int K, int batch, int cutoff_bits, const int32_t* lam_sorted, int32_t* Wt, int* kept, cudaStream_t s);
int mps_take(int n, int K, int batch, const int32_t* Xs, int32_t* Lnew, cudaStream_t s);
int mps_scales(int batch, const int* sl, const int* sr, const int* sg, int t, int u, int* s_theta, int* s_w, cudaStream_t s);
// S6 pieces on their own: out[:, rank[j]] = x_j with the phase convention A9 applied (out: FxC batch N N)
int phase_sorted(int N, int batch, const int32_t* X, const int* rank, int32_t* out, cudaStream_t s);

// lu.cu (NEXT-3, S4a')
// P A = L U in place for nprob N x N problems stored consecutively (complex FX planes over nprob N N elements); perm: [nprob][N];
// invd: complex FX [nprob][N] (1 / u_kk); flags: [nprob] (1 singular, 2 a pivot too small to invert, 4 the last pivot too small)
int lu_factor(int N, int nprob, int32_t* Mx, int* perm, int32_t* invd, int* flags, cudaStream_t s);
// B (complex FX planes over nprob N nrhs elements) <- A^-1 B (mode 0) or the unit-norm direction of A^-1 b (mode 1, nrhs = 1)
int lu_solve(int N, int nrhs, int nprob, int mode, const int32_t* Mx, const int* perm, const int32_t* invd, int32_t* B, int* flags,
             cudaStream_t s);
int rqi_setup(int N, int batch, const int32_t* A, const int32_t* theta, const int32_t* X, int32_t* Mx, int32_t* rhs, cudaStream_t s);
int rqi_scatter(int N, int batch, const int32_t* rhs, const int* flags, int32_t* X, cudaStream_t s);

}  // namespace zkd

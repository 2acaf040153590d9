/* include/zkd.h — C ABI of libzkd: 768-bit Hermitian eigendecomposition on one B200 (sm_100a).
 *
 * The operation: "diagonalizing N x N Hermitian matrix ... The 768-bit precision was used" (section
 * 2.1), by the route of ZKCM_CUS: a double-precision eigendecomposition followed by "the Rayleigh quotient
 * iteration ... to recover the precision" (section 2).  Every stage runs in hand-written CUDA
 * kernels; there is no CPU fallback.  DESIGN.md describes the path, the data layout and each kernel.
 *
 * Conventions
 *   - Plain C types only.  "device" pointers are CUDA device pointers, 16-byte aligned, owned by the caller;
 *     the library keeps no pointer after the work enqueued by a call has completed on `stream`.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).
 *   - Functions return 0 (ZKD_OK) or a negative ZKD_ERR_* code.  They never abort, throw or print.
 *   - Data-dependent outcomes are reported per matrix in zkd_info.status.
 *
 * API number layout (one real, zkd_real_bytes(prec) = 16 + prec/8 bytes; 112 at 768 bit; MPFR-like semantics):
 *     int32 sign   : -1, 0, +1
 *     int32 flags  : must be 0 (nonzero => malformed)
 *     int64 exp
 *     uint64 limb[prec/64], little-endian limb order
 *   value = sign * (sum_k limb[k] 2^(64k)) * 2^(exp - prec); nonzero numbers are normalised (top bit of the top
 *   limb set, mantissa in [1/2,1)); zero has every field zero.  No NaN/Inf.  Complex = (re, im) consecutive.
 * Array layout
 *   A[b][i][j]       row-major, complex; only the upper triangle (i <= j) and Re a_ii are read (LAPACK 'U').
 *   eigvals[b][j]    real, ascending.
 *   eigvecs[b][i][j] complex, component i of eigenvector j (so A X = X diag(lambda)); unit 2-norm; phase: the
 *                    first component of largest modulus is real positive.
 */
#ifndef ZKD_H
#define ZKD_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define ZKD_OK 0
#define ZKD_ERR_INVALID_ARG (-1)      /* N < 1, batch < 1, NULL or misaligned pointer, N > ZKD_MAX_N */
#define ZKD_ERR_UNSUPPORTED_PREC (-2) /* prec_bits is not a multiple of 64 in 128 .. 768 */
#define ZKD_ERR_WORKSPACE (-3)        /* workspace too small / allocation failed */
#define ZKD_ERR_CUDA (-4)             /* a CUDA call failed (the sticky error is cleared) */
#define ZKD_ERR_ARCH (-5)             /* device is not sm_100 */
#define ZKD_ERR_CLUSTERED (-7)        /* zkd_diag_herm_rqi_lu only: the spectrum has clusters, which per-vector RQI cannot separate */
#define ZKD_ERR_STATIC_LIMIT (-8)     /* zkd_seed_fp64_static only: N > ZKD_SEED_STATIC_MAX_N (its scratch is a fixed device array) */
#define ZKD_ERR_INTERNAL (-6)         /* internal consistency check failed (window overflow that could not be repaired) */

#define ZKD_MAX_N 2048
#define ZKD_SEED_STATIC_MAX_N 512 /* largest N of zkd_seed_fp64_static */

/* Per-matrix outcome, written to device memory by the call (one record per matrix of the batch).
 * status, n_clusters, max_cluster, log2_resid and log2_orth are per matrix.  `steps` is per CALL: the refinement loop runs
 * the whole batch until its slowest matrix stops, so every matrix of a call reports the same number.  A matrix whose own
 * residual is at or below the tolerance reports status 0 even when another matrix of the batch hit the floor (1) or the
 * step limit (2).  Failures that are not data-dependent outcomes (a window overflow the retry could not repair, a CUDA
 * error) fail the whole call through its return code. */
typedef struct {
  int32_t status;      /* 0 converged; 1 stopped at the precision floor above tolerance; 2 max steps; 3 malformed input */
  int32_t steps;       /* refinement passes of the top level (S4), the same for every matrix of the call */
  int32_t n_clusters;  /* clusters (incl. singletons) found by S2 at the top level */
  int32_t max_cluster; /* size of the largest cluster */
  float log2_resid;    /* log2 of max_ij |(A X - X S)_ij| of THIS matrix (S = the cluster-block Rayleigh quotients; the
                          residuals of the S5 sub-problems of its clusters folded in), in units where max|a_ij| is in
                          [1/8,1/4); -812 when the residual is exactly zero */
  float log2_orth;     /* log2 of max |X_c^H X_c - I| over the cluster blocks of THIS matrix after the last
                          orthonormalisation: twice the log2 measured before that Newton-Schulz step (which squares it),
                          not below -800 */
} zkd_info;

/* ---- the hot path -------------------------------------------------------------
 * prec_bits: the significand length of the API numbers, a multiple of 64 from 128 to 768 (the paper's settings: 768
 * PAPER.md:41, 256 PAPER.md:61, 128 PAPER.md:65).  Results are accurate to 2^-(prec_bits - 28) ||A||_F (eigenvalues,
 * residuals; 2^-(prec_bits - 28) for orthonormality) and rounded to prec_bits on export; internally every precision
 * runs on the same 840-bit fixed-point planes, with everything below 2^-(prec_bits + 44) left uncomputed. */

/* Bytes of one real in the API layout at `prec_bits` of significand ("The 768-bit precision was used", PAPER.md:41,
 * section 2.1; 256 bit: section 3.1; 128 bit: section 3.2): 16 + prec_bits/8.  Returns 0 if
 * prec_bits is unsupported.  Host call, no CUDA work, no error state. */
size_t zkd_real_bytes(int prec_bits);

/* Size in bytes of the device workspace zkd_diag_herm_ws needs for (N, batch); *workspace_bytes is a
 * host pointer.  Host call, no CUDA work.  Errors: ZKD_ERR_INVALID_ARG (N < 1, N > ZKD_MAX_N, batch < 1 or > 65535,
 * NULL), ZKD_ERR_UNSUPPORTED_PREC. */
int zkd_diag_herm_bufsize(int N, int batch, int prec_bits, size_t *workspace_bytes);

/* The operation of the paper's diag_H / zkcm_cus::cus_diag_H: "diagonalizing N x N Hermitian matrix" at multiprecision
 * (section 2.1) by "the Rayleigh quotient iteration ... to recover the precision from the result of
 * double-precision calculations" (section 2).
 * Eigendecomposition of `batch` Hermitian N x N matrices (S0 ingest .. S6 export, all on `stream`).
 *   A, eigvals, eigvecs, workspace, info: DEVICE pointers (info may be NULL).  A is not modified and may not
 *   alias the outputs.  The call synchronises `stream` internally a few times (cluster table and one
 *   convergence scalar per refinement step) and returns after all work has been enqueued; outputs are valid
 *   once `stream` is synchronised. */
int zkd_diag_herm_ws(int N, int batch, int prec_bits, const void *A, void *eigvals, void *eigvecs, void *workspace,
                     size_t workspace_bytes, zkd_info *info, void *stream);

/* The same operation (PAPER.md:41 / :33; north_star's example call) with a workspace obtained from, and returned to, the
 * stream-ordered CUDA allocator.  A, eigvals, eigvecs: DEVICE pointers, caller-owned, 16-byte aligned.  Same errors as
 * zkd_diag_herm_ws plus ZKD_ERR_WORKSPACE when the allocation fails. */
int zkd_diag_herm(int N, int batch, int prec_bits, const void *A, void *eigvals, void *eigvecs, void *stream);

/* End-to-end convenience for the same operation (PAPER.md:41 / :33): HOST buffers in the API layout (pageable or pinned,
 * caller-owned); copies H2D, runs zkd_diag_herm_ws on the legacy default stream, copies D2H, and synchronises.
 * info_host (host, `batch` records) may be NULL.  Keeps one grow-only device buffer per calling thread between calls. */
int zkd_diag_herm_host(int N, int batch, int prec_bits, const void *A_host, void *eigvals_host, void *eigvecs_host,
                       zkd_info *info_host);

/* ---- singular value decomposition ----------------------------------------------------
 * The second routine of the paper's ZKCM_CUS: "Hermitian matrix diagonalization and singular value decomposition"
 * (section 2; switched by ZKCM_QC, section 2.2).  Thin SVD of `batch` complex M x N
 * matrices, K = min(M, N):  A V = U diag(S), A^H U = V diag(S), S descending and >= 0, U (M x K) and V (N x K) with
 * orthonormal columns; phase: the first component of largest modulus of every v_j is real positive.  Computed through
 * the same hot path on the Hermitian matrix [[0, A], [A^H, 0]], so singular values are good to ABSOLUTE
 * 2^-(prec_bits - 28) ||A||_F: Schmidt weights far below sqrt(epsilon) are resolved.  Rank-deficient input is fine.
 *   A[b][i][j] (M x N), U[b][i][j] (M x K), V[b][i][j] (N x K): row-major complex API numbers; S[b][j]: real.
 *   All pointers DEVICE, 16-byte aligned, caller-owned; info (device, `batch` records, may be NULL) as for
 *   zkd_diag_herm_ws (clusters and residual refer to the (M+N) x (M+N) eigenproblem).  M + N <= ZKD_MAX_N.
 *   Errors as for zkd_diag_herm_ws.  zkd_svd obtains its workspace from the stream-ordered allocator. */
int zkd_svd_bufsize(int M, int N, int batch, int prec_bits, size_t *workspace_bytes);
int zkd_svd_ws(int M, int N, int batch, int prec_bits, const void *A, void *S, void *U, void *V, void *workspace,
               size_t workspace_bytes, zkd_info *info, void *stream);
int zkd_svd(int M, int N, int batch, int prec_bits, const void *A, void *S, void *U, void *V, void *stream);

/* ---- linear systems by multiprecision LU and exact RQI on top of it (8(a) S4a') --------
 * "Gaussian elimination, LU decomposition" are among ZKCM_OMP's main routines (section 2).
 * zkd_lu_solve: X with A X = B for `batch` complex N x N systems with nrhs right-hand sides each, by LU with partial
 * pivoting in the library's block fixed point: A and B are scaled by powers of two (max entry in [1/8, 1/4)), so the
 * accuracy is ABSOLUTE, about cond(A) 2^-(prec_bits+2) relative to ||X||-scale, and pivots below 2^-26 max|a_ij| cannot
 * be inverted.  A[b][i][j] (N x N), B[b][i][j], X[b][i][j] (N x nrhs): row-major complex API numbers, DEVICE pointers,
 * 16-byte aligned, caller-owned; status (device int[batch], may be NULL): 0 solved, 1 singular to working precision,
 * 2 pivot too small for the format, 3 malformed input number.  N <= ZKD_MAX_N. */
int zkd_lu_solve_bufsize(int N, int nrhs, int batch, int prec_bits, size_t *workspace_bytes);
int zkd_lu_solve(int N, int nrhs, int batch, int prec_bits, const void *A, const void *B, void *X, void *workspace,
                 size_t workspace_bytes, int *status, void *stream);
/* zkd_diag_herm_rqi_lu: the operation of zkd_diag_herm_ws by the paper's route taken literally:
 * fp64 eigendecomposition, then for every eigenpair the Rayleigh quotient iteration sigma = x^H A x,
 * y = (A - sigma I)^-1 x by one multiprecision LU per eigenpair and iteration, x = y / ||y|| (cubic: three iterations from
 * an fp64 start).  O(N^4); isolated eigenvalues only (returns ZKD_ERR_CLUSTERED otherwise); N <= 64.  It exists as the
 * in-product cross-check of the production path.  Arguments as zkd_diag_herm_ws. */
int zkd_diag_herm_rqi_lu_bufsize(int N, int batch, int prec_bits, size_t *workspace_bytes);
int zkd_diag_herm_rqi_lu(int N, int batch, int prec_bits, const void *A, void *eigvals, void *eigvecs, void *workspace,
                         size_t workspace_bytes, zkd_info *info, void *stream);

/* ---- minimal MPS two-site update around the eigensolver ------------------------------
 * An MPS is a "nested Schmidt decomposition" (section 1); its simulation cost is dominated by "Hermitian matrix
 * diagonalization" (section 2.1), and Schmidt weights of order epsilon ~ 2^(-n+1) must survive
 * (footnote) - hence the precision.  One update of `batch` independent bonds:
 *     Theta0 = L R;   Theta[(a,i'),(j',c)] = sum_ij G[(i'j'),(ij)] Theta0[(a,i),(j,c)];   rho = Theta Theta^H;
 *     rho = U diag(w) U^H  (zkd's Hermitian eigendecomposition);   L' = U[:, 0:K];   R' = L'^H Theta
 *   L[b]   : (chiL d) x chiC, rows (a, i);     R[b]  : chiC x (d chiR), columns (j, c);     G[b] : d^2 x d^2, rows (i' j'),
 *            columns (i j): the two-site gate.  All row-major complex API numbers.
 *   W[b]   : K reals, the Schmidt weights (eigenvalues of rho) in DESCENDING order, K = min(chiL d, max_keep) (max_keep <= 0:
 *            no limit); good to absolute 2^-(prec_bits - 28) trace(rho).
 *   Lnew[b]: (chiL d) x K, orthonormal columns (phase: first component of largest modulus real positive);
 *   Rnew[b]: K x (d chiR), so that Theta = Lnew Rnew up to the discarded weights.
 *   kept   : device int[batch]: how many leading weights exceed 2^-cutoff_bits trace(rho) (the caller truncates to that).
 * All pointers DEVICE, 16-byte aligned, caller-owned; info as for zkd_diag_herm_ws (may be NULL).  chiL d <= ZKD_MAX_N. */
int zkd_mps_two_site_update_bufsize(int chiL, int chiC, int chiR, int d, int batch, int prec_bits, size_t *workspace_bytes);
int zkd_mps_two_site_update(int chiL, int chiC, int chiR, int d, int batch, int prec_bits, const void *L, const void *R,
                            const void *G, int max_keep, int cutoff_bits, void *W, void *Lnew, void *Rnew, int *kept,
                            zkd_info *info, void *workspace, size_t workspace_bytes, void *stream);

/* Tunables.  PROCESS-WIDE and unsynchronised: set them before, not during, calls of zkd_diag_herm* from
 * other threads; the library may be used from several host threads with distinct workspaces as long as the options, the
 * counters and the kernel timing are left alone meanwhile, and it serves ONE device per process (the device current at
 * the first call).  Keys: "tau_bits" (cluster threshold 2^-tau ||A||_F,
 * default 20), "tol_bits" (stop when max|R_ij| <= 2^-tol, default 770), "max_steps" (default 120),
 * "gemm_path" (engine of the digit GEMM: 0 = automatic [default]: limb-sliced int8 tcgen05 MMAs when M, N, K >= 128,
 * the IMAD kernel otherwise; 1 = IMAD only; 2 = int8 tcgen05 wherever its tiles can be formed),
 * "gemm_tile" (tile of the IMAD digit GEMM: 0 automatic - 8 x 8 x 8 where 16-wide tiles
 * would be filled more than 1.25 x worse, e.g. 24- or 29-dimensional cluster blocks -, 8, 16), "min_split_ctas" (split-K target, default 296; every split keeps at least 32 of K), "early_split" (S4h: split clusters whose internal structure stands
 * above the noise of the projected matrix; default 1; 0 leaves every cluster to the S5 recursion),
 * "split_margin_bits" (that margin, default 40), "seed_sweeps" (cap on the fp64 Jacobi sweeps, default 12),
 * "seed_path" / "seed_cluster" (seed kernel selection), "cluster_tiles" (default 1: on levels where
 * no cluster straddles a multiple of 128 columns, most columns are clustered and the clusters average more than 51 columns,
 * the cluster-block products of a pass run as 128-column tile products on the int8 tcgen05 engine; 0: always per cluster on
 * the IMAD engine; 2: tiles wherever they can be formed), "i8_bdiag" (default 1: in those tile products the block-diagonal
 * operand M_t / S_t - no cluster straddling a multiple of 32 columns - is multiplied with 128 x 32 x 32 MMAs, one per 32-column
 * block, instead of full-width ones; 0: full width; same integers either way),
 * "block_correction" (default 1: the correction between clusters takes
 * one fixed-point step with the off-diagonal parts of the cluster blocks of X^H A X, which squares the spread / gap factor
 * that otherwise caps the gain of a pass), "seed_ring_block" (columns per block of the block-ring fp64 seed for N <= 256:
 * 2 or 4, 0 = the column ring, default -1 = 4 from N = 96 on), "seed_tma" (default 1: the blocked fp64 seed moves its columns by TMA bulk copies),
 * "seed_block_warps" (8 or 16), "seed_gram" (default 0; 1 / 2: the blocked seed finds a round's rotations on the 8 x 8 Gram
 * matrix of the CTA's two column blocks and applies them in one pass, for 256 < N <= 1600; measured slower),
 * "seed_degenerate_skip" (default 1: inside the path the fp64 seed leaves column pairs of one numerically multiple eigenvalue -
 * estimates closer than 2^-(tau_bits + 2) sigma / sqrt N, cosine below 2^-10 - unrotated, which keeps the Jacobi sweeps quadratically
 * convergent on spectra with multiplicities; such a pair always lies inside one cluster of S2; 0: off; >= 8: the exponent itself;
 * zkd_seed_fp64 and zkd_seed_fp64_static never apply the rule), "combine_path" (epilogue of the IMAD GEMM: 0 automatic,
 * 1 digit-serial, 2 warp-cooperative), "sstep_cpb" (matrix columns per CTA of the fused singleton step, 0 automatic), "sstep_par" (default 1: for N <= 96 and
 * one column per CTA the products of a row are spread over four threads), "sstep_warp" (1: its
 * warp-per-element variant for N <= 64, default 0), "sstep_cache" (shared-memory staging of the column, default 1),
 * "verbose" (1: one line per refinement pass on stderr).  All routes give the same results to the stated tolerances;
 * the defaults are the measured-fastest ones.  Returns ZKD_ERR_INVALID_ARG for an unknown key. */
int zkd_set_option(const char *key, double value);
int zkd_get_option(const char *key, double *value);

/* Text of a ZKD_ERR_* code (static storage); library version (major * 100 + minor).  SURVEY.md 8(b). */
const char *zkd_strerror(int code);
int zkd_version(void);

/* Counters since process start / last reset: kernels launched by this library and 28x28-bit digit products
 * (IMAD.WIDE) issued by its GEMM kernels, algorithmic count.  Host call. */
void zkd_counters(uint64_t *kernel_launches, uint64_t *gemm_digit_macs);
void zkd_counters_reset(void);

/* Per-launch device timing of the dominant kernel (the digit GEMM), for roofline reporting: zkd_kernel_timing(1)
 * resets and arms it (every digit-GEMM launch is then bracketed by a CUDA event pair on its own stream, up to 16384
 * launches), zkd_kernel_timing(0) disarms; zkd_kernel_timing_read waits for the recorded events and returns the summed
 * kernel time in ms, the number of timed launches and the digit products they performed.  Host calls. */
int zkd_kernel_timing(int enable);
int zkd_kernel_timing_read(double *gemm_ms, uint64_t *gemm_launches, uint64_t *gemm_digit_macs);
/* The same for the int8 tcgen05 engine (S4b): summed kernel time, timed launches, and the s8 x s8 multiply-accumulates
 * its tcgen05.mma instructions performed (full 128 x 128 x 128 blocks, padding included). */
int zkd_kernel_timing_read_i8(double *gemm_ms, uint64_t *gemm_launches, uint64_t *int8_macs);

/* Per-category timing of EVERY kernel of the hot path (same arming as above): category indices 0 .. categories-1, each
 * with a name (the kernel or kernel family), the summed device time of its launches, their number, and two work counts in
 * the category's unit - "executed" (what the launches performed, tile and instance padding included) and "algorithmic"
 * (what the requests needed).  Units: gemm_digits_kernel, singleton_step_kernel, ecalc_kernel, lu_kernels: 28x28-bit digit
 * products; gemm_i8_kernel: s8 x s8 multiply-accumulates; prep / combine / slice / combine_i8 / ingest_export: bytes
 * moved (algorithmic = executed); seed_fp64: 0 (use zkd_seed_stats).  Host calls. */
int zkd_kernel_timing_categories(void);
const char *zkd_kernel_timing_name(int category);
int zkd_kernel_timing_read_cat(int category, double *ms, uint64_t *launches, uint64_t *work_executed, uint64_t *work_algorithmic);
/* Work of the fp64 seed kernels (S1) since the last reset: column elements whose pair of columns was checked (three dot
 * products = 8 DFMA per element) and elements whose pair was also rotated (12 more DFMA per element).  Synchronises. */
int zkd_seed_stats(uint64_t *elems_checked, uint64_t *elems_rotated, int reset);

/* ---- host-side helpers (no CUDA): one real between the API layout and (sign, exp, limbs) / double (the
 * layout follows MPFR's, the library the paper's ZKCM is built on).  dst / src: host pointers to
 * zkd_real_bytes(prec_bits) bytes; limbs_le: prec_bits/64 words, least significant first.  ZKD_ERR_INVALID_ARG for NULL,
 * an unsupported precision, a sign outside -1..1, an unnormalised mantissa or a non-finite double. ---- */
int zkd_pack(void *dst, int prec_bits, int sign, int64_t exp, const uint64_t *limbs_le);
int zkd_unpack(const void *src, int prec_bits, int *sign, int64_t *exp, uint64_t *limbs_le);
int zkd_from_double(void *dst, int prec_bits, double v);
double zkd_to_double(const void *src, int prec_bits);

/* ---- building blocks exported for tests and measurement (device pointers; see DESIGN.md section "Kernels") ---- */

/* Internal fixed-point format ("FX"): ZKD_FX_DIGITS radix-2^28 digits per real, int32 each, digit-major planes:
 * real array of `count` numbers = int32[ZKD_FX_DIGITS][count]; digits 0..28 in [0,2^28), digit 29 signed;
 * value = (sum_d digit[d] 2^(28 d)) 2^-812.  Complex array = re planes followed by im planes. */
#define ZKD_FX_DIGITS 30
#define ZKD_FX_FRAC_BITS 812

/* API reals -> FX (value * 2^scale_bits, truncated toward zero at 2^-812) and back (rounded to nearest even). */
int zkd_fx_from_api(int count, int prec_bits, const void *src_api, int32_t *dst_fx, int scale_bits, void *stream);
int zkd_fx_to_api(int count, int prec_bits, const int32_t *src_fx, void *dst_api, int scale_bits, void *stream);

/* Element-wise multi-digit primitives on real FX arrays of `count` numbers (north_star (b); SURVEY.md 8(a) "MP
 * primitives"): out[e] = a[e] (op) b[e].  The hot path uses the same device functions inside its kernels; this entry exists
 * so that each primitive can be checked against exact integer arithmetic.  a, b, out: DEVICE pointers to int32[30][count]
 * (b may be NULL for the unary ones; out may alias a or b).
 *   ADD, SUB : exact modulo 2^840 (wraps like the top digit).      HALF : floor(a / 2).
 *   MUL      : sum of the digit products a_i b_j with i + j >= 28, + 2^(28*28 + 27), shifted right by 28*29 bits (floor):
 *              the exact product rounded at the guard column, minus the digit columns below the guard column, i.e.
 *              within [-28, +1/2] units of 2^-812 of the exact product for non-negative low digits.
 *   RECIP    : a in [1/4, 1/2] -> 1/a in [2, 4] by Newton from an fp64 start (error <= 64 units of 2^-812).
 *   RSQRT    : a > 0 -> 1/sqrt(a) (error <= 64 units of 2^-812 times max(1, 1/sqrt(a))); a <= 0 -> 0.
 *   MSB      : digit 0 of out = 1 + position of the highest bit of a that differs from its sign (0 for 0 and -1).
 *   FROM_DOUBLE : out = fx(double(a)): the FX -> fp64 -> FX round trip used by the seed (S1 / S3). */
#define ZKD_PRIM_ADD 0
#define ZKD_PRIM_SUB 1
#define ZKD_PRIM_MUL 2
#define ZKD_PRIM_RECIP 3
#define ZKD_PRIM_RSQRT 4
#define ZKD_PRIM_MSB 5
#define ZKD_PRIM_HALF 6
#define ZKD_PRIM_FROM_DOUBLE 7
int zkd_fx_prim(int op, int count, const int32_t *a_fx, const int32_t *b_fx, int32_t *out_fx, void *stream);

/* C (+)= op(A) * B for complex FX matrices (S4a/S4d/S4e), A: M x K, B: K x N, C: M x N (row-major element order,
 * `batch` problems stored consecutively).  op_a: 0 = A, 1 = A^H (then A is stored K x M).  mode: 0 assign, 1 add,
 * 2 subtract.  Only the window [top_bit - 28*digits, top_bit) of each operand takes part (FX bit 0 = 2^-812; every
 * element must fit the window with two spare bits, else *err_flag |= 1); the product is exact on those windows
 * except that digit columns more than (instance NP + 1) digits below the top are dropped.
 * out_cut_bit > 0 clears result bits below that FX bit.  err_flag, msb_out: device ints, may be NULL; msb_out
 * receives atomicMax of (1 + position of the highest significant bit) over the result elements.
 * path: 0 IMAD digit GEMM.  workspace from zkd_gemm_fx_bufsize. */
int zkd_gemm_fx_bufsize(int M, int N, int K, int batch, size_t *workspace_bytes);
int zkd_gemm_fx(int M, int N, int K, int batch, int op_a, const int32_t *A_fx, int a_top_bit, int a_digits,
                const int32_t *B_fx, int b_top_bit, int b_digits, int32_t *C_fx, int mode, int out_cut_bit, int path,
                void *workspace, size_t workspace_bytes, int *err_flag, int *msb_out, void *stream);

/* fp64 seed (S1; the "double-precision calculations" RQI starts from, PAPER.md:33 - hand-written, no cuSOLVER):
 * Hermitian eigendecomposition of batch N x N matrices given as complex doubles (row-major,
 * interleaved re/im); mu ascending, V[i][j] = component i of vector j. */
int zkd_seed_fp64(int N, int batch, const double *A64, double *mu, double *V, void *stream);
/* The same seed for callers that must not allocate (code under CUDA graph capture, serving loops, harnesses that forbid
 * cudaMalloc): same arguments, layouts and result as zkd_seed_fp64, but the call makes no cudaMalloc / cudaFree / event or
 * stream creation.  zkd_seed_fp64 keeps G = A + sigma I (N^2 complex doubles), sigma, the unsorted eigenvalues and the sweep
 * flags in a cudaMalloc'ed buffer when N > 256; this entry point runs that same blocked one-sided Jacobi kernel for every
 * 1 <= N <= ZKD_SEED_STATIC_MAX_N (= 512) with that scratch in a static __device__ array of 4 MiB + 8 KiB, which every GPU that
 * loads libzkd.so holds until the process exits.  Errors: ZKD_ERR_STATIC_LIMIT for N > 512 (nothing is launched),
 * ZKD_ERR_INVALID_ARG, ZKD_ERR_ARCH, ZKD_ERR_CUDA.  A64, mu, V: device pointers owned by the caller; the batch is processed
 * one matrix at a time on `stream`.  ALL calls on a device share the one array: calls on the same stream are ordered and
 * safe, calls that overlap on the GPU (different streams, different host threads without ordering) race on it and give
 * undefined results.  The array keeps the previous call's contents; the call clears what has to start at zero itself. */
int zkd_seed_fp64_static(int N, int batch, const double *A64, double *mu, double *V, void *stream);

/* Measured integer-multiply peak: runs a register-only IMAD.WIDE loop on every SM for about `millis`
 * milliseconds and returns wide (32x32+64) multiply-adds per second (host double). */
int zkd_measure_imad_peak(double millis, double *imad_wide_per_sec, void *stream);
/* Measured fp64 peak (roofline denominator of the seed): register-only DFMA loop on every SM; returns flop/s (2 per FMA). */
int zkd_measure_dfma_peak(double millis, double *fp64_flops_per_sec, void *stream);
/* Measured issue peak of the int8 tensor-core shape S4b uses (tcgen05.mma kind::i8, 128 x 128 x 32, one CTA per SM, operands
 * resident in shared memory, no loads): returns int8 op/s (2 per multiply-add).  Reported by bench.py beside the bf16-derived
 * peak of MEASURED_PEAKS.json. */
int zkd_measure_i8_mma_peak(double millis, double *int8_ops_per_sec, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* ZKD_H */

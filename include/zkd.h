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
#define ZKD_ERR_UNSUPPORTED_PREC (-2) /* this build: prec_bits == 768 only */
#define ZKD_ERR_WORKSPACE (-3)        /* workspace too small / allocation failed */
#define ZKD_ERR_CUDA (-4)             /* a CUDA call failed (the sticky error is cleared) */
#define ZKD_ERR_ARCH (-5)             /* device is not sm_100 */
#define ZKD_ERR_INTERNAL (-6)         /* internal consistency check failed (window overflow that could not be repaired) */

#define ZKD_MAX_N 2048

/* per-matrix outcome, written to device memory by the call */
typedef struct {
  int32_t status;      /* 0 converged; 1 stopped at the precision floor above tolerance; 2 max steps; 3 malformed input */
  int32_t steps;       /* refinement steps taken at the top level (S4) */
  int32_t n_clusters;  /* clusters (incl. singletons) found by S2 at the top level */
  int32_t max_cluster; /* size of the largest cluster */
  float log2_resid;    /* log2 of max_ij |(A X - X diag(lambda))_ij| in units where max|a_ij| is in [1/8,1/4) */
  float log2_orth;     /* log2 of max |X_c^H X_c - I| over cluster blocks after the last orthonormalisation: twice the
                          log2 measured before that Newton-Schulz step (which squares it), not below -800 */
} zkd_info;

/* ---- the hot path ------------------------------------------------------------- */

/* bytes of one real in the API layout; 0 if prec_bits is unsupported */
size_t zkd_real_bytes(int prec_bits);

/* Size of the device workspace zkd_diag_herm_ws needs for (N, batch).  Host call, no CUDA work. */
int zkd_diag_herm_bufsize(int N, int batch, int prec_bits, size_t *workspace_bytes);

/* Eigendecomposition of `batch` Hermitian N x N matrices (S0 ingest .. S6 export, all on `stream`).
 *   A, eigvals, eigvecs, workspace, info: DEVICE pointers (info may be NULL).  A is not modified and may not
 *   alias the outputs.  The call synchronises `stream` internally a few times (cluster table and one
 *   convergence scalar per refinement step) and returns after all work has been enqueued; outputs are valid
 *   once `stream` is synchronised. */
int zkd_diag_herm_ws(int N, int batch, int prec_bits, const void *A, void *eigvals, void *eigvecs, void *workspace,
                     size_t workspace_bytes, zkd_info *info, void *stream);

/* Same with a workspace obtained from (and returned to) the stream-ordered CUDA allocator. */
int zkd_diag_herm(int N, int batch, int prec_bits, const void *A, void *eigvals, void *eigvecs, void *stream);

/* End-to-end convenience: HOST buffers in the API layout; copies H2D, runs zkd_diag_herm, copies D2H, and
 * synchronises.  info_host may be NULL. */
int zkd_diag_herm_host(int N, int batch, int prec_bits, const void *A_host, void *eigvals_host, void *eigvecs_host,
                       zkd_info *info_host);

/* Tunables (process-wide; call before zkd_diag_herm*).  Keys: "tau_bits" (cluster threshold 2^-tau ||A||_F,
 * default 20), "tol_bits" (stop when max|R_ij| <= 2^-tol, default 770), "max_steps" (default 120),
 * "gemm_path" (engine of the digit GEMM: 0 = automatic [default]: limb-sliced int8 tcgen05 MMAs when M, N, K >= 128,
 * the IMAD kernel otherwise; 1 = IMAD only; 2 = int8 tcgen05 wherever its tiles can be formed),
 * "min_split_ctas" (split-K target, default 296; every split keeps at least 32 of K), "early_split" (S4h: split clusters whose internal structure stands
 * above the noise of the projected matrix; default 1; 0 leaves every cluster to the S5 recursion),
 * "split_margin_bits" (that margin, default 40), "seed_sweeps" (cap on the fp64 Jacobi sweeps, default 12),
 * "seed_path" / "seed_cluster" (seed kernel selection), "combine_path" (epilogue of the IMAD GEMM: 0 automatic,
 * 1 digit-serial, 2 warp-cooperative), "sstep_cpb" (matrix columns per CTA of the fused singleton step, 0 automatic), "sstep_warp" (1: its
 * warp-per-element variant for N <= 64, default 0), "sstep_cache" (shared-memory staging of the column, default 1),
 * "verbose" (1: one line per refinement pass on stderr).  All routes give the same results to the stated tolerances;
 * the defaults are the measured-fastest ones.  Returns ZKD_ERR_INVALID_ARG for an unknown key. */
int zkd_set_option(const char *key, double value);
int zkd_get_option(const char *key, double *value);

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

/* ---- host-side helpers (no CUDA): one real between the API layout and (sign, exp, limbs) / double ---- */
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

/* fp64 seed (S1): Hermitian eigendecomposition of batch N x N matrices given as complex doubles (row-major,
 * interleaved re/im); mu ascending, V[i][j] = component i of vector j. */
int zkd_seed_fp64(int N, int batch, const double *A64, double *mu, double *V, void *stream);

/* Measured integer-multiply peak: runs a register-only IMAD.WIDE loop on every SM for about `millis`
 * milliseconds and returns wide (32x32+64) multiply-adds per second (host double). */
int zkd_measure_imad_peak(double millis, double *imad_wide_per_sec, void *stream);
/* Measured fp64 peak (roofline denominator of the seed): register-only DFMA loop on every SM; returns flop/s (2 per FMA). */
int zkd_measure_dfma_peak(double millis, double *fp64_flops_per_sec, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* ZKD_H */

// zkd_internal.h — declarations shared between the translation units of libzkd (not part of the public ABI).
#pragma once
#include <cstddef>
#include <cstdint>
#include <cuda_runtime.h>

#include "../../include/zkd.h"

namespace zkd {

constexpr int kND = ZKD_FX_DIGITS;   // 30
constexpr int kDB = 28;
constexpr int kFRAC = ZKD_FX_FRAC_BITS;
constexpr int kFxBits = kND * kDB;   // 840 (the top digit really has 32 bits)
constexpr int kPrec = 768;                      // the largest (and default) API precision
constexpr int kApiRealBytes = 16 + kPrec / 8;  // 112, at kPrec

// ---- error plumbing ---------------------------------------------------------------------------------------------
#define ZKD_CUDA_TRY(expr)                         \
  do {                                             \
    cudaError_t _e = (expr);                       \
    if (_e != cudaSuccess) {                       \
      (void)cudaGetLastError();                    \
      return ZKD_ERR_CUDA;                         \
    }                                              \
  } while (0)
#define ZKD_TRY(expr)          \
  do {                         \
    int _rc = (expr);          \
    if (_rc != ZKD_OK) return _rc; \
  } while (0)

void count_launch(uint64_t n = 1);
void count_macs(uint64_t n);
inline int launch_check() {
  cudaError_t e = cudaGetLastError();
  return e == cudaSuccess ? ZKD_OK : ZKD_ERR_CUDA;
}

struct Options {
  int tau_bits = 20;
  int tol_bits = 770;
  int max_steps = 120;
  int gemm_path = 0;
  int gemm_tile = 0;         // IMAD digit GEMM: 0 automatic (8 x 8 x 8 tiles where 16-wide tiles fill badly), 8, 16
  int min_split_ctas = 296;  // split K until a product has about this many CTAs (two per SM), see pick_splits
  int seed_sweeps = 12;
  int seed_cluster = 0;  // ring seed: largest cluster size to use (0 = 16, falling back to 8 when refused)
  int seed_ring_block = -1;   // ring seed (N <= 256): columns per block of the block ring (2 or 4); 0: the column ring; -1: 4 for N >= 96
  int seed_tma = 1;           // blocked seed: columns move between L2 and shared memory by 1-D TMA bulk copies
  int seed_block_warps = 8;   // blocked seed (N > 256): warps per CTA (8 or 16)
  int seed_gram = 0;          // blocked seed: 1 / 2: a round's rotations found on the 8 x 8 Gram matrix of the CTA's two blocks (seed_blockg_kernel; 1: where the classic kernel would use W = 4, 2: up to N = 1600); measured slower (N = 1024: 44.1 vs 41.7 ms), off
  int seed_degenerate_skip = 1;  // fp64 seed: leave column pairs of one (numerically) multiple eigenvalue unrotated (rot_params)
  int seed_dbuf = 1;     // ring seed: two slot sets, one cluster barrier per round (when they fit shared memory)
  int seed_path = 0;     // 0: auto; 2: always the ring kernel for N <= 256; 3: unblocked cooperative kernel for N > 256
  int early_split = 1;        // S4h: split clusters as soon as their internal structure stands above the noise
  int split_margin_bits = 40; // ... by this many bits
  int block_correction = 1;   // S4d: one fixed-point step with the off-diagonal parts of the cluster blocks (second order in spread / gap)
  int i8_packed = 1;          // int8 GEMM output: 1 = one int64 per entry and group of four columns (combine_i8_packed_kernel), 0 = int32 columns
  int i8_slice = 0;           // int8 GEMM re-slicing kernel: 0 = four k per thread, seven slices per step; 1 = one element per thread
  int i8_step = 0;            // int8 GEMM: slices a per barrier round trip: 0 / 2 = two (rings <4, 9>), 1 = one (rings <5, 8>)
  int i8_bdiag = 1;           // int8 GEMM: quarter-width MMAs for block-diagonal Q tiles (GemmSide::bdiag32)
  int cluster_tiles = 1;      // cluster passes as 128-column tile products on the int8 engine when no cluster straddles a tile
  int combine_path = 0;       // IMAD GEMM epilogue: 0 auto, 1 digit-serial thread per element, 2 warp-cooperative (digit per lane)
  int sstep_warp = 0;         // singleton_step: 1: warp-per-element kernel (digit per lane) when one column per CTA and n <= 64; measured 1 % faster at N = 16, 3 % slower at N = 64: off by default
  int sstep_par = 1;          // singleton_step, one column per CTA, n <= 96: the products of a row spread over several threads
  int sstep_cache = 1;        // singleton_step: stage the column's x, w digits in shared memory (one column per CTA, n <= 96)
  int sstep_cpb = 0;          // singleton_step: matrix columns per CTA (0: auto)
  int verbose = 0;
};
Options& options();

// ---- complex FX matrices in device memory ------------------------------------------------------------------------
// A complex FX array with `count` elements: int32[2][kND][count] (re planes then im planes).
struct FxC {
  int32_t* p = nullptr;
  size_t count = 0;
  __host__ __device__ int32_t* re() const { return p; }
  __host__ __device__ int32_t* im() const { return p + (size_t)kND * count; }
  static size_t bytes(size_t count) { return sizeof(int32_t) * 2 * kND * count; }
};
struct FxR {
  int32_t* p = nullptr;
  size_t count = 0;
  static size_t bytes(size_t count) { return sizeof(int32_t) * kND * count; }
};

// ---- digit GEMM (gemm_digits.cu) ---------------------------------------------------------------------------------
// One side of a complex product C = op(P) * Q.  The window of the FX operand that takes part is
// bits [top_bit - 28*nw, top_bit) (FX bit 0 = 2^-812); bits above must be sign extension (checked on device).
struct GemmSide {
  const int32_t* fx = nullptr;  // complex FX array of batch*rows*cols elements, row-major
  int rows = 0, cols = 0;       // as stored
  bool conj_transpose = false;  // P only: use A^H (stored K x M)
  int top_bit = 0;
  int nw = 0;
  // optional view: batch element v is the rows x cols sub-matrix that starts at complex element off[v] of an array of
  // plane_count complex elements with row stride ld (cluster blocks and column slices of X, W, S)
  int ld = 0;                // 0: cols
  const int* off = nullptr;  // device, [batch]; null: v * rows * cols
  size_t plane_count = 0;    // 0: batch * rows * cols
  // Q only, a promise of the caller: the 128 x 128 matrices are block diagonal in aligned 32 x 32 blocks (cluster-tile products);
  // the int8 engine then issues 128 x 32 x 32 MMAs (gemm_i8.cu)
  bool bdiag32 = false;
};
struct GemmDstView {         // the same for the destination (M x N per batch element)
  int ld = 0;
  const int* off = nullptr;
  size_t plane_count = 0;
};
enum class GemmMode : int { Assign = 0, Add = 1, Sub = 2 };
// Timing bookkeeping only (KtScope work counters): the share of the products issued inside the scope that the caller needs
// (cluster passes run as 128-column tiles need sum m^2 / 128^2 per tile); thread-local, nests by restoring the old value.
double gemm_useful_fraction();
struct GemmUsefulScope {
  explicit GemmUsefulScope(double f);
  ~GemmUsefulScope();
  GemmUsefulScope(const GemmUsefulScope&) = delete;
  GemmUsefulScope& operator=(const GemmUsefulScope&) = delete;

 private:
  double old_;
};

size_t gemm_workspace_bytes(int M, int N, int K, int batch);
// dst (+)= op(P) * Q ; bits of the product below out_cut_bit are cleared (use a negative value for none).
// err_flag (device int, may be null) receives bit 1 when an operand does not fit its window.
// msb_out (device int, may be null): atomicMax of the msb position of |result| elements.
int gemm_complex(int M, int N, int K, int batch, const GemmSide& P, const GemmSide& Q, int32_t* dst_fx, GemmMode mode,
                 int out_cut_bit, int path, void* workspace, size_t workspace_bytes, int* err_flag, int* msb_out,
                 cudaStream_t stream, const GemmDstView* dst_view = nullptr);
// number of 28x28-bit digit products one call performs (algorithmic, after instance selection)
uint64_t gemm_complex_macs(int M, int N, int K, int batch, int nwP, int nwQ, int* inst_np, int* inst_nq);

// ---- pipeline pieces --------------------------------------------------------------------------------------------
int fx_from_api(int count, const void* src_api, int32_t* dst_fx, int scale_bits, cudaStream_t s, int prec = kPrec);
int fx_to_api(int count, const int32_t* src_fx, void* dst_api, int scale_bits, cudaStream_t s, int prec = kPrec);
// supported API precisions: multiples of 64 from 128 to 768 bits (PAPER.md:41 768, :61 256, :65 128)
inline bool prec_supported(int prec) { return prec >= 128 && prec <= kPrec && (prec & 63) == 0; }
inline size_t api_real_bytes(int prec) { return 16 + (size_t)prec / 8; }
// degenerate_skip: leave column pairs of one numerically multiple eigenvalue unrotated (rot_params in seed.cu); only for callers
// that treat the clusters of S2 as blocks afterwards (solve_level)
int seed_fp64(int N, int batch, const double* A64, double* mu, double* V, int max_sweeps, cudaStream_t s, bool degenerate_skip = false);
// the same with its scratch in a static device array (N <= ZKD_SEED_STATIC_MAX_N): allocates nothing
int seed_fp64_static(int N, int batch, const double* A64, double* mu, double* V, int max_sweeps, cudaStream_t s);

size_t diag_workspace_bytes(int N, int batch);
int diag_herm_device(int N, int batch, int prec, const void* A_api, void* eigvals_api, void* eigvecs_api, void* ws, size_t ws_bytes,
                     zkd_info* info, cudaStream_t s);

size_t lu_workspace_bytes(int N, int nrhs, int batch);
int lu_solve_device(int N, int nrhs, int batch, int prec, const void* A_api, const void* B_api, void* X_api, void* ws, size_t ws_bytes,
                    int* status_dev, cudaStream_t s);
size_t rqi_lu_workspace_bytes(int N, int batch);
int diag_herm_rqi_lu_device(int N, int batch, int prec, const void* A_api, void* eigvals_api, void* eigvecs_api, void* ws, size_t ws_bytes,
                            zkd_info* info, cudaStream_t s);
size_t mps_workspace_bytes(int chiL, int chiC, int chiR, int d, int batch);
int mps_update_device(int chiL, int chiC, int chiR, int d, int batch, int prec, const void* L_api, const void* R_api, const void* G_api,
                      int max_keep, int cutoff_bits, void* W_api, void* Lnew_api, void* Rnew_api, int* kept_dev, zkd_info* info, void* ws,
                      size_t ws_bytes, cudaStream_t s);
size_t svd_workspace_bytes(int M, int N, int batch);
int svd_device(int M, int N, int batch, int prec, const void* A_api, void* S_api, void* U_api, void* V_api, void* ws, size_t ws_bytes,
               zkd_info* info, cudaStream_t s);

}  // namespace zkd

namespace zkd {
int fx_from_api_scaled(size_t count, const void* src_api, int32_t* dst_fx, int scale_bits, const int* scale_dev,
                       int scale_stride, size_t per_scale, int* status, cudaStream_t s, int prec = kPrec);
int fx_to_api_scaled(size_t count, const int32_t* src_fx, void* dst_api, int scale_bits, const int* scale_dev, int scale_stride,
                     size_t per_scale, cudaStream_t s, int prec = kPrec);
int fxc_to_api(size_t count, const int32_t* src_fxc, void* dst_api, cudaStream_t s, int prec = kPrec);
int fxc_to_api_scaled(size_t count, const int32_t* src_fxc, void* dst_api, const int* scale_dev, size_t per_scale, cudaStream_t s, int prec = kPrec);
int fx_prim(int op, size_t count, const int32_t* a, const int32_t* b, int32_t* out, cudaStream_t s);
int measure_imad_peak(double millis, double* per_sec, cudaStream_t s);
int measure_dfma_peak(double millis, double* flops_per_sec, cudaStream_t s);
int seed_stats(uint64_t* elems_checked, uint64_t* elems_rotated, bool reset);
void kernel_timing_enable(bool on);
int kernel_timing_read(double* ms, uint64_t* launches, uint64_t* macs);
}  // namespace zkd

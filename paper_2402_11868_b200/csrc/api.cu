// api.cu — the C ABI of libzkd (include/zkd.h): argument validation, options, counters, host-side number helpers,
// and the measured integer-multiply peak.  No arithmetic of the method lives here.
#include <atomic>
#include <cmath>
#include <cstring>

#include "gemm_i8.h"
#include "timing.h"
#include "zkd_internal.h"

namespace zkd {

static std::atomic<uint64_t> g_launches{0}, g_macs{0}, g_i8_macs{0};
void count_launch(uint64_t n) { g_launches.fetch_add(n, std::memory_order_relaxed); }
void count_macs(uint64_t n) { g_macs.fetch_add(n, std::memory_order_relaxed); }
void count_i8_macs(uint64_t n) { g_i8_macs.fetch_add(n, std::memory_order_relaxed); }
Options& options() {
  static Options o;
  return o;
}

static int check_device() {
  static int cached = 1;  // 1 = unknown
  if (cached != 1) return cached;
  int dev = 0;
  cudaDeviceProp prop;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) {
    (void)cudaGetLastError();
    return ZKD_ERR_CUDA;
  }
  cached = (prop.major == 10) ? ZKD_OK : ZKD_ERR_ARCH;
  return cached;
}

// ---- measured IMAD peak -------------------------------------------------------------------------------------------
// Register-only loop of independent signed IMAD.WIDE (32x32+64 -> 64), the instruction the digit GEMM is made of:
// 8 accumulators x 4 multipliers per thread, 1024 threads per SM.  Every product of an iteration has distinct
// operands and the multipliers change every iteration (one IADD on the ALU pipe per 8 multiplies), so ptxas can
// neither merge nor hoist the multiplies: the SASS loop body holds exactly 32 IMAD.WIDE (cuobjdump -sass).
__global__ void __launch_bounds__(256) imad_peak_kernel(uint32_t* out, int32_t a0, int32_t b0, int iters) {
  int32_t a[8], b[4];
  int64_t acc[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) { a[i] = a0 + 3 * i + (int)threadIdx.x; acc[i] = i; }
#pragma unroll
  for (int u = 0; u < 4; ++u) b[u] = b0 + 5 * u + (int)blockIdx.x;
#pragma unroll 1
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < 4; ++u) {
#pragma unroll
      for (int i = 0; i < 8; ++i) acc[i] += (int64_t)a[i] * (int64_t)b[u];
      b[u] += it;
    }
  }
  int64_t s = 0;
#pragma unroll
  for (int i = 0; i < 8; ++i) s += acc[i];
  out[blockIdx.x * blockDim.x + threadIdx.x] = (uint32_t)s ^ (uint32_t)((uint64_t)s >> 32);
}

int measure_imad_peak(double millis, double* per_sec, cudaStream_t s) {
  int dev = 0, sms = 0;
  ZKD_CUDA_TRY(cudaGetDevice(&dev));
  ZKD_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  const int blocks = sms * 4, threads = 256;
  uint32_t* d = nullptr;
  ZKD_CUDA_TRY(cudaMalloc(&d, sizeof(uint32_t) * blocks * threads));
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  int iters = 2000;
  double best = 0;
  imad_peak_kernel<<<blocks, threads, 0, s>>>(d, 3, 5, 200);  // warm-up
  const int reps = millis > 20 ? 5 : 3;
  // size one launch to about millis/reps
  for (int r = 0; r < reps + 1; ++r) {
    cudaEventRecord(e0, s);
    imad_peak_kernel<<<blocks, threads, 0, s>>>(d, 3, 5, iters);
    cudaEventRecord(e1, s);
    if (cudaEventSynchronize(e1) != cudaSuccess) {
      (void)cudaGetLastError();
      cudaFree(d);
      return ZKD_ERR_CUDA;
    }
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    const double ops = (double)blocks * threads * (double)iters * 32.0;
    if (r > 0 && ops / (ms * 1e-3) > best) best = ops / (ms * 1e-3);
    if (r == 0 && ms > 0) {
      double scale = (millis / reps) / ms;
      if (scale > 50) scale = 50;
      if (scale < 0.05) scale = 0.05;
      iters = (int)(iters * scale) + 1;
    }
  }
  count_launch(reps + 2);
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(d);
  *per_sec = best;
  return ZKD_OK;
}

// ---- measured fp64 FMA peak (roofline denominator of the fp64 seed) -------------------------------------------------
// Register-only loop of independent DFMA chains: 8 accumulators per thread, 1024 threads per SM.
__global__ void __launch_bounds__(256) dfma_peak_kernel(double* out, double a0, double b0, int iters) {
  double acc[8], a[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) { acc[i] = (double)i + (double)threadIdx.x; a[i] = a0 + 1e-9 * (double)(i + blockIdx.x); }
  double b = b0;
#pragma unroll 1
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < 4; ++u) {
#pragma unroll
      for (int i = 0; i < 8; ++i) acc[i] = fma(acc[i], a[i], b);
    }
    b += 1e-12;
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < 8; ++i) s += acc[i];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

int measure_dfma_peak(double millis, double* flops_per_sec, cudaStream_t s) {
  int dev = 0, sms = 0;
  ZKD_CUDA_TRY(cudaGetDevice(&dev));
  ZKD_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  const int blocks = sms * 4, threads = 256;
  double* d = nullptr;
  ZKD_CUDA_TRY(cudaMalloc(&d, sizeof(double) * blocks * threads));
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  int iters = 2000;
  double best = 0;
  dfma_peak_kernel<<<blocks, threads, 0, s>>>(d, 0.999999, 1e-3, 200);  // warm-up
  const int reps = millis > 20 ? 5 : 3;
  for (int r = 0; r < reps + 1; ++r) {
    cudaEventRecord(e0, s);
    dfma_peak_kernel<<<blocks, threads, 0, s>>>(d, 0.999999, 1e-3, iters);
    cudaEventRecord(e1, s);
    if (cudaEventSynchronize(e1) != cudaSuccess) {
      (void)cudaGetLastError();
      cudaFree(d);
      return ZKD_ERR_CUDA;
    }
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    const double flops = (double)blocks * threads * (double)iters * 32.0 * 2.0;
    if (r > 0 && flops / (ms * 1e-3) > best) best = flops / (ms * 1e-3);
    if (r == 0 && ms > 0) {
      double scale = (millis / reps) / ms;
      if (scale > 50) scale = 50;
      if (scale < 0.05) scale = 0.05;
      iters = (int)(iters * scale) + 1;
    }
  }
  count_launch(reps + 2);
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(d);
  *flops_per_sec = best;
  return ZKD_OK;
}

}  // namespace zkd

using namespace zkd;

extern "C" {

size_t zkd_real_bytes(int prec_bits) { return prec_supported(prec_bits) ? api_real_bytes(prec_bits) : 0; }

const char* zkd_strerror(int code) {
  switch (code) {
    case ZKD_OK: return "ok";
    case ZKD_ERR_INVALID_ARG: return "invalid argument";
    case ZKD_ERR_UNSUPPORTED_PREC: return "unsupported precision (multiples of 64 from 128 to 768 bits)";
    case ZKD_ERR_WORKSPACE: return "workspace too small or allocation failed";
    case ZKD_ERR_CUDA: return "CUDA error";
    case ZKD_ERR_ARCH: return "device is not sm_100";
    case ZKD_ERR_INTERNAL: return "internal consistency check failed";
    case ZKD_ERR_CLUSTERED: return "clustered spectrum: exact per-vector RQI does not apply";
    case ZKD_ERR_STATIC_LIMIT: return "size exceeds the static scratch of the no-allocation entry point (N <= 512)";
    default: return "unknown error";
  }
}
int zkd_version(void) { return 100; }

void zkd_counters(uint64_t* kernel_launches, uint64_t* gemm_digit_macs) {
  if (kernel_launches) *kernel_launches = g_launches.load();
  if (gemm_digit_macs) *gemm_digit_macs = g_macs.load();
}
void zkd_counters_reset(void) {
  g_launches.store(0);
  g_macs.store(0);
  g_i8_macs.store(0);
}

static int* option_slot(const char* key) {
  Options& o = options();
  if (!key) return nullptr;
  if (!strcmp(key, "tau_bits")) return &o.tau_bits;
  if (!strcmp(key, "tol_bits")) return &o.tol_bits;
  if (!strcmp(key, "max_steps")) return &o.max_steps;
  if (!strcmp(key, "gemm_path")) return &o.gemm_path;
  if (!strcmp(key, "min_split_ctas")) return &o.min_split_ctas;
  if (!strcmp(key, "gemm_tile")) return &o.gemm_tile;
  if (!strcmp(key, "seed_sweeps")) return &o.seed_sweeps;
  if (!strcmp(key, "seed_path")) return &o.seed_path;
  if (!strcmp(key, "seed_dbuf")) return &o.seed_dbuf;
  if (!strcmp(key, "seed_block_warps")) return &o.seed_block_warps;
  if (!strcmp(key, "seed_tma")) return &o.seed_tma;
  if (!strcmp(key, "seed_gram")) return &o.seed_gram;
  if (!strcmp(key, "i8_bdiag")) return &o.i8_bdiag;
  if (!strcmp(key, "seed_degenerate_skip")) return &o.seed_degenerate_skip;
  if (!strcmp(key, "seed_ring_block")) return &o.seed_ring_block;
  if (!strcmp(key, "seed_cluster")) return &o.seed_cluster;
  if (!strcmp(key, "early_split")) return &o.early_split;
  if (!strcmp(key, "split_margin_bits")) return &o.split_margin_bits;
  if (!strcmp(key, "sstep_cpb")) return &o.sstep_cpb;
  if (!strcmp(key, "sstep_cache")) return &o.sstep_cache;
  if (!strcmp(key, "sstep_par")) return &o.sstep_par;
  if (!strcmp(key, "sstep_warp")) return &o.sstep_warp;
  if (!strcmp(key, "combine_path")) return &o.combine_path;
  if (!strcmp(key, "cluster_tiles")) return &o.cluster_tiles;
  if (!strcmp(key, "i8_step")) return &o.i8_step;
  if (!strcmp(key, "i8_slice")) return &o.i8_slice;
  if (!strcmp(key, "i8_packed")) return &o.i8_packed;
  if (!strcmp(key, "block_correction")) return &o.block_correction;
  if (!strcmp(key, "verbose")) return &o.verbose;
  return nullptr;
}
int zkd_set_option(const char* key, double value) {
  int* s = option_slot(key);
  if (!s || !std::isfinite(value)) return ZKD_ERR_INVALID_ARG;
  *s = (int)value;
  return ZKD_OK;
}
int zkd_get_option(const char* key, double* value) {
  int* s = option_slot(key);
  if (!s || !value) return ZKD_ERR_INVALID_ARG;
  *value = *s;
  return ZKD_OK;
}

// ---- host-side number helpers -------------------------------------------------------------------------------------
int zkd_pack(void* dst, int prec_bits, int sign, int64_t exp, const uint64_t* limbs_le) {
  if (!dst || !prec_supported(prec_bits) || sign < -1 || sign > 1) return ZKD_ERR_INVALID_ARG;
  unsigned char* o = (unsigned char*)dst;
  memset(o, 0, api_real_bytes(prec_bits));
  if (sign == 0) return ZKD_OK;
  if (!limbs_le || !(limbs_le[prec_bits / 64 - 1] >> 63)) return ZKD_ERR_INVALID_ARG;
  int32_t s32 = sign;
  memcpy(o, &s32, 4);
  memcpy(o + 8, &exp, 8);
  memcpy(o + 16, limbs_le, prec_bits / 8);
  return ZKD_OK;
}
int zkd_unpack(const void* src, int prec_bits, int* sign, int64_t* exp, uint64_t* limbs_le) {
  if (!src || !prec_supported(prec_bits)) return ZKD_ERR_INVALID_ARG;
  const unsigned char* s = (const unsigned char*)src;
  int32_t s32, fl;
  int64_t e;
  memcpy(&s32, s, 4);
  memcpy(&fl, s + 4, 4);
  memcpy(&e, s + 8, 8);
  if (fl != 0 || s32 < -1 || s32 > 1) return ZKD_ERR_INVALID_ARG;
  uint64_t top;
  memcpy(&top, s + 16 + prec_bits / 8 - 8, 8);
  if (s32 != 0 && !(top >> 63)) return ZKD_ERR_INVALID_ARG;
  if (sign) *sign = s32;
  if (exp) *exp = e;
  if (limbs_le) memcpy(limbs_le, s + 16, prec_bits / 8);
  return ZKD_OK;
}
int zkd_from_double(void* dst, int prec_bits, double v) {
  if (!dst || !prec_supported(prec_bits) || !std::isfinite(v)) return ZKD_ERR_INVALID_ARG;
  uint64_t limbs[kPrec / 64] = {0};
  if (v == 0.0) return zkd_pack(dst, prec_bits, 0, 0, nullptr);
  int e;
  double m = frexp(fabs(v), &e);  // m in [1/2, 1)
  limbs[prec_bits / 64 - 1] = (uint64_t)ldexp(m, 64);  // exact: m has 53 bits
  return zkd_pack(dst, prec_bits, v < 0 ? -1 : 1, e, limbs);
}
double zkd_to_double(const void* src, int prec_bits) {
  int sign;
  int64_t e;
  uint64_t limbs[kPrec / 64];
  if (zkd_unpack(src, prec_bits, &sign, &e, limbs) != ZKD_OK) return NAN;
  if (sign == 0) return 0.0;
  // round to nearest even on the top 64 bits + sticky
  uint64_t top = limbs[prec_bits / 64 - 1];
  bool sticky = false;
  for (int k = 0; k < prec_bits / 64 - 1; ++k) sticky |= limbs[k] != 0;
  uint64_t keep = top >> 11, rem = top & 0x7ff;
  if (rem > 0x400 || (rem == 0x400 && (sticky || (keep & 1)))) keep += 1;
  double m = ldexp((double)keep, -53);
  double r = ldexp(m, (int)e);
  return sign < 0 ? -r : r;
}

// ---- building blocks ----------------------------------------------------------------------------------------------
int zkd_fx_from_api(int count, int prec_bits, const void* src_api, int32_t* dst_fx, int scale_bits, void* stream) {
  if (!prec_supported(prec_bits)) return ZKD_ERR_UNSUPPORTED_PREC;
  if (count < 0 || !src_api || !dst_fx) return ZKD_ERR_INVALID_ARG;
  ZKD_TRY(check_device());
  return fx_from_api(count, src_api, dst_fx, scale_bits, (cudaStream_t)stream, prec_bits);
}
int zkd_fx_to_api(int count, int prec_bits, const int32_t* src_fx, void* dst_api, int scale_bits, void* stream) {
  if (!prec_supported(prec_bits)) return ZKD_ERR_UNSUPPORTED_PREC;
  if (count < 0 || !src_fx || !dst_api) return ZKD_ERR_INVALID_ARG;
  ZKD_TRY(check_device());
  return fx_to_api(count, src_fx, dst_api, scale_bits, (cudaStream_t)stream, prec_bits);
}
int zkd_fx_prim(int op, int count, const int32_t* a_fx, const int32_t* b_fx, int32_t* out_fx, void* stream) {
  if (count < 0 || !a_fx || !out_fx || op < 0 || op > ZKD_PRIM_FROM_DOUBLE) return ZKD_ERR_INVALID_ARG;
  if (!b_fx && (op == ZKD_PRIM_ADD || op == ZKD_PRIM_SUB || op == ZKD_PRIM_MUL)) return ZKD_ERR_INVALID_ARG;
  ZKD_TRY(check_device());
  return fx_prim(op, (size_t)count, a_fx, b_fx, out_fx, (cudaStream_t)stream);
}
int zkd_gemm_fx_bufsize(int M, int N, int K, int batch, size_t* workspace_bytes) {
  if (M < 1 || N < 1 || K < 1 || batch < 1 || !workspace_bytes) return ZKD_ERR_INVALID_ARG;
  *workspace_bytes = gemm_workspace_bytes(M, N, K, batch);
  return ZKD_OK;
}
int zkd_gemm_fx(int M, int N, int K, int batch, int op_a, const int32_t* A_fx, int a_top_bit, int a_digits,
                const int32_t* B_fx, int b_top_bit, int b_digits, int32_t* C_fx, int mode, int out_cut_bit, int path,
                void* workspace, size_t workspace_bytes, int* err_flag, int* msb_out, void* stream) {
  if (M < 1 || N < 1 || K < 1 || batch < 1 || !A_fx || !B_fx || !C_fx || !workspace || mode < 0 || mode > 2 ||
      a_digits < 1 || a_digits > kND || b_digits < 1 || b_digits > kND)
    return ZKD_ERR_INVALID_ARG;
  ZKD_TRY(check_device());
  GemmSide P, Q;
  P.fx = A_fx; P.rows = op_a ? K : M; P.cols = op_a ? M : K; P.conj_transpose = op_a != 0; P.top_bit = a_top_bit; P.nw = a_digits;
  Q.fx = B_fx; Q.rows = K; Q.cols = N; Q.top_bit = b_top_bit; Q.nw = b_digits;
  return gemm_complex(M, N, K, batch, P, Q, C_fx, (GemmMode)mode, out_cut_bit, path, workspace, workspace_bytes, err_flag,
                      msb_out, (cudaStream_t)stream);
}
int zkd_seed_fp64(int N, int batch, const double* A64, double* mu, double* V, void* stream) {
  if (N < 1 || N > ZKD_MAX_N || batch < 1 || !A64 || !mu || !V) return ZKD_ERR_INVALID_ARG;
  ZKD_TRY(check_device());
  return seed_fp64(N, batch, A64, mu, V, options().seed_sweeps, (cudaStream_t)stream);
}
int zkd_seed_fp64_static(int N, int batch, const double* A64, double* mu, double* V, void* stream) {
  if (N < 1 || batch < 1 || !A64 || !mu || !V) return ZKD_ERR_INVALID_ARG;
  if (N > ZKD_SEED_STATIC_MAX_N) return ZKD_ERR_STATIC_LIMIT;
  ZKD_TRY(check_device());
  return seed_fp64_static(N, batch, A64, mu, V, options().seed_sweeps, (cudaStream_t)stream);
}
int zkd_measure_imad_peak(double millis, double* imad_wide_per_sec, void* stream) {
  if (!imad_wide_per_sec || !(millis > 0)) return ZKD_ERR_INVALID_ARG;
  ZKD_TRY(check_device());
  return measure_imad_peak(millis, imad_wide_per_sec, (cudaStream_t)stream);
}

int zkd_measure_i8_mma_peak(double millis, double* int8_ops_per_sec, void* stream) {
  if (!int8_ops_per_sec || !(millis > 0) || millis > 10000) return ZKD_ERR_INVALID_ARG;
  return measure_i8_mma_peak(millis, int8_ops_per_sec, (cudaStream_t)stream);
}

int zkd_measure_dfma_peak(double millis, double* fp64_flops_per_sec, void* stream) {
  if (!fp64_flops_per_sec || !(millis > 0)) return ZKD_ERR_INVALID_ARG;
  ZKD_TRY(check_device());
  return measure_dfma_peak(millis, fp64_flops_per_sec, (cudaStream_t)stream);
}
int zkd_seed_stats(uint64_t* elems_checked, uint64_t* elems_rotated, int reset) {
  ZKD_TRY(check_device());
  return seed_stats(elems_checked, elems_rotated, reset != 0);
}
int zkd_kernel_timing_categories(void) { return KC_NUM; }
const char* zkd_kernel_timing_name(int category) { return kcat_name(category); }
int zkd_kernel_timing_read_cat(int category, double* ms, uint64_t* launches, uint64_t* work_executed, uint64_t* work_algorithmic) {
  return kt_read(category, ms, launches, work_executed, work_algorithmic);
}

int zkd_kernel_timing(int enable) {
  kernel_timing_enable(enable != 0);
  return ZKD_OK;
}
int zkd_kernel_timing_read(double* gemm_ms, uint64_t* gemm_launches, uint64_t* gemm_digit_macs) {
  return kernel_timing_read(gemm_ms, gemm_launches, gemm_digit_macs);
}
int zkd_kernel_timing_read_i8(double* gemm_ms, uint64_t* gemm_launches, uint64_t* int8_macs) {
  return kernel_timing_read_i8(gemm_ms, gemm_launches, int8_macs);
}

// ---- the hot path -------------------------------------------------------------------------------------------------
static int check_diag_args(int N, int batch, int prec_bits) {
  if (!prec_supported(prec_bits)) return ZKD_ERR_UNSUPPORTED_PREC;
  if (N < 1 || N > ZKD_MAX_N || batch < 1 || batch > 65535) return ZKD_ERR_INVALID_ARG;  // batch is a grid dimension (y / z)
  return ZKD_OK;
}
int zkd_diag_herm_bufsize(int N, int batch, int prec_bits, size_t* workspace_bytes) {
  ZKD_TRY(check_diag_args(N, batch, prec_bits));
  if (!workspace_bytes) return ZKD_ERR_INVALID_ARG;
  *workspace_bytes = diag_workspace_bytes(N, batch);
  return ZKD_OK;
}
int zkd_diag_herm_ws(int N, int batch, int prec_bits, const void* A, void* eigvals, void* eigvecs, void* workspace,
                     size_t workspace_bytes, zkd_info* info, void* stream) {
  ZKD_TRY(check_diag_args(N, batch, prec_bits));
  if (!A || !eigvals || !eigvecs || !workspace) return ZKD_ERR_INVALID_ARG;
  if (((uintptr_t)A | (uintptr_t)eigvals | (uintptr_t)eigvecs | (uintptr_t)workspace) & 15) return ZKD_ERR_INVALID_ARG;
  if (workspace_bytes < diag_workspace_bytes(N, batch)) return ZKD_ERR_WORKSPACE;
  ZKD_TRY(check_device());
  return diag_herm_device(N, batch, prec_bits, A, eigvals, eigvecs, workspace, workspace_bytes, info, (cudaStream_t)stream);
}
int zkd_diag_herm(int N, int batch, int prec_bits, const void* A, void* eigvals, void* eigvecs, void* stream) {
  ZKD_TRY(check_diag_args(N, batch, prec_bits));
  if (!A || !eigvals || !eigvecs) return ZKD_ERR_INVALID_ARG;
  ZKD_TRY(check_device());
  const size_t bytes = diag_workspace_bytes(N, batch);
  void* ws = nullptr;
  cudaStream_t s = (cudaStream_t)stream;
  if (cudaMallocAsync(&ws, bytes, s) != cudaSuccess) {
    (void)cudaGetLastError();
    return ZKD_ERR_WORKSPACE;
  }
  int rc = zkd_diag_herm_ws(N, batch, prec_bits, A, eigvals, eigvecs, ws, bytes, nullptr, stream);
  cudaFreeAsync(ws, s);
  return rc;
}
static int check_svd_args(int M, int N, int batch, int prec_bits) {
  if (!prec_supported(prec_bits)) return ZKD_ERR_UNSUPPORTED_PREC;
  if (M < 1 || N < 1 || M + N > ZKD_MAX_N || batch < 1 || batch > 65535) return ZKD_ERR_INVALID_ARG;
  return ZKD_OK;
}
int zkd_svd_bufsize(int M, int N, int batch, int prec_bits, size_t* workspace_bytes) {
  ZKD_TRY(check_svd_args(M, N, batch, prec_bits));
  if (!workspace_bytes) return ZKD_ERR_INVALID_ARG;
  *workspace_bytes = svd_workspace_bytes(M, N, batch);
  return ZKD_OK;
}
int zkd_svd_ws(int M, int N, int batch, int prec_bits, const void* A, void* S, void* U, void* V, void* workspace, size_t workspace_bytes,
               zkd_info* info, void* stream) {
  ZKD_TRY(check_svd_args(M, N, batch, prec_bits));
  if (!A || !S || !U || !V || !workspace) return ZKD_ERR_INVALID_ARG;
  if (((uintptr_t)A | (uintptr_t)S | (uintptr_t)U | (uintptr_t)V | (uintptr_t)workspace) & 15) return ZKD_ERR_INVALID_ARG;
  if (workspace_bytes < svd_workspace_bytes(M, N, batch)) return ZKD_ERR_WORKSPACE;
  ZKD_TRY(check_device());
  return svd_device(M, N, batch, prec_bits, A, S, U, V, workspace, workspace_bytes, info, (cudaStream_t)stream);
}
int zkd_svd(int M, int N, int batch, int prec_bits, const void* A, void* S, void* U, void* V, void* stream) {
  ZKD_TRY(check_svd_args(M, N, batch, prec_bits));
  if (!A || !S || !U || !V) return ZKD_ERR_INVALID_ARG;
  ZKD_TRY(check_device());
  const size_t bytes = svd_workspace_bytes(M, N, batch);
  void* ws = nullptr;
  cudaStream_t s = (cudaStream_t)stream;
  if (cudaMallocAsync(&ws, bytes, s) != cudaSuccess) {
    (void)cudaGetLastError();
    return ZKD_ERR_WORKSPACE;
  }
  int rc = zkd_svd_ws(M, N, batch, prec_bits, A, S, U, V, ws, bytes, nullptr, stream);
  cudaFreeAsync(ws, s);
  return rc;
}
int zkd_lu_solve_bufsize(int N, int nrhs, int batch, int prec_bits, size_t* workspace_bytes) {
  if (!prec_supported(prec_bits)) return ZKD_ERR_UNSUPPORTED_PREC;
  if (N < 1 || N > ZKD_MAX_N || nrhs < 1 || batch < 1 || batch > 65535 || !workspace_bytes) return ZKD_ERR_INVALID_ARG;
  *workspace_bytes = lu_workspace_bytes(N, nrhs, batch);
  return ZKD_OK;
}
int zkd_lu_solve(int N, int nrhs, int batch, int prec_bits, const void* A, const void* B, void* X, void* workspace, size_t workspace_bytes,
                 int* status, void* stream) {
  if (!prec_supported(prec_bits)) return ZKD_ERR_UNSUPPORTED_PREC;
  if (N < 1 || N > ZKD_MAX_N || nrhs < 1 || batch < 1 || batch > 65535 || !A || !B || !X || !workspace) return ZKD_ERR_INVALID_ARG;
  if (((uintptr_t)A | (uintptr_t)B | (uintptr_t)X | (uintptr_t)workspace) & 15) return ZKD_ERR_INVALID_ARG;
  if (workspace_bytes < lu_workspace_bytes(N, nrhs, batch)) return ZKD_ERR_WORKSPACE;
  ZKD_TRY(check_device());
  return lu_solve_device(N, nrhs, batch, prec_bits, A, B, X, workspace, workspace_bytes, status, (cudaStream_t)stream);
}
int zkd_diag_herm_rqi_lu_bufsize(int N, int batch, int prec_bits, size_t* workspace_bytes) {
  ZKD_TRY(check_diag_args(N, batch, prec_bits));
  if (N > 64 || !workspace_bytes) return ZKD_ERR_INVALID_ARG;
  *workspace_bytes = rqi_lu_workspace_bytes(N, batch);
  return ZKD_OK;
}
int zkd_diag_herm_rqi_lu(int N, int batch, int prec_bits, const void* A, void* eigvals, void* eigvecs, void* workspace,
                         size_t workspace_bytes, zkd_info* info, void* stream) {
  ZKD_TRY(check_diag_args(N, batch, prec_bits));
  if (N > 64 || !A || !eigvals || !eigvecs || !workspace) return ZKD_ERR_INVALID_ARG;
  if (((uintptr_t)A | (uintptr_t)eigvals | (uintptr_t)eigvecs | (uintptr_t)workspace) & 15) return ZKD_ERR_INVALID_ARG;
  if (workspace_bytes < rqi_lu_workspace_bytes(N, batch)) return ZKD_ERR_WORKSPACE;
  ZKD_TRY(check_device());
  return diag_herm_rqi_lu_device(N, batch, prec_bits, A, eigvals, eigvecs, workspace, workspace_bytes, info, (cudaStream_t)stream);
}
static int check_mps_args(int chiL, int chiC, int chiR, int d, int batch, int prec_bits) {
  if (!prec_supported(prec_bits)) return ZKD_ERR_UNSUPPORTED_PREC;
  if (chiL < 1 || chiC < 1 || chiR < 1 || d < 1 || d > 16 || batch < 1 || batch > 65535) return ZKD_ERR_INVALID_ARG;
  if ((long)chiL * d > ZKD_MAX_N || (long)d * chiR > 65536 || chiC > 65536) return ZKD_ERR_INVALID_ARG;
  return ZKD_OK;
}
int zkd_mps_two_site_update_bufsize(int chiL, int chiC, int chiR, int d, int batch, int prec_bits, size_t* workspace_bytes) {
  ZKD_TRY(check_mps_args(chiL, chiC, chiR, d, batch, prec_bits));
  if (!workspace_bytes) return ZKD_ERR_INVALID_ARG;
  *workspace_bytes = mps_workspace_bytes(chiL, chiC, chiR, d, batch);
  return ZKD_OK;
}
int zkd_mps_two_site_update(int chiL, int chiC, int chiR, int d, int batch, int prec_bits, const void* L, const void* R, const void* G,
                            int max_keep, int cutoff_bits, void* W, void* Lnew, void* Rnew, int* kept, zkd_info* info, void* workspace,
                            size_t workspace_bytes, void* stream) {
  ZKD_TRY(check_mps_args(chiL, chiC, chiR, d, batch, prec_bits));
  if (!L || !R || !G || !W || !Lnew || !Rnew || !kept || !workspace || cutoff_bits < 0 || cutoff_bits > 800) return ZKD_ERR_INVALID_ARG;
  if (((uintptr_t)L | (uintptr_t)R | (uintptr_t)G | (uintptr_t)W | (uintptr_t)Lnew | (uintptr_t)Rnew | (uintptr_t)workspace) & 15)
    return ZKD_ERR_INVALID_ARG;
  if (workspace_bytes < mps_workspace_bytes(chiL, chiC, chiR, d, batch)) return ZKD_ERR_WORKSPACE;
  ZKD_TRY(check_device());
  return mps_update_device(chiL, chiC, chiR, d, batch, prec_bits, L, R, G, max_keep, cutoff_bits, W, Lnew, Rnew, kept, info, workspace,
                           workspace_bytes, (cudaStream_t)stream);
}
int zkd_diag_herm_host(int N, int batch, int prec_bits, const void* A_host, void* eigvals_host, void* eigvecs_host,
                       zkd_info* info_host) {
  ZKD_TRY(check_diag_args(N, batch, prec_bits));
  if (!A_host || !eigvals_host || !eigvecs_host) return ZKD_ERR_INVALID_ARG;
  ZKD_TRY(check_device());
  const size_t nA = (size_t)batch * N * N * 2 * api_real_bytes(prec_bits), nL = (size_t)batch * N * api_real_bytes(prec_bits);
  const size_t wsb = diag_workspace_bytes(N, batch);
  const size_t offL = (nA + 255) / 256 * 256, offX = offL + (nL + 255) / 256 * 256, offI = offX + offL,
               offW = offI + ((sizeof(zkd_info) * batch + 255) / 256 * 256);
  // grow-only device buffer kept between calls (cudaMalloc/cudaFree cost more than a whole N=64 decomposition)
  static thread_local char* buf = nullptr;
  static thread_local size_t buf_bytes = 0;
  if (offW + wsb > buf_bytes) {
    if (buf) cudaFree(buf);
    buf = nullptr;
    buf_bytes = 0;
    if (cudaMalloc(&buf, offW + wsb) != cudaSuccess) {
      (void)cudaGetLastError();
      return ZKD_ERR_WORKSPACE;
    }
    buf_bytes = offW + wsb;
  }
  int rc = ZKD_OK;
  cudaStream_t s = 0;
  if (cudaMemcpyAsync(buf, A_host, nA, cudaMemcpyHostToDevice, s) != cudaSuccess) rc = ZKD_ERR_CUDA;
  if (rc == ZKD_OK)
    rc = zkd_diag_herm_ws(N, batch, prec_bits, buf, buf + offL, buf + offX, buf + offW, wsb, (zkd_info*)(buf + offI), s);
  if (rc == ZKD_OK) {
    if (cudaMemcpyAsync(eigvals_host, buf + offL, nL, cudaMemcpyDeviceToHost, s) != cudaSuccess ||
        cudaMemcpyAsync(eigvecs_host, buf + offX, nA, cudaMemcpyDeviceToHost, s) != cudaSuccess ||
        (info_host && cudaMemcpyAsync(info_host, buf + offI, sizeof(zkd_info) * batch, cudaMemcpyDeviceToHost, s) != cudaSuccess) ||
        cudaStreamSynchronize(s) != cudaSuccess)
      rc = ZKD_ERR_CUDA;
  }
  if (rc == ZKD_ERR_CUDA) (void)cudaGetLastError();
  return rc;
}

}  // extern "C"

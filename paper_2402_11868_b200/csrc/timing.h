// timing.h — per-launch device timing of the library's kernels by category (zkd_kernel_timing*, include/zkd.h), for the
// roofline objects of bench.py.  When armed, every kernel launch of the hot path is bracketed by a CUDA event pair on the
// stream it is launched on; the read call sums the elapsed times, launch counts and work counters per category.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace zkd {

enum KCat : int {
  KC_GEMM_DIGITS = 0,  // gemm_digits_kernel<NP,NQ>: work = 28x28-bit digit products (IMAD.WIDE)
  KC_GEMM_I8,          // gemm_i8_kernel: work = s8 x s8 multiply-accumulates
  KC_SEED,             // fp64 seed kernels: work = fp64 flops (rotations actually applied are not known on the host:
                       //   the bound "every pair of every sweep" is NOT used; see seed_stats)
  KC_SSTEP,            // singleton_step kernels: work = digit products
  KC_PREP,             // prep_kernel (+ cached-plane variants): work = bytes moved
  KC_COMBINE,          // combine_kernel / combine_warp_kernel: work = bytes moved
  KC_SLICE_I8,         // slice_i8_kernel: bytes
  KC_COMBINE_I8,       // combine_i8_kernel: bytes
  KC_ECALC,            // ecalc_kernel: digit products
  KC_LU,               // multiprecision LU / triangular solves (S4a', NEXT-3): digit products
  KC_IO,               // ingest / export / conversions: bytes
  KC_OTHER,
  KC_NUM
};

const char* kcat_name(int cat);
bool kt_armed();
// one timed region; work_exec = units the launch executes (padding included), work_alg = units the request needs
struct KtScope {
  KtScope(int cat, cudaStream_t s, uint64_t work_exec = 0, uint64_t work_alg = 0);
  ~KtScope();
  KtScope(const KtScope&) = delete;
  KtScope& operator=(const KtScope&) = delete;

 private:
  int slot_;
  cudaStream_t s_;
};

void kt_enable(bool on);
int kt_read(int cat, double* ms, uint64_t* launches, uint64_t* work_exec, uint64_t* work_alg);

}  // namespace zkd

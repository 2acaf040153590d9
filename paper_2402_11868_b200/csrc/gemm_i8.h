// gemm_i8.h — the int8 tcgen05 engine of the digit GEMM (S4b); see gemm_i8.cu.
#pragma once
#include "zkd_internal.h"

namespace zkd {

// path: 0 = auto (int8 where a matrix fills 128 x 128 x 128 tiles), 1 = IMAD only, 2 = int8 forced
bool gemm_i8_eligible(int path, int M, int N, int K, int batch);
size_t gemm_i8_workspace_bytes(int M, int N, int K, int batch);
// Pc / Qc: compact balanced radix-2^28 planes from prep_kernel ([3*batch][np][M][K] and [3*batch][nq][K][N]) whose digit 0
// sits at FX bit lsbP / lsbQ.  Writes dst (+)= P*Q like combine_kernel.
int gemm_i8_finish(int M, int N, int K, int batch, const int32_t* Pc, const int32_t* Qc, int np, int nq, int lsbP, int lsbQ,
                   int32_t* dst_fx, int mode, int cut_bit, void* ws, size_t ws_bytes, int* err_flag, int* msb_out,
                   cudaStream_t stream, const GemmDstView* dst_view = nullptr, bool q_bdiag32 = false);
void kernel_timing_enable_i8(bool on);
int kernel_timing_read_i8(double* ms, uint64_t* launches, uint64_t* i8_macs);
void count_i8_macs(uint64_t n);
// issue peak of the kernel's MMA shape (128 x 128 x 32 kind::i8, one CTA per SM, operands resident): int8 op/s
int measure_i8_mma_peak(double millis, double* ops_per_sec, cudaStream_t s);

}  // namespace zkd

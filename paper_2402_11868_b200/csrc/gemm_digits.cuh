// gemm_digits.cuh — the IMAD digit GEMM kernel template (S4a / S4d / S4e of SURVEY.md section 8(a)).
//
// Computes, for every plane g (3 real products of the 3M complex scheme x batch), the exact integer product
//     S[g][i][j] = sum_k P[g][i][k] * Q[g][k][j]
// of matrices whose entries are short multi-digit integers: NP (resp. NQ) balanced radix-2^28 digits in int32
// words, digit-major planes.  Every digit product is one IMAD.WIDE into a 64-bit column accumulator
// (column c = i_digit + j_digit); products whose column lies below LOW = NQ - 2 are skipped (truncated product:
// their total is < 2^-17 of the lowest kept column after the guard column is dropped by the caller).
// Carries are resolved once per 16-deep K tile, off the multiply loop.
//
// Roofline: compute-bound on the integer-multiply pipe (30.5 IMAD.WIDE / clk / SM measured by zkd_measure_imad_peak);
// operands are staged through shared memory, each tile word is reused by 16 threads.
#pragma once
#include "fx.cuh"

namespace zkd {

constexpr int GT = 16;  // default output tile GT x GT, K tile GT deep; the kernel is also built with 8 x 8 x 8 tiles (TG = 8)
// for shapes that fill 16-wide tiles badly: a 24 x 24 x 24 cluster product fills (24/32)^3 = 42 % of its 16-tiles and 100 % of its
// 8-tiles (c4's clusters are 24- to 29-dimensional).  The tile size changes the reuse of a staged word (TG times) and nothing
// else: the multiply loop and the output layout are the same.

template <int NP, int NQ, int TG = GT>
struct GemmShape {
  static constexpr int LOW = NQ >= 2 ? NQ - 2 : 0;
  static constexpr int NC = NP + NQ + 1 - LOW;  // kept columns LOW .. NP+NQ
  static constexpr size_t SMEM = sizeof(int32_t) * (NP + NQ) * TG * TG;
  static constexpr int COST = NP * NQ - (LOW * (LOW + 1)) / 2;  // digit products per (i, j, k) (valid while LOW <= min(NP, NQ))
  static constexpr int KUNROLL = COST <= 64 ? 8 : COST <= 160 ? 4 : COST <= 400 ? 2 : 1;
};

struct GemmKArgs {
  const int32_t* P;  // [g][d][M][K]
  const int32_t* Q;  // [g][d][K][N]
  int32_t* Out;      // [split][g][c][M][N]
  size_t p_gstride, p_dstride, q_gstride, q_dstride;
  int M, N, K, G, ksplit, nsplit;
};

template <int NP, int NQ, int TG>
__global__ void __launch_bounds__(TG * TG) gemm_digits_kernel(GemmKArgs a) {
  using S = GemmShape<NP, NQ, TG>;
  extern __shared__ int32_t smem[];
  int32_t* Ps = smem;                    // [NP][TG][TG]   (i, k)
  int32_t* Qs = smem + NP * TG * TG;     // [NQ][TG][TG]   (k, j)
  const int tx = threadIdx.x, ty = threadIdx.y;
  const int g = blockIdx.z / a.nsplit, sp = blockIdx.z % a.nsplit;
  const int i0 = blockIdx.y * TG, j0 = blockIdx.x * TG;
  const int kbeg = sp * a.ksplit, kend = min(a.K, kbeg + a.ksplit);
  const int32_t* Pg = a.P + (size_t)g * a.p_gstride;
  const int32_t* Qg = a.Q + (size_t)g * a.q_gstride;

  int64_t acc[S::NC];
#pragma unroll
  for (int c = 0; c < S::NC; ++c) acc[c] = 0;

  for (int k0 = kbeg; k0 < kend; k0 += TG) {
    // stage the tiles: thread (ty,tx) loads P[i0+ty][k0+tx] and Q[k0+ty][j0+tx] for every digit
    {
      const bool pin = (i0 + ty) < a.M && (k0 + tx) < kend;
      const bool qin = (k0 + ty) < kend && (j0 + tx) < a.N;
      const size_t po = (size_t)(i0 + ty) * a.K + (k0 + tx);
      const size_t qo = (size_t)(k0 + ty) * a.N + (j0 + tx);
#pragma unroll
      for (int d = 0; d < NP; ++d) Ps[(d * TG + ty) * TG + tx] = pin ? Pg[(size_t)d * a.p_dstride + po] : 0;
#pragma unroll
      for (int d = 0; d < NQ; ++d) Qs[(d * TG + ty) * TG + tx] = qin ? Qg[(size_t)d * a.q_dstride + qo] : 0;
    }
    __syncthreads();
    // unrolled for the small instances: with one kk per iteration ptxas shuffles the 64-bit accumulator pairs around the back
    // edge (~0.5 IMAD.MOV per product at <8,8>), which costs issue slots on the pipe the products need
#pragma unroll S::KUNROLL
    for (int kk = 0; kk < TG; ++kk) {
      int32_t p[NP], q[NQ];
#pragma unroll
      for (int d = 0; d < NQ; ++d) q[d] = Qs[(d * TG + kk) * TG + tx];
#pragma unroll
      for (int d = 0; d < NP; ++d) p[d] = Ps[(d * TG + ty) * TG + kk];
      mac_cols<NP, NQ, S::LOW, S::NC, false>(acc, p, q);
    }
    carry_balanced(acc);  // <= 16 * min(NP,NQ) products of <= 2^54 per column since the last ripple: < 2^63
    __syncthreads();
  }
  if (i0 + ty < a.M && j0 + tx < a.N) {
    const size_t mn = (size_t)a.M * a.N;
    int32_t* o = a.Out + ((size_t)(sp * a.G + g) * S::NC) * mn + (size_t)(i0 + ty) * a.N + (j0 + tx);
#pragma unroll
    for (int c = 0; c < S::NC; ++c) o[(size_t)c * mn] = (int32_t)acc[c];
  }
}

using GemmLaunchFn = cudaError_t (*)(const GemmKArgs&, dim3 grid, cudaStream_t);

template <int NP, int NQ, int TG>
cudaError_t gemm_digits_launch(const GemmKArgs& a, dim3 grid, cudaStream_t s) {
  using S = GemmShape<NP, NQ, TG>;
  if (S::SMEM > 48 * 1024) {  // per device and cheap: set on every launch rather than cached in a process-wide flag
    cudaError_t e = cudaFuncSetAttribute(gemm_digits_kernel<NP, NQ, TG>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)S::SMEM);
    if (e != cudaSuccess) return e;
  }
  gemm_digits_kernel<NP, NQ, TG><<<grid, dim3(TG, TG), S::SMEM, s>>>(a);
  return cudaGetLastError();
}

struct GemmInstance {
  int np, nq, low, nc;
  GemmLaunchFn launch;   // 16 x 16 x 16 tiles
  GemmLaunchFn launch8;  // 8 x 8 x 8 tiles
};

}  // namespace zkd

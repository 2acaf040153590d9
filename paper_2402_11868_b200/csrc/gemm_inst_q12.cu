// gemm_inst_q12.cu — instantiations of the digit GEMM for NQ = 12 (one translation unit per NQ so that the
// fully unrolled kernels compile in parallel).  Shape list: DESIGN.md, section "GEMM instances".
#include "gemm_digits.cuh"

namespace zkd {
#define ZKD_INST(NP, NQ) {NP, NQ, GemmShape<NP, NQ>::LOW, GemmShape<NP, NQ>::NC, &gemm_digits_launch<NP, NQ, 16>, &gemm_digits_launch<NP, NQ, 8>}
extern const GemmInstance kGemmInstQ12[] = {
    ZKD_INST(12, 12),
    ZKD_INST(16, 12),
    ZKD_INST(20, 12),
    ZKD_INST(24, 12),
    ZKD_INST(30, 12),
};
extern const int kGemmInstQ12Count = sizeof(kGemmInstQ12) / sizeof(GemmInstance);
}  // namespace zkd

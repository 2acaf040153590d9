// gemm_inst_q4.cu — instantiations of the digit GEMM for NQ = 4 (one translation unit per NQ so that the
// fully unrolled kernels compile in parallel).  Shape list: DESIGN.md, section "GEMM instances".
#include "gemm_digits.cuh"

namespace zkd {
#define ZKD_INST(NP, NQ) {NP, NQ, GemmShape<NP, NQ>::LOW, GemmShape<NP, NQ>::NC, &gemm_digits_launch<NP, NQ, 16>, &gemm_digits_launch<NP, NQ, 8>}
extern const GemmInstance kGemmInstQ4[] = {
    ZKD_INST(4, 4),
    ZKD_INST(6, 4),
    ZKD_INST(8, 4),
    ZKD_INST(12, 4),
    ZKD_INST(16, 4),
    ZKD_INST(20, 4),
    ZKD_INST(24, 4),
    ZKD_INST(27, 4),
    ZKD_INST(30, 4),
};
extern const int kGemmInstQ4Count = sizeof(kGemmInstQ4) / sizeof(GemmInstance);
}  // namespace zkd

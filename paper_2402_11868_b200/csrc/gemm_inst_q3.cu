// gemm_inst_q3.cu — instantiations of the digit GEMM for NQ = 3 (one translation unit per NQ so that the
// fully unrolled kernels compile in parallel).  Shape list: DESIGN.md, section "GEMM instances".
#include "gemm_digits.cuh"

namespace zkd {
#define ZKD_INST(NP, NQ) {NP, NQ, GemmShape<NP, NQ>::LOW, GemmShape<NP, NQ>::NC, &gemm_digits_launch<NP, NQ, 16>, &gemm_digits_launch<NP, NQ, 8>}
extern const GemmInstance kGemmInstQ3[] = {
    ZKD_INST(3, 3),
    ZKD_INST(4, 3),
    ZKD_INST(6, 3),
    ZKD_INST(8, 3),
    ZKD_INST(12, 3),
    ZKD_INST(16, 3),
    ZKD_INST(20, 3),
    ZKD_INST(24, 3),
    ZKD_INST(27, 3),
    ZKD_INST(30, 3),
};
extern const int kGemmInstQ3Count = sizeof(kGemmInstQ3) / sizeof(GemmInstance);
}  // namespace zkd

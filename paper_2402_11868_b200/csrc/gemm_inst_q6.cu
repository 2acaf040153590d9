// gemm_inst_q6.cu — instantiations of the digit GEMM for NQ = 6 (one translation unit per NQ so that the
// fully unrolled kernels compile in parallel).  Shape list: DESIGN.md, section "GEMM instances".
#include "gemm_digits.cuh"

namespace zkd {
#define ZKD_INST(NP, NQ) {NP, NQ, GemmShape<NP, NQ>::LOW, GemmShape<NP, NQ>::NC, &gemm_digits_launch<NP, NQ, 16>, &gemm_digits_launch<NP, NQ, 8>}
extern const GemmInstance kGemmInstQ6[] = {
    ZKD_INST(6, 6),
    ZKD_INST(8, 6),
    ZKD_INST(12, 6),
    ZKD_INST(16, 6),
    ZKD_INST(20, 6),
    ZKD_INST(24, 6),
    ZKD_INST(27, 6),
    ZKD_INST(30, 6),
};
extern const int kGemmInstQ6Count = sizeof(kGemmInstQ6) / sizeof(GemmInstance);
}  // namespace zkd

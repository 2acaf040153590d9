// gemm_inst_q5.cu — instantiations of the digit GEMM for NQ = 5 (one translation unit per NQ so that the
// fully unrolled kernels compile in parallel).  Shape list: DESIGN.md, section "GEMM instances".
#include "gemm_digits.cuh"

namespace zkd {
#define ZKD_INST(NP, NQ) {NP, NQ, GemmShape<NP, NQ>::LOW, GemmShape<NP, NQ>::NC, &gemm_digits_launch<NP, NQ, 16>, &gemm_digits_launch<NP, NQ, 8>}
extern const GemmInstance kGemmInstQ5[] = {
    ZKD_INST(5, 5),
    ZKD_INST(8, 5),
    ZKD_INST(12, 5),
    ZKD_INST(16, 5),
    ZKD_INST(20, 5),
    ZKD_INST(24, 5),
    ZKD_INST(27, 5),
    ZKD_INST(30, 5),
};
extern const int kGemmInstQ5Count = sizeof(kGemmInstQ5) / sizeof(GemmInstance);
}  // namespace zkd

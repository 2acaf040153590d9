// gemm_inst_q10.cu — instantiations of the digit GEMM for NQ = 10 (one translation unit per NQ so that the
// fully unrolled kernels compile in parallel).  Shape list: DESIGN.md, section "GEMM instances".
#include "gemm_digits.cuh"

namespace zkd {
#define ZKD_INST(NP, NQ) {NP, NQ, GemmShape<NP, NQ>::LOW, GemmShape<NP, NQ>::NC, &gemm_digits_launch<NP, NQ, 16>, &gemm_digits_launch<NP, NQ, 8>}
extern const GemmInstance kGemmInstQ10[] = {
    ZKD_INST(10, 10),
    ZKD_INST(12, 10),
    ZKD_INST(16, 10),
    ZKD_INST(20, 10),
    ZKD_INST(24, 10),
    ZKD_INST(30, 10),
};
extern const int kGemmInstQ10Count = sizeof(kGemmInstQ10) / sizeof(GemmInstance);
}  // namespace zkd

// gemm_inst_q15.cu — instantiations of the digit GEMM for NQ = 15 (one translation unit per NQ so that the
// fully unrolled kernels compile in parallel).  Shape list: DESIGN.md, section "GEMM instances".
#include "gemm_digits.cuh"

namespace zkd {
#define ZKD_INST(NP, NQ) {NP, NQ, GemmShape<NP, NQ>::LOW, GemmShape<NP, NQ>::NC, &gemm_digits_launch<NP, NQ, 16>, &gemm_digits_launch<NP, NQ, 8>}
extern const GemmInstance kGemmInstQ15[] = {
    ZKD_INST(15, 15),
    ZKD_INST(16, 15),
    ZKD_INST(20, 15),
    ZKD_INST(24, 15),
    ZKD_INST(30, 15),
};
extern const int kGemmInstQ15Count = sizeof(kGemmInstQ15) / sizeof(GemmInstance);
}  // namespace zkd

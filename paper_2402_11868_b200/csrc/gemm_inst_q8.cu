// gemm_inst_q8.cu — instantiations of the digit GEMM for NQ = 8 (one translation unit per NQ so that the
// fully unrolled kernels compile in parallel).  Shape list: DESIGN.md, section "GEMM instances".
#include "gemm_digits.cuh"

namespace zkd {
#define ZKD_INST(NP, NQ) {NP, NQ, GemmShape<NP, NQ>::LOW, GemmShape<NP, NQ>::NC, &gemm_digits_launch<NP, NQ, 16>, &gemm_digits_launch<NP, NQ, 8>}
extern const GemmInstance kGemmInstQ8[] = {
    ZKD_INST(8, 8),
    ZKD_INST(12, 8),
    ZKD_INST(16, 8),
    ZKD_INST(20, 8),
    ZKD_INST(24, 8),
    ZKD_INST(27, 8),
    ZKD_INST(30, 8),
};
extern const int kGemmInstQ8Count = sizeof(kGemmInstQ8) / sizeof(GemmInstance);
}  // namespace zkd

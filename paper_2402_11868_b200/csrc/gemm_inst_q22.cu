// gemm_inst_q22.cu — instantiations of the digit GEMM for NQ = 22 (one translation unit per NQ so that the
// fully unrolled kernels compile in parallel).  Shape list: DESIGN.md, section "GEMM instances".
#include "gemm_digits.cuh"

namespace zkd {
#define ZKD_INST(NP, NQ) {NP, NQ, GemmShape<NP, NQ>::LOW, GemmShape<NP, NQ>::NC, &gemm_digits_launch<NP, NQ, 16>, &gemm_digits_launch<NP, NQ, 8>}
extern const GemmInstance kGemmInstQ22[] = {
    ZKD_INST(22, 22),
    ZKD_INST(30, 22),
};
extern const int kGemmInstQ22Count = sizeof(kGemmInstQ22) / sizeof(GemmInstance);
}  // namespace zkd

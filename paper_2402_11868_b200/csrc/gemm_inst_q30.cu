// gemm_inst_q30.cu — instantiations of the digit GEMM for NQ = 30 (one translation unit per NQ so that the
// fully unrolled kernels compile in parallel).  Shape list: DESIGN.md, section "GEMM instances".
#include "gemm_digits.cuh"

namespace zkd {
#define ZKD_INST(NP, NQ) {NP, NQ, GemmShape<NP, NQ>::LOW, GemmShape<NP, NQ>::NC, &gemm_digits_launch<NP, NQ, 16>, &gemm_digits_launch<NP, NQ, 8>}
extern const GemmInstance kGemmInstQ30[] = {
    ZKD_INST(30, 30),
};
extern const int kGemmInstQ30Count = sizeof(kGemmInstQ30) / sizeof(GemmInstance);
}  // namespace zkd

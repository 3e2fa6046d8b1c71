// Stage 3/4, mm_mode = NNP_MM_3XTF32_TC / NNP_MM_TF32_TC: tcgen05 + TMA grouped GEMMs.  (Placeholder until the
// tensor-core kernels land: fails loudly, never falls back.)
#include "nnp_internal.cuh"

int nnp_launch_gemm_tc(nnp_ctx *c, const GemmBatch &, int, int)
{
    c->err = "mm_mode 1/2 (tcgen05 path) is not built in this revision; use NNP_MM_FP32_SIMT";
    return NNP_EINVAL;
}

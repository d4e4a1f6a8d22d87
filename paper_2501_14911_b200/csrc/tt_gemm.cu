// tt_gemm.cu - k-RHS per-frequency complex GEMMs (step D of DESIGN.md).  Placeholder translation
// unit: the k-RHS entry points currently run the single-vector kernels once per right-hand side.
#include "tt_common.cuh"
#include "tt_internal.h"

namespace tt {

cudaError_t gemm_fwd_launch(int, const void*, const void*, void*, const GemmGeom&, cudaStream_t) {
    return cudaErrorNotSupported;
}
cudaError_t gemm_adj_launch(int, const void*, const void*, void*, const GemmGeom&, cudaStream_t) {
    return cudaErrorNotSupported;
}

}  // namespace tt

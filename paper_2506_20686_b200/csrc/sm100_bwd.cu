// bf16 backward on tcgen05 (under construction: currently routes to the CUDA-core kernels).
#include "sm100_common.cuh"
#include "tri_common.cuh"

namespace tri {

size_t sm100_bwd_workspace(const Problem& p) { return simt_bwd_workspace(p); }

tri_status sm100_bwd(const Problem& p, const void* dO, const void* Q, const void* K, const void* V, const void* G,
                     const void* bias, const unsigned char* mask, const void* O, const float* LSE, void* dQ, void* dK,
                     void* dV, void* dG, float* dBias, void* ws, cudaStream_t st) {
    return simt_bwd(p, TRI_BF16, dO, Q, K, V, G, bias, mask, O, LSE, dQ, dK, dV, dG, dBias, ws, st);
}

}  // namespace tri

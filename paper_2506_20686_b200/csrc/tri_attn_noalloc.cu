// tri_attn_fwd_noalloc: the forward (Listing 1 P:L153-185 + gate + mask) for callers that cannot allocate device
// memory and do not want to carry a workspace -- code under CUDA graph capture, tight serving loops, harnesses that
// forbid cudaMalloc.  The forward's scratch (the packed mask words and the fp32 log2e * bias planes of the tensor-core
// path; see sm100_fwd_workspace) lives in ONE file-scope device array of TRI_NOALLOC_SCRATCH_BYTES, which every GPU
// that loads the library holds until the process exits.  No cudaMalloc, cudaFree or allocating library routine is
// called here or below (tri_attn_fwd launches kernels and encodes tensor maps only).
//
// The array is shared by every call and keeps the last call's contents.  Nothing in it has to start at zero: the
// mask words and the bias planes a call reads are all written by that call's own preparation kernels first (TMA never
// reads beyond the planes it was given the extent of), so no clearing pass is needed.  Two calls that overlap on the
// GPU (different streams, or different host threads without stream ordering between them) race on the array.
#include <cstdint>
#include <mutex>

#include "tri_common.cuh"

namespace {
// In host code this name is a host-side stand-in for the symbol, NOT a device address: the address comes from
// cudaGetSymbolAddress, once per device, with that device current (below).
static __device__ __align__(256) unsigned char g_noalloc_scratch[TRI_NOALLOC_SCRATCH_BYTES];

std::mutex g_noalloc_mu;
void* g_noalloc_ptr[64];  // per device ordinal; nullptr = not looked up yet

tri_status noalloc_scratch(void** out) {
    int dev = 0;
    TRI_CUDA_CHECK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return TRI_ERR_UNSUPPORTED;
    std::lock_guard<std::mutex> lock(g_noalloc_mu);
    if (!g_noalloc_ptr[dev]) {
        void* ptr = nullptr;
        TRI_CUDA_CHECK(cudaGetSymbolAddress(&ptr, g_noalloc_scratch));
        if (!ptr || ((uintptr_t)ptr & 255)) return ::tri::cuda_fail(cudaErrorInvalidSymbol, "tri_attn_fwd_noalloc: scratch symbol");
        g_noalloc_ptr[dev] = ptr;
    }
    *out = g_noalloc_ptr[dev];
    return TRI_OK;
}
}  // namespace

extern "C" {

size_t tri_attn_noalloc_scratch_bytes(void) { return (size_t)TRI_NOALLOC_SCRATCH_BYTES; }

tri_status tri_attn_fwd_noalloc(const void* Q, const void* K, const void* V, const void* G, const void* bias,
                                const unsigned char* mask, void* O, float* LSE, int B, int N, int H, int d,
                                tri_variant variant, tri_dtype dtype, void* cuda_stream) {
    // 0 = bad or unsupported arguments: tri_attn_fwd below returns the precise status for those before any launch
    const size_t need = tri_attn_fwd_workspace_bytes(B, N, H, d, variant, dtype);
    if (need > (size_t)TRI_NOALLOC_SCRATCH_BYTES) return TRI_ERR_TOO_LARGE;
    if (!Q || !K || !V || !G || !bias || !O || !LSE) return TRI_ERR_INVALID_ARG;  // before the first CUDA call
    void* scratch = nullptr;
    if (need > 0) {
        const tri_status s = noalloc_scratch(&scratch);
        if (s != TRI_OK) return s;
    }
    return tri_attn_fwd(Q, K, V, G, bias, mask, O, LSE, B, N, H, d, variant, dtype, scratch, need ? (size_t)TRI_NOALLOC_SCRATCH_BYTES : 0,
                        cuda_stream);
}

}  // extern "C"

// placeholder, replaced by the tcgen05 forward
#include "tri_common.cuh"
namespace tri {
bool sm100_supported(const Problem&, tri_dtype) { return false; }
size_t sm100_fwd_workspace(const Problem&) { return 0; }
size_t sm100_bwd_workspace(const Problem&) { return 0; }
tri_status sm100_fwd(const Problem&, const void*, const void*, const void*, const void*, const void*, const unsigned char*, void*, float*, void*, cudaStream_t) { return TRI_ERR_UNSUPPORTED; }
tri_status sm100_bwd(const Problem&, const void*, const void*, const void*, const void*, const void*, const void*, const unsigned char*, const void*, const float*, void*, void*, void*, void*, float*, void*, cudaStream_t) { return TRI_ERR_UNSUPPORTED; }
}

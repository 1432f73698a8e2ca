// Host side of TMA: builds CUtensorMap descriptors with the driver's cuTensorMapEncodeTiled, resolved at run
// time through the runtime API (no link-time dependency on libcuda).
#include <mutex>
#include <string.h>
#include <unordered_map>

#include "sm100_common.cuh"
#include "tri_common.cuh"

namespace tri {
namespace {

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn() {
    static EncodeTiledFn fn = nullptr;
    static std::once_flag once;
    std::call_once(once, [] {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
    });
    return fn;
}

// Descriptor cache: a CUtensorMap is a pure function of (kind, base pointer, shape, variant, box), and a training loop
// calls with the same buffers every step, so the driver's encode runs once per distinct key (bounded: flushed at 4096 keys).
struct TmapKey {
    int kind;
    const void* base;
    int a, b, c, d, e, f;
    bool operator==(const TmapKey& o) const { return memcmp(this, &o, sizeof(TmapKey)) == 0; }
};
struct TmapKeyHash {
    size_t operator()(const TmapKey& k) const {
        size_t h = (size_t)k.base * 1099511628211ull;
        const int v[7] = {k.kind, k.a, k.b, k.c, k.d, k.e, k.f};
        for (int x : v) h = (h ^ (size_t)x) * 1099511628211ull;
        return h;
    }
};
std::mutex g_tmap_mu;
std::unordered_map<TmapKey, CUtensorMap, TmapKeyHash> g_tmap_cache;

template <typename F>
bool cached(const TmapKey& key, CUtensorMap* out, F&& encode) {
    {
        std::lock_guard<std::mutex> lock(g_tmap_mu);
        auto it = g_tmap_cache.find(key);
        if (it != g_tmap_cache.end()) {
            *out = it->second;
            return true;
        }
    }
    if (!encode(out)) return false;
    std::lock_guard<std::mutex> lock(g_tmap_mu);
    if (g_tmap_cache.size() >= 4096) g_tmap_cache.clear();
    g_tmap_cache.emplace(key, *out);
    return true;
}

}  // namespace

bool make_tmap_u(CUtensorMap* out_, const void* base, int B, int N, int H, int d, int variant, int box_pos, int rows) {
    const int R = rows < 0 ? N : rows;  // broadcast rows (starting node: the first N axis)
    TmapKey key;
    memset(&key, 0, sizeof(key));
    key.kind = 0; key.base = base; key.a = B; key.b = N; key.c = H; key.d = d; key.e = variant * 65536 + R; key.f = box_pos;
    return cached(key, out_, [&](CUtensorMap* out) {
    EncodeTiledFn fn = encode_fn();
    if (!fn) return false;
    const cuuint64_t es = 2;
    const cuuint64_t s_c = (cuuint64_t)d * es, s_h = (cuuint64_t)N * d * es, s_a = (cuuint64_t)H * N * d * es,
                     s_b = (cuuint64_t)R * H * N * d * es;
    // dims: (d, pos, row, h, b)
    cuuint64_t dims[5] = {(cuuint64_t)d, (cuuint64_t)N, (cuuint64_t)R, (cuuint64_t)H, (cuuint64_t)B};
    cuuint64_t strides[4];
    if (variant == TRI_STARTING) { strides[0] = s_c; strides[1] = s_a; } else { strides[0] = s_a; strides[1] = s_c; }
    strides[2] = s_h;
    strides[3] = s_b;
    cuuint32_t box[5] = {(cuuint32_t)d, (cuuint32_t)box_pos, 1, 1, 1};
    cuuint32_t estr[5] = {1, 1, 1, 1, 1};
    CUresult r = fn(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 5, const_cast<void*>(base), dims, strides, box, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_64B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS;
    });
}

bool make_tmap_plane(CUtensorMap* out_, const void* base, int BH, int N, int box_rows) {
    TmapKey key;
    memset(&key, 0, sizeof(key));
    key.kind = 1; key.base = base; key.a = BH; key.b = N; key.c = box_rows;
    return cached(key, out_, [&](CUtensorMap* out) {
    EncodeTiledFn fn = encode_fn();
    if (!fn) return false;
    cuuint64_t dims[3] = {(cuuint64_t)N, (cuuint64_t)N, (cuuint64_t)BH};
    cuuint64_t strides[2] = {(cuuint64_t)N * 2, (cuuint64_t)N * N * 2};
    cuuint32_t box[3] = {64, (cuuint32_t)box_rows, 1};
    cuuint32_t estr[3] = {1, 1, 1};
    CUresult r = fn(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(base), dims, strides, box, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS;
    });
}

bool make_tmap_plane_f32(CUtensorMap* out_, const void* base, int BH, int N, int box_rows) {
    TmapKey key;
    memset(&key, 0, sizeof(key));
    key.kind = 2; key.base = base; key.a = BH; key.b = N; key.c = box_rows;
    return cached(key, out_, [&](CUtensorMap* out) {
    EncodeTiledFn fn = encode_fn();
    if (!fn) return false;
    cuuint64_t dims[3] = {(cuuint64_t)N, (cuuint64_t)N, (cuuint64_t)BH};
    cuuint64_t strides[2] = {(cuuint64_t)N * 4, (cuuint64_t)N * N * 4};
    cuuint32_t box[3] = {32, (cuuint32_t)box_rows, 1};
    cuuint32_t estr[3] = {1, 1, 1};
    CUresult r = fn(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<void*>(base), dims, strides, box, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS;
    });
}

}  // namespace tri

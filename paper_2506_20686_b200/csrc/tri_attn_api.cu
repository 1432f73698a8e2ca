// C-ABI entry points of libtri_attn.so (include/tri_attn.h): argument validation, workspace
// accounting, kernel-family selection, and the host-buffer end-to-end step.
#include <atomic>
#include <stdio.h>
#include <string.h>

#include "tri_common.cuh"

namespace tri {

static std::atomic<unsigned long long> g_launches{0};
static thread_local char g_err[256] = "";

void count_launch(int n) { g_launches.fetch_add((unsigned long long)n, std::memory_order_relaxed); }

tri_status cuda_fail(cudaError_t e, const char* where) {
    snprintf(g_err, sizeof(g_err), "%s: %s", where, cudaGetErrorString(e));
    return TRI_ERR_CUDA;
}

// ---- per-kernel event timing --------------------------------------------------------------------
namespace {
struct ProfRec { const char* name; cudaEvent_t a, b; };
constexpr int kMaxProf = 8192;
ProfRec g_prof[kMaxProf];
int g_prof_n = 0;
int g_prof_created = 0;
bool g_prof_on = false;
}  // namespace

ProfScope::ProfScope(const char* name, cudaStream_t s) : idx(-1), st(s) {
    if (!g_prof_on || g_prof_n >= kMaxProf) return;
    idx = g_prof_n++;
    if (idx >= g_prof_created) {
        cudaEventCreate(&g_prof[idx].a);
        cudaEventCreate(&g_prof[idx].b);
        g_prof_created = idx + 1;
    }
    g_prof[idx].name = name;
    cudaEventRecord(g_prof[idx].a, st);
}
ProfScope::~ProfScope() {
    if (idx >= 0) cudaEventRecord(g_prof[idx].b, st);
}

static bool shape_ok(int B, int N, int H, int d) { return B > 0 && N > 0 && H > 0 && d > 0; }
static bool enums_ok(int variant, int dtype) {
    return (variant == TRI_STARTING || variant == TRI_ENDING) && (dtype == TRI_F32 || dtype == TRI_BF16);
}
static bool d_ok(int d) { return d == 16 || d == 32 || d == 64; }
static bool size_ok(int B, int N, int H, int d) {
    // all element counts must fit comfortably in 63 bits and slice counts in a 31-bit grid dimension
    const double u = (double)B * N * H * N * d;
    return u < 9.0e15 && (double)B * N * H < 2.0e9;
}
static bool al16(const void* p) { return ((uintptr_t)p & 15) == 0; }

}  // namespace tri

using namespace tri;

extern "C" {

size_t tri_attn_fwd_workspace_bytes(int B, int N, int H, int d, tri_variant variant, tri_dtype dtype) {
    if (!shape_ok(B, N, H, d) || !enums_ok(variant, dtype) || !d_ok(d) || !size_ok(B, N, H, d)) return 0;
    Problem p = make_problem(B, N, H, d, variant);
    size_t w = sm100_supported(p, dtype) ? sm100_fwd_workspace(p) : simt_fwd_workspace(p);
    return w < 256 ? 256 : w;
}

size_t tri_attn_bwd_workspace_bytes(int B, int N, int H, int d, tri_variant variant, tri_dtype dtype) {
    if (!shape_ok(B, N, H, d) || !enums_ok(variant, dtype) || !d_ok(d) || !size_ok(B, N, H, d)) return 0;
    Problem p = make_problem(B, N, H, d, variant);
    size_t w = sm100_supported(p, dtype) ? sm100_bwd_workspace(p) : simt_bwd_workspace(p);
    return w < 256 ? 256 : w;
}

tri_status tri_attn_fwd(const void* Q, const void* K, const void* V, const void* G, const void* bias,
                        const unsigned char* mask, void* O, float* LSE, int B, int N, int H, int d,
                        tri_variant variant, tri_dtype dtype, void* workspace, size_t workspace_bytes,
                        void* cuda_stream) {
    if (!shape_ok(B, N, H, d) || !enums_ok(variant, dtype)) return TRI_ERR_INVALID_ARG;
    if (!Q || !K || !V || !G || !bias || !O || !LSE) return TRI_ERR_INVALID_ARG;
    if (!al16(Q) || !al16(K) || !al16(V) || !al16(G) || !al16(bias) || !al16(O) || !al16(LSE)) return TRI_ERR_INVALID_ARG;
    if (!d_ok(d) || !size_ok(B, N, H, d)) return TRI_ERR_UNSUPPORTED;
    const size_t need = tri_attn_fwd_workspace_bytes(B, N, H, d, variant, dtype);
    if (!workspace || ((uintptr_t)workspace & 255) || workspace_bytes < need) return TRI_ERR_WORKSPACE;
    Problem p = make_problem(B, N, H, d, variant);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (sm100_supported(p, dtype)) return sm100_fwd(p, Q, K, V, G, bias, mask, O, LSE, workspace, st);
    return simt_fwd(p, dtype, Q, K, V, G, bias, mask, O, LSE, workspace, st);
}

tri_status tri_attn_bwd(const void* dO, const void* Q, const void* K, const void* V, const void* G,
                        const void* bias, const unsigned char* mask, const void* O, const float* LSE,
                        void* dQ, void* dK, void* dV, void* dG, float* dBias, int B, int N, int H, int d,
                        tri_variant variant, tri_dtype dtype, void* workspace, size_t workspace_bytes,
                        void* cuda_stream) {
    if (!shape_ok(B, N, H, d) || !enums_ok(variant, dtype)) return TRI_ERR_INVALID_ARG;
    if (!dO || !Q || !K || !V || !G || !bias || !O || !LSE || !dQ || !dK || !dV || !dG || !dBias) return TRI_ERR_INVALID_ARG;
    if (!al16(dO) || !al16(Q) || !al16(K) || !al16(V) || !al16(G) || !al16(bias) || !al16(O) || !al16(LSE) ||
        !al16(dQ) || !al16(dK) || !al16(dV) || !al16(dG) || !al16(dBias))
        return TRI_ERR_INVALID_ARG;
    if (!d_ok(d) || !size_ok(B, N, H, d)) return TRI_ERR_UNSUPPORTED;
    const size_t need = tri_attn_bwd_workspace_bytes(B, N, H, d, variant, dtype);
    if (!workspace || ((uintptr_t)workspace & 255) || workspace_bytes < need) return TRI_ERR_WORKSPACE;
    Problem p = make_problem(B, N, H, d, variant);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (sm100_supported(p, dtype))
        return sm100_bwd(p, dO, Q, K, V, G, bias, mask, O, LSE, dQ, dK, dV, dG, dBias, workspace, st);
    return simt_bwd(p, dtype, dO, Q, K, V, G, bias, mask, O, LSE, dQ, dK, dV, dG, dBias, workspace, st);
}

// ---- host-buffer end-to-end step --------------------------------------------------------------
namespace {
struct Arena {
    size_t U, biasB, maskB, lseB, dbiasB, ws, total;
    size_t off[16];
};
Arena arena_layout(int B, int N, int H, int d, tri_variant variant, tri_dtype dtype) {
    Arena a;
    const size_t es = dtype == TRI_F32 ? 4 : 2;
    a.U = align_up((size_t)B * N * H * N * d * es, 256);
    a.biasB = align_up((size_t)B * H * N * N * es, 256);
    a.maskB = align_up((size_t)B * N * N, 256);
    a.lseB = align_up((size_t)B * N * H * N * 4, 256);
    a.dbiasB = align_up((size_t)B * H * N * N * 4, 256);
    size_t wf = tri_attn_fwd_workspace_bytes(B, N, H, d, variant, dtype);
    size_t wb = tri_attn_bwd_workspace_bytes(B, N, H, d, variant, dtype);
    a.ws = align_up(wf > wb ? wf : wb, 256);
    // order: Q K V G dO O dQ dK dV dG (10 x U) | bias | mask | LSE | dBias | ws
    size_t o = 0;
    for (int i = 0; i < 10; ++i) { a.off[i] = o; o += a.U; }
    a.off[10] = o; o += a.biasB;
    a.off[11] = o; o += a.maskB;
    a.off[12] = o; o += a.lseB;
    a.off[13] = o; o += a.dbiasB;
    a.off[14] = o; o += a.ws;
    a.total = o;
    return a;
}
}  // namespace

size_t tri_attn_step_host_arena_bytes(int B, int N, int H, int d, tri_variant variant, tri_dtype dtype) {
    if (!shape_ok(B, N, H, d) || !enums_ok(variant, dtype) || !d_ok(d) || !size_ok(B, N, H, d)) return 0;
    return arena_layout(B, N, H, d, variant, dtype).total;
}

tri_status tri_attn_step_host(const void* hQ, const void* hK, const void* hV, const void* hG, const void* hbias,
                              const unsigned char* hmask, const void* hdO, void* hO, float* hLSE, void* hdQ,
                              void* hdK, void* hdV, void* hdG, float* hdBias, int B, int N, int H, int d,
                              tri_variant variant, tri_dtype dtype, void* arena, size_t arena_bytes,
                              void* cuda_stream) {
    if (!shape_ok(B, N, H, d) || !enums_ok(variant, dtype)) return TRI_ERR_INVALID_ARG;
    if (!hQ || !hK || !hV || !hG || !hbias || !hdO || !hO || !hLSE || !hdQ || !hdK || !hdV || !hdG || !hdBias)
        return TRI_ERR_INVALID_ARG;
    if (!d_ok(d) || !size_ok(B, N, H, d)) return TRI_ERR_UNSUPPORTED;
    const Arena a = arena_layout(B, N, H, d, variant, dtype);
    if (!arena || ((uintptr_t)arena & 255) || arena_bytes < a.total) return TRI_ERR_WORKSPACE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    char* base = (char*)arena;
    const size_t es = dtype == TRI_F32 ? 4 : 2;
    const size_t Ub = (size_t)B * N * H * N * d * es;
    const void* hin[5] = {hQ, hK, hV, hG, hdO};
    for (int i = 0; i < 5; ++i) TRI_CUDA_CHECK(cudaMemcpyAsync(base + a.off[i], hin[i], Ub, cudaMemcpyHostToDevice, st));
    TRI_CUDA_CHECK(cudaMemcpyAsync(base + a.off[10], hbias, (size_t)B * H * N * N * es, cudaMemcpyHostToDevice, st));
    unsigned char* dmask = nullptr;
    if (hmask) {
        dmask = (unsigned char*)(base + a.off[11]);
        TRI_CUDA_CHECK(cudaMemcpyAsync(dmask, hmask, (size_t)B * N * N, cudaMemcpyHostToDevice, st));
    }
    void *dQ_ = base + a.off[0], *dK_ = base + a.off[1], *dV_ = base + a.off[2], *dG_ = base + a.off[3];
    void *ddO = base + a.off[4], *dO_ = base + a.off[5];
    void *gQ = base + a.off[6], *gK = base + a.off[7], *gV = base + a.off[8], *gG = base + a.off[9];
    void* dbias_in = base + a.off[10];
    float* dLSE = (float*)(base + a.off[12]);
    float* gBias = (float*)(base + a.off[13]);
    void* ws = base + a.off[14];
    tri_status s = tri_attn_fwd(dQ_, dK_, dV_, dG_, dbias_in, dmask, dO_, dLSE, B, N, H, d, variant, dtype, ws, a.ws, st);
    if (s != TRI_OK) return s;
    s = tri_attn_bwd(ddO, dQ_, dK_, dV_, dG_, dbias_in, dmask, dO_, dLSE, gQ, gK, gV, gG, gBias, B, N, H, d, variant,
                     dtype, ws, a.ws, st);
    if (s != TRI_OK) return s;
    TRI_CUDA_CHECK(cudaMemcpyAsync(hO, dO_, Ub, cudaMemcpyDeviceToHost, st));
    TRI_CUDA_CHECK(cudaMemcpyAsync(hLSE, dLSE, (size_t)B * N * H * N * 4, cudaMemcpyDeviceToHost, st));
    void* hout[4] = {hdQ, hdK, hdV, hdG};
    void* dout[4] = {gQ, gK, gV, gG};
    for (int i = 0; i < 4; ++i) TRI_CUDA_CHECK(cudaMemcpyAsync(hout[i], dout[i], Ub, cudaMemcpyDeviceToHost, st));
    TRI_CUDA_CHECK(cudaMemcpyAsync(hdBias, gBias, (size_t)B * H * N * N * 4, cudaMemcpyDeviceToHost, st));
    return TRI_OK;
}

void tri_attn_profile_begin(void) {
    g_prof_n = 0;
    g_prof_on = true;
}

int tri_attn_profile_end(char* buf, size_t buflen) {
    g_prof_on = false;
    struct Agg { const char* name; int n; double ms; } agg[64];
    int na = 0;
    for (int i = 0; i < g_prof_n; ++i) {
        if (cudaEventSynchronize(g_prof[i].b) != cudaSuccess) return -1;
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, g_prof[i].a, g_prof[i].b) != cudaSuccess) return -1;
        int j = 0;
        while (j < na && strcmp(agg[j].name, g_prof[i].name) != 0) ++j;
        if (j == na) {
            if (na == 64) continue;
            agg[na++] = Agg{g_prof[i].name, 0, 0.0};
        }
        agg[j].n += 1;
        agg[j].ms += ms;
    }
    size_t off = 0;
    if (buf && buflen) buf[0] = 0;
    for (int j = 0; j < na && buf; ++j) {
        int w = snprintf(buf + off, off < buflen ? buflen - off : 0, "%s %d %.6f\n", agg[j].name, agg[j].n, agg[j].ms);
        if (w < 0 || off + (size_t)w >= buflen) break;
        off += (size_t)w;
    }
    g_prof_n = 0;
    return na;
}

unsigned long long tri_attn_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

const char* tri_status_string(tri_status s) {
    switch (s) {
        case TRI_OK: return "TRI_OK";
        case TRI_ERR_INVALID_ARG: return "TRI_ERR_INVALID_ARG: null/misaligned pointer, non-positive size or bad enum";
        case TRI_ERR_UNSUPPORTED: return "TRI_ERR_UNSUPPORTED: shape or dtype outside the supported set";
        case TRI_ERR_WORKSPACE: return "TRI_ERR_WORKSPACE: workspace null, misaligned or too small";
        case TRI_ERR_CUDA: return "TRI_ERR_CUDA: a CUDA call or kernel launch failed";
    }
    return "unknown tri_status";
}

const char* tri_attn_last_cuda_error(void) { return g_err; }

}  // extern "C"

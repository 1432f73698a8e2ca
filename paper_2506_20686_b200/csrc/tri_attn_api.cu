// C-ABI entry points of libtri_attn.so (include/tri_attn.h): argument validation, workspace
// accounting, kernel-family selection, and the host-buffer end-to-end step.
#include <atomic>
#include <mutex>
#include <vector>
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

// byte ranges of the tensors of a call; outputs must not overlap inputs or each other (include/tri_attn.h)
struct Range { const void* p; size_t n; bool out; };
static bool overlap(const Range& a, const Range& b) {
    const uintptr_t a0 = (uintptr_t)a.p, b0 = (uintptr_t)b.p;
    return a.p && b.p && a0 < b0 + b.n && b0 < a0 + a.n;
}
static bool aliasing(const Range* r, int n) {
    for (int i = 0; i < n; ++i)
        for (int j = i + 1; j < n; ++j)
            if ((r[i].out || r[j].out) && overlap(r[i], r[j])) return true;
    return false;
}

}  // namespace tri

using namespace tri;

extern "C" {

size_t tri_attn_fwd_workspace_bytes(int B, int N, int H, int d, tri_variant variant, tri_dtype dtype) {
    if (!shape_ok(B, N, H, d) || !enums_ok(variant, dtype) || !d_ok(d) || !size_ok(B, N, H, d)) return 0;
    Problem p = make_problem(B, N, H, d, variant);
    size_t w = sm100_fwd_supported(p, dtype) ? sm100_fwd_workspace(p) : simt_fwd_workspace(p);
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
    {
        const size_t es = dtype == TRI_F32 ? 4 : 2, U = (size_t)B * N * H * N * d * es, P = (size_t)B * H * N * N;
        const Range r[] = {{Q, U, false}, {K, U, false}, {V, U, false}, {G, U, false}, {bias, P * es, false},
                           {mask, (size_t)B * N * N, false}, {O, U, true}, {LSE, (size_t)B * N * H * N * 4, true},
                           {workspace, need, true}};
        if (aliasing(r, 9)) return TRI_ERR_INVALID_ARG;
    }
    Problem p = make_problem(B, N, H, d, variant);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (sm100_fwd_supported(p, dtype)) return sm100_fwd(p, Q, K, V, G, bias, mask, O, LSE, workspace, st);
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
    {
        const size_t es = dtype == TRI_F32 ? 4 : 2, U = (size_t)B * N * H * N * d * es, P = (size_t)B * H * N * N;
        const Range r[] = {{dO, U, false}, {Q, U, false}, {K, U, false}, {V, U, false}, {G, U, false}, {bias, P * es, false},
                           {mask, (size_t)B * N * N, false}, {O, U, false}, {LSE, (size_t)B * N * H * N * 4, false},
                           {dQ, U, true}, {dK, U, true}, {dV, U, true}, {dG, U, true}, {dBias, P * 4, true},
                           {workspace, need, true}};
        if (aliasing(r, 15)) return TRI_ERR_INVALID_ARG;
    }
    Problem p = make_problem(B, N, H, d, variant);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (sm100_supported(p, dtype))
        return sm100_bwd(p, dO, Q, K, V, G, bias, mask, O, LSE, dQ, dK, dV, dG, dBias, workspace, st);
    return simt_bwd(p, dtype, dO, Q, K, V, G, bias, mask, O, LSE, dQ, dK, dV, dG, dBias, workspace, st);
}

// ---- decoupled row count (starting node): R broadcast rows that attend over N positions with one [B,H,N,N] bias ----
static bool rows_ok(int B, int R, int N, int H, int d, tri_dtype dtype, bool fwd_only = false) {
    if (!shape_ok(B, N, H, d) || R <= 0 || !d_ok(d) || !size_ok(B, R > N ? R : N, H, d)) return false;
    const Problem p = make_problem(B, N, H, d, TRI_STARTING, R);
    return fwd_only ? sm100_fwd_supported(p, dtype) : sm100_supported(p, dtype);
}

size_t tri_attn_rows_fwd_workspace_bytes(int B, int R, int N, int H, int d, tri_dtype dtype) {
    if (!rows_ok(B, R, N, H, d, dtype, true)) return 0;
    const size_t w = sm100_fwd_workspace(make_problem(B, N, H, d, TRI_STARTING, R));
    return w < 256 ? 256 : w;
}

size_t tri_attn_rows_bwd_workspace_bytes(int B, int R, int N, int H, int d, tri_dtype dtype) {
    if (!rows_ok(B, R, N, H, d, dtype)) return 0;
    const size_t w = sm100_bwd_workspace(make_problem(B, N, H, d, TRI_STARTING, R));
    return w < 256 ? 256 : w;
}

tri_status tri_attn_rows_fwd(const void* Q, const void* K, const void* V, const void* G, const void* bias,
                             const unsigned char* mask, void* O, float* LSE, int B, int R, int N, int H, int d,
                             tri_dtype dtype, void* workspace, size_t workspace_bytes, void* cuda_stream) {
    if (!shape_ok(B, N, H, d) || R <= 0 || !enums_ok(TRI_STARTING, dtype)) return TRI_ERR_INVALID_ARG;
    if (!Q || !K || !V || !G || !bias || !O || !LSE) return TRI_ERR_INVALID_ARG;
    if (!al16(Q) || !al16(K) || !al16(V) || !al16(G) || !al16(bias) || !al16(O) || !al16(LSE)) return TRI_ERR_INVALID_ARG;
    if (!rows_ok(B, R, N, H, d, dtype, true)) return TRI_ERR_UNSUPPORTED;
    const size_t need = tri_attn_rows_fwd_workspace_bytes(B, R, N, H, d, dtype);
    if (!workspace || ((uintptr_t)workspace & 255) || workspace_bytes < need) return TRI_ERR_WORKSPACE;
    {
        const size_t U = (size_t)B * R * H * N * d * 2, P = (size_t)B * H * N * N;
        const Range r[] = {{Q, U, false}, {K, U, false}, {V, U, false}, {G, U, false}, {bias, P * 2, false},
                           {mask, (size_t)B * R * N, false}, {O, U, true}, {LSE, (size_t)B * R * H * N * 4, true},
                           {workspace, need, true}};
        if (aliasing(r, 9)) return TRI_ERR_INVALID_ARG;
    }
    return sm100_fwd(make_problem(B, N, H, d, TRI_STARTING, R), Q, K, V, G, bias, mask, O, LSE, workspace, (cudaStream_t)cuda_stream);
}

tri_status tri_attn_rows_bwd(const void* dO, const void* Q, const void* K, const void* V, const void* G, const void* bias,
                             const unsigned char* mask, const void* O, const float* LSE, void* dQ, void* dK, void* dV,
                             void* dG, float* dBias, int B, int R, int N, int H, int d, tri_dtype dtype, void* workspace,
                             size_t workspace_bytes, void* cuda_stream) {
    if (!shape_ok(B, N, H, d) || R <= 0 || !enums_ok(TRI_STARTING, dtype)) return TRI_ERR_INVALID_ARG;
    if (!dO || !Q || !K || !V || !G || !bias || !O || !LSE || !dQ || !dK || !dV || !dG || !dBias) return TRI_ERR_INVALID_ARG;
    if (!al16(dO) || !al16(Q) || !al16(K) || !al16(V) || !al16(G) || !al16(bias) || !al16(O) || !al16(LSE) ||
        !al16(dQ) || !al16(dK) || !al16(dV) || !al16(dG) || !al16(dBias))
        return TRI_ERR_INVALID_ARG;
    if (!rows_ok(B, R, N, H, d, dtype)) return TRI_ERR_UNSUPPORTED;
    const size_t need = tri_attn_rows_bwd_workspace_bytes(B, R, N, H, d, dtype);
    if (!workspace || ((uintptr_t)workspace & 255) || workspace_bytes < need) return TRI_ERR_WORKSPACE;
    {
        const size_t U = (size_t)B * R * H * N * d * 2, P = (size_t)B * H * N * N;
        const Range r[] = {{dO, U, false}, {Q, U, false}, {K, U, false}, {V, U, false}, {G, U, false}, {bias, P * 2, false},
                           {mask, (size_t)B * R * N, false}, {O, U, false}, {LSE, (size_t)B * R * H * N * 4, false},
                           {dQ, U, true}, {dK, U, true}, {dV, U, true}, {dG, U, true}, {dBias, P * 4, true},
                           {workspace, need, true}};
        if (aliasing(r, 15)) return TRI_ERR_INVALID_ARG;
    }
    return sm100_bwd(make_problem(B, N, H, d, TRI_STARTING, R), dO, Q, K, V, G, bias, mask, O, LSE, dQ, dK, dV, dG, dBias, workspace,
                     (cudaStream_t)cuda_stream);
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

namespace {
// copy streams and fork / join events of tri_attn_step_host (created once per process, never destroyed)
struct HostPipe {
    std::mutex mu;
    cudaStream_t in = nullptr, out = nullptr;
    std::vector<cudaEvent_t> ev;
    bool ready = false;
    bool init() {
        if (ready) return true;
        if (cudaStreamCreateWithFlags(&in, cudaStreamNonBlocking) != cudaSuccess) return false;
        if (cudaStreamCreateWithFlags(&out, cudaStreamNonBlocking) != cudaSuccess) return false;
        ready = true;
        return true;
    }
    cudaEvent_t event(size_t i) {
        while (ev.size() <= i) {
            cudaEvent_t e = nullptr;
            if (cudaEventCreateWithFlags(&e, cudaEventDisableTiming) != cudaSuccess) return nullptr;
            ev.push_back(e);
        }
        return ev[i];
    }
};
HostPipe g_pipes[64];  // one per device ordinal
}  // namespace

// Batch elements are independent problems (every tensor has B as its outermost axis), and on the tensor-core path of
// the starting-node variant so are the broadcast rows of one element (all tensors but bias / dBias have the row as
// their second axis; dBias is accumulated chunk after chunk, in row order).  The step therefore runs as a three-stage
// pipeline over chunks: H2D of chunk c+1 (copy stream) || forward + backward of chunk c (the caller's stream) || D2H
// of chunk c-1 (second copy stream).  Inside a chunk the dO copy overlaps the forward and the O / LSE read-back overlaps
// the backward.  Everything is forked from and joined back into `cuda_stream` with events, so the call still behaves
// as one unit of work enqueued on that stream, and the host is never blocked.
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
    int dev = 0;
    TRI_CUDA_CHECK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return TRI_ERR_UNSUPPORTED;
    HostPipe& g_pipe = g_pipes[dev];
    std::lock_guard<std::mutex> lock(g_pipe.mu);
    if (!g_pipe.init()) return cuda_fail(cudaGetLastError(), "tri_attn_step_host: stream creation");
    cudaStream_t sin = g_pipe.in, sout = g_pipe.out;
    char* base = (char*)arena;
    const size_t es = dtype == TRI_F32 ? 4 : 2;
    // Pipeline chunk.  Row chunks (about eight per element, at least 4 MB per tensor) when the tensor-core kernels can run
    // a [1, rc, H, N, d] problem; else one batch element when its slices keep the 16-byte pointer alignment; else all.
    int rc = N, cb = B;
    if (variant == TRI_STARTING && sm100_supported(make_problem(1, N, H, d, variant), dtype)) {
        rc = ((N + 7) / 8 + 3) / 4 * 4;
        while (rc < N && (size_t)rc * H * N * d * es < ((size_t)4 << 20)) rc *= 2;
        if (rc > N) rc = N;
        cb = 1;
    } else if (B > 1 && ((size_t)H * N * N * es) % 16 == 0 && ((size_t)N * H * N * 4) % 16 == 0) {
        cb = 1;
    }
    const bool by_rows = rc < N;
    // per-row and per-element sizes (bytes)
    const size_t u_row = (size_t)H * N * d * es, l_row = (size_t)H * N * 4, m_row = (size_t)N;
    const size_t pb = (size_t)H * N * N * es, gb = (size_t)H * N * N * 4;
    // arena regions: 0-3 Q K V G | 4 dO | 5 O | 6-9 dQ dK dV dG | 10 bias | 11 mask | 12 LSE | 13 dBias | 14 workspace
    size_t ne = 0;
    cudaEvent_t e0 = g_pipe.event(ne++);
    if (!e0) return cuda_fail(cudaGetLastError(), "tri_attn_step_host: event creation");
    // fork: the copy streams start after everything already enqueued on the caller's stream (the arena may be in use)
    TRI_CUDA_CHECK(cudaEventRecord(e0, st));
    TRI_CUDA_CHECK(cudaStreamWaitEvent(sin, e0, 0));
    TRI_CUDA_CHECK(cudaStreamWaitEvent(sout, e0, 0));
    const void* hin[4] = {hQ, hK, hV, hG};
    void* hout[4] = {hdQ, hdK, hdV, hdG};
    const size_t wf = tri_attn_fwd_workspace_bytes(cb, N, H, d, variant, dtype), wb = tri_attn_bwd_workspace_bytes(cb, N, H, d, variant, dtype);
    void* ws = base + a.off[14];
    for (int b = 0; b < B; b += cb) {
        for (int r0 = 0; r0 < N; r0 += rc) {
            const int nr = N - r0 < rc ? N - r0 : rc;
            const size_t row = (size_t)b * N + r0;                                 // first global row of the chunk
            const size_t uo = row * u_row, u = (size_t)cb * nr * u_row;            // offset / size in a [B,N,H,N,d] tensor
            const size_t lo = row * l_row, lb = (size_t)cb * nr * l_row;           // LSE
            const size_t mo = row * m_row, mb = (size_t)cb * nr * m_row;           // mask
            const bool first = r0 == 0, last = r0 + nr == N;
            auto U_ = [&](int r) { return (void*)(base + a.off[r] + uo); };
            cudaEvent_t e_inA = g_pipe.event(ne++), e_inB = g_pipe.event(ne++), e_f = g_pipe.event(ne++), e_b = g_pipe.event(ne++);
            if (!e_inA || !e_inB || !e_f || !e_b) return cuda_fail(cudaGetLastError(), "tri_attn_step_host: event creation");
            // ---- H2D of the chunk (copy stream): forward inputs, then dO
            for (int i = 0; i < 4; ++i)
                TRI_CUDA_CHECK(cudaMemcpyAsync(U_(i), (const char*)hin[i] + uo, u, cudaMemcpyHostToDevice, sin));
            void* dbias_in = base + a.off[10] + (size_t)b * pb;
            if (first) TRI_CUDA_CHECK(cudaMemcpyAsync(dbias_in, (const char*)hbias + (size_t)b * pb, (size_t)cb * pb, cudaMemcpyHostToDevice, sin));
            unsigned char* dmask = nullptr;
            if (hmask) {
                dmask = (unsigned char*)(base + a.off[11] + mo);
                TRI_CUDA_CHECK(cudaMemcpyAsync(dmask, hmask + mo, mb, cudaMemcpyHostToDevice, sin));
            }
            TRI_CUDA_CHECK(cudaEventRecord(e_inA, sin));
            TRI_CUDA_CHECK(cudaMemcpyAsync(U_(4), (const char*)hdO + uo, u, cudaMemcpyHostToDevice, sin));
            TRI_CUDA_CHECK(cudaEventRecord(e_inB, sin));
            // ---- compute of the chunk (caller's stream)
            float* dLSE = (float*)(base + a.off[12] + lo);
            float* gBias = (float*)(base + a.off[13] + (size_t)b * gb);
            TRI_CUDA_CHECK(cudaStreamWaitEvent(st, e_inA, 0));
            tri_status s;
            if (by_rows)
                s = sm100_fwd(make_problem(1, N, H, d, variant, nr), U_(0), U_(1), U_(2), U_(3), dbias_in, dmask, U_(5), dLSE, ws, st);
            else
                s = tri_attn_fwd(U_(0), U_(1), U_(2), U_(3), dbias_in, dmask, U_(5), dLSE, cb, N, H, d, variant, dtype, ws, wf, st);
            if (s != TRI_OK) return s;
            TRI_CUDA_CHECK(cudaEventRecord(e_f, st));
            TRI_CUDA_CHECK(cudaStreamWaitEvent(st, e_inB, 0));
            if (by_rows)
                s = sm100_bwd(make_problem(1, N, H, d, variant, nr), U_(4), U_(0), U_(1), U_(2), U_(3), dbias_in, dmask, U_(5), dLSE, U_(6),
                              U_(7), U_(8), U_(9), gBias, ws, st, /*accumulate_dbias=*/!first);
            else
                s = tri_attn_bwd(U_(4), U_(0), U_(1), U_(2), U_(3), dbias_in, dmask, U_(5), dLSE, U_(6), U_(7), U_(8), U_(9), gBias, cb, N, H,
                                 d, variant, dtype, ws, wb, st);
            if (s != TRI_OK) return s;
            TRI_CUDA_CHECK(cudaEventRecord(e_b, st));
            // ---- D2H of the chunk (second copy stream): O, LSE while the backward runs, gradients after it
            TRI_CUDA_CHECK(cudaStreamWaitEvent(sout, e_f, 0));
            TRI_CUDA_CHECK(cudaMemcpyAsync((char*)hO + uo, U_(5), u, cudaMemcpyDeviceToHost, sout));
            TRI_CUDA_CHECK(cudaMemcpyAsync((char*)hLSE + lo, dLSE, lb, cudaMemcpyDeviceToHost, sout));
            TRI_CUDA_CHECK(cudaStreamWaitEvent(sout, e_b, 0));
            for (int i = 0; i < 4; ++i)
                TRI_CUDA_CHECK(cudaMemcpyAsync((char*)hout[i] + uo, U_(6 + i), u, cudaMemcpyDeviceToHost, sout));
            if (last)
                TRI_CUDA_CHECK(cudaMemcpyAsync((char*)hdBias + (size_t)b * gb, gBias, (size_t)cb * gb, cudaMemcpyDeviceToHost, sout));
        }
    }
    // join: later work on the caller's stream waits for the last read-back (and for the copy-in stream, trivially done)
    cudaEvent_t e1 = g_pipe.event(ne++), e2 = g_pipe.event(ne++);
    if (!e1 || !e2) return cuda_fail(cudaGetLastError(), "tri_attn_step_host: event creation");
    TRI_CUDA_CHECK(cudaEventRecord(e1, sout));
    TRI_CUDA_CHECK(cudaStreamWaitEvent(st, e1, 0));
    TRI_CUDA_CHECK(cudaEventRecord(e2, sin));
    TRI_CUDA_CHECK(cudaStreamWaitEvent(st, e2, 0));
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

int tri_attn_uses_tensor_cores(int B, int N, int H, int d, tri_variant variant, tri_dtype dtype) {
    if (!shape_ok(B, N, H, d) || !enums_ok(variant, dtype) || !d_ok(d)) return 0;
    return sm100_supported(make_problem(B, N, H, d, variant), dtype) ? 1 : 0;
}

unsigned long long tri_attn_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

const char* tri_status_string(tri_status s) {
    switch (s) {
        case TRI_OK: return "TRI_OK";
        case TRI_ERR_INVALID_ARG: return "TRI_ERR_INVALID_ARG: null/misaligned pointer, non-positive size or bad enum";
        case TRI_ERR_UNSUPPORTED: return "TRI_ERR_UNSUPPORTED: shape or dtype outside the supported set";
        case TRI_ERR_WORKSPACE: return "TRI_ERR_WORKSPACE: workspace null, misaligned or too small";
        case TRI_ERR_CUDA: return "TRI_ERR_CUDA: a CUDA call or kernel launch failed";
        case TRI_ERR_TOO_LARGE: return "TRI_ERR_TOO_LARGE: the problem needs more scratch than the library's built-in array holds (tri_attn_fwd_noalloc); use the workspace entry point";
    }
    return "unknown tri_status";
}

const char* tri_attn_last_cuda_error(void) { return g_err; }

}  // extern "C"

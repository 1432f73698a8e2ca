// Internal declarations shared by the translation units of libtri_attn.so (not part of the ABI).
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "tri_attn.h"

namespace tri {

// One problem instance.  Index conventions (include/tri_attn.h): a "slice" is one (b, r, h) where r
// runs over the broadcast axis of the variant (i for starting, j for ending); inside a slice,
// queries q and keys k run over the other pair axis.
struct Problem {
    int B, N, H, d;
    int variant;  // tri_variant
    int R;        // broadcast rows (= N for the square pair-tensor problem; decoupled row counts: starting node only)
    // element strides of the [B,N,H,N,d] tensors
    long long sB;      // N*H*N*d
    long long sH;      // N*d
    long long sSlice;  // starting: H*N*d (axis a)   ending: d (axis c)
    long long sPos;    // starting: d     (axis c)   ending: H*N*d (axis a)
    // bias[b,h,.,.] : element (q,k) at q*bQ + k*bK
    int bQ, bK;
    // mask[b,.,.]   : element (r,k) at r*mR + k*mK
    int mR, mK;
    // LSE / D [B,R,H,N]: element (r,q) at r*lR + q*lQ (+ b*lB + h*N)
    long long lR, lQ;
    long long lB;  // R*H*N
    long long mB;  // mask batch stride R*N
};

inline Problem make_problem(int B, int N, int H, int d, int variant, int R = -1) {
    Problem p;
    if (R < 0) R = N;
    p.B = B; p.N = N; p.H = H; p.d = d; p.variant = variant; p.R = R;
    p.sB = (long long)R * H * N * d;
    p.lB = (long long)R * H * N;
    p.mB = (long long)R * N;
    p.sH = (long long)N * d;
    if (variant == TRI_STARTING) {
        p.sSlice = (long long)H * N * d; p.sPos = d;
        p.bQ = N; p.bK = 1;
        p.mR = N; p.mK = 1;
        p.lR = (long long)H * N; p.lQ = 1;
    } else {
        p.sSlice = d; p.sPos = (long long)H * N * d;
        p.bQ = 1; p.bK = N;
        p.mR = 1; p.mK = N;
        p.lR = 1; p.lQ = (long long)H * N;
    }
    return p;
}

// launch accounting + error capture (tri_attn_api.cu)
void count_launch(int n = 1);
tri_status cuda_fail(cudaError_t e, const char* where);
#define TRI_CUDA_CHECK(expr)                                   \
    do {                                                       \
        cudaError_t _e = (expr);                               \
        if (_e != cudaSuccess) return ::tri::cuda_fail(_e, #expr); \
    } while (0)
#define TRI_LAUNCH_CHECK(where)                                \
    do {                                                       \
        ::tri::count_launch();                                 \
        cudaError_t _e = cudaGetLastError();                   \
        if (_e != cudaSuccess) return ::tri::cuda_fail(_e, where); \
    } while (0)

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// Per-kernel CUDA-event timing (tri_attn_profile_begin / _end in the ABI).  Declare one in the scope
// of a launch: records an event before and after it on `st` while profiling is on, else does nothing.
struct ProfScope {
    ProfScope(const char* name, cudaStream_t st);
    ~ProfScope();
    int idx;
    cudaStream_t st;
};

// ---- fp32 CUDA-core path (simt_kernels.cu) -------------------------------------------------
size_t simt_fwd_workspace(const Problem& p);
size_t simt_bwd_workspace(const Problem& p);
tri_status simt_fwd(const Problem& p, tri_dtype dt, const void* Q, const void* K, const void* V,
                    const void* G, const void* bias, const unsigned char* mask, void* O, float* LSE,
                    void* ws, cudaStream_t st);
tri_status simt_bwd(const Problem& p, tri_dtype dt, const void* dO, const void* Q, const void* K,
                    const void* V, const void* G, const void* bias, const unsigned char* mask,
                    const void* O, const float* LSE, void* dQ, void* dK, void* dV, void* dG,
                    float* dBias, void* ws, cudaStream_t st);

// ---- bf16 tcgen05 / TMA path (sm100_fwd.cu, sm100_bwd.cu) ------------------------------------
bool sm100_supported(const Problem& p, tri_dtype dt);      // forward + backward on the tensor-core kernels
bool sm100_fwd_supported(const Problem& p, tri_dtype dt);  // forward only (a superset: N up to 16384)
tri_status sm100_transpose_planes(const void* in, void* out, int BH, int N, cudaStream_t st);  // bf16 [BH,N,N]
// fp32 planes f*bias: nat (same orientation) and / or tr (transposed); either may be null
tri_status sm100_bias_planes(const void* in, float* nat, float* tr, int BH, int N, float f, cudaStream_t st);
// keep flags -> one 64-bit word per (b, row, 64-key tile), rows / keys in the variant's sense
tri_status sm100_pack_mask(const Problem& p, const unsigned char* mask, void* bits, cudaStream_t st);
size_t sm100_maskbits_bytes(const Problem& p);
bool sm100_needs_maskbits(const Problem& p, const unsigned char* mask);
// dK / dV stage (sm100_dkdv.cu): NL / ND are fp32 [B,N,H,N] scratch arrays of sm100_dkdv2_aux_bytes() each, filled by
// sm100_lse_prep; a launch covers work items [item_begin, item_begin + item_count) of sm100_dkdv2_items() on <= max_ctas CTAs
size_t sm100_dkdv2_aux_bytes(const Problem& p);
long long sm100_dkdv2_items(const Problem& p);
tri_status sm100_lse_prep(const Problem& p, const float* LSE, const float* Dws, float* NL, float* ND, cudaStream_t st);
tri_status sm100_dkdv2_launch(const Problem& p, const void* Q, const void* dA, const void* K, const void* V, const void* bias_kq,
                              const unsigned long long* maskbits, const float* NL, const float* ND, void* dK, void* dV,
                              long long item_begin, long long item_count, int max_ctas, const char* prof_name, cudaStream_t st);
// fused dQ + dBias stage (sm100_dqdb.cu): cluster size (0 = shape not covered), row split, persistent grid, launch
// one launch of the fused dQ + dBias stage over a slice of the key axis (the whole axis when N <= 2048)
struct DqdbPass {
    int tile_base, tiles;  // first 64-key tile and tile count of the slice
    int last;              // the last slice: dQ is finished (scaled, bf16); otherwise the fp32 running sum goes to dq_part
    float* dq_part;        // fp32 running sum of dQ between the slices, same element order as dQ (unused when there is one slice)
};
int sm100_dqdb_passes(int N);
DqdbPass sm100_dqdb_pass(int N, int i, float* dq_part);
int sm100_dqdb_cluster(int tiles);
constexpr int kDqdbMaxSplit = 8;  // the workspace holds this many partial dBias planes
bool sm100_dqdb_plan(const Problem& p, int tiles, int forceG, int* C, int* G, int* grid);
tri_status sm100_dqdb_launch(const Problem& p, int C, int G, int grid, const void* Q, const void* dA, const void* K,
                             const void* V, const float* biasL_qk, const unsigned long long* maskbits, const float* LSE,
                             const float* Dws, void* dQ, float* dBias, float* planes, DqdbPass pass, cudaStream_t st);
int sm100_sm_count();
size_t sm100_fwd_workspace(const Problem& p);
size_t sm100_bwd_workspace(const Problem& p);
tri_status sm100_fwd(const Problem& p, const void* Q, const void* K, const void* V, const void* G,
                     const void* bias, const unsigned char* mask, void* O, float* LSE, void* ws,
                     cudaStream_t st);
tri_status sm100_bwd(const Problem& p, const void* dO, const void* Q, const void* K, const void* V,
                     const void* G, const void* bias, const unsigned char* mask, const void* O,
                     const float* LSE, void* dQ, void* dK, void* dV, void* dG, float* dBias,
                     void* ws, cudaStream_t st, bool accumulate_dbias = false);  // true: dBias += (starting node only)

}  // namespace tri

// bf16 backward on tcgen05 / TMEM / TMA (sm_100a).  Listing 2, Table I, gate from the task
// statement.  P is recomputed from the saved LSE; nothing of size N^3 is stored.
//
//   pre      D = rowsum(dO . O), dG = dO . O . (1 - sigmoid G), dA = dO . sigmoid G (bf16, workspace)
//   dkdv     (sm100_dkdv.cu) key-stationary (thread = key): S^T = K Q^T, dP^T = V dA^T, P^T, dS^T -> bf16 -> TMEM,
//            dV += P^T dA, dK += dS^T Q
//   dqdb     (sm100_dqdb.cu) dQ and dBias from one recomputation, tile-stationary, cluster reduce of dQ
//   reduce   level 2 of the dBias reduction: adds the row-split partial planes in ascending order
#include <mutex>

#include "sm100_common.cuh"
#include "tri_common.cuh"

namespace tri {
using namespace sm100;

namespace {

constexpr int DH = 32;
constexpr int T128 = 128 * DH * 2;  // 8 KB tile (128 positions)
constexpr int T64 = 64 * DH * 2;    // 4 KB tile (64 positions)

__device__ __forceinline__ float sigmoid_fast(float g) { return __fdividef(1.0f, 1.0f + ex2(-g * kLog2e)); }

// ------------------------------------------------------------------------------------------------------------
// pre-process: 4 threads per 32-channel row (16 B each): coalesced 64-byte rows, D via two shuffles.
// ------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) sm100_bwd_pre_kernel(long long rows, const uint4* __restrict__ dO,
                                                            const uint4* __restrict__ O, const uint4* __restrict__ G,
                                                            uint4* __restrict__ dG, uint4* __restrict__ dA,
                                                            float* __restrict__ Dws) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;  // 16-byte chunk index
    if (i >= rows * 4) return;
    const uint4 a = __ldg(dO + i), o = __ldg(O + i), g = __ldg(G + i);
    const uint32_t aw[4] = {a.x, a.y, a.z, a.w}, ow[4] = {o.x, o.y, o.z, o.w}, gw[4] = {g.x, g.y, g.z, g.w};
    uint32_t dgw[4], daw[4];
    float acc = 0.0f;
#pragma unroll
    for (int e = 0; e < 4; ++e) {
        const float a0 = bf16_lo(aw[e]), a1 = bf16_hi(aw[e]);
        const float x0 = a0 * bf16_lo(ow[e]), x1 = a1 * bf16_hi(ow[e]);
        const float s0 = sigmoid_fast(bf16_lo(gw[e])), s1 = sigmoid_fast(bf16_hi(gw[e]));
        acc += x0 + x1;
        dgw[e] = pack_bf16(x0 * (1.0f - s0), x1 * (1.0f - s1));
        daw[e] = pack_bf16(a0 * s0, a1 * s1);
    }
    dG[i] = make_uint4(dgw[0], dgw[1], dgw[2], dgw[3]);
    dA[i] = make_uint4(daw[0], daw[1], daw[2], daw[3]);
    acc += __shfl_xor_sync(0xffffffffu, acc, 1);
    acc += __shfl_xor_sync(0xffffffffu, acc, 2);
    if ((threadIdx.x & 3) == 0) Dws[i >> 2] = acc;
}

// level 2 of the dBias reduction (only when the row axis was split): dBias[bh][q*bQ + k*bK] = sum over planes, in
// ascending order, of plane[g][bh][q][k]; the ending-node variant wants the transpose (bQ = 1), via a 32x32 smem tile.
// accumulate != 0 (starting node only): the sum starts from the value dBias already holds (row-chunked callers).
__global__ void __launch_bounds__(256) sm100_dbias_reduce_kernel(const float* __restrict__ planes, float* __restrict__ dBias,
                                                                 int BH, int N, int G, int transpose, int accumulate) {
    __shared__ float tile[32][33];
    const int bh = blockIdx.z, q0 = blockIdx.y * 32, k0 = blockIdx.x * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    const long long pstride = (long long)BH * N * N;
    for (int j = ty; j < 32; j += 8) {
        if (q0 + j >= N || k0 + tx >= N) continue;
        const long long o = (long long)bh * N * N + (long long)(q0 + j) * N + k0 + tx;
        float acc = accumulate ? dBias[o] + planes[o] : planes[o];
        for (int g = 1; g < G; ++g) acc += planes[o + g * pstride];
        if (transpose) tile[j][tx] = acc; else dBias[o] = acc;
    }
    if (transpose) {
        __syncthreads();
        for (int j = ty; j < 32; j += 8)
            if (k0 + j < N && q0 + tx < N) dBias[(long long)bh * N * N + (long long)(k0 + j) * N + q0 + tx] = tile[tx][j];
    }
}

}  // namespace

// ---- host side ------------------------------------------------------------------------------------------------
namespace {
struct BwdWs {
    size_t d_off, da_off, biast_off, biasl_off, mask_off, nl_off, nd_off, planes_off, dqpart_off, total;
};
BwdWs bwd_ws_layout(const Problem& p) {
    BwdWs w;
    size_t o = 0;
    w.d_off = o; o += align_up((size_t)p.B * p.R * p.H * p.N * sizeof(float), 256);          // D = rowsum(dO . O)
    w.da_off = o; o += align_up((size_t)p.B * p.R * p.H * p.N * p.d * 2, 256);               // dA = dO . sigmoid(G)
    w.biast_off = o; o += align_up((size_t)p.B * p.H * p.N * p.N * 2, 256);                  // bias^T, bf16 (dkdv)
    w.biasl_off = o; o += align_up((size_t)p.B * p.H * p.N * p.N * 4, 256);                  // log2e * bias[q][k], fp32 (dqdb)
    w.mask_off = o; o += sm100_maskbits_bytes(p);
    w.nl_off = o; o += sm100_dkdv2_aux_bytes(p);                                             // -LSE*log2e per (row, query)
    w.nd_off = o; o += sm100_dkdv2_aux_bytes(p);                                             // -D per (row, query)
    // partial dBias planes: the fused kernel picks its row split (<= kDqdbMaxSplit) at launch from the device's
    // resident cluster count, so the workspace always holds the maximum
    w.planes_off = o; o += align_up((size_t)kDqdbMaxSplit * p.B * p.H * p.N * p.N * sizeof(float), 256);
    // N > 2048: fp32 running sum of dQ between the key passes of the fused stage (one U-shaped tensor)
    w.dqpart_off = o;
    if (sm100_dqdb_passes(p.N) > 1) o += align_up((size_t)p.B * p.R * p.H * p.N * p.d * sizeof(float), 256);
    w.total = o;
    return w;
}
// one side stream + fork / join events per device (created on first use, never destroyed)
struct SideStream {
    cudaStream_t stream = nullptr;
    cudaEvent_t fork = nullptr, join = nullptr;    // stage-1 slice beside stage 2
    cudaEvent_t fork0 = nullptr, join0 = nullptr;  // bias / mask preparation beside the pre-process kernel
    cudaStream_t hi = nullptr;                     // high-priority stream of the dBias plane reduction
    cudaEvent_t stage2 = nullptr, join2 = nullptr; // stage 2 done -> reduction (beside the rest of stage 1) -> joined
    bool ready = false;
    std::mutex enqueue;  // held while one call enqueues: the stream and the events are shared by all callers on the device
};
std::mutex g_side_mu;
SideStream g_side[64];
SideStream* side_stream() {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return nullptr;
    std::lock_guard<std::mutex> lock(g_side_mu);
    SideStream& s = g_side[dev];
    if (!s.ready) {
        if (cudaStreamCreateWithFlags(&s.stream, cudaStreamNonBlocking) != cudaSuccess) return nullptr;
        if (cudaEventCreateWithFlags(&s.fork, cudaEventDisableTiming) != cudaSuccess) return nullptr;
        if (cudaEventCreateWithFlags(&s.join, cudaEventDisableTiming) != cudaSuccess) return nullptr;
        if (cudaEventCreateWithFlags(&s.fork0, cudaEventDisableTiming) != cudaSuccess) return nullptr;
        if (cudaEventCreateWithFlags(&s.join0, cudaEventDisableTiming) != cudaSuccess) return nullptr;
        if (cudaEventCreateWithFlags(&s.stage2, cudaEventDisableTiming) != cudaSuccess) return nullptr;
        if (cudaEventCreateWithFlags(&s.join2, cudaEventDisableTiming) != cudaSuccess) return nullptr;
        int lo = 0, hi = 0;  // numerically lower = higher priority
        if (cudaDeviceGetStreamPriorityRange(&lo, &hi) != cudaSuccess) return nullptr;
        if (cudaStreamCreateWithPriority(&s.hi, cudaStreamNonBlocking, hi) != cudaSuccess) return nullptr;
        s.ready = true;
    }
    return &s;
}
template <typename K>
tri_status set_smem(K kern, int bytes) {
    TRI_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
    return TRI_OK;
}
}  // namespace

size_t sm100_bwd_workspace(const Problem& p) { return bwd_ws_layout(p).total; }

tri_status sm100_bwd(const Problem& p, const void* dO, const void* Q, const void* K, const void* V, const void* G,
                     const void* bias, const unsigned char* mask, const void* O, const float* LSE, void* dQ, void* dK,
                     void* dV, void* dG, float* dBias, void* ws, cudaStream_t st, bool accumulate_dbias) {
    if (accumulate_dbias && p.variant != TRI_STARTING) return TRI_ERR_UNSUPPORTED;
    const BwdWs w = bwd_ws_layout(p);
    float* Dws = (float*)((char*)ws + w.d_off);
    void* dA = (char*)ws + w.da_off;
    void* biasT = (char*)ws + w.biast_off;
    const long long rows = (long long)p.B * p.R * p.H * p.N;
    // Library-owned side stream, forked from and joined back into `st` with events (to the caller the call is one unit of
    // work on `st`).  It carries (1) the bias / mask preparation, which is independent of the HBM-bound pre-process kernel,
    // (2) a slice of stage 1 beside stage 2, (3) the dBias plane reduction beside the rest of stage 1.
    SideStream* side = side_stream();
    // Host threads that call on one device share the side streams and their events: their enqueues take turns (a stream wait
    // captures the event's state when it is enqueued, so a later re-record by another caller does not disturb it).
    std::unique_lock<std::mutex> enqueue_lock;
    if (side) enqueue_lock = std::unique_lock<std::mutex>(side->enqueue);
    cudaStream_t sp = side ? side->stream : st;  // where the preparation kernels go
    if (side) {
        TRI_CUDA_CHECK(cudaEventRecord(side->fork0, st));
        TRI_CUDA_CHECK(cudaStreamWaitEvent(side->stream, side->fork0, 0));
    }
    {
        ProfScope ps("sm100_bwd_pre_kernel", st);
        sm100_bwd_pre_kernel<<<(unsigned)((rows * 4 + 255) / 256), 256, 0, st>>>(rows, (const uint4*)dO, (const uint4*)O,
                                                                               (const uint4*)G, (uint4*)dG, (uint4*)dA, Dws);
    }
    TRI_LAUNCH_CHECK("sm100_bwd_pre_kernel");
    tri_status s = sm100_transpose_planes(bias, biasT, p.B * p.H, p.N, sp);
    if (s != TRI_OK) return s;
    TRI_LAUNCH_CHECK("sm100_transpose_bf16");
    const void* bias_kq = p.variant == TRI_STARTING ? biasT : bias;  // [k][q]

    unsigned long long* maskbits = nullptr;
    if (sm100_needs_maskbits(p, mask)) {
        maskbits = (unsigned long long*)((char*)ws + w.mask_off);
        if ((s = sm100_pack_mask(p, mask, maskbits, sp)) != TRI_OK) return s;
        TRI_LAUNCH_CHECK("pack_mask_kernel");
    }
    float* biasL = (float*)((char*)ws + w.biasl_off);
    {
        const bool tr = p.variant == TRI_ENDING;
        if ((s = sm100_bias_planes(bias, tr ? nullptr : biasL, tr ? biasL : nullptr, p.B * p.H, p.N, kLog2e, sp)) != TRI_OK) return s;
        TRI_LAUNCH_CHECK("bias_planes_kernel");
    }
    if (side) {
        TRI_CUDA_CHECK(cudaEventRecord(side->join0, side->stream));
        TRI_CUDA_CHECK(cudaStreamWaitEvent(st, side->join0, 0));
    }
    float* NL = (float*)((char*)ws + w.nl_off);
    float* ND = (float*)((char*)ws + w.nd_off);
    if ((s = sm100_lse_prep(p, LSE, Dws, NL, ND, st)) != TRI_OK) return s;
    // Stage 2 (dQ + dBias, one recomputation of P / dS) runs as clusters and leaves some SMs empty (132 of 148 at N = 768:
    // cudaOccupancyMaxActiveClusters).  Stage 1 (dK, dV) is independent of it, so a first slice of stage 1's work items runs
    // on those SMs at the same time on the side stream; the rest of stage 1 follows on all SMs.
    float* planes = (float*)((char*)ws + w.planes_off);
    int Gs = 1, C2 = 0, grid2 = 0;
    const int npass = sm100_dqdb_passes(p.N);
    float* dq_part = (float*)((char*)ws + w.dqpart_off);
    const DqdbPass pass0 = sm100_dqdb_pass(p.N, 0, dq_part);
    if (!sm100_dqdb_plan(p, pass0.tiles, 0, &C2, &Gs, &grid2))
        return cuda_fail(cudaErrorLaunchFailure, "sm100_dqdb_plan: no resident cluster of the needed size");
    const long long items1 = sm100_dkdv2_items(p);
    const int sms = sm100_sm_count();
    const int spare = sms - grid2;
    long long itemsA = 0;
    if (side && spare >= 4 && items1 > 4 * sms) {
        // the spare SMs work for about the duration of stage 2, which is ~1.4x stage 1's on the whole chip
        itemsA = (long long)((double)items1 * spare / sms * 1.4);
    }
    const bool reduce = Gs > 1 || accumulate_dbias;
    if (itemsA > 0) {
        TRI_CUDA_CHECK(cudaEventRecord(side->fork, st));
        TRI_CUDA_CHECK(cudaStreamWaitEvent(side->stream, side->fork, 0));
    }
    float* dbias_out = accumulate_dbias ? planes : dBias;
    if ((s = sm100_dqdb_launch(p, C2, Gs, grid2, Q, dA, K, V, biasL, maskbits, LSE, Dws, dQ, dbias_out, planes, pass0, st)) != TRI_OK) return s;
    for (int i = 1; i < npass; ++i) {  // N > 2048: the further slices of the key axis, same row split
        const DqdbPass ps = sm100_dqdb_pass(p.N, i, dq_part);
        int Ci = 0, Gi = 0, gridi = 0;
        if (!sm100_dqdb_plan(p, ps.tiles, Gs, &Ci, &Gi, &gridi) || Gi != Gs)
            return cuda_fail(cudaErrorLaunchFailure, "sm100_dqdb_plan: no resident cluster of the needed size");
        if ((s = sm100_dqdb_launch(p, Ci, Gs, gridi, Q, dA, K, V, biasL, maskbits, LSE, Dws, dQ, dbias_out, planes, ps, st)) != TRI_OK) return s;
    }
    if (itemsA > 0) {
        if ((s = sm100_dkdv2_launch(p, Q, dA, K, V, bias_kq, maskbits, NL, ND, dK, dV, 0, itemsA, spare, "sm100_dkdv_kernel(side)",
                                    side->stream)) != TRI_OK)
            return s;
    }
    if (reduce) {
        // level 2 of the dBias reduction needs stage 2 only.  On a high-priority stream its (small, memory-bound) blocks
        // take the SMs that stage 2 frees ahead of the persistent CTAs of the rest of stage 1, and finish beside them;
        // enqueued behind stage 1 they would wait for its last CTA.
        cudaStream_t sr = side ? side->hi : st;
        if (side) {
            TRI_CUDA_CHECK(cudaEventRecord(side->stage2, st));
            TRI_CUDA_CHECK(cudaStreamWaitEvent(side->hi, side->stage2, 0));
        }
        {
            ProfScope ps("sm100_dbias_reduce_kernel", sr);
            sm100_dbias_reduce_kernel<<<dim3((p.N + 31) / 32, (p.N + 31) / 32, p.B * p.H), 256, 0, sr>>>(
                planes, dBias, p.B * p.H, p.N, Gs, p.variant == TRI_ENDING ? 1 : 0, accumulate_dbias ? 1 : 0);
        }
        TRI_LAUNCH_CHECK("sm100_dbias_reduce_kernel");
        if (side) TRI_CUDA_CHECK(cudaEventRecord(side->join2, side->hi));
    }
    if ((s = sm100_dkdv2_launch(p, Q, dA, K, V, bias_kq, maskbits, NL, ND, dK, dV, itemsA, items1 - itemsA, sms, "sm100_dkdv_kernel", st)) !=
        TRI_OK)
        return s;
    if (itemsA > 0) {
        TRI_CUDA_CHECK(cudaEventRecord(side->join, side->stream));
        TRI_CUDA_CHECK(cudaStreamWaitEvent(st, side->join, 0));
    }
    if (side && reduce) TRI_CUDA_CHECK(cudaStreamWaitEvent(st, side->join2, 0));
    return TRI_OK;
}

}  // namespace tri

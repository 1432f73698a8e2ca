// tri_attn_bias_all_gather / tri_attn_dbias_reduce_scatter: the two exchanges of EvoSP-3D's bias over peer memory.
// The all-gather is a pull: every rank copies the N / P query lines of each peer's shard into its own full bias.
// The reduce-scatter of dBias as ONE kernel
// over peer memory.  Each rank of the SP group holds a partial dBias [B,H,N,N] fp32 (the sum over its own broadcast rows, written
// by tri_attn_rows_bwd); rank r needs the query lines [r n, (r+1) n), n = N / P, summed over all ranks.  The kernel reads
// those lines straight out of every peer's buffer (NVLink / NVSwitch P2P loads of 16 bytes, coalesced) and adds them in
// ascending rank order -- a fixed order, so the result is bitwise reproducible and the same on every run, which NCCL's
// reduce-scatter does not promise across algorithms.  No staging copy, no second pass: reduction and exchange are one launch.
//
// Synchronisation is the caller's (evosp.py does it with the symmetric-memory handle's barrier on the stream): every peer's
// tri_attn_rows_bwd must have completed before the launch, and no peer may overwrite its buffer before all ranks have read it.
#include <cstdint>

#include "tri_common.cuh"

namespace {
constexpr int kMaxPeers = 16;
struct PeerPtrs { const float* p[kMaxPeers]; };

__global__ void __launch_bounds__(256) dbias_reduce_scatter_kernel(PeerPtrs peers, int P, int rank, float* __restrict__ out, int BH,
                                                                   int N, int n) {
    const long long total4 = (long long)BH * n * (N / 4);
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < total4; i += (long long)gridDim.x * blockDim.x) {
        const int k4 = (int)(i % (N / 4));
        const long long t = i / (N / 4);
        const int l = (int)(t % n);
        const long long bh = t / n;
        const long long src = ((bh * N + (long long)rank * n + l) * N) / 4 + k4;
        float4 acc = __ldg((const float4*)peers.p[0] + src);
        for (int q = 1; q < P; ++q) {
            const float4 v = __ldg((const float4*)peers.p[q] + src);
            acc.x += v.x; acc.y += v.y; acc.z += v.z; acc.w += v.w;
        }
        ((float4*)out)[i] = acc;
    }
}

// all-gather of the bias by pulling: out[bh][p n + l][:] = peer p's shard [bh][l][:]; 16 bytes per thread, the row of N
// elements (es bytes each) is a whole number of 16-byte chunks
__global__ void __launch_bounds__(256) bias_all_gather_kernel(PeerPtrs peers, int P, uint4* __restrict__ out, int BH, int N, int n,
                                                              int row16) {
    const long long total = (long long)BH * N * row16;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
        const int c = (int)(i % row16);
        const long long t = i / row16;
        const int line = (int)(t % N);
        const long long bh = t / N;
        const int q = line / n, l = line - q * n;
        out[i] = __ldg((const uint4*)peers.p[q] + (bh * n + l) * row16 + c);
    }
}
}  // namespace

extern "C" tri_status tri_attn_bias_all_gather(const void* const* peer_shards, int P, void* out_bias, int B, int H, int N,
                                               tri_dtype dtype, void* cuda_stream) {
    if (!peer_shards || !out_bias || P <= 0 || B <= 0 || H <= 0 || N <= 0 || (dtype != TRI_F32 && dtype != TRI_BF16))
        return TRI_ERR_INVALID_ARG;
    const int es = dtype == TRI_F32 ? 4 : 2;
    if (P > kMaxPeers || N % P != 0 || ((long long)N * es) % 16 != 0) return TRI_ERR_UNSUPPORTED;
    PeerPtrs pp;
    for (int q = 0; q < kMaxPeers; ++q) pp.p[q] = nullptr;
    for (int q = 0; q < P; ++q) {
        if (!peer_shards[q] || ((uintptr_t)peer_shards[q] & 15)) return TRI_ERR_INVALID_ARG;
        pp.p[q] = (const float*)peer_shards[q];
    }
    if ((uintptr_t)out_bias & 15) return TRI_ERR_INVALID_ARG;
    const int row16 = N * es / 16;
    const long long total = (long long)B * H * N * row16;
    const int sms = ::tri::sm100_sm_count();
    const long long want = (total + 255) / 256;
    const int grid = (int)(want < (long long)sms * 8 ? want : (long long)sms * 8);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    {
        ::tri::ProfScope ps("bias_all_gather_kernel", st);
        bias_all_gather_kernel<<<grid, 256, 0, st>>>(pp, P, (uint4*)out_bias, B * H, N, N / P, row16);
    }
    TRI_LAUNCH_CHECK("bias_all_gather_kernel");
    return TRI_OK;
}

extern "C" tri_status tri_attn_dbias_reduce_scatter(const float* const* peer_dbias, int P, int rank, float* out_shard, int B, int H,
                                                    int N, void* cuda_stream) {
    if (!peer_dbias || !out_shard || P <= 0 || rank < 0 || rank >= P || B <= 0 || H <= 0 || N <= 0) return TRI_ERR_INVALID_ARG;
    if (P > kMaxPeers || N % P != 0 || N % 4 != 0) return TRI_ERR_UNSUPPORTED;
    PeerPtrs pp;
    for (int q = 0; q < kMaxPeers; ++q) pp.p[q] = nullptr;
    for (int q = 0; q < P; ++q) {
        if (!peer_dbias[q] || ((uintptr_t)peer_dbias[q] & 15)) return TRI_ERR_INVALID_ARG;
        pp.p[q] = peer_dbias[q];
    }
    if ((uintptr_t)out_shard & 15) return TRI_ERR_INVALID_ARG;
    const int n = N / P;
    const long long total4 = (long long)B * H * n * (N / 4);
    const int sms = ::tri::sm100_sm_count();
    const long long want = (total4 + 255) / 256;
    const int grid = (int)(want < (long long)sms * 8 ? want : (long long)sms * 8);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    {
        ::tri::ProfScope ps("dbias_reduce_scatter_kernel", st);
        dbias_reduce_scatter_kernel<<<grid, 256, 0, st>>>(pp, P, rank, out_shard, B * H, N, n);
    }
    TRI_LAUNCH_CHECK("dbias_reduce_scatter_kernel");
    return TRI_OK;
}

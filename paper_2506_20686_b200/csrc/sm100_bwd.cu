// bf16 backward on tcgen05 / TMEM / TMA (sm_100a).  Listing 2, Table I, gate from the task
// statement.  P is recomputed from the saved LSE; nothing of size N^3 is stored.
//
//   pre      D = rowsum(dO . O), dG = dO . O . (1 - sigmoid G), dA = dO . sigmoid G (bf16, workspace)
//   dkdv     key-stationary (thread = key): S^T = K Q^T, dP^T = V dA^T (SS), P^T, dS^T -> bf16 -> TMEM,
//            dV += P^T dA, dK += dS^T Q (TS, B operand MN-major)
//   dqdb     (sm100_dqdb.cu) dQ and dBias from one recomputation, tile-stationary, cluster reduce of dQ
//   reduce   level 2 of the dBias reduction: adds the row-split partial planes in ascending order
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

// p = exp(x - LSE), ds = p (dp - D) for 32 score columns held as raw TMEM words.
//   sraw / dpraw : fp32 bit patterns of S and dP;  bw[16] : 32 bf16 bias values;  nl[c], dd[c] : -LSE*log2e and D of
//   the column (dkdv: per query column)  or scalars broadcast by the caller (dq / dbias).

// ------------------------------------------------------------------------------------------------------------
// dkdv: CTA = (b, row pair, h, 128-key block); loop over 64-query tiles (outer) and the R_ rows (inner).
// ------------------------------------------------------------------------------------------------------------
template <int R_>
struct DkdvSmem {
    static constexpr int kv_off = 0;                          // R_ x (K, V) 128x32
    static constexpr int qa_off = kv_off + R_ * 2 * T128;     // 2 stages x (Q, dA) 64x32
    static constexpr int bias_off = qa_off + 2 * 2 * T64;     // [128 k][64 q] bf16, SWIZZLE_128B
    static constexpr int ld_off = bias_off + 2 * 16384;       // (bias double buffered) ; 2 stages x (nl[64], D[64]) floats
    static constexpr int bar_off = ld_off + 2 * 128 * 4;
    static constexpr int total = bar_off + 64 + 1024;
};

template <int R_>
__global__ void __launch_bounds__(256, 2) sm100_dkdv_kernel(const __grid_constant__ CUtensorMap tmQ64,
                                                         const __grid_constant__ CUtensorMap tmA64,
                                                         const __grid_constant__ CUtensorMap tmK128,
                                                         const __grid_constant__ CUtensorMap tmV128,
                                                         const __grid_constant__ CUtensorMap tmBiasKQ, Problem p,
                                                         const unsigned char* __restrict__ mask,
                                                         const float* __restrict__ LSE, const float* __restrict__ Dws,
                                                         __nv_bfloat16* __restrict__ dK, __nv_bfloat16* __restrict__ dV) {
    using L = DkdvSmem<R_>;
    constexpr int TCOLS = (128 + 64 * R_) <= 256 ? 256 : 512;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    uint8_t* sKV = smem + L::kv_off;
    uint8_t* sQA = smem + L::qa_off;
    uint8_t* sBias = smem + L::bias_off;
    float* sLD = (float*)(smem + L::ld_off);
    uint64_t* bars = (uint64_t*)(smem + L::bar_off);
    uint64_t* bar_kv = bars + 0;
    uint64_t* bar_qa = bars + 1;  // [2]
    uint64_t* bar_bias = bars + 5;  // [2]
    uint64_t* bar_mma = bars + 4;
    uint32_t* tmem_slot = (uint32_t*)(bars + 7);

    // 256 threads: a key row (TMEM lane) is shared by two threads, warps w and w+4, 32 query columns each
    const int tid = threadIdx.x, warp = tid >> 5, chalf = warp >> 2;
    const int row = (warp & 3) * 32 + (tid & 31);
    const int NKB = p.N / 128, NQT = p.N / 64, NG = p.N / R_;
    int idx = blockIdx.x;
    const int kb = idx % NKB; idx /= NKB;
    const int h = idx % p.H; idx /= p.H;
    const int g = idx % NG;
    const int b = idx / NG;
    const int r0 = g * R_, k0 = kb * 128, bh = b * p.H + h;

    if (tid == 0) {
        prefetch_tmap(&tmQ64); prefetch_tmap(&tmA64); prefetch_tmap(&tmK128); prefetch_tmap(&tmV128); prefetch_tmap(&tmBiasKQ);
        mbar_init(bar_kv, 1); mbar_init(bar_qa, 1); mbar_init(bar_qa + 1, 1); mbar_init(bar_bias, 1); mbar_init(bar_bias + 1, 1);
        mbar_init(bar_mma, 1);
        fence_barrier_init();
    }
    if (warp == 0) tmem_alloc<TCOLS>(tmem_slot);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    const uint32_t lane_off = (uint32_t)((warp & 3) * 32) << 16;
    const uint32_t tS = tmem, tDP = tmem + 64;
    const int T = NQT * R_;

    auto load_qa = [&](int t) {
        const int qt = t / R_, r = t % R_, st = t & 1;
        mbar_expect_tx(bar_qa + st, 2 * T64);
        tma_load_5d(sQA + st * 2 * T64, &tmQ64, bar_qa + st, 0, qt * 64, r0 + r, h, b);
        tma_load_5d(sQA + st * 2 * T64 + T64, &tmA64, bar_qa + st, 0, qt * 64, r0 + r, h, b);
    };
    if (tid == 0) {
        mbar_expect_tx(bar_kv, R_ * 2 * T128);
        for (int r = 0; r < R_; ++r) {
            tma_load_5d(sKV + r * 2 * T128, &tmK128, bar_kv, 0, k0, r0 + r, h, b);
            tma_load_5d(sKV + r * 2 * T128 + T128, &tmV128, bar_kv, 0, k0, r0 + r, h, b);
        }
        load_qa(0);
        mbar_expect_tx(bar_bias, 16384);
        tma_load_3d(sBias, &tmBiasKQ, bar_bias, 0, k0, bh);
        if (NQT > 1) {
            mbar_expect_tx(bar_bias + 1, 16384);
            tma_load_3d(sBias + 16384, &tmBiasKQ, bar_bias + 1, 64, k0, bh);
        }
    }
    // per-tile LSE / D of the 64 query columns: threads 0..63 fetch LSE, 64..127 fetch D
    auto ld_val = [&](int t) -> float {
        const int qt = t / R_, r = t % R_, q = qt * 64 + (tid & 63);
        const long long o = (long long)b * p.N * p.H * p.N + (long long)h * p.N + (long long)(r0 + r) * p.lR + (long long)q * p.lQ;
        if (tid < 64) {
            const float l = __ldg(LSE + o);
            return l == -INFINITY ? -INFINITY : -l * kLog2e;
        }
        return -__ldg(Dws + o);
    };
    if (tid < 128) sLD[tid] = ld_val(0);
    bool keep[R_];
#pragma unroll
    for (int r = 0; r < R_; ++r)
        keep[r] = !mask || mask[(long long)b * p.N * p.N + (long long)(r0 + r) * p.mR + (long long)(k0 + row) * p.mK];
    __syncthreads();

    constexpr uint32_t idescS = make_idesc(128, 64, false, false);
    constexpr uint32_t idescO = make_idesc(128, DH, false, true);
    const float scale = rsqrtf((float)DH);
    const uint64_t scale2 = pack2(scale, scale), l2e2 = pack2(kLog2e, kLog2e);

    for (int qt = 0; qt < NQT; ++qt) {
#pragma unroll
        for (int r = 0; r < R_; ++r) {
            const int t = qt * R_ + r, st = t & 1;
            if (warp == 0) {  // warp-uniform so the descriptors stay in uniform registers; one elected lane issues
                if (t == 0) mbar_wait(bar_kv, 0);
                mbar_wait(bar_qa + st, (t >> 1) & 1);
                tc_fence_after();
                const uint64_t dk = make_desc_sw64(smem_u32(sKV + r * 2 * T128));
                const uint64_t dv = make_desc_sw64(smem_u32(sKV + r * 2 * T128 + T128));
                const uint64_t dq = make_desc_sw64(smem_u32(sQA + st * 2 * T64));
                const uint64_t da = make_desc_sw64(smem_u32(sQA + st * 2 * T64 + T64));
                if (elect_one()) {
                    mma_ss(tS, dk, dq, idescS, 0);
                    mma_ss(tS, dk + 2, dq + 2, idescS, 1);
                    mma_ss(tDP, dv, da, idescS, 0);
                    mma_ss(tDP, dv + 2, da + 2, idescS, 1);
                    mma_commit(bar_mma);
                }
                __syncwarp();
            }
            float ldnext = 0.0f;
            if (t + 1 < T && tid < 128) ldnext = ld_val(t + 1);
            mbar_wait(bar_mma, t & 1);
            tc_fence_after();
            if (tid == 32 && t + 1 < T) load_qa(t + 1);  // warp 1 issues the TMA loads, warp 0 the MMAs
            if (r == 0) mbar_wait(bar_bias + (qt & 1), (qt >> 1) & 1);
            const uint8_t* sB = sBias + (qt & 1) * 16384;
            const float* nlq = sLD + st * 128;
            const float* ddq = nlq + 64;
            {
                const int c32 = chalf;
                uint32_t sraw[32], dpraw[32];
                tmem_ld32(tS + lane_off + c32 * 32, sraw);
                tmem_ld32(tDP + lane_off + c32 * 32, dpraw);
                uint4 bv[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) bv[j] = lds128(sB + row * 128 + (((c32 * 4 + j) ^ (row & 7)) << 4));
                tmem_ld_wait();
                uint32_t pp[16], ds[16];
                if (keep[r]) {
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        const uint32_t w[4] = {bv[j].x, bv[j].y, bv[j].z, bv[j].w};
                        const float4 n0 = lds128f(nlq + c32 * 32 + j * 8), n1 = lds128f(nlq + c32 * 32 + j * 8 + 4);
                        const float4 d0 = lds128f(ddq + c32 * 32 + j * 8), d1 = lds128f(ddq + c32 * 32 + j * 8 + 4);
                        const uint64_t nn[4] = {pack2(n0.x, n0.y), pack2(n0.z, n0.w), pack2(n1.x, n1.y), pack2(n1.z, n1.w)};
                        const uint64_t dn[4] = {pack2(d0.x, d0.y), pack2(d0.z, d0.w), pack2(d1.x, d1.y), pack2(d1.z, d1.w)};
#pragma unroll
                        for (int e = 0; e < 4; ++e) {
                            const int c = j * 8 + e * 2;
                            const uint64_t x2 = fma2(pack2(__uint_as_float(sraw[c]), __uint_as_float(sraw[c + 1])), scale2,
                                                     pack2(bf16_lo(w[e]), bf16_hi(w[e])));
                            float a0, a1, s0, s1;
                            unpack2(fma2(x2, l2e2, nn[e]), a0, a1);
                            const float p0 = ex2(a0), p1 = ex2(a1);
                            // sLD holds -D: ds = p * (dp - D)
                            unpack2(mul2(pack2(p0, p1), add2(pack2(__uint_as_float(dpraw[c]), __uint_as_float(dpraw[c + 1])), dn[e])), s0, s1);
                            pp[j * 4 + e] = pack_bf16(p0, p1);
                            ds[j * 4 + e] = pack_bf16(s0, s1);
                        }
                    }
                } else {  // masked key: its whole row of P^T and dS^T is zero
#pragma unroll
                    for (int e = 0; e < 16; ++e) { pp[e] = 0u; ds[e] = 0u; }
                }
                tmem_st16(tS + lane_off + c32 * 32, pp);   // packed into my own fp32 columns [32*c32, +16)
                tmem_st16(tDP + lane_off + c32 * 32, ds);
            }
            if (t + 1 < T && tid < 128) sLD[((t + 1) & 1) * 128 + tid] = ldnext;
            tmem_st_wait();
            tc_fence_before();
            __syncthreads();
            if (warp == 0) {
                tc_fence_after();
                const uint64_t dq = make_desc_sw64(smem_u32(sQA + st * 2 * T64));
                const uint64_t da = make_desc_sw64(smem_u32(sQA + st * 2 * T64 + T64));
                const uint32_t tdV = tmem + 128 + r * 64, tdK = tdV + 32;
                if (elect_one()) {
#pragma unroll
                    for (int ks = 0; ks < 4; ++ks)  // A columns: k-steps 0,1 at [0,16), k-steps 2,3 at [32,48)
                        mma_ts(tdV, tS + (ks >> 1) * 32 + (ks & 1) * 8, da + (uint64_t)ks * 64, idescO, (qt > 0 || ks > 0) ? 1u : 0u);
#pragma unroll
                    for (int ks = 0; ks < 4; ++ks)
                        mma_ts(tdK, tDP + (ks >> 1) * 32 + (ks & 1) * 8, dq + (uint64_t)ks * 64, idescO, (qt > 0 || ks > 0) ? 1u : 0u);
                    if (r == R_ - 1 && qt + 2 < NQT) {  // every thread is past its reads of buffer qt&1: refill it with qt+2
                        mbar_expect_tx(bar_bias + (qt & 1), 16384);
                        tma_load_3d(sBias + (qt & 1) * 16384, &tmBiasKQ, bar_bias + (qt & 1), (qt + 2) * 64, k0, bh);
                    }
                }
                __syncwarp();
            }
        }
    }
    if (tid == 0) mma_commit(bar_mma);
    mbar_wait(bar_mma, T & 1);
    tc_fence_after();
#pragma unroll
    for (int r = 0; r < R_; ++r) {  // warps 0-3 write dV_r, warps 4-7 write dK_r (scaled)
        uint32_t v[32];
        tmem_ld32(tmem + lane_off + 128 + r * 64 + chalf * 32, v);
        tmem_ld_wait();
        const long long off = (long long)b * p.sB + (long long)h * p.sH + (long long)(r0 + r) * p.sSlice + (long long)(k0 + row) * p.sPos;
        uint4* po = (uint4*)((chalf ? dK : dV) + off);
        const float sc = chalf ? scale : 1.0f;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            uint32_t a[4];
#pragma unroll
            for (int e = 0; e < 4; ++e)
                a[e] = pack_bf16(__uint_as_float(v[j * 8 + 2 * e]) * sc, __uint_as_float(v[j * 8 + 2 * e + 1]) * sc);
            po[j] = make_uint4(a[0], a[1], a[2], a[3]);
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc<TCOLS>(tmem);
}


// level 2 of the dBias reduction (only when the row axis was split): dBias[bh][q*bQ + k*bK] = sum over planes, in
// ascending order, of plane[g][bh][q][k]; the ending-node variant wants the transpose (bQ = 1), via a 32x32 smem tile.
__global__ void __launch_bounds__(256) sm100_dbias_reduce_kernel(const float* __restrict__ planes, float* __restrict__ dBias,
                                                                 int BH, int N, int G, int transpose) {
    __shared__ float tile[32][33];
    const int bh = blockIdx.z, q0 = blockIdx.y * 32, k0 = blockIdx.x * 32;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    const long long pstride = (long long)BH * N * N;
    for (int j = ty; j < 32; j += 8) {
        const long long o = (long long)bh * N * N + (long long)(q0 + j) * N + k0 + tx;
        float acc = planes[o];
        for (int g = 1; g < G; ++g) acc += planes[o + g * pstride];
        if (transpose) tile[j][tx] = acc; else dBias[o] = acc;
    }
    if (transpose) {
        __syncthreads();
        for (int j = ty; j < 32; j += 8) dBias[(long long)bh * N * N + (long long)(k0 + j) * N + q0 + tx] = tile[tx][j];
    }
}

}  // namespace

// ---- host side ------------------------------------------------------------------------------------------------
namespace {
struct BwdWs {
    size_t d_off, da_off, biast_off, biasl_off, mask_off, planes_off, total;
};
BwdWs bwd_ws_layout(const Problem& p) {
    BwdWs w;
    size_t o = 0;
    w.d_off = o; o += align_up((size_t)p.B * p.N * p.H * p.N * sizeof(float), 256);          // D = rowsum(dO . O)
    w.da_off = o; o += align_up((size_t)p.B * p.N * p.H * p.N * p.d * 2, 256);               // dA = dO . sigmoid(G)
    w.biast_off = o; o += align_up((size_t)p.B * p.H * p.N * p.N * 2, 256);                  // bias^T, bf16 (dkdv)
    w.biasl_off = o; o += align_up((size_t)p.B * p.H * p.N * p.N * 4, 256);                  // log2e * bias[q][k], fp32 (dqdb)
    w.mask_off = o; o += sm100_maskbits_bytes(p);
    // partial dBias planes: the fused kernel picks its row split (<= kDqdbMaxSplit) at launch from the device's
    // resident cluster count, so the workspace always holds the maximum
    w.planes_off = o; o += align_up((size_t)kDqdbMaxSplit * p.B * p.H * p.N * p.N * sizeof(float), 256);
    w.total = o;
    return w;
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
                     void* dV, void* dG, float* dBias, void* ws, cudaStream_t st) {
    constexpr int RKV = 2;
    const BwdWs w = bwd_ws_layout(p);
    float* Dws = (float*)((char*)ws + w.d_off);
    void* dA = (char*)ws + w.da_off;
    void* biasT = (char*)ws + w.biast_off;
    const long long rows = (long long)p.B * p.N * p.H * p.N;
    {
        ProfScope ps("sm100_bwd_pre_kernel", st);
        sm100_bwd_pre_kernel<<<(unsigned)((rows * 4 + 255) / 256), 256, 0, st>>>(rows, (const uint4*)dO, (const uint4*)O,
                                                                               (const uint4*)G, (uint4*)dG, (uint4*)dA, Dws);
    }
    TRI_LAUNCH_CHECK("sm100_bwd_pre_kernel");
    tri_status s = sm100_transpose_planes(bias, biasT, p.B * p.H, p.N, st);
    if (s != TRI_OK) return s;
    TRI_LAUNCH_CHECK("sm100_transpose_bf16");
    const void* bias_kq = p.variant == TRI_STARTING ? biasT : bias;  // [k][q]

    CUtensorMap tQ64, tA64, tK128, tV128, tBkq;
    bool ok = make_tmap_u(&tQ64, Q, p.B, p.N, p.H, p.d, p.variant, 64) && make_tmap_u(&tA64, dA, p.B, p.N, p.H, p.d, p.variant, 64) &&
              make_tmap_u(&tK128, K, p.B, p.N, p.H, p.d, p.variant, 128) && make_tmap_u(&tV128, V, p.B, p.N, p.H, p.d, p.variant, 128) &&
              make_tmap_plane(&tBkq, bias_kq, p.B * p.H, p.N, 128);
    if (!ok) return cuda_fail(cudaErrorUnknown, "cuTensorMapEncodeTiled");

    // the opt-in shared-memory size is a per-device function attribute: set it on every launch (cheap, thread-safe)
    if ((s = set_smem(sm100_dkdv_kernel<RKV>, DkdvSmem<RKV>::total)) != TRI_OK) return s;
    {
        ProfScope ps("sm100_dkdv_kernel", st);
        const unsigned grid = (unsigned)((long long)p.B * (p.N / RKV) * p.H * (p.N / 128));
        sm100_dkdv_kernel<RKV><<<grid, 256, DkdvSmem<RKV>::total, st>>>(tQ64, tA64, tK128, tV128, tBkq, p, mask, LSE, Dws,
                                                                       (__nv_bfloat16*)dK, (__nv_bfloat16*)dV);
    }
    TRI_LAUNCH_CHECK("sm100_dkdv_kernel");
    // stage 2, fused: dQ and dBias from one recomputation of P / dS (cluster over the key tiles of a query block)
    float* planes = (float*)((char*)ws + w.planes_off);
    int Gs = 1, C2 = 0, grid2 = 0;
    if (!sm100_dqdb_plan(p, &C2, &Gs, &grid2)) return cuda_fail(cudaErrorLaunchFailure, "sm100_dqdb_plan: no resident cluster of the needed size");
    unsigned long long* maskbits = nullptr;
    if (mask) {
        maskbits = (unsigned long long*)((char*)ws + w.mask_off);
        if ((s = sm100_pack_mask(p, mask, maskbits, st)) != TRI_OK) return s;
        TRI_LAUNCH_CHECK("pack_mask_kernel");
    }
    float* biasL = (float*)((char*)ws + w.biasl_off);
    {
        const bool tr = p.variant == TRI_ENDING;
        if ((s = sm100_bias_planes(bias, tr ? nullptr : biasL, tr ? biasL : nullptr, p.B * p.H, p.N, kLog2e, st)) != TRI_OK) return s;
        TRI_LAUNCH_CHECK("bias_planes_kernel");
    }
    if ((s = sm100_dqdb_launch(p, C2, Gs, grid2, Q, dA, K, V, biasL, maskbits, LSE, Dws, dQ, dBias, planes, st)) != TRI_OK) return s;
    if (Gs > 1) {
        {
            ProfScope ps("sm100_dbias_reduce_kernel", st);
            sm100_dbias_reduce_kernel<<<dim3(p.N / 32, p.N / 32, p.B * p.H), 256, 0, st>>>(
                planes, dBias, p.B * p.H, p.N, Gs, p.variant == TRI_ENDING ? 1 : 0);
        }
        TRI_LAUNCH_CHECK("sm100_dbias_reduce_kernel");
    }
    return TRI_OK;
}

}  // namespace tri

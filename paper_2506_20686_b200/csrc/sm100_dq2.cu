// dQ, software-pipelined (sm_100a): one CTA per SM = two independent "slots" of 256 threads that share the bias tile.
//
// The CTA owns a 128-query block of 4 broadcast rows of one (b,h); slot s takes rows 2s, 2s+1 and 224 TMEM columns:
//     [0,64)    S  = Q_r K^T        (tcgen05.mma SS, M=128 N=64 K=2x16)
//     [64,128)  dP = dA_r V^T       (SS)
//     [128,160) dS = P*(dP - D) as bf16 pairs (NOT aliased on dP), A operand of
//     [160,224) dQ_r += dS K        (TS, N=32, K=4x16), one 32-column accumulator per row
// Listing 2's stage 2 is serial per tile; here a tile's S/dP leave TMEM for registers first, the slot
// meets at a named barrier, and its thread 0 immediately issues S/dP of the NEXT tile, so the tensor pipe and the
// mbarrier round trip run under the exponentials of the current tile.  K/V tiles ride a 4-stage TMA ring per slot.
// A query row (TMEM lane) is shared by two threads (warps w and w+4 of the slot), 32 key columns each.
#include "sm100_common.cuh"
#include "tri_common.cuh"

namespace tri {
using namespace sm100;

namespace {

constexpr int DH = 32;
constexpr int T128 = 128 * DH * 2;  // 8 KB
constexpr int T64 = 64 * DH * 2;    // 4 KB
constexpr int RS = 2, RT = 4;       // rows per slot / per CTA
constexpr int NST = 4;              // K/V ring depth per slot

struct Dq2Smem {
    static constexpr int qa_off = 0;                            // RT x (Q, dA) 128x32
    static constexpr int kv_off = qa_off + RT * 2 * T128;       // [slot][NST] x (K, V) 64x32
    static constexpr int bias_off = kv_off + 2 * NST * 2 * T64; // [2 buffers] [128 q][64 k] bf16, SWIZZLE_128B
    static constexpr int mask_off = bias_off + 2 * 16384;       // [slot][2] x 64 floats
    static constexpr int bar_off = mask_off + 2 * 2 * 64 * 4;
    static constexpr int total = bar_off + 256 + 1024;
};
enum { D_QA = 0 /*[slot]*/, D_KV = 2 /*[slot][NST]*/, D_BIAS_FULL = 10 /*[2]*/, D_BIAS_EMPTY = 12 /*[2]*/, D_MMA = 14 /*[slot]*/,
       D_TS = 16 /*[slot]*/, D_COUNT = 18 };

__global__ void __launch_bounds__(512, 1) sm100_dq2_kernel(const __grid_constant__ CUtensorMap tmQ128,
                                                           const __grid_constant__ CUtensorMap tmA128,
                                                           const __grid_constant__ CUtensorMap tmK64,
                                                           const __grid_constant__ CUtensorMap tmV64,
                                                           const __grid_constant__ CUtensorMap tmBiasQK, Problem p,
                                                           const unsigned char* __restrict__ mask,
                                                           const float* __restrict__ LSE, const float* __restrict__ Dws,
                                                           __nv_bfloat16* __restrict__ dQ) {
    using L = Dq2Smem;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    uint8_t* sQA = smem + L::qa_off;
    uint8_t* sBias = smem + L::bias_off;
    uint64_t* bars = (uint64_t*)(smem + L::bar_off);
    uint32_t* tmem_slot = (uint32_t*)(bars + D_COUNT);

    const int tid = threadIdx.x, warp = tid >> 5;
    const int slot = warp >> 3, chalf = (warp >> 2) & 1;
    const int row = (warp & 3) * 32 + (tid & 31);
    const int stid = tid & 255;  // thread index inside the slot
    const int swarp = warp & 7;   // warp index inside the slot (warp 0 also issues the slot's MMAs)
    const int bar_id = 1 + slot;
    const int NQB = p.N / 128, NKT = p.N / 64, NG = p.N / RT;
    int idx = blockIdx.x;
    const int qb = idx % NQB; idx /= NQB;
    const int h = idx % p.H; idx /= p.H;
    const int g = idx % NG;
    const int b = idx / NG;
    const int r0 = g * RT + slot * RS, q0 = qb * 128, bh = b * p.H + h;
    const int T = NKT * RS;  // tiles of this slot: key tile kt OUTER, row r INNER

    uint8_t* sKV = smem + L::kv_off + slot * NST * 2 * T64;
    float* sMask = (float*)(smem + L::mask_off) + slot * 2 * 64;
    uint64_t* bar_qa = bars + D_QA + slot;
    uint64_t* bar_kv = bars + D_KV + slot * NST;
    uint64_t* bar_mma = bars + D_MMA + slot;  // S, dP of a tile ready
    uint64_t* bar_ts = bars + D_TS + slot;    // dQ += dS K of a tile done: dS buffer and the tile's K/V ring slot are free

    if (tid == 0) {
        prefetch_tmap(&tmQ128); prefetch_tmap(&tmA128); prefetch_tmap(&tmK64); prefetch_tmap(&tmV64); prefetch_tmap(&tmBiasQK);
        for (int i = 0; i < D_COUNT; ++i) mbar_init(bars + i, (i >= D_BIAS_EMPTY && i < D_MMA) ? 2 : 1);
        fence_barrier_init();
    }
    if (warp == 0) tmem_alloc<512>(tmem_slot);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot + slot * 256;
    const uint32_t lane_off = (uint32_t)((warp & 3) * 32) << 16;
    const uint32_t tS = tmem, tDP = tmem + 64, tDS = tmem + 128, tDQ = tmem + 160;

    auto load_kv = [&](int t) {
        const int kt = t / RS, r = t % RS, st = t % NST;
        mbar_expect_tx(bar_kv + st, 2 * T64);
        tma_load_5d(sKV + st * 2 * T64, &tmK64, bar_kv + st, 0, kt * 64, r0 + r, h, b);
        tma_load_5d(sKV + st * 2 * T64 + T64, &tmV64, bar_kv + st, 0, kt * 64, r0 + r, h, b);
    };
    auto load_bias = [&](int kt) {
        mbar_expect_tx(bars + D_BIAS_FULL + (kt & 1), 16384);
        tma_load_3d(sBias + (kt & 1) * 16384, &tmBiasQK, bars + D_BIAS_FULL + (kt & 1), kt * 64, q0, bh);
    };
    constexpr uint32_t idescS = make_idesc(128, 64, false, false);
    constexpr uint32_t idescO = make_idesc(128, DH, false, true);
    auto issue_ss = [&](int t) {  // S, dP of tile t: called by the whole first warp of the slot (warp-uniform)
        const int r = t % RS, st = t % NST;
        mbar_wait(bar_kv + st, (t / NST) & 1);
        tc_fence_after();
        const uint64_t dq = make_desc_sw64(smem_u32(sQA + (slot * RS + r) * 2 * T128));
        const uint64_t da = make_desc_sw64(smem_u32(sQA + (slot * RS + r) * 2 * T128 + T128));
        const uint64_t dk = make_desc_sw64(smem_u32(sKV + st * 2 * T64));
        const uint64_t dv = make_desc_sw64(smem_u32(sKV + st * 2 * T64 + T64));
        if (elect_one()) {
            mma_ss(tS, dq, dk, idescS, 0);
            mma_ss(tS, dq + 2, dk + 2, idescS, 1);
            mma_ss(tDP, da, dv, idescS, 0);
            mma_ss(tDP, da + 2, dv + 2, idescS, 1);
            mma_commit(bar_mma);
        }
        __syncwarp();
    };

    if (stid == 0) {
        mbar_expect_tx(bar_qa, RS * 2 * T128);
        for (int r = 0; r < RS; ++r) {
            tma_load_5d(sQA + (slot * RS + r) * 2 * T128, &tmQ128, bar_qa, 0, q0, r0 + r, h, b);
            tma_load_5d(sQA + (slot * RS + r) * 2 * T128 + T128, &tmA128, bar_qa, 0, q0, r0 + r, h, b);
        }
        for (int t = 0; t < NST - 1 && t < T; ++t) load_kv(t);
        if (slot == 0) {
            load_bias(0);
            if (NKT > 1) load_bias(1);
        }
    }
    if (swarp == 0) {
        mbar_wait(bar_qa, 0);
        issue_ss(0);
    }
    auto mask_val = [&](int t) -> float {  // key (kt*64 + stid%64) of the tile's broadcast row
        const int kt = t / RS, r = t % RS;
        const unsigned char mk = mask[(long long)b * p.N * p.N + (long long)(r0 + r) * p.mR + (long long)(kt * 64 + (stid & 63)) * p.mK];
        return mk ? 0.0f : -INFINITY;
    };
    int anymask = 0;
    if (mask) {
        const float mv = mask_val(0);
        if (stid < 64) sMask[stid] = mv;
        anymask = named_bar_or(bar_id, 256, mv != 0.0f);
    }
    float nl[RS], dd[RS];
#pragma unroll
    for (int r = 0; r < RS; ++r) {
        const long long o = (long long)b * p.N * p.H * p.N + (long long)h * p.N + (long long)(r0 + r) * p.lR + (long long)(q0 + row) * p.lQ;
        const float l = __ldg(LSE + o);
        nl[r] = l == -INFINITY ? -INFINITY : -l * kLog2e;
        dd[r] = __ldg(Dws + o);
    }
    const float scale = rsqrtf((float)DH);
    const uint64_t scale2 = pack2(scale, scale), l2e2 = pack2(kLog2e, kLog2e);
    int next_bias = 2;  // slot 0 / thread 0 only: next key tile whose bias has to be requested

    for (int kt = 0; kt < NKT; ++kt) {
#pragma unroll
        for (int r = 0; r < RS; ++r) {
            const int t = kt * RS + r, st = t % NST;
            float mnext = 0.0f;
            if (mask && t + 1 < T) mnext = mask_val(t + 1);
            mbar_wait(bar_mma, t & 1);  // S(t), dP(t) ready
            tc_fence_after();
            if (r == 0) mbar_wait(bars + D_BIAS_FULL + (kt & 1), (kt >> 1) & 1);
            uint32_t sraw[32], dpraw[32];
            tmem_ld32(tS + lane_off + chalf * 32, sraw);
            tmem_ld32(tDP + lane_off + chalf * 32, dpraw);
            const uint8_t* sB = sBias + (kt & 1) * 16384;
            uint4 bv[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) bv[j] = lds128(sB + row * 128 + (((chalf * 4 + j) ^ (row & 7)) << 4));
            tmem_ld_wait();
            tc_fence_before();
            named_bar_sync(bar_id, 256);  // [A] the whole tile is in registers: S / dP may be overwritten
            if (swarp == 0 && t + 1 < T) issue_ss(t + 1);

            if (anymask) {
                const float* mrow = sMask + (t & 1) * 64 + chalf * 32;
#pragma unroll
                for (int c4 = 0; c4 < 8; ++c4) {
                    const float4 mv = lds128f(mrow + c4 * 4);
                    sraw[c4 * 4] = __float_as_uint(__uint_as_float(sraw[c4 * 4]) + mv.x);  // -inf survives the scale
                    sraw[c4 * 4 + 1] = __float_as_uint(__uint_as_float(sraw[c4 * 4 + 1]) + mv.y);
                    sraw[c4 * 4 + 2] = __float_as_uint(__uint_as_float(sraw[c4 * 4 + 2]) + mv.z);
                    sraw[c4 * 4 + 3] = __float_as_uint(__uint_as_float(sraw[c4 * 4 + 3]) + mv.w);
                }
            }
            const uint64_t nl2 = pack2(nl[r], nl[r]), nd2 = pack2(-dd[r], -dd[r]);
            uint32_t ds[16];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const uint32_t w[4] = {bv[j].x, bv[j].y, bv[j].z, bv[j].w};
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const int c = j * 8 + e * 2;
                    const uint64_t x2 = fma2(pack2(__uint_as_float(sraw[c]), __uint_as_float(sraw[c + 1])), scale2,
                                             pack2(bf16_lo(w[e]), bf16_hi(w[e])));
                    float a0, a1, s0, s1;
                    unpack2(fma2(x2, l2e2, nl2), a0, a1);
                    const float p0 = ex2(a0), p1 = ex2(a1);
                    unpack2(mul2(pack2(p0, p1), add2(pack2(__uint_as_float(dpraw[c]), __uint_as_float(dpraw[c + 1])), nd2)), s0, s1);
                    ds[j * 4 + e] = pack_bf16(s0, s1);
                }
            }
            if (t >= 1) {  // dQ MMAs of tile t-1 done: dS buffer free, K/V ring slot (t-1)%NST free
                mbar_wait(bar_ts, (t - 1) & 1);
                tc_fence_after();
            }
            if (stid == 0 && t + NST - 1 < T) load_kv(t + NST - 1);
            tmem_st16(tDS + lane_off + chalf * 16, ds);
            if (mask && t + 1 < T && stid < 64) sMask[((t + 1) & 1) * 64 + stid] = mnext;
            tmem_st_wait();
            tc_fence_before();
            if (mask) anymask = named_bar_or(bar_id, 256, mnext != 0.0f); else named_bar_sync(bar_id, 256);  // [B]
            if (swarp == 0) {  // warp-uniform: the elected lane issues dQ_r += dS K
                tc_fence_after();
                const uint64_t dk = make_desc_sw64(smem_u32(sKV + st * 2 * T64));
                if (elect_one()) {
#pragma unroll
                    for (int ks = 0; ks < 4; ++ks)
                        mma_ts(tDQ + r * 32, tDS + ks * 8, dk + (uint64_t)ks * 64, idescO, (kt > 0 || ks > 0) ? 1u : 0u);
                    mma_commit(bar_ts);
                }
                __syncwarp();
                if (stid == 0) {
                    if (r == RS - 1) mbar_arrive(bars + D_BIAS_EMPTY + (kt & 1));  // this slot is past bias tile kt
                    if (slot == 0 && next_bias < NKT &&
                        mbar_test_wait(bars + D_BIAS_EMPTY + (next_bias & 1), ((next_bias >> 1) - 1) & 1)) {
                        load_bias(next_bias);
                        ++next_bias;
                    }
                }
            }
        }
    }
    mbar_wait(bar_ts, (T - 1) & 1);  // last dQ MMAs done
    tc_fence_after();
    {   // epilogue: warps 0-3 of the slot write row 0, warps 4-7 row 1 (scaled, P:L514 + reading A1)
        const int r = chalf;
        uint32_t v[32];
        tmem_ld32(tDQ + lane_off + r * 32, v);
        tmem_ld_wait();
        const long long off = (long long)b * p.sB + (long long)h * p.sH + (long long)(r0 + r) * p.sSlice + (long long)(q0 + row) * p.sPos;
        uint4* pq = (uint4*)(dQ + off);
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            uint32_t a[4];
#pragma unroll
            for (int e = 0; e < 4; ++e)
                a[e] = pack_bf16(__uint_as_float(v[j * 8 + 2 * e]) * scale, __uint_as_float(v[j * 8 + 2 * e + 1]) * scale);
            pq[j] = make_uint4(a[0], a[1], a[2], a[3]);
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc<512>(*tmem_slot);
}

}  // namespace

tri_status sm100_dq2_launch(const Problem& p, const CUtensorMap& tQ128, const CUtensorMap& tA128, const CUtensorMap& tK64,
                            const CUtensorMap& tV64, const CUtensorMap& tBqk, const unsigned char* mask, const float* LSE,
                            const float* Dws, void* dQ, cudaStream_t st) {
    // the opt-in shared-memory size is a per-device function attribute: set it on every launch (cheap, thread-safe)
    TRI_CUDA_CHECK(cudaFuncSetAttribute(sm100_dq2_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, Dq2Smem::total));
    const unsigned grid = (unsigned)((long long)p.B * (p.N / RT) * p.H * (p.N / 128));
    {
        ProfScope ps("sm100_dq2_kernel", st);
        sm100_dq2_kernel<<<grid, 512, Dq2Smem::total, st>>>(tQ128, tA128, tK64, tV64, tBqk, p, mask, LSE, Dws, (__nv_bfloat16*)dQ);
    }
    TRI_LAUNCH_CHECK("sm100_dq2_kernel");
    return TRI_OK;
}

}  // namespace tri

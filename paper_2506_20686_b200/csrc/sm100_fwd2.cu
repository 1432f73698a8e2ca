// bf16 forward, warp-specialised (sm_100a): one CTA per SM = 16 softmax warps + 2 MMA-issuer warps + 1 TMA warp.
//
// The CTA owns a 128-query block of 4 broadcast rows of one (b,h).  The rows are split over two "slots" (2 rows
// each); a slot = 8 softmax warps + its own issuer warp + 256 TMEM columns:
//     [0,128)   S  = Q_r K_r^T, fp32            (tcgen05.mma SS, M=128 N=128 K=2x16)
//     [128,192) P  = bf16 pairs, A operand of   O_r += P V_r (tcgen05.mma TS, N=32, K=8x16)
//     [192,256) O_r accumulators of the slot's 2 rows
// Software pipeline of a slot (Listing 1 P:L153-185 is the serial form): as soon as every softmax thread has
// pulled S(t) into registers (bar_sc) the issuer launches S(t+1), so the tensor pipe works under the exponentials
// of tile t; P V of tile t follows when P(t) is in TMEM (bar_p).  Tiles run key block kb OUTER, row r INNER, so a
// 128x128 bias tile (TMA, double buffered) serves all 4 rows ("on-the-fly broadcasting").
// A query row is handled by TWO threads (64 key columns each, warps w and w+4 of the slot); they exchange their
// partial row maxima through shared memory at a 256-thread named barrier; partial row sums are merged at the end.
#include "sm100_common.cuh"
#include "tri_common.cuh"

namespace tri {
using namespace sm100;

namespace {

constexpr int BQ = 128, BK = 128, DH = 32;
constexpr int TILE = BQ * DH * 2;  // 8 KB
constexpr int RS = 2;              // rows per slot
constexpr int RT = 4;              // rows per CTA
constexpr float kLazy = 5.0f;     // lazy-rescale threshold on the running max (natural-log units)
constexpr int NSOFT = 512;         // softmax threads (warps 0..15)
constexpr int NTHREADS = NSOFT + 96;  // + issuer warps 16,17 + TMA warp 18

struct F2Smem {
    static constexpr int q_off = 0;                             // RT x 8 KB
    static constexpr int k_off = q_off + RT * TILE;             // [slot][stage] 8 KB
    static constexpr int v_off = k_off + 4 * TILE;              // [slot][stage] 8 KB
    static constexpr int bias_off = v_off + 4 * TILE;           // [buf][key half] 16 KB each, SWIZZLE_128B
    static constexpr int m_off = bias_off + 2 * 32768;          // float m[slot][RS][128]
    static constexpr int l_off = m_off + 2 * RS * 128 * 4;      // float l[slot][RS][256]
    static constexpr int pmax_off = l_off + 2 * RS * 256 * 4;   // float pmax[slot][half][128]
    static constexpr int mask_off = pmax_off + 2 * 2 * 128 * 4; // float mask[slot][2][128]
    static constexpr int bar_off = mask_off + 2 * 2 * 128 * 4;
    static constexpr int total = bar_off + 256 + 1024;
};

// mbarrier indices
enum { B_Q = 0, B_K = 1 /*[slot][2]*/, B_V = 5 /*[slot][2]*/, B_BIAS_FULL = 9 /*[2]*/, B_BIAS_EMPTY = 11 /*[2]*/,
       B_S = 13 /*[slot]*/, B_SC = 15 /*[slot]*/, B_P = 17 /*[slot]*/, B_PV = 19 /*[slot]*/, B_COUNT = 21 };

__global__ void __launch_bounds__(NTHREADS, 1) sm100_fwd2_kernel(const __grid_constant__ CUtensorMap tmQ,
                                                                 const __grid_constant__ CUtensorMap tmK,
                                                                 const __grid_constant__ CUtensorMap tmV,
                                                                 const __grid_constant__ CUtensorMap tmBias, Problem p,
                                                                 const __nv_bfloat16* __restrict__ G,
                                                                 const unsigned char* __restrict__ mask,
                                                                 __nv_bfloat16* __restrict__ O, float* __restrict__ LSE) {
    using L = F2Smem;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    uint8_t* sQ = smem + L::q_off;
    uint8_t* sK = smem + L::k_off;
    uint8_t* sV = smem + L::v_off;
    uint8_t* sBias = smem + L::bias_off;
    float* sM = (float*)(smem + L::m_off);
    float* sL = (float*)(smem + L::l_off);
    float* sPmax = (float*)(smem + L::pmax_off);
    float* sMask = (float*)(smem + L::mask_off);
    uint64_t* bars = (uint64_t*)(smem + L::bar_off);
    uint32_t* tmem_slot = (uint32_t*)(bars + B_COUNT);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int NQB = p.N / BQ, NKB = p.N / BK, NG = p.N / RT;
    int idx = blockIdx.x;
    const int qb = idx % NQB; idx /= NQB;
    const int h = idx % p.H; idx /= p.H;
    const int g = idx % NG;
    const int b = idx / NG;
    const int r0 = g * RT, q0 = qb * BQ, bh = b * p.H + h;
    const int T = NKB * RS;  // tiles per slot

    if (tid == 0) {
        prefetch_tmap(&tmQ); prefetch_tmap(&tmK); prefetch_tmap(&tmV); prefetch_tmap(&tmBias);
        for (int i = 0; i < B_COUNT; ++i) {
            const bool warp_counted = (i >= B_SC && i < B_PV);           // 8 softmax-warp arrivals
            const bool two = (i >= B_BIAS_EMPTY && i < B_S);             // one arrival per slot
            mbar_init(bars + i, warp_counted ? 8 : (two ? 2 : 1));
        }
        fence_barrier_init();
    }
    if (warp == 18) tmem_alloc<512>(tmem_slot);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;

    if (warp == 18) {
        // =========================== TMA warp: Q once, bias tiles (shared by both slots) ===========================
        if (lane == 0) {
            mbar_expect_tx(bars + B_Q, RT * TILE);
            for (int r = 0; r < RT; ++r) tma_load_5d(sQ + r * TILE, &tmQ, bars + B_Q, 0, q0, r0 + r, h, b);
            for (int kb = 0; kb < NKB; ++kb) {
                const int buf = kb & 1;
                if (kb >= 2) mbar_wait(bars + B_BIAS_EMPTY + buf, ((kb >> 1) - 1) & 1);  // both slots done with kb-2
                mbar_expect_tx(bars + B_BIAS_FULL + buf, 32768);
                tma_load_3d(sBias + buf * 32768, &tmBias, bars + B_BIAS_FULL + buf, kb * BK, q0, bh);
                tma_load_3d(sBias + buf * 32768 + 16384, &tmBias, bars + B_BIAS_FULL + buf, kb * BK + 64, q0, bh);
            }
        }
        __syncwarp();
    } else if (warp >= 16) {
        // =========================== MMA issuer of slot (warp - 16): K/V TMA + every tcgen05.mma ===========================
        const int slot = warp - 16;
        if (lane == 0) {
            uint64_t* bK = bars + B_K + slot * 2;
            uint64_t* bV = bars + B_V + slot * 2;
            auto load_k = [&](int t) {
                const int kb = t / RS, r = t % RS, st = t & 1;
                mbar_expect_tx(bK + st, TILE);
                tma_load_5d(sK + (slot * 2 + st) * TILE, &tmK, bK + st, 0, kb * BK, r0 + slot * RS + r, h, b);
            };
            auto load_v = [&](int t) {
                const int kb = t / RS, r = t % RS, st = t & 1;
                mbar_expect_tx(bV + st, TILE);
                tma_load_5d(sV + (slot * 2 + st) * TILE, &tmV, bV + st, 0, kb * BK, r0 + slot * RS + r, h, b);
            };
            constexpr uint32_t idescS = make_idesc(128, 128, false, false);
            constexpr uint32_t idescO = make_idesc(128, DH, false, true);
            const uint32_t tS = tmem + slot * 256, tP = tS + 128, tO = tS + 192;
            auto issue_s = [&](int t) {
                const int r = t % RS, st = t & 1;
                mbar_wait(bK + st, (t >> 1) & 1);
                tc_fence_after();
                const uint64_t dq = make_desc_sw64(smem_u32(sQ + (slot * RS + r) * TILE));
                const uint64_t dk = make_desc_sw64(smem_u32(sK + (slot * 2 + st) * TILE));
                mma_ss(tS, dq, dk, idescS, 0);
                mma_ss(tS, dq + 2, dk + 2, idescS, 1);
                mma_commit(bars + B_S + slot);
            };
            load_k(0);
            if (T > 1) load_k(1);
            load_v(0);
            mbar_wait(bars + B_Q, 0);
            issue_s(0);
            for (int t = 0; t < T; ++t) {
                const int kb = t / RS, r = t % RS, st = t & 1;
                // every softmax thread holds S(t) in registers: K stage st and the S columns are free
                mbar_wait(bars + B_SC + slot, t & 1);
                if (t + 2 < T) load_k(t + 2);
                if (t + 1 < T) issue_s(t + 1);
                // P(t) is in TMEM
                mbar_wait(bars + B_P + slot, t & 1);
                if (t >= 1) mbar_wait(bars + B_PV + slot, (t - 1) & 1);  // (must precede this tile's commit)
                mbar_wait(bV + st, (t >> 1) & 1);
                tc_fence_after();
                const uint64_t dv = make_desc_sw64(smem_u32(sV + (slot * 2 + st) * TILE));
#pragma unroll
                for (int ks = 0; ks < BK / 16; ++ks)
                    mma_ts(tO + r * 32, tP + ks * 8, dv + (uint64_t)ks * 64, idescO, (kb > 0 || ks > 0) ? 1u : 0u);
                mma_commit(bars + B_PV + slot);
                if (t + 1 < T) load_v(t + 1);  // P V(t-1) is done (waited above): V stage (t+1)&1 is free
                if (r == RS - 1) mbar_arrive(bars + B_BIAS_EMPTY + (kb & 1));  // this slot is past bias tile kb
            }
        }
        __syncwarp();
    } else {
        // =========================== softmax warps ===========================
        const int slot = warp >> 3, half = (warp >> 2) & 1, quarter = warp & 3;
        const int row = quarter * 32 + lane;   // query row inside the block = TMEM lane
        const int bar_id = 1 + slot;           // named barrier of the slot (0 is __syncthreads)
        const uint32_t lane_off = (uint32_t)(quarter * 32) << 16;
        const uint32_t tS = tmem + slot * 256 + lane_off, tP = tS + 128, tO = tS + 192;
        float* myM = sM + slot * RS * 128 + row;               // + r*128
        float* myL = sL + slot * RS * 256 + half * 128 + row;  // + r*256
        float* pmax_mine = sPmax + (slot * 2 + half) * 128 + row;
        const float* pmax_other = sPmax + (slot * 2 + (half ^ 1)) * 128 + row;
        float* maskS = sMask + slot * 2 * 128;                 // [2][128]
        uint64_t* bar_s = bars + B_S + slot;
        uint64_t* bar_sc = bars + B_SC + slot;
        uint64_t* bar_p = bars + B_P + slot;
        uint64_t* bar_pv = bars + B_PV + slot;
        const float scale = rsqrtf((float)DH);
        for (int r = 0; r < RS; ++r) { myM[r * 128] = -INFINITY; myL[r * 256] = 0.0f; }

        auto mask_val = [&](int t) -> float {  // half-0 threads: key (kb*128 + row) of the tile's broadcast row
            const int kb = t / RS, r = t % RS;
            const unsigned char mk = mask[(long long)b * p.N * p.N + (long long)(r0 + slot * RS + r) * p.mR +
                                          (long long)(kb * BK + row) * p.mK];
            return mk ? 0.0f : -INFINITY;
        };
        int anymask = 0;
        if (mask) {
            float mv = 0.0f;
            if (half == 0) { mv = mask_val(0); maskS[row] = mv; }
            anymask = named_bar_or(bar_id, 256, mv != 0.0f);
        }

        for (int kb = 0; kb < NKB; ++kb) {
#pragma unroll 1
            for (int r = 0; r < RS; ++r) {
                const int t = kb * RS + r, st = t & 1;
                float mnext = 0.0f;
                if (mask && half == 0 && t + 1 < T) mnext = mask_val(t + 1);
                mbar_wait(bar_s, t & 1);
                tc_fence_after();
                float x[64];
                {
                    uint32_t* raw = (uint32_t*)x;
                    tmem_ld32(tS + half * 64, *(uint32_t(*)[32])raw);
                    tmem_ld32(tS + half * 64 + 32, *(uint32_t(*)[32])(raw + 32));
                    tmem_ld_wait();
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(bar_sc);  // S(t) is in registers: the issuer may overwrite it with S(t+1)
                if (r == 0) mbar_wait(bars + B_BIAS_FULL + (kb & 1), (kb >> 1) & 1);
                const float m_old = myM[r * 128];

                // ---- my 64 score columns: x = scale*S + bias (+ mask) ---------------------------------------------
                const uint8_t* brow = sBias + (kb & 1) * 32768 + half * 16384 + row * 128;
                const uint64_t scale2 = pack2(scale, scale);
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    const uint4 bv = *(const uint4*)(brow + ((j ^ (row & 7)) << 4));
                    const uint32_t w[4] = {bv.x, bv.y, bv.z, bv.w};
#pragma unroll
                    for (int e = 0; e < 4; ++e) {
                        const int c = j * 8 + e * 2;
                        unpack2(fma2(pack2(x[c], x[c + 1]), scale2, pack2(bf16_lo(w[e]), bf16_hi(w[e]))), x[c], x[c + 1]);
                    }
                }
                if (anymask) {
                    const float4* mrow = (const float4*)(maskS + st * 128 + half * 64);
#pragma unroll
                    for (int c4 = 0; c4 < 16; ++c4) {
                        const float4 mv = mrow[c4];
                        x[c4 * 4] += mv.x; x[c4 * 4 + 1] += mv.y; x[c4 * 4 + 2] += mv.z; x[c4 * 4 + 3] += mv.w;
                    }
                }
                float mx = x[0];
#pragma unroll
                for (int c = 1; c < 64; ++c) mx = fmaxf(mx, x[c]);
                *pmax_mine = mx;
                if (mask && half == 0 && t + 1 < T) maskS[(st ^ 1) * 128 + row] = mnext;
                if (mask) anymask = named_bar_or(bar_id, 256, mnext != 0.0f); else named_bar_sync(bar_id, 256);

                // ---- online softmax, -inf guard of reading A6.  The running reference m only moves when
                // the tile maximum exceeds it by more than kLazy (O and l share the reference, so the result is
                // exact either way); this keeps the O rescale out of almost every tile.
                const float mt = fmaxf(mx, *pmax_other);
                const bool bump = mt > m_old + kLazy;
                const float m_new = bump ? mt : m_old;
                const float m_safe = (m_new == -INFINITY) ? 0.0f : m_new;
                const float alpha = bump ? ex2((m_old - m_safe) * kLog2e) : 1.0f;
                const float mneg = -m_safe * kLog2e;
                const uint64_t l2e2 = pack2(kLog2e, kLog2e), mneg2 = pack2(mneg, mneg);
                uint64_t lacc = pack2(0.0f, 0.0f);
                uint32_t* pk = (uint32_t*)x;  // packed in place: pk[e] <- (x[2e], x[2e+1])
#pragma unroll
                for (int e = 0; e < 32; ++e) {
                    float a0, a1;
                    unpack2(fma2(pack2(x[2 * e], x[2 * e + 1]), l2e2, mneg2), a0, a1);
                    const float p0 = ex2(a0), p1 = ex2(a1);
                    lacc = add2(lacc, pack2(p0, p1));
                    pk[e] = pack_bf16(p0, p1);
                }
                float l0, l1;
                unpack2(lacc, l0, l1);
                myL[r * 256] = myL[r * 256] * alpha + (l0 + l1);
                if (half == 0 && bump) myM[r * 128] = m_new;
                if (t >= 1) { mbar_wait(bar_pv, (t - 1) & 1); tc_fence_after(); }  // P V(t-1) done: P buffer and O are free
                tmem_st32(tP + half * 32, *(uint32_t(*)[32])pk);
                if (kb > 0 && __any_sync(0xffffffffu, bump)) {  // rescale my 16 columns of O_r
                    uint32_t o[16];
                    tmem_ld16(tO + r * 32 + half * 16, o);
                    tmem_ld_wait();
#pragma unroll
                    for (int c = 0; c < 16; ++c) o[c] = __float_as_uint(__uint_as_float(o[c]) * alpha);
                    tmem_st16(tO + r * 32 + half * 16, o);
                }
                tmem_st_wait();
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(bar_p);
            }
        }
        mbar_wait(bar_pv, (T - 1) & 1);  // last P V of the slot complete
        tc_fence_after();
        named_bar_sync(bar_id, 256);     // partial row sums of both halves visible

        // ---- epilogue: O = sigmoid(G) * O_r / l ; LSE = m + ln l; half h takes row r = h ----------------
        for (int r = half; r < RS; r += 2) {
            uint32_t o[32];
            tmem_ld32(tO + r * 32, o);
            const int rr = r0 + slot * RS + r;
            const long long off = (long long)b * p.sB + (long long)h * p.sH + (long long)rr * p.sSlice + (long long)(q0 + row) * p.sPos;
            const uint4* gp = (const uint4*)(G + off);
            uint4 gv[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) gv[j] = __ldg(gp + j);
            tmem_ld_wait();
            const float l = sL[slot * RS * 256 + r * 256 + row] + sL[slot * RS * 256 + r * 256 + 128 + row];
            const float inv = l > 0.0f ? 1.0f / l : 0.0f;
            uint4* op = (uint4*)(O + off);
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const uint32_t gw[4] = {gv[j].x, gv[j].y, gv[j].z, gv[j].w};
                uint32_t ow[4];
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const float g0 = bf16_lo(gw[e]), g1 = bf16_hi(gw[e]);
                    const float s0 = __fdividef(1.0f, 1.0f + ex2(-g0 * kLog2e)), s1 = __fdividef(1.0f, 1.0f + ex2(-g1 * kLog2e));
                    ow[e] = pack_bf16(__uint_as_float(o[j * 8 + 2 * e]) * inv * s0, __uint_as_float(o[j * 8 + 2 * e + 1]) * inv * s1);
                }
                op[j] = make_uint4(ow[0], ow[1], ow[2], ow[3]);
            }
            const long long loff = (long long)b * p.N * p.H * p.N + (long long)h * p.N + (long long)rr * p.lR + (long long)(q0 + row) * p.lQ;
            LSE[loff] = l > 0.0f ? sM[slot * RS * 128 + r * 128 + row] + __logf(l) : -INFINITY;
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 18) tmem_dealloc<512>(tmem);
}

}  // namespace

tri_status sm100_fwd2_launch(const Problem& p, const CUtensorMap& tQ, const CUtensorMap& tK, const CUtensorMap& tV,
                             const CUtensorMap& tB, const void* G, const unsigned char* mask, void* O, float* LSE,
                             cudaStream_t st) {
    static bool attr_done = false;
    if (!attr_done) {
        TRI_CUDA_CHECK(cudaFuncSetAttribute(sm100_fwd2_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, F2Smem::total));
        attr_done = true;
    }
    const unsigned grid = (unsigned)((long long)p.B * (p.N / RT) * p.H * (p.N / BQ));
    {
        ProfScope ps("sm100_fwd2_kernel", st);
        sm100_fwd2_kernel<<<grid, NTHREADS, F2Smem::total, st>>>(tQ, tK, tV, tB, p, (const __nv_bfloat16*)G, mask,
                                                                 (__nv_bfloat16*)O, LSE);
    }
    TRI_LAUNCH_CHECK("sm100_fwd2_kernel");
    return TRI_OK;
}

}  // namespace tri

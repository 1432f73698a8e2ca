// bf16 forward, warp-specialised with register reallocation (sm_100a): one CTA per SM, three warpgroups.
//
//   WG0, WG1 : softmax warpgroups ("slots"), one thread per query row = TMEM lane, the whole 128-key row of a score tile
//              in registers (setmaxnreg raises them to 240 registers/thread); slot s owns rows 2s, 2s+1 of the CTA's
//              4 broadcast rows and 256 TMEM columns: [0,128) S fp32, [128,192) P bf16 pairs, [192,256) O_r (2 x 32).
//   WG2      : warp 8 / 9 = MMA + K/V-TMA issuer of slot 0 / 1 (whole warp runs the loop, elect.sync picks the lane, it
//              also stages the key mask), warp 10 = Q and bias TMA, warp 11 idle; setmaxnreg drops them to 24 registers.
// Pipeline of a slot (Listing 1 P:L153-185 is the serial form): S(t+1) = Q K^T is issued as soon as every softmax
// thread has S(t) in registers; O_r += P V follows when P(t) is in TMEM.  Key block OUTER, row INNER: one 128x128 bias
// tile (TMA, double buffered) serves the CTA's 4 rows.  No CTA-wide barrier in the main loop.
#include "sm100_common.cuh"
#include "tri_common.cuh"

namespace tri {
using namespace sm100;

namespace {

constexpr int BQ = 128, BK = 128, DH = 32;
constexpr int TILE = BQ * DH * 2;  // 8 KB
constexpr int RS = 2, RT = 4;      // rows per slot / per CTA
constexpr float kLazy = 5.0f;      // lazy-rescale threshold on the running max (natural-log units)
constexpr int NTHREADS = 384;

struct F3Smem {
    static constexpr int q_off = 0;                               // RT x 8 KB
    static constexpr int k_off = q_off + RT * TILE;               // [slot][2] 8 KB
    static constexpr int v_off = k_off + 4 * TILE;                // [slot][2] 8 KB
    static constexpr int bias_off = v_off + 4 * TILE;             // [buf][key half] 16 KB each, SWIZZLE_128B
    static constexpr int mask_off = bias_off + 2 * 32768;         // float mask[slot][2][128] + int any[slot][2]
    static constexpr int bar_off = mask_off + 2 * 2 * 128 * 4 + 16;
    static constexpr int total = bar_off + 256 + 1024;
};
enum { B_Q = 0, B_K = 1 /*[slot][2]*/, B_V = 5 /*[slot][2]*/, B_BIAS_FULL = 9 /*[2]*/, B_BIAS_EMPTY = 11 /*[2]*/,
       B_S = 13 /*[slot]*/, B_SC = 15 /*[slot]*/, B_P = 17 /*[slot]*/, B_PV = 19 /*[slot]*/, B_COUNT = 21 };

template <int N_>
__device__ __forceinline__ void setmaxnreg_inc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(N_)); }
template <int N_>
__device__ __forceinline__ void setmaxnreg_dec() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(N_)); }

__global__ void __launch_bounds__(NTHREADS, 1) sm100_fwd3_kernel(const __grid_constant__ CUtensorMap tmQ,
                                                                 const __grid_constant__ CUtensorMap tmK,
                                                                 const __grid_constant__ CUtensorMap tmV,
                                                                 const __grid_constant__ CUtensorMap tmBias, Problem p,
                                                                 const __nv_bfloat16* __restrict__ G,
                                                                 const unsigned char* __restrict__ mask,
                                                                 __nv_bfloat16* __restrict__ O, float* __restrict__ LSE) {
    using L = F3Smem;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    uint8_t* sQ = smem + L::q_off;
    uint8_t* sK = smem + L::k_off;
    uint8_t* sV = smem + L::v_off;
    uint8_t* sBias = smem + L::bias_off;
    float* sMask = (float*)(smem + L::mask_off);
    int* sAny = (int*)(sMask + 2 * 2 * 128);
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
            const bool warp_counted = (i >= B_SC && i < B_PV);  // 4 softmax-warp arrivals
            const bool two = (i >= B_BIAS_EMPTY && i < B_S);    // one arrival per slot
            mbar_init(bars + i, warp_counted ? 4 : (two ? 2 : 1));
        }
        fence_barrier_init();
    }
    if (warp == 8) tmem_alloc<512>(tmem_slot);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;

    if (warp >= 8) {
        setmaxnreg_dec<24>();
        if (warp == 10) {
            // ---------------- Q once, bias tiles (shared by both slots) ----------------
            if (elect_one()) {
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
        } else if (warp < 10) {
            // ---------------- issuer of slot (warp - 8): K/V TMA, mask staging, every tcgen05.mma ----------------
            const int slot = warp - 8;
            uint64_t* bK = bars + B_K + slot * 2;
            uint64_t* bV = bars + B_V + slot * 2;
            float* maskS = sMask + slot * 2 * 128;
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
            auto issue_s = [&](int t) {  // whole warp; mask slot t&1 and the S columns are free here
                const int kb = t / RS, r = t % RS, st = t & 1;
                if (mask) {
                    int any = 0;
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        const int k = lane * 4 + i;
                        const unsigned char mk = mask[(long long)b * p.N * p.N + (long long)(r0 + slot * RS + r) * p.mR +
                                                      (long long)(kb * BK + k) * p.mK];
                        maskS[st * 128 + k] = mk ? 0.0f : -INFINITY;
                        any |= !mk;
                    }
                    any = __any_sync(0xffffffffu, any);
                    if (lane == 0) sAny[slot * 2 + st] = any;
                    __syncwarp();
                }
                mbar_wait(bK + st, (t >> 1) & 1);
                tc_fence_after();
                const uint64_t dq = make_desc_sw64(smem_u32(sQ + (slot * RS + r) * TILE));
                const uint64_t dk = make_desc_sw64(smem_u32(sK + (slot * 2 + st) * TILE));
                if (elect_one()) {
                    mma_ss(tS, dq, dk, idescS, 0);
                    mma_ss(tS, dq + 2, dk + 2, idescS, 1);
                    mma_commit(bars + B_S + slot);
                }
                __syncwarp();
            };
            if (elect_one()) {
                load_k(0);
                if (T > 1) load_k(1);
                load_v(0);
            }
            __syncwarp();
            mbar_wait(bars + B_Q, 0);
            issue_s(0);
            for (int t = 0; t < T; ++t) {
                const int kb = t / RS, r = t % RS, st = t & 1;
                mbar_wait(bars + B_SC + slot, t & 1);  // S(t) is in registers: K stage st and the S columns are free
                if (t + 2 < T && elect_one()) load_k(t + 2);
                __syncwarp();
                if (t + 1 < T) issue_s(t + 1);
                mbar_wait(bars + B_P + slot, t & 1);   // P(t) is in TMEM
                if (t >= 1) mbar_wait(bars + B_PV + slot, (t - 1) & 1);  // (must precede this tile's commit)
                mbar_wait(bV + st, (t >> 1) & 1);
                tc_fence_after();
                const uint64_t dv = make_desc_sw64(smem_u32(sV + (slot * 2 + st) * TILE));
                if (elect_one()) {
#pragma unroll
                    for (int ks = 0; ks < BK / 16; ++ks)
                        mma_ts(tO + r * 32, tP + ks * 8, dv + (uint64_t)ks * 64, idescO, (kb > 0 || ks > 0) ? 1u : 0u);
                    mma_commit(bars + B_PV + slot);
                    if (t + 1 < T) load_v(t + 1);  // P V(t-1) is done (waited above): V stage (t+1)&1 is free
                    if (r == RS - 1) mbar_arrive(bars + B_BIAS_EMPTY + (kb & 1));  // this slot is past bias tile kb
                }
                __syncwarp();
            }
        }
    } else {
        setmaxnreg_inc<240>();
        // =========================== softmax warpgroups ===========================
        const int slot = warp >> 2;
        const int row = (warp & 3) * 32 + lane;  // query row inside the block = TMEM lane
        const uint32_t lane_off = (uint32_t)((warp & 3) * 32) << 16;
        const uint32_t tS = tmem + slot * 256 + lane_off, tP = tS + 128, tO = tS + 192;
        const float* maskS = sMask + slot * 2 * 128;
        uint64_t* bar_s = bars + B_S + slot;
        uint64_t* bar_sc = bars + B_SC + slot;
        uint64_t* bar_p = bars + B_P + slot;
        uint64_t* bar_pv = bars + B_PV + slot;
        const float scale = rsqrtf((float)DH);
        const uint64_t scale2 = pack2(scale, scale), l2e2 = pack2(kLog2e, kLog2e);
        float m_run[RS], l_run[RS];
#pragma unroll
        for (int r = 0; r < RS; ++r) { m_run[r] = -INFINITY; l_run[r] = 0.0f; }

        for (int kb = 0; kb < NKB; ++kb) {
#pragma unroll
            for (int r = 0; r < RS; ++r) {
                const int t = kb * RS + r, st = t & 1;
                mbar_wait(bar_s, t & 1);
                tc_fence_after();
                float x[BK];
#pragma unroll
                for (int c32 = 0; c32 < 4; ++c32) tmem_ld32(tS + c32 * 32, *(uint32_t(*)[32])((uint32_t*)x + c32 * 32));
                tmem_ld_wait();
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(bar_sc);  // S(t) is in registers: the issuer may overwrite it with S(t+1)
                if (r == 0) mbar_wait(bars + B_BIAS_FULL + (kb & 1), (kb >> 1) & 1);

                // ---- x = scale*S + bias (+ mask), row maximum ------------------------------------------------------
                const uint8_t* brow = sBias + (kb & 1) * 32768 + row * 128;
#pragma unroll
                for (int j = 0; j < 16; ++j) {
                    const uint4 bv = lds128(brow + (j >> 3) * 16384 + (((j & 7) ^ (row & 7)) << 4));
                    const uint32_t w[4] = {bv.x, bv.y, bv.z, bv.w};
#pragma unroll
                    for (int e = 0; e < 4; ++e) {
                        const int c = j * 8 + e * 2;
                        unpack2(fma2(pack2(x[c], x[c + 1]), scale2, pack2(bf16_lo(w[e]), bf16_hi(w[e]))), x[c], x[c + 1]);
                    }
                }
                if (mask && sAny[slot * 2 + st]) {
                    const float4* mrow = (const float4*)(maskS + st * 128);
#pragma unroll
                    for (int c4 = 0; c4 < BK / 4; ++c4) {
                        const float4 mv = lds128f(mrow + c4);
                        x[c4 * 4] += mv.x; x[c4 * 4 + 1] += mv.y; x[c4 * 4 + 2] += mv.z; x[c4 * 4 + 3] += mv.w;
                    }
                }
                float mx = x[0];
#pragma unroll
                for (int c = 1; c < BK; ++c) mx = fmaxf(mx, x[c]);

                // ---- online softmax, lazily updated reference, -inf guard of reading A6 ----------------
                const float m_old = m_run[r];
                const bool bump = mx > m_old + kLazy;
                const float m_new = bump ? mx : m_old;
                const float m_safe = (m_new == -INFINITY) ? 0.0f : m_new;
                const float alpha = bump ? ex2((m_old - m_safe) * kLog2e) : 1.0f;
                const float mneg = -m_safe * kLog2e;
                const uint64_t mneg2 = pack2(mneg, mneg);
                uint64_t lacc = pack2(0.0f, 0.0f);
                uint32_t* pk = (uint32_t*)x;  // packed in place: pk[e] <- (x[2e], x[2e+1])
#pragma unroll
                for (int e = 0; e < BK / 2; ++e) {
                    float a0, a1;
                    unpack2(fma2(pack2(x[2 * e], x[2 * e + 1]), l2e2, mneg2), a0, a1);
                    const float p0 = ex2(a0), p1 = ex2(a1);
                    lacc = add2(lacc, pack2(p0, p1));
                    pk[e] = pack_bf16(p0, p1);
                }
                float l0, l1;
                unpack2(lacc, l0, l1);
                l_run[r] = l_run[r] * alpha + (l0 + l1);
                m_run[r] = m_new;
                if (t >= 1) { mbar_wait(bar_pv, (t - 1) & 1); tc_fence_after(); }  // P V(t-1) done: P buffer and O are free
                tmem_st32(tP, *(uint32_t(*)[32])pk);
                tmem_st32(tP + 32, *(uint32_t(*)[32])(pk + 32));
                if (kb > 0 && __any_sync(0xffffffffu, bump)) {  // rescale O_r
                    uint32_t o[32];
                    tmem_ld32(tO + r * 32, o);
                    tmem_ld_wait();
#pragma unroll
                    for (int c = 0; c < 32; ++c) o[c] = __float_as_uint(__uint_as_float(o[c]) * alpha);
                    tmem_st32(tO + r * 32, o);
                }
                tmem_st_wait();
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(bar_p);
            }
        }
        mbar_wait(bar_pv, (T - 1) & 1);  // last P V of the slot complete
        tc_fence_after();

        // ---- epilogue: O = sigmoid(G) * O_r / l ; LSE = m + ln l -------------------------------------------
#pragma unroll
        for (int r = 0; r < RS; ++r) {
            uint32_t o[32];
            tmem_ld32(tO + r * 32, o);
            const int rr = r0 + slot * RS + r;
            const long long off = (long long)b * p.sB + (long long)h * p.sH + (long long)rr * p.sSlice + (long long)(q0 + row) * p.sPos;
            const uint4* gp = (const uint4*)(G + off);
            uint4 gv[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) gv[j] = __ldg(gp + j);
            tmem_ld_wait();
            const float l = l_run[r];
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
            LSE[loff] = l > 0.0f ? m_run[r] + __logf(l) : -INFINITY;
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 8) tmem_dealloc<512>(tmem);
}

}  // namespace

tri_status sm100_fwd3_launch(const Problem& p, const CUtensorMap& tQ, const CUtensorMap& tK, const CUtensorMap& tV,
                             const CUtensorMap& tB, const void* G, const unsigned char* mask, void* O, float* LSE,
                             cudaStream_t st) {
    // the opt-in shared-memory size is a per-device function attribute: set it on every launch (cheap, thread-safe)
    TRI_CUDA_CHECK(cudaFuncSetAttribute(sm100_fwd3_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, F3Smem::total));
    const unsigned grid = (unsigned)((long long)p.B * (p.N / RT) * p.H * (p.N / BQ));
    {
        ProfScope ps("sm100_fwd3_kernel", st);
        sm100_fwd3_kernel<<<grid, NTHREADS, F3Smem::total, st>>>(tQ, tK, tV, tB, p, (const __nv_bfloat16*)G, mask,
                                                                 (__nv_bfloat16*)O, LSE);
    }
    TRI_LAUNCH_CHECK("sm100_fwd3_kernel");
    return TRI_OK;
}

}  // namespace tri

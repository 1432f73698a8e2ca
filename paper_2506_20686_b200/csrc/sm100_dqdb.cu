// Stage 2 of the bf16 backward on tcgen05 / TMEM / TMA (sm_100a): dQ and dBias from ONE recomputation of P and dS
// (Listing 2 stage 2; Table I).  The paper adds its dS tiles into dBias with tl.atomic_add
// (P:L488); here the reduction over the broadcast rows is deterministic and on-chip:
//
//   * tile-stationary: a CTA owns the dBias tiles (128 queries x up to 3 x 64 keys) of one (b, h) in REGISTERS and
//     streams over the broadcast rows r in ascending order (level 1 of the dBias reduction; level 2, only when the
//     row axis is split over G CTAs to fill the SMs, is sm100_dbias_reduce_kernel);
//   * the CTAs that own the key tiles of one 128-query block form a thread-block CLUSTER; each accumulates its
//     partial dQ_r = sum over its keys of dS K in TMEM, and the partials of a row are added in rank order through
//     distributed shared memory (rank c receives the running sum of ranks < c, adds its own, passes it on; the last
//     rank scales and stores dQ).  No floating-point atomics anywhere; every output is bitwise reproducible.
//
// Persistent, warp-specialised CTA of 640 threads:
//   warps 0-11   three compute groups (128 threads = 128 query rows = 128 TMEM lanes); group g owns key tile g of the
//                CTA: p = exp2(S*scale*log2e + log2e*bias - LSE*log2e), dS = p (dP - D), dBias += dS (fp32 registers),
//                dS -> bf16 -> TMEM;
//   warp 12      TMA producer: per row Q_r, dA_r (128 x 32) and K_r, V_r (192 x 32) into a 2-stage ring; per work item
//                the fp32 log2e*bias tiles of the groups;
//   warp 13      tcgen05.mma issuer: S = Q K^T, dP = dA V^T (SS, M128 N64 K2x16) per group, then dQ += dS K (TS, M128 N32
//                K4x16) in group order into a double-buffered accumulator;
//   warps 16-19  dQ reducer: TMEM partial -> registers -> + inbox -> next rank's inbox (st.shared::cluster) or global.
#include <cuda_runtime.h>

#include "sm100_common.cuh"
#include "tri_common.cuh"

namespace tri {
using namespace sm100;

namespace {

constexpr int NGB = 3;                                    // compute groups (64-key tiles) per CTA
constexpr int BQ = 128, BK = 64, DH = 32;
constexpr int NST = 2;                                    // operand ring stages (one broadcast row each)
constexpr int QT_BYTES = BQ * DH * 2;                     // 8 KB
constexpr int KT_BYTES = BK * DH * 2;                     // 4 KB
constexpr int STAGE_BYTES = 2 * QT_BYTES + 2 * NGB * KT_BYTES;  // Q, dA, K[192], V[192] = 40 KB
constexpr int BIAS_BYTES = BQ * BK * 4;                   // 32 KB per group: two [128 q][32 k] fp32 boxes, SWIZZLE_128B
constexpr int INBOX_BYTES = BQ * DH * 4;                  // 16 KB: running dQ sum of the lower ranks
constexpr int NIN = 2;                                    // inbox ring depth
constexpr int DQDB_THREADS = (NGB + 2) * 128;

struct DqdbSmem {
    static constexpr int op_off = 0;
    static constexpr int bias_off = op_off + NST * STAGE_BYTES;
    static constexpr int inbox_off = bias_off + NGB * BIAS_BYTES;
    static constexpr int bar_off = inbox_off + NIN * INBOX_BYTES;
    static constexpr int b_full = 0;                      // [NST] TMA -> issuer
    static constexpr int b_free = b_full + NST;           // [NST] MMAs of the row done -> producer
    static constexpr int b_bias_full = b_free + NST;
    static constexpr int b_bias_free = b_bias_full + 1;
    static constexpr int b_s_full = b_bias_free + 1;      // [NGB] S, dP of the row in TMEM
    static constexpr int b_ds_ready = b_s_full + NGB;     // [NGB] dS of the row in TMEM
    static constexpr int b_dq_full = b_ds_ready + NGB;    // [2] partial dQ of the row complete
    static constexpr int b_dq_free = b_dq_full + 2;       // [2] reducer has it in registers
    static constexpr int b_in_full = b_dq_free + 2;       // [NIN] lower rank wrote my inbox slot (remote arrivals)
    static constexpr int b_out_free = b_in_full + NIN;    // [NIN] upper rank read its inbox slot (remote arrivals)
    static constexpr int n_bars = b_out_free + NIN;
    static constexpr int total = bar_off + n_bars * 8 + 16 + 1024;
};

// ---- cluster / distributed shared memory primitives ----------------------------------------------------------
__device__ __forceinline__ uint32_t cluster_ctarank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ uint32_t cluster_nctarank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ uint32_t map_to_rank(uint32_t saddr, uint32_t rank) {
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(saddr), "r"(rank));
    return r;
}
__device__ __forceinline__ void st_cluster_v4(uint32_t addr, float a, float b, float c, float d) {
    asm volatile("st.shared::cluster.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
}
__device__ __forceinline__ void mbar_arrive_remote(uint32_t addr) {  // release at cluster scope: my earlier DSMEM stores
    asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(addr) : "memory");
}
__device__ __forceinline__ void mbar_wait_cluster(uint64_t* bar, uint32_t parity) {  // acquire at cluster scope
    uint32_t ok;
    do {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%1], %2, %3;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(ok)
            : "r"(smem_u32(bar)), "r"(parity), "r"(0x989680u)
            : "memory");
    } while (!ok);
}

struct Item2 { int b, h, q0, rb; };
__device__ __forceinline__ Item2 decode_item2(int item, int N, int H, int G, int NR) {
    Item2 it;
    const int NQB = N / BQ;
    it.rb = (item % G) * NR;
    int t = item / G;
    it.q0 = (t % NQB) * BQ;
    const int bh = t / NQB;
    it.b = bh / H;
    it.h = bh % H;
    return it;
}

__global__ void __launch_bounds__(DQDB_THREADS, 1)
sm100_dqdb_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmA,
                  const __grid_constant__ CUtensorMap tmK, const __grid_constant__ CUtensorMap tmV,
                  const __grid_constant__ CUtensorMap tmBias, Problem p, const unsigned long long* __restrict__ maskbits,
                  const float* __restrict__ LSE, const float* __restrict__ Dws, __nv_bfloat16* __restrict__ dQ,
                  float* __restrict__ dBias, float* __restrict__ planes, int G, int n_items, int kbox) {
    using L = DqdbSmem;
    extern __shared__ uint8_t smem_raw[];
    // the dynamic shared-memory window starts at the same offset in every CTA of the cluster, so the aligned layout
    // (and therefore every mapa-translated address) is identical across ranks
    uint8_t* smem = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    uint8_t* sOp = smem + L::op_off;
    uint8_t* sBias = smem + L::bias_off;
    uint8_t* sInbox = smem + L::inbox_off;
    uint64_t* bars = (uint64_t*)(smem + L::bar_off);
    uint64_t* full = bars + L::b_full;
    uint64_t* freeb = bars + L::b_free;
    uint64_t* bias_full = bars + L::b_bias_full;
    uint64_t* bias_free = bars + L::b_bias_free;
    uint64_t* s_full = bars + L::b_s_full;
    uint64_t* ds_ready = bars + L::b_ds_ready;
    uint64_t* dq_full = bars + L::b_dq_full;
    uint64_t* dq_free = bars + L::b_dq_free;
    uint64_t* in_full = bars + L::b_in_full;
    uint64_t* out_free = bars + L::b_out_free;
    uint32_t* tmem_slot = (uint32_t*)(bars + L::n_bars);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int N = p.N, NW = N / BK;
    const int C = (int)cluster_nctarank(), c = (int)cluster_ctarank();
    // key tiles of this rank: the N/64 tiles are dealt to the C ranks as evenly as possible (at most NGB each)
    const int base_t = NW / C, rem_t = NW % C;
    const int nt = base_t + (c < rem_t ? 1 : 0);
    const int t0 = c * base_t + (c < rem_t ? c : rem_t);
    const int k0 = t0 * BK;
    const int NR = N / G;  // broadcast rows per work item
    const int cid = (int)blockIdx.x / C, ncl = (int)gridDim.x / C;
    const int n_my = (n_items - cid + ncl - 1) / ncl;
    const int NRtot = n_my * NR;

    if (tid == 0) {
        prefetch_tmap(&tmQ); prefetch_tmap(&tmA); prefetch_tmap(&tmK); prefetch_tmap(&tmV); prefetch_tmap(&tmBias);
        for (int i = 0; i < NST; ++i) { mbar_init(full + i, 1); mbar_init(freeb + i, 1); }
        mbar_init(bias_full, 1);
        mbar_init(bias_free, nt * 4);
        for (int i = 0; i < NGB; ++i) { mbar_init(s_full + i, 1); mbar_init(ds_ready + i, 4); }
        for (int i = 0; i < 2; ++i) { mbar_init(dq_full + i, 1); mbar_init(dq_free + i, 4); }
        for (int i = 0; i < NIN; ++i) { mbar_init(in_full + i, 128); mbar_init(out_free + i, 4); }
        fence_barrier_init();
    }
    if (warp == 0) tmem_alloc<512>(tmem_slot);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    cluster_sync_all();  // every rank's barriers are initialised before any remote arrive / store

    if (warp >= NGB * 4 && warp < NGB * 4 + 4) {
        // =============================== helper warpgroup ===============================
        setmaxnreg_dec<40>();
        if (warp == NGB * 4) {
            // ---- TMA producer ----
            int n = 0;
            for (int il = 0; il < n_my; ++il) {
                const Item2 it = decode_item2(cid + il * ncl, N, p.H, G, NR);
                const int bh = it.b * p.H + it.h;
                if (il > 0) mbar_wait(bias_free, (il - 1) & 1);
                if (elect_one()) {
                    mbar_expect_tx(bias_full, nt * BIAS_BYTES);
                    for (int g = 0; g < nt; ++g) {
                        tma_load_3d(sBias + g * BIAS_BYTES, &tmBias, bias_full, k0 + g * BK, it.q0, bh);
                        tma_load_3d(sBias + g * BIAS_BYTES + BIAS_BYTES / 2, &tmBias, bias_full, k0 + g * BK + 32, it.q0, bh);
                    }
                }
                __syncwarp();
                for (int r = 0; r < NR; ++r, ++n) {
                    const int s = n % NST;
                    if (n >= NST) mbar_wait(freeb + s, ((n / NST) - 1) & 1);
                    if (elect_one()) {
                        uint8_t* st = sOp + s * STAGE_BYTES;
                        mbar_expect_tx(full + s, 2 * QT_BYTES + 2 * kbox * DH * 2);
                        tma_load_5d(st, &tmQ, full + s, 0, it.q0, it.rb + r, it.h, it.b);
                        tma_load_5d(st + QT_BYTES, &tmA, full + s, 0, it.q0, it.rb + r, it.h, it.b);
                        tma_load_5d(st + 2 * QT_BYTES, &tmK, full + s, 0, k0, it.rb + r, it.h, it.b);
                        tma_load_5d(st + 2 * QT_BYTES + NGB * KT_BYTES, &tmV, full + s, 0, k0, it.rb + r, it.h, it.b);
                    }
                    __syncwarp();
                }
            }
        } else if (warp == NGB * 4 + 1) {
            // ---- MMA issuer (warp-uniform control flow; one elected lane issues and commits) ----
            constexpr uint32_t idescS = make_idesc(128, BK, false, false);
            constexpr uint32_t idescO = make_idesc(128, DH, false, true);
            const uint32_t opbase = smem_u32(sOp);
            auto issue_sdp = [&](int s, int g) {
                const uint32_t st = opbase + s * STAGE_BYTES;
                const uint64_t dq = make_desc_sw64(st), da = make_desc_sw64(st + QT_BYTES);
                const uint64_t dk = make_desc_sw64(st + 2 * QT_BYTES + g * KT_BYTES);
                const uint64_t dv = make_desc_sw64(st + 2 * QT_BYTES + (NGB + g) * KT_BYTES);
                const uint32_t tS = tmem + g * 128, tDP = tS + 64;
                if (elect_one()) {
                    mma_ss(tS, dq, dk, idescS, 0);
                    mma_ss(tS, dq + 2, dk + 2, idescS, 1);
                    mma_ss(tDP, da, dv, idescS, 0);
                    mma_ss(tDP, da + 2, dv + 2, idescS, 1);
                    mma_commit(s_full + g);
                }
                __syncwarp();
            };
            if (NRtot > 0) {
                mbar_wait(full + 0, 0);
                tc_fence_after();
                for (int g = 0; g < nt; ++g) issue_sdp(0, g);
            }
            for (int n = 0; n < NRtot; ++n) {
                const int s = n % NST, j = n & 1;
                for (int g = 0; g < nt; ++g) {
                    mbar_wait(ds_ready + g, n & 1);
                    if (g == 0 && n >= 2) mbar_wait(dq_free + j, ((n >> 1) - 1) & 1);
                    tc_fence_after();
                    const uint64_t dk = make_desc_sw64(opbase + s * STAGE_BYTES + 2 * QT_BYTES + g * KT_BYTES);
                    const uint32_t tDS = tmem + g * 128 + 64, tDQ = tmem + NGB * 128 + j * 32;
                    if (elect_one()) {
#pragma unroll
                        for (int ks = 0; ks < BK / 16; ++ks)
                            mma_ts(tDQ, tDS + ks * 8, dk + (uint64_t)ks * 64, idescO, (g > 0 || ks > 0) ? 1u : 0u);
                        if (g == nt - 1) {
                            mma_commit(dq_full + j);
                            mma_commit(freeb + s);
                        }
                    }
                    __syncwarp();
                    if (n + 1 < NRtot) {
                        const int s1 = (n + 1) % NST;
                        if (g == 0) {
                            mbar_wait(full + s1, ((n + 1) / NST) & 1);
                            tc_fence_after();
                        }
                        issue_sdp(s1, g);
                    }
                }
            }
        }
    } else if (warp < NGB * 4) {
        // =============================== compute groups ===============================
        setmaxnreg_inc<128>();
        const int g = warp >> 2;
        if (g < nt) {
            const int row = tid & 127;  // query row inside the block = TMEM lane
            const uint32_t lane_off = (uint32_t)((warp & 3) * 32) << 16;
            const uint32_t tS = tmem + g * 128 + lane_off, tDP = tS + 64;
            const float sl = rsqrtf((float)DH) * kLog2e;
            const uint64_t sl2 = pack2(sl, sl);
            const uint8_t* brow = sBias + g * BIAS_BYTES + row * 128;
            const int tile = t0 + g;
            uint64_t acc2[BK / 2];
#pragma unroll
            for (int i = 0; i < BK / 2; ++i) acc2[i] = pack2(0.0f, 0.0f);
            int n = 0;
            for (int il = 0; il < n_my; ++il) {
                const Item2 it = decode_item2(cid + il * ncl, N, p.H, G, NR);
                const long long lbase = (long long)it.b * N * p.H * N + (long long)it.h * N + (long long)(it.q0 + row) * p.lQ;
                const unsigned long long* mcol = maskbits ? maskbits + ((long long)it.b * N + it.rb) * NW + tile : nullptr;
                float lse_n = __ldg(LSE + lbase + (long long)it.rb * p.lR), dd_n = __ldg(Dws + lbase + (long long)it.rb * p.lR);
                uint64_t mb_n = mcol ? ldg_u64(mcol) : ~0ull;
                mbar_wait(bias_full, il & 1);
                for (int r = 0; r < NR; ++r, ++n) {
                    const float nl = lse_n == -INFINITY ? -INFINITY : -lse_n * kLog2e;
                    const uint64_t nl2 = pack2(nl, nl), nd2 = pack2(-dd_n, -dd_n);
                    const uint64_t mb = mb_n;
                    if (r + 1 < NR) {
                        lse_n = __ldg(LSE + lbase + (long long)(it.rb + r + 1) * p.lR);
                        dd_n = __ldg(Dws + lbase + (long long)(it.rb + r + 1) * p.lR);
                        if (mcol) mb_n = ldg_u64(mcol + (long long)(r + 1) * NW);
                    }
                    mbar_wait(s_full + g, n & 1);
                    tc_fence_after();
                    uint32_t dsb[16];
#pragma unroll
                    for (int ch = 0; ch < 4; ++ch) {  // 16 key columns at a time
                        uint32_t sr[16], dp[16];
                        tmem_ld16(tS + ch * 16, sr);
                        tmem_ld16(tDP + ch * 16, dp);
                        float4 bv[4];
#pragma unroll
                        for (int i = 0; i < 4; ++i)
                            bv[i] = lds128f(brow + (ch >> 1) * (BIAS_BYTES / 2) + (((((ch & 1) << 2) + i) ^ (row & 7)) << 4));
                        tmem_ld_wait();
#pragma unroll
                        for (int i = 0; i < 4; ++i) {
                            const float bb[4] = {bv[i].x, bv[i].y, bv[i].z, bv[i].w};
#pragma unroll
                            for (int e = 0; e < 2; ++e) {
                                const int cc = i * 4 + e * 2;  // column inside the chunk
                                float x0, x1;
                                unpack2(fma2(pack2(__uint_as_float(sr[cc]), __uint_as_float(sr[cc + 1])), sl2, pack2(bb[e * 2], bb[e * 2 + 1])), x0, x1);
                                if (mb != ~0ull) {
                                    if (!((mb >> (ch * 16 + cc)) & 1ull)) x0 = -INFINITY;
                                    if (!((mb >> (ch * 16 + cc + 1)) & 1ull)) x1 = -INFINITY;
                                }
                                float a0, a1, s0, s1;
                                unpack2(add2(pack2(x0, x1), nl2), a0, a1);
                                const uint64_t p2 = pack2(ex2(a0), ex2(a1));
                                const uint64_t ds2 = mul2(p2, add2(pack2(__uint_as_float(dp[cc]), __uint_as_float(dp[cc + 1])), nd2));
                                acc2[ch * 8 + (cc >> 1)] = add2(acc2[ch * 8 + (cc >> 1)], ds2);
                                unpack2(ds2, s0, s1);
                                dsb[(ch & 1) * 8 + (cc >> 1)] = pack_bf16(s0, s1);
                            }
                        }
                        if (ch & 1) tmem_st16(tDP + (ch >> 1) * 16, dsb);  // dS (bf16 pairs) over the dP columns already read
                    }
                    tmem_st_wait();
                    tc_fence_before();
                    warp_arrive(ds_ready + g);
                }
                // ---- item done: my 64 dBias values of query row q0+row (level-1 sum over rows rb..rb+NR-1, ascending) ----
                float acc[BK];
#pragma unroll
                for (int i = 0; i < BK / 2; ++i) {
                    unpack2(acc2[i], acc[2 * i], acc[2 * i + 1]);
                    acc2[i] = pack2(0.0f, 0.0f);
                }
                const int bh = it.b * p.H + it.h;
                if (G > 1) {
                    float* out = planes + ((long long)(it.rb / NR) * p.B * p.H + bh) * N * N + (long long)(it.q0 + row) * N + tile * BK;
#pragma unroll
                    for (int i = 0; i < BK; i += 4) *(float4*)(out + i) = make_float4(acc[i], acc[i + 1], acc[i + 2], acc[i + 3]);
                } else {
                    float* out = dBias + (long long)bh * N * N + (long long)(it.q0 + row) * p.bQ + (long long)(tile * BK) * p.bK;
                    if (p.bK == 1) {
#pragma unroll
                        for (int i = 0; i < BK; i += 4) *(float4*)(out + i) = make_float4(acc[i], acc[i + 1], acc[i + 2], acc[i + 3]);
                    } else {
#pragma unroll
                        for (int i = 0; i < BK; ++i) out[(long long)i * p.bK] = acc[i];
                    }
                }
                // my generic-proxy reads of the bias tiles are complete before the producer's TMA may overwrite them
                fence_proxy_async();
                warp_arrive(bias_free);
            }
        }
    } else {
        // =============================== dQ reducer warpgroup ===============================
        setmaxnreg_dec<56>();
        const int row = tid & 127;
        const uint32_t lane_off = (uint32_t)((warp & 3) * 32) << 16;
        const float scale = rsqrtf((float)DH);
        const uint32_t inbox_local = smem_u32(sInbox);
        const uint32_t inbox_next = (c + 1 < C) ? map_to_rank(inbox_local, (uint32_t)(c + 1)) : 0u;
        const uint32_t infull_next = (c + 1 < C) ? map_to_rank(smem_u32(in_full), (uint32_t)(c + 1)) : 0u;
        const uint32_t outfree_prev = (c > 0) ? map_to_rank(smem_u32(out_free), (uint32_t)(c - 1)) : 0u;
        int n = 0;
        for (int il = 0; il < n_my; ++il) {
            const Item2 it = decode_item2(cid + il * ncl, N, p.H, G, NR);
            for (int r = 0; r < NR; ++r, ++n) {
                const int j = n & 1, ph = (n >> 1) & 1;
                mbar_wait(dq_full + j, ph);
                tc_fence_after();
                uint32_t v[32];
                tmem_ld32(tmem + NGB * 128 + j * 32 + lane_off, v);
                tmem_ld_wait();
                tc_fence_before();
                warp_arrive(dq_free + j);
                float f[32];
#pragma unroll
                for (int i = 0; i < 32; ++i) f[i] = __uint_as_float(v[i]);
                if (c > 0) {  // running sum of ranks 0..c-1 (fixed order: deterministic)
                    mbar_wait_cluster(in_full + j, ph);
                    const uint8_t* src = sInbox + j * INBOX_BYTES + row * 128;
#pragma unroll
                    for (int i = 0; i < 8; ++i) {
                        const float4 t = lds128f(src + ((i ^ (row & 7)) << 4));
                        f[4 * i] = t.x + f[4 * i]; f[4 * i + 1] = t.y + f[4 * i + 1];
                        f[4 * i + 2] = t.z + f[4 * i + 2]; f[4 * i + 3] = t.w + f[4 * i + 3];
                    }
                    __syncwarp();
                    if (lane == 0) mbar_arrive_remote(outfree_prev + j * 8);  // the slot may be rewritten
                }
                if (c + 1 < C) {
                    if (n >= NIN) mbar_wait_cluster(out_free + j, (ph ^ 1));
                    const uint32_t dst = inbox_next + j * INBOX_BYTES + row * 128;
#pragma unroll
                    for (int i = 0; i < 8; ++i)
                        st_cluster_v4(dst + ((i ^ (row & 7)) << 4), f[4 * i], f[4 * i + 1], f[4 * i + 2], f[4 * i + 3]);
                    mbar_arrive_remote(infull_next + j * 8);
                } else {  // last rank: dQ = scale * sum
                    const long long off = (long long)it.b * p.sB + (long long)it.h * p.sH + (long long)(it.rb + r) * p.sSlice +
                                          (long long)(it.q0 + row) * p.sPos;
                    uint4* pq = (uint4*)(dQ + off);
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        uint32_t a[4];
#pragma unroll
                        for (int e = 0; e < 4; ++e) a[e] = pack_bf16(f[i * 8 + 2 * e] * scale, f[i * 8 + 2 * e + 1] * scale);
                        pq[i] = make_uint4(a[0], a[1], a[2], a[3]);
                    }
                }
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();  // no rank exits while a peer may still write its inbox or arrive on its barriers
    if (warp == 0) tmem_dealloc<512>(tmem);
}

}  // namespace

// cluster size for N/64 key tiles at <= NGB tiles per rank, from the sizes the launch code accepts
int sm100_dqdb_cluster(int N) {
    const int T = N / BK, need = (T + NGB - 1) / NGB;
    const int sizes[] = {1, 2, 3, 4, 6, 8, 12, 16};
    for (int s : sizes)
        if (s >= need) return s;
    return 0;
}

// Row slices per (b, h, query block): device-independent (the workspace size depends on it), assuming 148 / C resident
// clusters; minimises waves * rows per item.
int sm100_dqdb_split(const Problem& p) {
    const int C = sm100_dqdb_cluster(p.N);
    if (C == 0) return 1;
    const int ncl = 148 / C;
    const long long base = (long long)p.B * p.H * (p.N / BQ);
    int bestG = 1;
    double best = 1e30;
    for (int G = 1; G <= 8; ++G) {
        if (p.N % G) continue;
        const double waves = (double)((base * G + ncl - 1) / ncl);
        const double cost = waves * (p.N / G + 16);
        if (cost < best * 0.98) { best = cost; bestG = G; }
    }
    return bestG;
}

// persistent grid (a multiple of the cluster size C), 0 if the kernel cannot run on this device / shape
int sm100_dqdb_grid(const Problem& p, int C, int G) {
    if (C == 0) return 0;
    if (cudaFuncSetAttribute(sm100_dqdb_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, DqdbSmem::total) != cudaSuccess) return 0;
    if (C > 8 && cudaFuncSetAttribute(sm100_dqdb_kernel, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) != cudaSuccess) return 0;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(C * 64));
    cfg.blockDim = dim3(DQDB_THREADS);
    cfg.dynamicSmemBytes = DqdbSmem::total;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = (unsigned)C; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    int ncl = 0;
    if (cudaOccupancyMaxActiveClusters(&ncl, sm100_dqdb_kernel, &cfg) != cudaSuccess || ncl <= 0) {
        cudaGetLastError();
        return 0;
    }
    const long long items = (long long)p.B * p.H * (p.N / BQ) * G;
    return (int)((items < ncl ? items : ncl) * C);
}

tri_status sm100_dqdb_launch(const Problem& p, int C, int G, int grid, const void* Q, const void* dA, const void* K, const void* V,
                             const float* biasL_qk, const unsigned long long* maskbits, const float* LSE, const float* Dws,
                             void* dQ, float* dBias, float* planes, cudaStream_t st) {
    const int kbox = p.N < NGB * BK ? p.N : NGB * BK;
    CUtensorMap tQ, tA, tK, tV, tB;
    if (!make_tmap_u(&tQ, Q, p.B, p.N, p.H, p.d, p.variant, BQ) || !make_tmap_u(&tA, dA, p.B, p.N, p.H, p.d, p.variant, BQ) ||
        !make_tmap_u(&tK, K, p.B, p.N, p.H, p.d, p.variant, kbox) || !make_tmap_u(&tV, V, p.B, p.N, p.H, p.d, p.variant, kbox) ||
        !make_tmap_plane_f32(&tB, biasL_qk, p.B * p.H, p.N, BQ))
        return cuda_fail(cudaErrorUnknown, "cuTensorMapEncodeTiled");
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3(DQDB_THREADS);
    cfg.dynamicSmemBytes = DqdbSmem::total;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = (unsigned)C; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    const int n_items = p.B * p.H * (p.N / BQ) * G;
    {
        ProfScope ps("sm100_dqdb_kernel", st);
        TRI_CUDA_CHECK(cudaLaunchKernelEx(&cfg, sm100_dqdb_kernel, tQ, tA, tK, tV, tB, p, maskbits, LSE, Dws, (__nv_bfloat16*)dQ,
                                          dBias, planes, G, n_items, kbox));
    }
    TRI_LAUNCH_CHECK("sm100_dqdb_kernel");
    return TRI_OK;
}

}  // namespace tri

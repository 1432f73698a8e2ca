// Stage 2 of the bf16 backward on tcgen05 / TMEM / TMA (sm_100a): dQ and dBias from ONE recomputation of P and dS
// (Listing 2 stage 2; Table I).  The paper adds its dS tiles into dBias with tl.atomic_add
// (P:L488); here the reduction over the broadcast rows is deterministic and on-chip:
//
//   * tile-stationary: a CTA owns the dBias tiles (128 queries x up to 2 x 64 keys) of one (b, h) in REGISTERS and
//     streams over the broadcast rows r in ascending order (level 1 of the dBias reduction; level 2, only when the
//     row axis is split over G CTAs to fill the SMs, is sm100_dbias_reduce_kernel);
//   * the CTAs that own the key tiles of one 128-query block form a thread-block CLUSTER; each accumulates its
//     partial dQ_r = sum over its keys of dS K in TMEM, and the partials of a row are added in rank order through
//     distributed shared memory (rank c receives the running sum of ranks < c, adds its own, passes it on; the last
//     rank scales and stores dQ).  No floating-point atomics anywhere; every output is bitwise reproducible.
//     A cluster has at most 16 ranks = 2048 keys; N > 2048 runs ceil(N / 2048) launches over slices of the key axis
//     (DqdbPass, template flag kPasses): dBias columns are disjoint per slice, dQ is carried as an fp32 sum in global memory.
//
// Persistent, warp-specialised CTA of 512 threads:
//   warps 0-7    two compute groups (128 threads = 128 query rows = 128 TMEM lanes); group g owns key tile g of the CTA,
//                keeps its fp32 log2e*bias tile and its dBias tile in REGISTERS for the whole work item, and walks the two
//                32-key halves of the tile per row (S / dP ping-pong in TMEM, so the MMAs of one half run under the math
//                of the other): p = exp2(S*scale*log2e + log2e*bias - LSE*log2e), dS = p (dP - D), dBias += dS,
//                dS -> bf16 -> TMEM;
//   warp 8       feeder: TMA of Q_r, dA_r (128 x 32) and K_r, V_r (128 x 32) into a 3-stage ring, the bias tiles of the
//                groups per work item, and the shared memory -> TMEM copy (tcgen05.cp) of Q_r, dA_r one row ahead;
//   warps 9-10   one S / dP issuer per group: S = Q K^T, dP = dA V^T per half (TS form: A = Q_r / dA_r in TMEM, so shared
//                memory only serves the 32-key B operands);
//   warp 11      dQ issuer: dQ += dS K (TS, M128 N32 K2x16) in a fixed (half, group) order into one of four accumulators.
//                (Measured on this B200: one thread issues a tcgen05.mma every ~50 clk, a tcgen05.cp every ~107 clk and a
//                tcgen05.commit every ~142 clk, and different warps issue concurrently -- so the tensor work of a row is
//                spread over four warps and commits are kept to one per hand-off.)
//   warps 12-15  dQ reducer: partial dQ of a row: TMEM -> registers -> + inbox -> next rank's inbox (st.async into
//                distributed shared memory, completion counted on the receiver's mbarrier) or, on the last rank, global.
#include <cuda_runtime.h>

#include "sm100_common.cuh"
#include "tri_common.cuh"

namespace tri {
using namespace sm100;

namespace {

constexpr int NGB = 2;                                    // compute groups (64-key tiles) per CTA
constexpr int BQ = 128, BK = 64, BH = 32, DH = 32;        // BH: keys per half tile (one MMA / softmax unit)
constexpr int NST = 3;                                    // operand ring stages (one broadcast row each)
constexpr int QT_BYTES = BQ * DH * 2;                     // 8 KB
constexpr int KT_BYTES = BK * DH * 2;                     // 4 KB
constexpr int STAGE_BYTES = 2 * QT_BYTES + 2 * NGB * KT_BYTES;  // Q, dA, K[128], V[128] = 32 KB
constexpr int BIAS_BYTES = BQ * BK * 4;                   // 32 KB per group: two [128 q][32 k] fp32 boxes, SWIZZLE_128B
constexpr int INBOX_BYTES = BQ * DH * 4;                  // 16 KB: running dQ sum of the lower ranks
constexpr int NIN = 2;                                    // inbox ring depth
constexpr int DQDB_THREADS = (NGB + 2) * 128;
// TMEM columns: group g at 160 g: half h at +80 h: S [0,32) | dP [32,64) | dS bf16 [64,80)
constexpr int TM_GROUP = 160, TM_HALF = 80;
constexpr int NDQ = 4;                                    // dQ accumulators in flight (rows the reducer may lag behind)
constexpr int TM_DQ = NGB * TM_GROUP;                     // NDQ 32-column dQ accumulators
constexpr int TM_QA = TM_DQ + NDQ * 32;                         // two buffers of Q bf16 [0,16) | dA bf16 [16,32)

struct DqdbSmem {
    static constexpr int op_off = 0;
    static constexpr int bias_off = op_off + NST * STAGE_BYTES;
    static constexpr int inbox_off = bias_off + NGB * BIAS_BYTES;
    static constexpr int bar_off = inbox_off + NIN * INBOX_BYTES;
    static constexpr int b_full = 0;                      // [NST] TMA -> issuer, stager
    static constexpr int b_free = b_full + NST;           // [NST] MMAs of the row done -> producer
    static constexpr int b_bias_full = b_free + NST;
    static constexpr int b_bias_free = b_bias_full + 1;
    static constexpr int b_s_full = b_bias_free + 1;      // [NGB][2] S, dP of the half in TMEM
    static constexpr int b_consumed = b_s_full + 2 * NGB; // [NGB][2] S, dP of the half are in registers
    static constexpr int b_ds_ready = b_consumed + 2 * NGB;  // [NGB][2] dS of the half in TMEM
    static constexpr int b_qa_ready = b_ds_ready + 2 * NGB;  // [2] Q_r, dA_r of a row copied into TMEM
    static constexpr int b_qa_free = b_qa_ready + 2;         // [2] every S / dP MMA that reads the buffer has completed
    static constexpr int b_dq_full = b_qa_free + 2;       // [NDQ] partial dQ of the row complete (= its dS halves are free)
    static constexpr int b_dq_free = b_dq_full + NDQ;     // [NDQ] reducer has it in registers
    static constexpr int b_in_full = b_dq_free + NDQ;       // [NIN] lower rank's st.async bytes landed in my inbox slot
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
// 16-byte asynchronous store into a peer's shared memory; its bytes are counted on the peer's mbarrier (no fences)
__device__ __forceinline__ void st_async_v4(uint32_t addr, float a, float b, float c, float d, uint32_t mbar) {
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v4.f32 [%0], {%1, %2, %3, %4}, [%5];"
                 ::"r"(addr), "f"(a), "f"(b), "f"(c), "f"(d), "r"(mbar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_remote(uint32_t addr) {  // credit return: no data is published by it
    asm volatile("mbarrier.arrive.relaxed.cluster.shared::cluster.b64 _, [%0];" ::"r"(addr) : "memory");
}

// 16 key columns of one query row: x = S*scale*log2e + log2e*bias (+ -inf mask), p = exp2(x - LSE*log2e), dS = p (dP - D);
// dBias accumulators += dS (fp32), dS -> bf16 pairs.  sr / dp: raw fp32 bits of S / dP from TMEM.
__device__ __forceinline__ void dqdb_chunk(const uint32_t (&sr)[16], const uint32_t (&dp)[16], uint32_t (&dsb)[8], uint64_t* acc2,
                                           const uint64_t* bias2, uint64_t sl2, uint64_t nl2, uint64_t nd2, uint32_t mc, bool masked) {
#pragma unroll
    for (int e = 0; e < 8; ++e) {
        float x0, x1;
        unpack2(fma2(pack2(__uint_as_float(sr[e * 2]), __uint_as_float(sr[e * 2 + 1])), sl2, bias2[e]), x0, x1);
        if (masked) {
            if (!((mc >> (e * 2)) & 1u)) x0 = -INFINITY;
            if (!((mc >> (e * 2 + 1)) & 1u)) x1 = -INFINITY;
        }
        float a0, a1, s0, s1;
        unpack2(add2(pack2(x0, x1), nl2), a0, a1);
        const uint64_t p2 = pack2(ex2(a0), ex2(a1));
        const uint64_t ds2 = mul2(p2, add2(pack2(__uint_as_float(dp[e * 2]), __uint_as_float(dp[e * 2 + 1])), nd2));
        acc2[e] = add2(acc2[e], ds2);
        unpack2(ds2, s0, s1);
        dsb[e] = pack_bf16(s0, s1);
    }
}

struct Item2 { int b, h, q0, rb; };
// query block fastest: clusters that run concurrently work on the same rows (K_r, V_r shared through L2)
template <bool kAligned>
__device__ __forceinline__ Item2 decode_item2(int item, int N, int H, int G, int NR) {
    Item2 it;
    const int NQB = kAligned ? N / BQ : (N + BQ - 1) / BQ;
    it.q0 = (item % NQB) * BQ;
    int t = item / NQB;
    it.rb = (t % G) * NR;
    const int bh = t / G;
    it.b = bh / H;
    it.h = bh % H;
    return it;
}

// kAligned: N % 128 == 0 (no partial tile anywhere: the bounds checks fold away).  kPasses: N > 2048, the launch covers a
// slice of the key axis (`pass`) and dQ is carried between the launches; false keeps that code out of the common kernel.
template <bool kAligned, bool kPasses>
__global__ void __launch_bounds__(DQDB_THREADS, 1)
sm100_dqdb_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmA,
                  const __grid_constant__ CUtensorMap tmK, const __grid_constant__ CUtensorMap tmV,
                  const __grid_constant__ CUtensorMap tmBias, Problem p, const unsigned long long* __restrict__ maskbits,
                  const float* __restrict__ LSE, const float* __restrict__ Dws, __nv_bfloat16* __restrict__ dQ,
                  float* __restrict__ dBias, float* __restrict__ planes, int G, int n_items, int kbox, DqdbPass pass) {
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
    uint64_t* consumed = bars + L::b_consumed;
    uint64_t* ds_ready = bars + L::b_ds_ready;
    uint64_t* qa_ready = bars + L::b_qa_ready;
    uint64_t* qa_free = bars + L::b_qa_free;
    uint64_t* dq_full = bars + L::b_dq_full;
    uint64_t* dq_free = bars + L::b_dq_free;
    uint64_t* in_full = bars + L::b_in_full;
    uint64_t* out_free = bars + L::b_out_free;
    uint32_t* tmem_slot = (uint32_t*)(bars + L::n_bars);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int N = p.N, NW = kAligned ? N / BK : (N + BK - 1) / BK;  // the last tile / query block may be partial (TMA zero-fill + mask bits)
    const int C = (int)cluster_nctarank(), c = (int)cluster_ctarank();
    // key tiles of this rank: the pass's tiles (all N/64 of them when N <= 2048) are dealt to the C ranks as evenly as
    // possible (at most NGB each)
    const int ptiles = kPasses ? pass.tiles : NW, pbase = kPasses ? pass.tile_base : 0;
    const int base_t = ptiles / C, rem_t = ptiles % C;
    const int nt = base_t + (c < rem_t ? 1 : 0);
    const int t0 = pbase + c * base_t + (c < rem_t ? c : rem_t);
    const int k0 = t0 * BK;
    const int NR = p.R / G;  // broadcast rows per work item
    const int cid = (int)blockIdx.x / C, ncl = (int)gridDim.x / C;
    const int n_my = (n_items - cid + ncl - 1) / ncl;
    const int NRtot = n_my * NR;

    if (tid == 0) {
        prefetch_tmap(&tmQ); prefetch_tmap(&tmA); prefetch_tmap(&tmK); prefetch_tmap(&tmV); prefetch_tmap(&tmBias);
        for (int i = 0; i < NST; ++i) { mbar_init(full + i, 1); mbar_init(freeb + i, 1); }
        mbar_init(bias_full, 1);
        mbar_init(bias_free, nt * 4);
        for (int i = 0; i < 2 * NGB; ++i) {
            mbar_init(s_full + i, 1); mbar_init(consumed + i, 4); mbar_init(ds_ready + i, 4);
        }
        for (int i = 0; i < 2; ++i) { mbar_init(qa_ready + i, 1); mbar_init(qa_free + i, nt * 4); }
        for (int i = 0; i < NDQ; ++i) { mbar_init(dq_full + i, 1); mbar_init(dq_free + i, 4); }
        for (int i = 0; i < NIN; ++i) { mbar_init(in_full + i, 1); mbar_init(out_free + i, 4); }
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
        const uint32_t opbase = smem_u32(sOp);
        if (warp == NGB * 4) {
            // ---- feeder: TMA loads NST - 1 rows ahead, tcgen05.cp of Q_r / dA_r one row ahead ----
            auto stage_qa = [&](int m) {  // Q_r, dA_r of row m (this CTA's m-th row): ring stage -> TMEM buffer m & 1
                const int s = m % NST;
                mbar_wait(full + s, (m / NST) & 1);
                if (m >= 2) mbar_wait(qa_free + (m & 1), ((m >> 1) - 1) & 1);  // the S / dP MMAs of row m - 2 are done with it
                tc_fence_after();
                const uint32_t st = opbase + s * STAGE_BYTES;
                const uint64_t dq = make_desc_sw64(st), da = make_desc_sw64(st + QT_BYTES);
                const uint32_t tQ = tmem + TM_QA + (m & 1) * 32;
                if (elect_one()) {
                    tmem_cp_128x256b(tQ, dq);
                    tmem_cp_128x256b(tQ + 8, dq + 2);
                    tmem_cp_128x256b(tQ + 16, da);
                    tmem_cp_128x256b(tQ + 24, da + 2);
                    mma_commit(qa_ready + (m & 1));
                }
                __syncwarp();
            };
            int n = 0;
            for (int il = 0; il < n_my; ++il) {
                const Item2 it = decode_item2<kAligned>(cid + il * ncl, N, p.H, G, NR);
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
                    // the row loaded NST - 2 iterations ago goes to TMEM (its TMA has landed; it is one row ahead of the MMAs)
                    if (n >= NST - 2) stage_qa(n - (NST - 2));
                }
            }
            for (int m = (NRtot > NST - 2 ? NRtot - (NST - 2) : 0); m < NRtot; ++m) stage_qa(m);
        } else if (warp <= NGB * 4 + NGB) {
            // ---- S / dP issuer of group g (warp-uniform control flow; one elected lane issues and commits) ----
            const int g = warp - (NGB * 4 + 1);
            constexpr uint32_t idesc = make_idesc(128, BH, false, false);  // B = K / V rows, K-major
            if (g < nt) {
                int s = 0;
                for (int n = 0; n < NRtot; ++n) {
                    mbar_wait(qa_ready + (n & 1), (n >> 1) & 1);  // Q_r, dA_r in TMEM (this also means the row's TMA has landed)
                    for (int h = 0; h < 2; ++h) {
                        if (n > 0) mbar_wait(consumed + g * 2 + h, (n - 1) & 1);
                        tc_fence_after();
                        const uint32_t st = opbase + s * STAGE_BYTES + 2 * QT_BYTES + g * KT_BYTES + h * (BH * DH * 2);
                        const uint64_t dk = make_desc_sw64(st), dv = make_desc_sw64(st + NGB * KT_BYTES);
                        const uint32_t tS = tmem + g * TM_GROUP + h * TM_HALF, tDP = tS + 32;
                        const uint32_t tQ = tmem + TM_QA + (n & 1) * 32, tA = tQ + 16;
                        if (elect_one()) {
                            mma_ts(tS, tQ, dk, idesc, 0);
                            mma_ts(tS, tQ + 8, dk + 2, idesc, 1);
                            mma_ts(tDP, tA, dv, idesc, 0);
                            mma_ts(tDP, tA + 8, dv + 2, idesc, 1);
                            mma_commit(s_full + g * 2 + h);
                        }
                        __syncwarp();
                    }
                    if (++s == NST) s = 0;
                }
            }
        } else {
            // ---- dQ issuer: dQ_r += dS(g, h) K_r[keys 32h .. 32h+31 of tile g], strictly in (row, half, group) order ----
            constexpr uint32_t idescO = make_idesc(128, DH, false, true);  // B = K rows as [key][d], MN-major
            int s = 0;
            for (int n = 0; n < NRtot; ++n) {
                const int j = n % NDQ;
                for (int h = 0; h < 2; ++h)
                    for (int g = 0; g < nt; ++g) {
                        const bool first = h == 0 && g == 0, last = h == 1 && g == nt - 1;
                        mbar_wait(ds_ready + g * 2 + h, n & 1);
                        if (first && n >= NDQ) mbar_wait(dq_free + j, ((n / NDQ) - 1) & 1);
                        tc_fence_after();
                        // 16 keys of the MN-major B operand = 1024 bytes
                        const uint64_t dk = make_desc_sw64(opbase + s * STAGE_BYTES + 2 * QT_BYTES + g * KT_BYTES + h * (BH * DH * 2));
                        const uint32_t tDS = tmem + g * TM_GROUP + h * TM_HALF + 64, tDQ = tmem + TM_DQ + j * 32;
                        if (elect_one()) {
                            mma_ts(tDQ, tDS, dk, idescO, first ? 0u : 1u);
                            mma_ts(tDQ, tDS + 8, dk + 64, idescO, 1u);
                            if (last) {
                                // one commit per hand-off: the row's partial dQ is complete -- which also tells the compute
                                // groups that every dS half of the row has been read -- and the ring stage is free (the
                                // S / dP MMAs and copies of the row completed before its dS existed)
                                mma_commit(dq_full + j);
                                mma_commit(freeb + s);
                            }
                        }
                        __syncwarp();
                    }
                if (++s == NST) s = 0;
            }
        }
    } else if (warp < NGB * 4) {
        // =============================== compute groups ===============================
        setmaxnreg_inc<200>();
        const int g = warp >> 2;
        if (g < nt) {
            const int row = tid & 127;  // query row inside the block = TMEM lane
            const uint32_t lane_off = (uint32_t)((warp & 3) * 32) << 16;
            const uint32_t tG = tmem + g * TM_GROUP + lane_off;
            const float sl = rsqrtf((float)DH) * kLog2e;
            const uint64_t sl2 = pack2(sl, sl);
            const uint8_t* brow = sBias + g * BIAS_BYTES + row * 128;
            const int sw = row & 7;
            const int tile = t0 + g;
            uint64_t acc2[BK / 2], bias2[BK / 2];
#pragma unroll
            for (int i = 0; i < BK / 2; ++i) acc2[i] = pack2(0.0f, 0.0f);
            int n = 0;
            for (int il = 0; il < n_my; ++il) {
                const Item2 it = decode_item2<kAligned>(cid + il * ncl, N, p.H, G, NR);
                const float* lp = LSE + (long long)it.b * p.lB + (long long)it.h * N + (long long)(it.q0 + row) * p.lQ +
                                  (long long)it.rb * p.lR;
                const float* dp_ = Dws + (lp - LSE);
                const unsigned long long* mp = maskbits ? maskbits + ((long long)it.b * p.R + it.rb) * NW + tile : nullptr;
                const bool inq = kAligned || it.q0 + row < N;  // queries beyond N (last, partial block): LSE = -inf makes p = dS = 0
                float lse_n = inq ? __ldg(lp) : -INFINITY, dd_n = inq ? __ldg(dp_) : 0.0f;
                uint64_t mb_n = mp ? ldg_u64(mp) : ~0ull;
                // my row of the bias tile -> registers for the whole item; the shared buffer goes back to the producer
                mbar_wait(bias_full, il & 1);
#pragma unroll
                for (int q4 = 0; q4 < 16; ++q4) {
                    const float4 bv = lds128f(brow + (q4 >> 3) * (BIAS_BYTES / 2) + (((q4 & 7) ^ sw) << 4));
                    bias2[q4 * 2] = pack2(bv.x, bv.y);
                    bias2[q4 * 2 + 1] = pack2(bv.z, bv.w);
                }
                fence_proxy_async();  // my generic-proxy reads are complete before the producer's TMA may overwrite the tile
                warp_arrive(bias_free);
                for (int r = 0; r < NR; ++r, ++n) {
                    const float nl = lse_n == -INFINITY ? -INFINITY : -lse_n * kLog2e;
                    const uint64_t nl2 = pack2(nl, nl), nd2 = pack2(-dd_n, -dd_n);
                    const uint64_t mb = mb_n;
                    if (r + 1 < NR) {
                        lp += p.lR; dp_ += p.lR;
                        if (inq) {
                            lse_n = __ldg(lp);
                            dd_n = __ldg(dp_);
                        }
                        if (mp) { mp += NW; mb_n = ldg_u64(mp); }
                    }
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        const uint32_t tS = tG + h * TM_HALF, tDP = tS + 32, tDS = tS + 64;
                        const uint32_t mh = (uint32_t)(mb >> (h * 32));
                        mbar_wait(s_full + g * 2 + h, n & 1);
                        tc_fence_after();
                        if (h == 1) warp_arrive(qa_free + (n & 1));  // my group's S / dP MMAs of the row are complete
                        uint32_t dsb[2][8];
#pragma unroll
                        for (int ch = 0; ch < 2; ++ch) {  // 16 key columns at a time
                            uint32_t sr[16], dp[16];
                            tmem_ld16(tS + ch * 16, sr);
                            tmem_ld16(tDP + ch * 16, dp);
                            tmem_ld_wait();
                            if (ch == 1) {  // S, dP of this half are in registers: the issuer may overwrite the columns
                                tc_fence_before();
                                warp_arrive(consumed + g * 2 + h);
                            }
                            // the select instructions of the mask path are predicated, not branched around: measured faster
                            // (2.39 vs 2.83 ms at cfg4) than a branch-free unmasked copy of the loop
                            dqdb_chunk(sr, dp, dsb[ch], &acc2[h * 16 + ch * 8], &bias2[h * 16 + ch * 8], sl2, nl2, nd2, mh >> (ch * 16),
                                       mh != 0xffffffffu);
                        }
                        if (n > 0) {  // the dQ MMAs of the previous row have read this half's dS columns
                            mbar_wait(dq_full + (n - 1) % NDQ, ((n - 1) / NDQ) & 1);
                            tc_fence_after();
                        }
                        tmem_st8(tDS, dsb[0]);
                        tmem_st8(tDS + 8, dsb[1]);
                        tmem_st_wait();
                        tc_fence_before();
                        warp_arrive(ds_ready + g * 2 + h);
                    }
                }
                // ---- item done: my 64 dBias values of query row q0+row (level-1 sum over rows rb..rb+NR-1, ascending) ----
                float acc[BK];
#pragma unroll
                for (int i = 0; i < BK / 2; ++i) {
                    unpack2(acc2[i], acc[2 * i], acc[2 * i + 1]);
                    acc2[i] = pack2(0.0f, 0.0f);
                }
                const int bh = it.b * p.H + it.h;
                const int nk = kAligned ? BK : N - tile * BK;  // keys of my tile that exist (>= BK except in the last tile; N % 8 == 0)
                if (!inq) {
                    // query row beyond N: nothing to store
                } else if (G > 1) {
                    float* out = planes + ((long long)(it.rb / NR) * p.B * p.H + bh) * N * N + (long long)(it.q0 + row) * N + tile * BK;
#pragma unroll
                    for (int i = 0; i < BK; i += 4)
                        if (i < nk) *(float4*)(out + i) = make_float4(acc[i], acc[i + 1], acc[i + 2], acc[i + 3]);
                } else {
                    float* out = dBias + (long long)bh * N * N + (long long)(it.q0 + row) * p.bQ + (long long)(tile * BK) * p.bK;
                    if (p.bK == 1) {
#pragma unroll
                        for (int i = 0; i < BK; i += 4)
                            if (i < nk) *(float4*)(out + i) = make_float4(acc[i], acc[i + 1], acc[i + 2], acc[i + 3]);
                    } else {
#pragma unroll
                        for (int i = 0; i < BK; ++i)
                            if (i < nk) out[(long long)i * p.bK] = acc[i];
                    }
                }
            }
        }
    } else {
        // =============================== dQ reducer warpgroup ===============================
        setmaxnreg_dec<72>();
        const int row = tid & 127;
        const int sw = row & 7;
        const uint32_t lane_off = (uint32_t)((warp & 3) * 32) << 16;
        const float scale = rsqrtf((float)DH);
        const uint32_t inbox_next = (c + 1 < C) ? map_to_rank(smem_u32(sInbox), (uint32_t)(c + 1)) : 0u;
        const uint32_t infull_next = (c + 1 < C) ? map_to_rank(smem_u32(in_full), (uint32_t)(c + 1)) : 0u;
        const uint32_t outfree_prev = (c > 0) ? map_to_rank(smem_u32(out_free), (uint32_t)(c - 1)) : 0u;
        if (c > 0 && tid == (NGB + 1) * 128)  // arm both inbox slots for their first use
            for (int i = 0; i < NIN && i < NRtot; ++i) mbar_expect_tx(in_full + i, INBOX_BYTES);
        int n = 0;
        for (int il = 0; il < n_my; ++il) {
            const Item2 it = decode_item2<kAligned>(cid + il * ncl, N, p.H, G, NR);
            __nv_bfloat16* qp = dQ + (long long)it.b * p.sB + (long long)it.h * p.sH + (long long)it.rb * p.sSlice + (long long)(it.q0 + row) * p.sPos;
            for (int r = 0; r < NR; ++r, ++n, qp += p.sSlice) {
                const int j = n & 1, ph = (n >> 1) & 1;  // inbox slot and its phase
                const int jd = n % NDQ;
                mbar_wait(dq_full + jd, (n / NDQ) & 1);
                tc_fence_after();
                uint32_t v[32];
                tmem_ld32(tmem + TM_DQ + jd * 32 + lane_off, v);
                tmem_ld_wait();
                tc_fence_before();
                warp_arrive(dq_free + jd);
                float f[32];
#pragma unroll
                for (int i = 0; i < 32; ++i) f[i] = __uint_as_float(v[i]);
                if (c > 0) {  // running sum of ranks 0..c-1 (fixed order: deterministic)
                    mbar_wait(in_full + j, ph);
                    const uint8_t* src = sInbox + j * INBOX_BYTES + row * 128;
#pragma unroll
                    for (int i = 0; i < 8; ++i) {
                        const float4 t = lds128f(src + ((i ^ sw) << 4));
                        f[4 * i] = t.x + f[4 * i]; f[4 * i + 1] = t.y + f[4 * i + 1];
                        f[4 * i + 2] = t.z + f[4 * i + 2]; f[4 * i + 3] = t.w + f[4 * i + 3];
                    }
                    // all 128 readers are done with the slot: re-arm it for row n + NIN, then hand the credit back
                    named_bar_sync(1, 128);
                    if (tid == (NGB + 1) * 128 && n + NIN < NRtot) mbar_expect_tx(in_full + j, INBOX_BYTES);
                    if (lane == 0) mbar_arrive_remote(outfree_prev + j * 8);
                }
                if (kPasses && c == 0 && pass.tile_base > 0 && (kAligned || it.q0 + row < N)) {
                    // a later key pass (N > 2048): the running sum starts from what the earlier passes left in global memory
                    const float4* src = (const float4*)(pass.dq_part + (qp - dQ));
#pragma unroll
                    for (int i = 0; i < 8; ++i) {
                        const float4 t = __ldg(src + i);
                        f[4 * i] = t.x + f[4 * i]; f[4 * i + 1] = t.y + f[4 * i + 1];
                        f[4 * i + 2] = t.z + f[4 * i + 2]; f[4 * i + 3] = t.w + f[4 * i + 3];
                    }
                }
                if (c + 1 < C) {
                    if (n >= NIN) mbar_wait(out_free + j, ph ^ 1);
                    const uint32_t dst = inbox_next + j * INBOX_BYTES + row * 128;
#pragma unroll
                    for (int i = 0; i < 8; ++i)
                        st_async_v4(dst + ((i ^ sw) << 4), f[4 * i], f[4 * i + 1], f[4 * i + 2], f[4 * i + 3], infull_next + j * 8);
                } else if (kPasses && !pass.last) {  // last rank of a key pass that is not the last: the fp32 sum goes to global memory
                    if (kAligned || it.q0 + row < N) {
                        float4* dst = (float4*)(pass.dq_part + (qp - dQ));
#pragma unroll
                        for (int i = 0; i < 8; ++i) dst[i] = make_float4(f[4 * i], f[4 * i + 1], f[4 * i + 2], f[4 * i + 3]);
                    }
                } else if (kAligned || it.q0 + row < N) {  // last rank: dQ = scale * sum (queries beyond N: nothing to store)
                    uint4* pq = (uint4*)qp;
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

// the instantiation for a problem size
static auto dqdb_kernel_for(int N) -> decltype(&sm100_dqdb_kernel<true, false>) {
    const bool al = N % 128 == 0, ps = (N + BK - 1) / BK > 16 * NGB;
    return al ? (ps ? sm100_dqdb_kernel<true, true> : sm100_dqdb_kernel<true, false>)
              : (ps ? sm100_dqdb_kernel<false, true> : sm100_dqdb_kernel<false, false>);
}

// Key passes: one cluster covers at most 16 ranks x NGB tiles = 2048 keys, so N > 2048 runs ceil(tiles / 32) launches over
// equal slices of the key axis; dBias columns are disjoint per pass, dQ is carried between passes as an fp32 sum.
int sm100_dqdb_passes(int N) { return ((N + BK - 1) / BK + 16 * NGB - 1) / (16 * NGB); }
DqdbPass sm100_dqdb_pass(int N, int i, float* dq_part) {
    const int T = (N + BK - 1) / BK, np = sm100_dqdb_passes(N), per = (T + np - 1) / np;
    DqdbPass ps;
    ps.tile_base = i * per;
    ps.tiles = T - ps.tile_base < per ? T - ps.tile_base : per;
    ps.last = i == np - 1 ? 1 : 0;
    ps.dq_part = dq_part;
    return ps;
}

// cluster size for T key tiles at <= NGB tiles per rank, from the sizes the launch code accepts
int sm100_dqdb_cluster(int T) {
    const int need = (T + NGB - 1) / NGB;
    const int sizes[] = {1, 2, 3, 4, 6, 8, 12, 16};
    for (int s : sizes)
        if (s >= need) return s;
    return 0;
}

// Launch plan on the current device: cluster size C, row slices G per (b, h, query block) (<= kDqdbMaxSplit, chosen to
// minimise waves * rows per item for the number of clusters the device can hold), persistent grid (a multiple of C).
// Returns false if the kernel cannot run on this device / shape.
bool sm100_dqdb_plan(const Problem& p, int tiles, int forceG, int* Cout, int* Gout, int* grid) {
    const int C = sm100_dqdb_cluster(tiles);
    if (C == 0) return false;
    auto kern = dqdb_kernel_for(p.N);
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, DqdbSmem::total) != cudaSuccess) return false;
    if (C > 8 && cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) != cudaSuccess) return false;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(C * 64));
    cfg.blockDim = dim3(DQDB_THREADS);
    cfg.dynamicSmemBytes = DqdbSmem::total;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = (unsigned)C; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    int ncl = 0;
    if (cudaOccupancyMaxActiveClusters(&ncl, kern, &cfg) != cudaSuccess || ncl <= 0) {
        cudaGetLastError();
        return false;
    }
    const long long base = (long long)p.B * p.H * ((p.N + BQ - 1) / BQ);
    int bestG = 1;
    double best = 1e30;
    for (int G = 1; G <= kDqdbMaxSplit; ++G) {
        if (p.R % G || (forceG > 0 && G != forceG)) continue;
        const double waves = (double)((base * G + ncl - 1) / ncl);
        const double cost = waves * (p.R / G + 12);  // + per-item fill / drain / dBias flush in row units
        if (cost < best * 0.99) { best = cost; bestG = G; }
    }
    const long long items = base * bestG;
    *Cout = C; *Gout = bestG;
    *grid = (int)((items < ncl ? items : ncl) * C);
    return true;
}

tri_status sm100_dqdb_launch(const Problem& p, int C, int G, int grid, const void* Q, const void* dA, const void* K, const void* V,
                             const float* biasL_qk, const unsigned long long* maskbits, const float* LSE, const float* Dws,
                             void* dQ, float* dBias, float* planes, DqdbPass pass, cudaStream_t st) {
    const int kbox = p.N < NGB * BK ? p.N : NGB * BK;
    CUtensorMap tQ, tA, tK, tV, tB;
    if (!make_tmap_u(&tQ, Q, p.B, p.N, p.H, p.d, p.variant, BQ, p.R) || !make_tmap_u(&tA, dA, p.B, p.N, p.H, p.d, p.variant, BQ, p.R) ||
        !make_tmap_u(&tK, K, p.B, p.N, p.H, p.d, p.variant, kbox, p.R) || !make_tmap_u(&tV, V, p.B, p.N, p.H, p.d, p.variant, kbox, p.R) ||
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
    const int n_items = p.B * p.H * ((p.N + BQ - 1) / BQ) * G;
    {
        ProfScope ps("sm100_dqdb_kernel", st);
        TRI_CUDA_CHECK(cudaLaunchKernelEx(&cfg, dqdb_kernel_for(p.N), tQ, tA, tK, tV, tB, p, maskbits, LSE, Dws, (__nv_bfloat16*)dQ,
                                          dBias, planes, G, n_items, kbox, pass));
    }
    TRI_LAUNCH_CHECK("sm100_dqdb_kernel");
    return TRI_OK;
}

}  // namespace tri

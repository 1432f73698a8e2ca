// Stage 1 of the bf16 backward on tcgen05 / TMEM / TMA (sm_100a): dK and dV (Listing 2 stage 1; Table I
// P:L508).  Key-stationary: a work item is (b, h, 128-key block, three broadcast rows); TMEM lane = key.
//
// Persistent, warp-specialised CTA of 512 threads:
//   warps 0-11   three compute groups (128 threads = 128 keys); group g owns row 3t + g of the item and walks the
//                queries of that row in units of 32:
//                  p^T = exp2(S^T*scale*log2e + log2e*bias^T - LSE_q*log2e), dS^T = p^T (dP^T - D_q)  -> bf16 -> TMEM
//                (LSE_q, D_q of the unit's queries come pre-scaled from a small fp32 side array, one broadcast
//                 ld.shared per four columns);
//   warp 12      TMA producer: K_r, V_r (128 x 32) of the three rows per item; per 64 queries a ring stage with Q_r,
//                dA_r (64 x 32) of the three rows, the bf16 bias^T tile [128 k][64 q] they share ("on-the-fly
//                broadcasting") and the LSE / D segments;
//   warps 13-15  one tcgen05 issuer per group: K_r, V_r go shared memory -> TMEM once per item (tcgen05.cp), then per
//                unit S^T = K Q^T, dP^T = V dA^T (TS, M128 N32 K2x16; shared memory only serves the 32-query B operand)
//                and dV += P^T dA, dK += dS^T Q (TS, A = the bf16 tiles the group stored, B = the same Q / dA tiles
//                read MN-major); accumulators dV, dK stay in TMEM for the whole row.
// Row epilogue (compute group): dV, dK -> registers -> bf16 -> global (dK scaled by 1/sqrt(d)).
#include "sm100_common.cuh"
#include "tri_common.cuh"

namespace tri {
using namespace sm100;

namespace {

constexpr int NGK = 3;                                   // compute groups = broadcast rows per work item
constexpr int BKEY = 128, BQS = 64, BU = 32, DH = 32;    // keys per item, queries per ring stage, queries per unit
constexpr int NSTG = 3;                                  // ring stages
constexpr int KV_BYTES = BKEY * DH * 2;                  // 8 KB
constexpr int QS_BYTES = BQS * DH * 2;                   // 4 KB: 64 queries x 32 channels
constexpr int BIAS_BYTES = BKEY * BQS * 2;               // 16 KB: [128 k][64 q] bf16, SWIZZLE_128B
constexpr int LD_BYTES = NGK * 2 * BQS * 4;              // per group: 64 x (-LSE*log2e), 64 x (-D)
constexpr int STAGE_BYTES = ((NGK * 2 * QS_BYTES + BIAS_BYTES + LD_BYTES + 1023) / 1024) * 1024;
constexpr int DKDV_THREADS = (NGK + 1) * 128;
// TMEM columns of group g at 160 g: S^T [0,32) (P^T bf16 over [0,16)) | dP^T [32,64) (dS^T bf16 over [32,48)) |
// dV [64,96) | dK [96,128) | K bf16 [128,144) | V bf16 [144,160)
constexpr int TMG = 160;

struct DkdvSmem {
    static constexpr int kv_off = 0;                                  // NGK x (K, V)
    static constexpr int st_off = kv_off + NGK * 2 * KV_BYTES;        // NSTG stages: NGK x (Q, dA) | bias^T | LD
    static constexpr int bar_off = st_off + NSTG * STAGE_BYTES;
    static constexpr int b_kv_full = 0;                               // [1] K, V of the item landed
    static constexpr int b_kv_free = 1;                               // [1] all groups copied them to TMEM
    static constexpr int b_full = 2;                                  // [NSTG]
    static constexpr int b_free = b_full + NSTG;                      // [NSTG] 3 issuers' MMAs + 12 compute warps
    static constexpr int b_s_full = b_free + NSTG;                    // [NGK] S^T, dP^T of the unit in TMEM
    static constexpr int b_p_ready = b_s_full + NGK;                  // [NGK] P^T, dS^T of the unit in TMEM
    static constexpr int b_acc_full = b_p_ready + NGK;                // [NGK] dV, dK of the row complete
    static constexpr int b_acc_free = b_acc_full + NGK;               // [NGK] the group has them in registers
    static constexpr int b_tok = b_acc_free + NGK;                    // [NGK][4] math-phase token of (group, scheduler quarter)
    static constexpr int n_bars = b_tok + NGK * 4;
    static constexpr int total = bar_off + n_bars * 8 + 16 + 1024;
};

struct ItemK { int b, h, k0, r0; };
// key block fastest: the CTAs that run concurrently share the Q / dA rows of a few row triples (read once from HBM,
// then from L2) instead of streaming the whole pair tensor once per key block
template <bool kAligned>
__device__ __forceinline__ ItemK decode_itemk(int item, int N, int H, int NT3) {
    ItemK it;
    const int NKB = kAligned ? N / BKEY : (N + BKEY - 1) / BKEY;
    it.k0 = (item % NKB) * BKEY;
    int t = item / NKB;
    it.r0 = (t % NT3) * NGK;
    const int bh = t / NT3;
    it.b = bh / H;
    it.h = bh % H;
    return it;
}

// 1-D bulk copy global -> shared, completion counted on an mbarrier (bytes: multiple of 16, both addresses 16-aligned)
__device__ __forceinline__ void bulk_load(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

// 16 query columns of one key row.  sr / dp: raw fp32 S^T / dP^T from TMEM; bw: 8 words = 16 bf16 bias values;
// nl / nd: -LSE*log2e and -D of the 16 queries (shared memory, same address for the whole warp).
__device__ __forceinline__ void dkdv_chunk(const uint32_t (&sr)[16], const uint32_t (&dp)[16], const uint32_t* bw, const float* nl,
                                           const float* nd, uint64_t sl2, uint64_t l2e2, uint32_t* pp, uint32_t* ds) {
#pragma unroll
    for (int c4 = 0; c4 < 4; ++c4) {
        const float4 n4 = lds128f(nl + c4 * 4), d4 = lds128f(nd + c4 * 4);
        const uint64_t nn[2] = {pack2(n4.x, n4.y), pack2(n4.z, n4.w)}, dd[2] = {pack2(d4.x, d4.y), pack2(d4.z, d4.w)};
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            const int c = c4 * 4 + e * 2;
            const uint32_t w = bw[c >> 1];
            const uint64_t t2 = fma2(pack2(bf16_lo(w), bf16_hi(w)), l2e2, nn[e]);
            float a0, a1, s0, s1;
            unpack2(fma2(pack2(__uint_as_float(sr[c]), __uint_as_float(sr[c + 1])), sl2, t2), a0, a1);
            const float p0 = ex2(a0), p1 = ex2(a1);
            unpack2(mul2(pack2(p0, p1), add2(pack2(__uint_as_float(dp[c]), __uint_as_float(dp[c + 1])), dd[e])), s0, s1);
            pp[c >> 1] = pack_bf16(p0, p1);
            ds[c >> 1] = pack_bf16(s0, s1);
        }
    }
}

// kAligned: N % 128 == 0 (no partial tile anywhere: the bounds checks fold away)
template <bool kAligned>
__global__ void __launch_bounds__(DKDV_THREADS, 1)
sm100_dkdv2_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmA,
                   const __grid_constant__ CUtensorMap tmK, const __grid_constant__ CUtensorMap tmV,
                   const __grid_constant__ CUtensorMap tmBiasKQ, Problem p, const unsigned long long* __restrict__ maskbits,
                   const float* __restrict__ NL, const float* __restrict__ ND, __nv_bfloat16* __restrict__ dK,
                   __nv_bfloat16* __restrict__ dV, int item_begin, int total_items) {
    using L = DkdvSmem;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    uint8_t* sKV = smem + L::kv_off;
    uint8_t* sSt = smem + L::st_off;
    uint64_t* bars = (uint64_t*)(smem + L::bar_off);
    uint64_t* kv_full = bars + L::b_kv_full;
    uint64_t* kv_free = bars + L::b_kv_free;
    uint64_t* full = bars + L::b_full;
    uint64_t* freeb = bars + L::b_free;
    uint64_t* s_full = bars + L::b_s_full;
    uint64_t* p_ready = bars + L::b_p_ready;
    uint64_t* acc_full = bars + L::b_acc_full;
    uint64_t* acc_free = bars + L::b_acc_free;
    uint64_t* tok = bars + L::b_tok;
    uint32_t* tmem_slot = (uint32_t*)(bars + L::n_bars);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int N = p.N, NW = kAligned ? N / 64 : (N + 63) / 64;
    const int NT3 = (p.R + NGK - 1) / NGK;  // row triples (the last one may be partial)
    const int NS = kAligned ? N / BQS : (N + BQS - 1) / BQS;   // ring stages per row (the last one may be partial: TMA zero-fills Q / dA / bias^T,
                                          // NL is -inf there, so P^T = dS^T = 0 for queries >= N;
                                          // NL / ND rows are padded to NS * BQS by lse_prep_kernel)
    const int n_items = (total_items - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;

    if (tid == 0) {
        prefetch_tmap(&tmQ); prefetch_tmap(&tmA); prefetch_tmap(&tmK); prefetch_tmap(&tmV); prefetch_tmap(&tmBiasKQ);
        mbar_init(kv_full, 1);
        mbar_init(kv_free, NGK);
        for (int i = 0; i < NSTG; ++i) { mbar_init(full + i, 1); mbar_init(freeb + i, NGK + NGK * 4); }
        for (int i = 0; i < NGK; ++i) {
            mbar_init(s_full + i, 1); mbar_init(p_ready + i, 4); mbar_init(acc_full + i, 1); mbar_init(acc_free + i, 4);
        }
        for (int i = 0; i < NGK * 4; ++i) mbar_init(tok + i, 1);
        fence_barrier_init();
    }
    if (warp == 0) tmem_alloc<512>(tmem_slot);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;

    if (warp >= NGK * 4) {
        // =============================== helper warpgroup ===============================
        setmaxnreg_dec<48>();
        if (warp == NGK * 4) {
            // ---- TMA producer ----
            int n = 0;  // stage counter over the CTA's life
            for (int il = 0; il < n_items; ++il) {
                const ItemK it = decode_itemk<kAligned>(item_begin + (int)blockIdx.x + il * (int)gridDim.x, N, p.H, NT3);
                const int bh = it.b * p.H + it.h;
                const int nr = min(NGK, p.R - it.r0);  // active rows of the item
                if (il > 0) mbar_wait(kv_free, (il - 1) & 1);
                if (elect_one()) {
                    mbar_expect_tx(kv_full, nr * 2 * KV_BYTES);
                    for (int g = 0; g < nr; ++g) {
                        tma_load_5d(sKV + g * 2 * KV_BYTES, &tmK, kv_full, 0, it.k0, it.r0 + g, it.h, it.b);
                        tma_load_5d(sKV + g * 2 * KV_BYTES + KV_BYTES, &tmV, kv_full, 0, it.k0, it.r0 + g, it.h, it.b);
                    }
                }
                __syncwarp();
                for (int sq = 0; sq < NS; ++sq, ++n) {
                    const int s = n % NSTG;
                    if (n >= NSTG) mbar_wait(freeb + s, ((n / NSTG) - 1) & 1);
                    if (elect_one()) {
                        uint8_t* st = sSt + s * STAGE_BYTES;
                        mbar_expect_tx(full + s, nr * (2 * QS_BYTES + 2 * BQS * 4) + BIAS_BYTES);
                        for (int g = 0; g < nr; ++g) {
                            tma_load_5d(st + g * 2 * QS_BYTES, &tmQ, full + s, 0, sq * BQS, it.r0 + g, it.h, it.b);
                            tma_load_5d(st + g * 2 * QS_BYTES + QS_BYTES, &tmA, full + s, 0, sq * BQS, it.r0 + g, it.h, it.b);
                            const long long o = ((((long long)it.b * p.R + it.r0 + g) * p.H + it.h) * NS + sq) * BQS;  // row pitch NS * BQS
                            float* ld = (float*)(st + NGK * 2 * QS_BYTES + BIAS_BYTES) + g * 2 * BQS;
                            bulk_load(ld, NL + o, BQS * 4, full + s);
                            bulk_load(ld + BQS, ND + o, BQS * 4, full + s);
                        }
                        tma_load_3d(st + NGK * 2 * QS_BYTES, &tmBiasKQ, full + s, sq * BQS, it.k0, bh);
                    }
                    __syncwarp();
                }
            }
        } else {
            // ---- tcgen05 issuer of group g (warp-uniform control flow; one elected lane issues and commits) ----
            const int g = warp - (NGK * 4 + 1);
            constexpr uint32_t idescS = make_idesc(128, BU, false, false);  // B = Q / dA rows, K-major
            constexpr uint32_t idescO = make_idesc(128, DH, false, true);   // B = dA / Q as [query][d], MN-major
            const uint32_t tG = tmem + g * TMG, tS = tG, tDP = tG + 32, tDV = tG + 64, tDK = tG + 96, tK = tG + 128, tV = tG + 144;
            const uint32_t stbase = smem_u32(sSt), kvbase = smem_u32(sKV) + g * 2 * KV_BYTES;
            int n = 0;   // stage counter
            int un = 0;  // unit counter (barrier phases of s_full / p_ready)
            int ia = 0;  // rows this group has processed (barrier phases of acc_full / acc_free)
            for (int il = 0; il < n_items; ++il) {
                const ItemK it = decode_itemk<kAligned>(item_begin + (int)blockIdx.x + il * (int)gridDim.x, N, p.H, NT3);
                const bool active = it.r0 + g < p.R;
                mbar_wait(kv_full, il & 1);
                tc_fence_after();
                if (active) {
                    const uint64_t dk = make_desc_sw64(kvbase), dv = make_desc_sw64(kvbase + KV_BYTES);
                    if (elect_one()) {
                        tmem_cp_128x256b(tK, dk);
                        tmem_cp_128x256b(tK + 8, dk + 2);
                        tmem_cp_128x256b(tV, dv);
                        tmem_cp_128x256b(tV + 8, dv + 2);
                        mma_commit(kv_free);  // the copies have read the shared-memory tiles
                    }
                    __syncwarp();
                } else {
                    if (elect_one()) mbar_arrive(kv_free);
                    __syncwarp();
                }
                for (int sq = 0; sq < NS; ++sq, ++n) {
                    const int s = n % NSTG;
                    mbar_wait(full + s, (n / NSTG) & 1);
                    tc_fence_after();
                    if (!active) {  // keep the ring's arrival count: this group has nothing to read in the stage
                        if (elect_one()) mbar_arrive(freeb + s);
                        __syncwarp();
                        continue;
                    }
                    const uint32_t st = stbase + s * STAGE_BYTES + g * 2 * QS_BYTES;
#pragma unroll
                    for (int hu = 0; hu < 2; ++hu, ++un) {
                        const int u = sq * 2 + hu;  // unit inside the row
                        const uint64_t dq = make_desc_sw64(st + hu * (BU * DH * 2)), da = make_desc_sw64(st + QS_BYTES + hu * (BU * DH * 2));
                        if (u > 0) {
                            // previous unit's P^T, dS^T are in TMEM: accumulate dV, dK with the previous unit's dA / Q tiles
                            const int sp = hu ? s : (n + NSTG - 1) % NSTG;
                            const uint32_t stp = stbase + sp * STAGE_BYTES + g * 2 * QS_BYTES + (hu ^ 1) * (BU * DH * 2);
                            const uint64_t dqp = make_desc_sw64(stp), dap = make_desc_sw64(stp + QS_BYTES);
                            mbar_wait(p_ready + g, (un - 1) & 1);
                            tc_fence_after();
                            if (elect_one()) {
                                mma_ts(tDV, tS, dap, idescO, u > 1 ? 1u : 0u);
                                mma_ts(tDV, tS + 8, dap + 64, idescO, 1u);
                                mma_ts(tDK, tDP, dqp, idescO, u > 1 ? 1u : 0u);
                                mma_ts(tDK, tDP + 8, dqp + 64, idescO, 1u);
                                if (hu == 0) mma_commit(freeb + sp);  // last reader of the previous stage's Q / dA tiles
                            }
                            __syncwarp();
                        }
                        if (elect_one()) {
                            mma_ts(tS, tK, dq, idescS, 0);
                            mma_ts(tS, tK + 8, dq + 2, idescS, 1);
                            mma_ts(tDP, tV, da, idescS, 0);
                            mma_ts(tDP, tV + 8, da + 2, idescS, 1);
                            mma_commit(s_full + g);
                        }
                        __syncwarp();
                    }
                }
                if (active) {
                    // last unit of the row
                    const int sp = (n + NSTG - 1) % NSTG;
                    const uint32_t stp = stbase + sp * STAGE_BYTES + g * 2 * QS_BYTES + (BU * DH * 2);
                    const uint64_t dqp = make_desc_sw64(stp), dap = make_desc_sw64(stp + QS_BYTES);
                    mbar_wait(p_ready + g, (un - 1) & 1);
                    tc_fence_after();
                    if (elect_one()) {
                        mma_ts(tDV, tS, dap, idescO, 1u);
                        mma_ts(tDV, tS + 8, dap + 64, idescO, 1u);
                        mma_ts(tDK, tDP, dqp, idescO, 1u);
                        mma_ts(tDK, tDP + 8, dqp + 64, idescO, 1u);
                        mma_commit(freeb + sp);
                        mma_commit(acc_full + g);
                    }
                    __syncwarp();
                    // the group reads dV, dK out before the next row's MMAs overwrite them
                    mbar_wait(acc_free + g, ia & 1);
                    ++ia;
                }
            }
        }
    } else {
        // =============================== compute groups ===============================
        setmaxnreg_inc<144>();
        const int g = warp >> 2;
        const int row = tid & 127;  // key inside the block = TMEM lane
        const uint32_t lane_off = (uint32_t)((warp & 3) * 32) << 16;
        const uint32_t tG = tmem + g * TMG + lane_off, tS = tG, tDP = tG + 32, tDV = tG + 64, tDK = tG + 96;
        const float scale = rsqrtf((float)DH);
        const float sl = scale * kLog2e;
        const uint64_t sl2 = pack2(sl, sl), l2e2 = pack2(kLog2e, kLog2e);
        const int sw = row & 7;
        int n = 0, un = 0, ia = 0;  // stage, unit and active-item counters
        int ut = 0;                  // units seen (active or not): phase of the math-phase token
        uint64_t* my_tok = tok + g * 4 + (warp & 3);
        uint64_t* next_tok = tok + ((g + 1) % NGK) * 4 + (warp & 3);
        for (int il = 0; il < n_items; ++il) {
            const ItemK it = decode_itemk<kAligned>(item_begin + (int)blockIdx.x + il * (int)gridDim.x, N, p.H, NT3);
            const int r = it.r0 + g;
            const bool active = r < p.R;
            bool keep = kAligned || it.k0 + row < N;  // keys beyond N of the last (partial) key block are TMA zero-fill
            if (active && keep && maskbits)
                keep = (ldg_u64(maskbits + ((long long)it.b * p.R + r) * NW + (it.k0 + row) / 64) >> ((it.k0 + row) & 63)) & 1ull;
            const bool allkeep = __all_sync(0xffffffffu, keep);
            for (int sq = 0; sq < NS; ++sq, ++n) {
                const int s = n % NSTG;
                mbar_wait(full + s, (n / NSTG) & 1);
                if (active) {
                    const uint8_t* st = sSt + s * STAGE_BYTES;
                    const uint8_t* brow = st + NGK * 2 * QS_BYTES + row * 128;
                    const float* ld = (const float*)(st + NGK * 2 * QS_BYTES + BIAS_BYTES) + g * 2 * BQS;
#pragma unroll
                    for (int hu = 0; hu < 2; ++hu, ++un, ++ut) {
                        uint32_t bw[16];
#pragma unroll
                        for (int j = 0; j < 4; ++j) {
                            const uint4 v = lds128(brow + (((hu * 4 + j) ^ sw) << 4));
                            bw[4 * j] = v.x; bw[4 * j + 1] = v.y; bw[4 * j + 2] = v.z; bw[4 * j + 3] = v.w;
                        }
                        mbar_wait(s_full + g, un & 1);
                        tc_fence_after();
                        uint32_t sr[32], dp[32], pp[16], ds[16];
                        tmem_ld32(tS, sr);
                        tmem_ld32(tDP, dp);
                        tmem_ld_wait();
                        // The three groups' warps of one scheduler share its MUFU unit.  Left alone they run their exp phases
                        // at the same time (each at a third of the rate) and then wait for their MMAs at the same time; the
                        // token makes the exp phases take turns, so one group's MMA round trip hides under the others' math.
                        if (g > 0 || ut > 0) mbar_wait(my_tok, (g > 0 ? ut : ut - 1) & 1);
                        dkdv_chunk(*(const uint32_t(*)[16])&sr[0], *(const uint32_t(*)[16])&dp[0], bw, ld + hu * BU, ld + BQS + hu * BU, sl2,
                                   l2e2, pp, ds);
                        dkdv_chunk(*(const uint32_t(*)[16])&sr[16], *(const uint32_t(*)[16])&dp[16], bw + 8, ld + hu * BU + 16,
                                   ld + BQS + hu * BU + 16, sl2, l2e2, pp + 8, ds + 8);
                        if (lane == 0) mbar_arrive(next_tok);
                        if (!allkeep && !keep) {  // masked key: its whole row of P^T and dS^T is zero
#pragma unroll
                            for (int e = 0; e < 16; ++e) { pp[e] = 0u; ds[e] = 0u; }
                        }
                        tmem_st16(tS, pp);    // P^T  (bf16 pairs) over the S^T columns already read
                        tmem_st16(tDP, ds);   // dS^T (bf16 pairs) over the dP^T columns already read
                        tmem_st_wait();
                        tc_fence_before();
                        warp_arrive(p_ready + g);
                    }
                } else {
                    // a row group without a row in this item still passes the token on, once per unit
                    for (int hu = 0; hu < 2; ++hu, ++ut) {
                        if (g > 0 || ut > 0) mbar_wait(my_tok, (g > 0 ? ut : ut - 1) & 1);
                        if (lane == 0) mbar_arrive(next_tok);
                    }
                }
                // my generic-proxy reads of the stage (bias^T, LSE / D) are complete before the producer may refill it
                fence_proxy_async();
                warp_arrive(freeb + s);
            }
            if (active) {
                // ---- row epilogue: dV, dK (scaled) -> bf16 -> global ----
                mbar_wait(acc_full + g, ia & 1);
                ++ia;
                tc_fence_after();
                uint32_t v[32], k[32];
                tmem_ld32(tDV, v);
                tmem_ld32(tDK, k);
                tmem_ld_wait();
                tc_fence_before();
                warp_arrive(acc_free + g);
                const long long off = (long long)it.b * p.sB + (long long)it.h * p.sH + (long long)r * p.sSlice + (long long)(it.k0 + row) * p.sPos;
                uint4* pv = (uint4*)(dV + off);
                uint4* pk = (uint4*)(dK + off);
                if (!kAligned && it.k0 + row >= N) continue;  // keys beyond N of the last (partial) key block: nothing to store
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    uint32_t a[4], c[4];
#pragma unroll
                    for (int e = 0; e < 4; ++e) {
                        a[e] = pack_bf16(__uint_as_float(v[j * 8 + 2 * e]), __uint_as_float(v[j * 8 + 2 * e + 1]));
                        c[e] = pack_bf16(__uint_as_float(k[j * 8 + 2 * e]) * scale, __uint_as_float(k[j * 8 + 2 * e + 1]) * scale);
                    }
                    pv[j] = make_uint4(a[0], a[1], a[2], a[3]);
                    pk[j] = make_uint4(c[0], c[1], c[2], c[3]);
                }
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc<512>(tmem);
}

// -LSE*log2e (-inf for fully masked queries) and -D as [B][row][H][query] in the variant's (row, query) sense, so a unit's
// 32 queries are contiguous for both variants.  The query axis is padded to whole 64-query stages with NL = -inf, ND = 0.
__global__ void __launch_bounds__(256) lse_prep_kernel(const float* __restrict__ LSE, const float* __restrict__ Dws,
                                                       float* __restrict__ NL, float* __restrict__ ND, Problem p) {
    const int NPQ = (p.N + BQS - 1) / BQS * BQS;
    const long long total = (long long)p.B * p.R * p.H * NPQ;
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= total) return;
    const int q = (int)(i % NPQ);
    long long t = i / NPQ;
    if (q >= p.N) {
        NL[i] = -INFINITY;
        ND[i] = 0.0f;
        return;
    }
    const int h = (int)(t % p.H);
    t /= p.H;
    const int r = (int)(t % p.R);
    const int b = (int)(t / p.R);
    const long long src = (long long)b * p.lB + (long long)h * p.N + (long long)r * p.lR + (long long)q * p.lQ;
    const float l = __ldg(LSE + src);
    NL[i] = l == -INFINITY ? -INFINITY : -l * kLog2e;
    ND[i] = -__ldg(Dws + src);
}

}  // namespace

size_t sm100_dkdv2_aux_bytes(const Problem& p) { return align_up((size_t)p.B * p.R * p.H * ((p.N + BQS - 1) / BQS * BQS) * 4, 256); }

long long sm100_dkdv2_items(const Problem& p) { return (long long)p.B * p.H * ((p.N + BKEY - 1) / BKEY) * ((p.R + NGK - 1) / NGK); }

tri_status sm100_lse_prep(const Problem& p, const float* LSE, const float* Dws, float* NL, float* ND, cudaStream_t st) {
    const long long total = (long long)p.B * p.R * p.H * ((p.N + BQS - 1) / BQS * BQS);
    {
        ProfScope ps("lse_prep_kernel", st);
        lse_prep_kernel<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(LSE, Dws, NL, ND, p);
    }
    TRI_LAUNCH_CHECK("lse_prep_kernel");
    return TRI_OK;
}

// work items [item_begin, item_begin + item_count) on at most max_ctas persistent CTAs
tri_status sm100_dkdv2_launch(const Problem& p, const void* Q, const void* dA, const void* K, const void* V, const void* bias_kq,
                              const unsigned long long* maskbits, const float* NL, const float* ND, void* dK, void* dV,
                              long long item_begin, long long item_count, int max_ctas, const char* prof_name, cudaStream_t st) {
    if (item_count <= 0) return TRI_OK;
    CUtensorMap tQ, tA, tK, tV, tB;
    if (!make_tmap_u(&tQ, Q, p.B, p.N, p.H, p.d, p.variant, BQS, p.R) || !make_tmap_u(&tA, dA, p.B, p.N, p.H, p.d, p.variant, BQS, p.R) ||
        !make_tmap_u(&tK, K, p.B, p.N, p.H, p.d, p.variant, BKEY, p.R) || !make_tmap_u(&tV, V, p.B, p.N, p.H, p.d, p.variant, BKEY, p.R) ||
        !make_tmap_plane(&tB, bias_kq, p.B * p.H, p.N, BKEY))
        return cuda_fail(cudaErrorUnknown, "cuTensorMapEncodeTiled");
    auto kern = p.N % 128 == 0 ? sm100_dkdv2_kernel<true> : sm100_dkdv2_kernel<false>;
    TRI_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, DkdvSmem::total));
    const int grid = (int)(item_count < max_ctas ? item_count : max_ctas);
    {
        ProfScope ps(prof_name, st);
        kern<<<grid, DKDV_THREADS, DkdvSmem::total, st>>>(tQ, tA, tK, tV, tB, p, maskbits, NL, ND, (__nv_bfloat16*)dK, (__nv_bfloat16*)dV,
                                                          (int)item_begin, (int)item_count);
    }
    TRI_LAUNCH_CHECK("sm100_dkdv_kernel");
    return TRI_OK;
}

}  // namespace tri

// bf16 forward on tcgen05 / TMEM / TMA (sm_100a): flash-style online softmax, the [B,N,H,N,N] map never leaves
// the SM (Listing 1, Sec. IV-A; gate, mask and 1/sqrt(d) from the task statement).
//
// Persistent, warp-specialised: one CTA per SM, 768 threads =
//   4 softmax warpgroups ("groups", 128 threads = 128 query rows = 128 TMEM lanes each) -- group g owns broadcast
//     row 4*rq + g of the current work item (b, h, 128-query block qb, row quad rq) and walks its 64-key tiles;
//   2 helper warpgroups: warp 16 = TMA producer, warps 17-20 = one in-order tcgen05.mma issuer per group (one elected
//     lane; they sleep in mbarrier.try_wait instead of polling), warps 21-23 idle.
// Registers are moved from the helpers to the softmax warpgroups with setmaxnreg.  The four groups of a CTA work on
// the same (b, h, qb), so one 128x64 bias tile (TMA, SWIZZLE_128B) serves four score tiles ("on-the-fly
// broadcasting").  Per (group, tile) with TMEM columns [128g, 128g+128) = S 64 | P 32 | O 32:
//   S = Q_r K_r^T          tcgen05.mma SS, M=128 N=64 K=2x16, operands TMA-staged (SWIZZLE_64B, K-major)
//   x = scale*S + bias (+ -inf mask); online max / sum; p = exp2((x - m) log2e)
//   P -> bf16 -> TMEM;  O_r += P V_r   tcgen05.mma TS, M=128 N=32 K=4x16, V MN-major
// S of tile n+1 is issued as soon as the group has S of tile n in registers ("consumed"), so the tensor pipe runs
// one tile ahead of the softmax and no group waits for an MMA in steady state.
// Row epilogue: O = sigmoid(G) * O_r / l, LSE = m + ln l.
#include "sm100_common.cuh"
#include "tri_common.cuh"

namespace tri {
using namespace sm100;

namespace {

constexpr int NG = 4;                      // softmax groups per CTA
constexpr int BQ = 128, BK = 64, DH = 32;
constexpr int KV_ST = 3;                   // K/V ring stages per group
constexpr int NB = 2;                      // bias ring stages (shared by the groups)
constexpr int QT_BYTES = BQ * DH * 2;      // 8 KB: 128 x 32 bf16
constexpr int KT_BYTES = BK * DH * 2;      // 4 KB:  64 x 32 bf16
constexpr int BIAS_BYTES = BQ * BK * 4;    // 32 KB: two [128 q][32 k] fp32 boxes (log2e * bias), SWIZZLE_128B
constexpr float kLazy = 7.0f;              // lazy-rescale threshold on the running max (log2 units)
constexpr int FWD_THREADS = (NG + 2) * 128;  // 4 softmax warpgroups + 2 helper warpgroups (TMA warp, 4 issuer warps)
constexpr int kTokRelease = 24;            // pair index (of 32) of the exp loop at which the MUFU token moves on

struct FwdSmem {
    static constexpr int q_off = 0;                                    // NG x 2 x Q tile
    static constexpr int kv_off = q_off + NG * 2 * QT_BYTES;           // NG x KV_ST x (K, V)
    static constexpr int bias_off = kv_off + NG * KV_ST * 2 * KT_BYTES;
    static constexpr int bar_off = bias_off + NB * BIAS_BYTES;
    // mbarriers (8 bytes each)
    static constexpr int b_kv_full = 0;                                // [NG][KV_ST]
    static constexpr int b_kv_free = b_kv_full + NG * KV_ST;           // [NG][KV_ST]
    static constexpr int b_bias_full = b_kv_free + NG * KV_ST;         // [NB]
    static constexpr int b_bias_free = b_bias_full + NB;               // [NB]
    static constexpr int b_s_full = b_bias_free + NB;                  // [NG]
    static constexpr int b_consumed = b_s_full + NG;                   // [NG]
    static constexpr int b_p_ready = b_consumed + NG;                  // [NG]
    static constexpr int b_pv_done = b_p_ready + NG;                   // [NG]
    static constexpr int b_tok = b_pv_done + NG;                       // [NG][4] exp-phase token of (group, scheduler quarter)
    static constexpr int n_bars = b_tok + NG * 4;
    static constexpr int total = bar_off + n_bars * 8 + 16 + 1024;     // + tmem slot + alignment slack
};

struct Item { int b, h, q0, r4; };
// row quad fastest (measured: query block fastest halves the K / V re-reads from HBM but is 4 % slower at cfg5, where
// the ending-node rows are 64-byte neighbours in memory and concurrent quads share DRAM pages)
template <bool kAligned>
__device__ __forceinline__ Item decode_item(int item, int N, int H, int R) {
    const int NRQ = (R + NG - 1) / NG, NQB = kAligned ? N / BQ : (N + BQ - 1) / BQ;  // the last row quad may be partial
    Item it;
    it.r4 = (item % NRQ) * NG;
    int t = item / NRQ;
    it.q0 = (t % NQB) * BQ;
    const int bh = t / NQB;
    it.b = bh / H;
    it.h = bh % H;
    return it;
}

// kAligned: N % 128 == 0 (no partial tile anywhere: the bounds checks fold away)
template <bool kAligned>
__global__ void __launch_bounds__(FWD_THREADS, 1)
sm100_fwd_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmK,
                 const __grid_constant__ CUtensorMap tmV, const __grid_constant__ CUtensorMap tmBias, Problem p,
                 const __nv_bfloat16* __restrict__ G, const unsigned long long* __restrict__ maskbits,
                 __nv_bfloat16* __restrict__ O, float* __restrict__ LSE, int total_items) {
    using L = FwdSmem;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    uint8_t* sQ = smem + L::q_off;
    uint8_t* sKV = smem + L::kv_off;
    uint8_t* sBias = smem + L::bias_off;
    uint64_t* bars = (uint64_t*)(smem + L::bar_off);
    uint64_t* kv_full = bars + L::b_kv_full;
    uint64_t* kv_free = bars + L::b_kv_free;
    uint64_t* bias_full = bars + L::b_bias_full;
    uint64_t* bias_free = bars + L::b_bias_free;
    uint64_t* s_full = bars + L::b_s_full;
    uint64_t* consumed = bars + L::b_consumed;
    uint64_t* p_ready = bars + L::b_p_ready;
    uint64_t* pv_done = bars + L::b_pv_done;
    uint64_t* tok = bars + L::b_tok;
    uint32_t* tmem_slot = (uint32_t*)(bars + L::n_bars);

    const int tid = threadIdx.x, warp = tid >> 5;
    const int N = p.N;
    const int TPR = kAligned ? N / BK : (N + BK - 1) / BK;  // key tiles per row (the last one may be partial: TMA zero-fills, the mask bits hide it)
    const int n_items = (total_items - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
    const int NT_all = n_items * TPR;  // tiles per group over the CTA's life

    if (tid == 0) {
        prefetch_tmap(&tmQ); prefetch_tmap(&tmK); prefetch_tmap(&tmV); prefetch_tmap(&tmBias);
        for (int i = 0; i < NG * KV_ST; ++i) { mbar_init(kv_full + i, 1); mbar_init(kv_free + i, 1); }
        for (int i = 0; i < NB; ++i) { mbar_init(bias_full + i, 1); mbar_init(bias_free + i, NG * 4); }
        for (int i = 0; i < NG; ++i) {
            mbar_init(s_full + i, 1); mbar_init(consumed + i, 4); mbar_init(p_ready + i, 4); mbar_init(pv_done + i, 1);
        }
        for (int i = 0; i < NG * 4; ++i) mbar_init(tok + i, 1);
        fence_barrier_init();
    }
    if (warp == 0) tmem_alloc<512>(tmem_slot);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;

    if (warp >= NG * 4) {
        // =============================== helper warpgroup ===============================
        setmaxnreg_dec<32>();
        if (warp == NG * 4) {
            // ---- TMA producer: bias tile of (item, kt) once, then (Q at kt = 0,) K, V of every group ----
            int kst = 0, kph = 0, bst = 0, bph = 0;
            for (int il = 0; il < n_items; ++il) {
                const Item it = decode_item<kAligned>((int)blockIdx.x + il * (int)gridDim.x, N, p.H, p.R);
                const int bh = it.b * p.H + it.h;
                for (int kt = 0; kt < TPR; ++kt) {
                    mbar_wait(bias_free + bst, bph ^ 1);
                    if (elect_one()) {
                        mbar_expect_tx(bias_full + bst, BIAS_BYTES);
                        tma_load_3d(sBias + bst * BIAS_BYTES, &tmBias, bias_full + bst, kt * BK, it.q0, bh);
                        tma_load_3d(sBias + bst * BIAS_BYTES + BIAS_BYTES / 2, &tmBias, bias_full + bst, kt * BK + 32, it.q0, bh);
                    }
                    __syncwarp();
#pragma unroll 1
                    for (int g = 0; g < NG; ++g) {
                        uint64_t* full = kv_full + g * KV_ST + kst;
                        mbar_wait(kv_free + g * KV_ST + kst, kph ^ 1);
                        if (elect_one()) {
                            uint8_t* kv = sKV + (g * KV_ST + kst) * 2 * KT_BYTES;
                            mbar_expect_tx(full, 2 * KT_BYTES + (kt == 0 ? QT_BYTES : 0));
                            if (kt == 0) tma_load_5d(sQ + (g * 2 + (il & 1)) * QT_BYTES, &tmQ, full, 0, it.q0, it.r4 + g, it.h, it.b);
                            tma_load_5d(kv, &tmK, full, 0, kt * BK, it.r4 + g, it.h, it.b);
                            tma_load_5d(kv + KT_BYTES, &tmV, full, 0, kt * BK, it.r4 + g, it.h, it.b);
                        }
                        __syncwarp();
                    }
                    if (++kst == KV_ST) { kst = 0; kph ^= 1; }
                    if (++bst == NB) { bst = 0; bph ^= 1; }
                }
            }
        } else if (warp <= NG * 4 + NG) {
            // ---- tcgen05 issuer of group g (warp-uniform control flow; one elected lane issues and commits) ----
            // In order, sleeping in mbarrier.try_wait: S(n) once the group has S(n-1) in registers and K(n) has landed, then
            // O += P(n-1) V(n-1) once P(n-1) is stored -- the order in which the group raises those events.
            const int g = warp - (NG * 4 + 1);
            constexpr uint32_t idescS = make_idesc(128, BK, false, false);
            constexpr uint32_t idescO = make_idesc(128, DH, false, true);
            const uint32_t qbase = smem_u32(sQ) + g * 2 * QT_BYTES, kvbase = smem_u32(sKV) + g * KV_ST * 2 * KT_BYTES;
            const uint32_t tS = tmem + g * 128, tP = tS + 64, tO = tS + 96;
            int st = 0, kt = 0, par = 0;     // ring stage, key tile and Q buffer of S(n)
            int pst = 0, pkt = 0;            // ring stage and key tile of P(n-1) V(n-1)
            for (int n = 0; n <= NT_all; ++n) {
                if (n < NT_all) {
                    mbar_wait(kv_full + g * KV_ST + st, (n / KV_ST) & 1);
                    if (n > 0) mbar_wait(consumed + g, (n - 1) & 1);
                    tc_fence_after();
                    const uint64_t dq = make_desc_sw64(qbase + par * QT_BYTES);
                    const uint64_t dk = make_desc_sw64(kvbase + st * 2 * KT_BYTES);
                    if (elect_one()) {
                        mma_ss(tS, dq, dk, idescS, 0);
                        mma_ss(tS, dq + 2, dk + 2, idescS, 1);
                        mma_commit(s_full + g);
                    }
                    __syncwarp();
                    if (++st == KV_ST) st = 0;
                    if (++kt == TPR) { kt = 0; par ^= 1; }
                }
                if (n > 0) {
                    mbar_wait(p_ready + g, (n - 1) & 1);
                    tc_fence_after();
                    const uint64_t dv = make_desc_sw64(kvbase + pst * 2 * KT_BYTES + KT_BYTES);
                    if (elect_one()) {
#pragma unroll
                        for (int ks = 0; ks < BK / 16; ++ks)
                            mma_ts(tO, tP + ks * 8, dv + (uint64_t)ks * 64, idescO, (pkt > 0 || ks > 0) ? 1u : 0u);
                        mma_commit(kv_free + g * KV_ST + pst);
                        mma_commit(pv_done + g);
                    }
                    __syncwarp();
                    if (++pst == KV_ST) pst = 0;
                    if (++pkt == TPR) pkt = 0;
                }
            }
        }
    } else {
        // =============================== softmax groups ===============================
        setmaxnreg_inc<104>();  // 512 x 104 + 256 x 32 = 768 x 80 (the launch allocation)
        const int g = warp >> 2;
        const int row = tid & 127;                                  // query row inside the block = TMEM lane
        const uint32_t lane_off = (uint32_t)((warp & 3) * 32) << 16;
        const uint32_t tS = tmem + g * 128 + lane_off, tP = tS + 64, tO = tS + 96;
        const float sl = rsqrtf((float)DH) * kLog2e;  // scores are kept in log2 units: x = S * scale * log2e + log2e * bias
        const uint64_t sl2 = pack2(sl, sl);
        const int NW = kAligned ? N / 64 : (N + 63) / 64;  // mask words per row
        int bst = 0, bph = 0;
        int n = 0;
        uint64_t* my_tok = tok + g * 4 + (warp & 3);
        uint64_t* next_tok = tok + ((g + 1) % NG) * 4 + (warp & 3);
        for (int il = 0; il < n_items; ++il) {
            const Item it = decode_item<kAligned>((int)blockIdx.x + il * (int)gridDim.x, N, p.H, p.R);
            const int r = it.r4 + g;
            const bool rin = r < p.R;  // a group beyond the last row (R % 4 != 0) works on TMA zero-fill and stores nothing
            const unsigned long long* mrow = maskbits && rin ? maskbits + ((long long)it.b * p.R + r) * NW : nullptr;
            uint64_t mb_next = mrow ? ldg_u64(mrow) : ~0ull;
            float m_run = -INFINITY, l_run = 0.0f;
            const long long off = (long long)it.b * p.sB + (long long)it.h * p.sH + (long long)r * p.sSlice + (long long)(it.q0 + row) * p.sPos;
            for (int kt = 0; kt < TPR; ++kt, ++n) {
                const uint64_t mb = mb_next;
                if (mrow && kt + 1 < TPR) mb_next = ldg_u64(mrow + kt + 1);
                mbar_wait(s_full + g, n & 1);
                tc_fence_after();
                uint32_t raw[BK];
                tmem_ld32(tS, *(uint32_t(*)[32])&raw[0]);
                tmem_ld32(tS + 32, *(uint32_t(*)[32])&raw[32]);
                mbar_wait(bias_full + bst, bph);
                const uint8_t* brow = sBias + bst * BIAS_BYTES + row * 128;  // my row in the two 32-column boxes
                tmem_ld_wait();
                tc_fence_before();
                warp_arrive(consumed + g);  // S(n) is in registers: the issuer may overwrite the S columns

                // ---- scores of my query row in log2 units: x = (scale*log2e)*S + log2e*bias (+ mask) -------------------
                float x[BK];
#pragma unroll
                for (int c4 = 0; c4 < BK / 4; ++c4) {
                    const float4 bv = lds128f(brow + (c4 >> 3) * (BIAS_BYTES / 2) + (((c4 & 7) ^ (row & 7)) << 4));
                    const int c = c4 * 4;
                    unpack2(fma2(pack2(__uint_as_float(raw[c]), __uint_as_float(raw[c + 1])), sl2, pack2(bv.x, bv.y)), x[c], x[c + 1]);
                    unpack2(fma2(pack2(__uint_as_float(raw[c + 2]), __uint_as_float(raw[c + 3])), sl2, pack2(bv.z, bv.w)), x[c + 2], x[c + 3]);
                }
                // my generic-proxy reads of the bias tile must be complete before the producer's TMA (async proxy) may
                // overwrite it: without the proxy fence the arrive can overtake the ld.shared of a busy warp
                fence_proxy_async();
                warp_arrive(bias_free + bst);
                if (++bst == NB) { bst = 0; bph ^= 1; }
                if (mb != ~0ull) {
#pragma unroll
                    for (int c = 0; c < BK; ++c)
                        if (!((mb >> c) & 1ull)) x[c] = -INFINITY;
                }
                float mx;
                {   // four independent max chains (ILP), merged at the end
                    float m4[4] = {x[0], x[1], x[2], x[3]};
#pragma unroll
                    for (int c = 4; c < BK; c += 4) {
                        m4[0] = fmaxf(m4[0], x[c]); m4[1] = fmaxf(m4[1], x[c + 1]);
                        m4[2] = fmaxf(m4[2], x[c + 2]); m4[3] = fmaxf(m4[3], x[c + 3]);
                    }
                    mx = fmaxf(fmaxf(m4[0], m4[1]), fmaxf(m4[2], m4[3]));
                }
                // ---- online softmax with the -inf guard of reading A6 ---------------------------------
                // The running reference m moves only when this tile's maximum exceeds it by more than kLazy (O and l
                // share the reference, so the result is exact either way): keeps the O rescale out of almost every tile.
                const float m_old = m_run;
                const bool bump = mx > m_old + kLazy;
                const float m_new = bump ? mx : m_old;
                const float m_safe = (m_new == -INFINITY) ? 0.0f : m_new;
                const float alpha = bump ? ex2(m_old - m_safe) : 1.0f;
                const uint64_t mneg2 = pack2(-m_safe, -m_safe);
                uint64_t lacc4[4] = {pack2(0.0f, 0.0f), pack2(0.0f, 0.0f), pack2(0.0f, 0.0f), pack2(0.0f, 0.0f)};
                // The four groups' warps of one scheduler share its MUFU unit, and one warp's exp loop saturates it.  Left
                // alone the groups run their exp loops at the same time (each at a quarter of the rate) and then their
                // score / max phases at the same time, with the unit idle; the token makes the exp loops take turns.
                if (g > 0 || n > 0) mbar_wait(my_tok, (g > 0 ? n : n - 1) & 1);
                uint32_t pk[BK / 2];
#pragma unroll
                for (int e = 0; e < BK / 2; ++e) {
                    if (e == kTokRelease) {  // hand the token on a little early: the next warp's wake-up hides under my last exps
                        __syncwarp();
                        if ((tid & 31) == 0) mbar_arrive(next_tok);
                    }
                    float a0, a1;
                    unpack2(add2(pack2(x[2 * e], x[2 * e + 1]), mneg2), a0, a1);
                    const float p0 = ex2(a0), p1 = ex2(a1);
                    lacc4[e & 3] = add2(lacc4[e & 3], pack2(p0, p1));
                    pk[e] = pack_bf16(p0, p1);
                }
                float l0, l1;
                unpack2(add2(add2(lacc4[0], lacc4[1]), add2(lacc4[2], lacc4[3])), l0, l1);
                l_run = l_run * alpha + (l0 + l1);
                m_run = m_new;
                // P(n-1) has been read and O(n-1) accumulated before P / O are touched again
                if (n > 0) {
                    mbar_wait(pv_done + g, (n - 1) & 1);
                    tc_fence_after();
                }
                if (kt > 0 && __any_sync(0xffffffffu, bump)) {  // rescale the accumulator O_r
                    uint32_t o[32];
                    tmem_ld32(tO, o);
                    tmem_ld_wait();
#pragma unroll
                    for (int c = 0; c < 32; ++c) o[c] = __float_as_uint(__uint_as_float(o[c]) * alpha);
                    tmem_st32(tO, o);
                }
                tmem_st32(tP, pk);
                tmem_st_wait();
                tc_fence_before();
                warp_arrive(p_ready + g);
            }
            // ---- row epilogue: O = sigmoid(G) * O_r / l ; LSE = m + ln l -------------------------------
            const bool inq = rin && (kAligned || it.q0 + row < N);  // the last query block may be partial
            uint4 gv[4];
            const uint4* gp = (const uint4*)(G + off);
#pragma unroll
            for (int j = 0; j < 4; ++j) gv[j] = inq ? __ldg(gp + j) : make_uint4(0u, 0u, 0u, 0u);
            mbar_wait(pv_done + g, (n - 1) & 1);
            tc_fence_after();
            uint32_t o[32];
            tmem_ld32(tO, o);
            tmem_ld_wait();
            const float inv = l_run > 0.0f ? 1.0f / l_run : 0.0f;
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
                if (inq) op[j] = make_uint4(ow[0], ow[1], ow[2], ow[3]);
            }
            const long long loff = (long long)it.b * p.lB + (long long)it.h * N + (long long)r * p.lR + (long long)(it.q0 + row) * p.lQ;
            if (inq) LSE[loff] = l_run > 0.0f ? m_run * kLn2 + __logf(l_run) : -INFINITY;
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc<512>(tmem);
}

// bf16 plane transpose out[bh][j][i] = in[bh][i][j]  (bias for the ending-node variant: bias[b,h,k,i] -> [q=i][k])
__global__ void transpose_bf16_kernel(const __nv_bfloat16* __restrict__ in, __nv_bfloat16* __restrict__ out, int N) {
    __shared__ __nv_bfloat16 tile[32][33];
    const long long plane = (long long)blockIdx.z * N * N;
    const int x = blockIdx.x * 32 + threadIdx.x, y0 = blockIdx.y * 32;
    for (int j = threadIdx.y; j < 32; j += 8)
        if (x < N && y0 + j < N) tile[j][threadIdx.x] = in[plane + (long long)(y0 + j) * N + x];
    __syncthreads();
    const int xo = blockIdx.y * 32 + threadIdx.x, yo0 = blockIdx.x * 32;
    for (int j = threadIdx.y; j < 32; j += 8)
        if (xo < N && yo0 + j < N) out[plane + (long long)(yo0 + j) * N + xo] = tile[threadIdx.x][j];
}

// fp32 planes of f * bias for the softmax warps (no bf16 unpacking in the inner loops): nat[bh][y][x] = f*in[bh][y][x],
// tr[bh][x][y] = f*in[bh][y][x]; either output may be null.  N^2 H B elements: negligible next to the N^3 work.
__global__ void bias_planes_kernel(const __nv_bfloat16* __restrict__ in, float* __restrict__ nat, float* __restrict__ tr,
                                   int N, float f) {
    __shared__ float tile[32][33];
    const long long plane = (long long)blockIdx.z * N * N;
    const int x = blockIdx.x * 32 + threadIdx.x, y0 = blockIdx.y * 32;
    for (int j = threadIdx.y; j < 32; j += 8) {
        if (x >= N || y0 + j >= N) continue;
        const float v = f * __bfloat162float(in[plane + (long long)(y0 + j) * N + x]);
        if (nat) nat[plane + (long long)(y0 + j) * N + x] = v;
        tile[j][threadIdx.x] = v;
    }
    if (!tr) return;
    __syncthreads();
    const int xo = blockIdx.y * 32 + threadIdx.x, yo0 = blockIdx.x * 32;
    for (int j = threadIdx.y; j < 32; j += 8)
        if (xo < N && yo0 + j < N) tr[plane + (long long)(yo0 + j) * N + xo] = tile[threadIdx.x][j];
}

// keep flags [B,N,N] (u8) -> one 64-bit word per (b, row r, 64-key tile): bit k = key 64*w + k of row r is visible.
// Rows / keys follow the variant (mask element (r,k) at r*mR + k*mK), so the kernels read one word per tile.
// Keys >= N of the last (partial) tile get a zero bit; mask == nullptr packs "every key < N visible" (ragged N only).
__global__ void __launch_bounds__(128) pack_mask_kernel(const unsigned char* __restrict__ mask,
                                                        unsigned long long* __restrict__ bits, Problem p) {
    const int lane = threadIdx.x & 31, w = blockIdx.x * 4 + (threadIdx.x >> 5);
    const int r = blockIdx.y, b = blockIdx.z, NW = (p.N + 63) / 64;
    if (w >= NW) return;
    const unsigned char* base = mask ? mask + (long long)b * p.mB + (long long)r * p.mR : nullptr;
    const int k_lo = w * 64 + lane, k_hi = k_lo + 32;
    const unsigned lo = __ballot_sync(0xffffffffu, k_lo < p.N && (!base || base[(long long)k_lo * p.mK] != 0));
    const unsigned hi = __ballot_sync(0xffffffffu, k_hi < p.N && (!base || base[(long long)k_hi * p.mK] != 0));
    if (lane == 0) bits[((long long)b * p.R + r) * NW + w] = (unsigned long long)lo | ((unsigned long long)hi << 32);
}

int sm_count() {
    static int n = 0;
    if (n == 0) {
        int dev = 0;
        if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0)
            n = 148;
    }
    return n;
}

}  // namespace

tri_status sm100_transpose_planes(const void* in, void* out, int BH, int N, cudaStream_t st) {
    ProfScope ps("transpose_bf16_kernel", st);
    transpose_bf16_kernel<<<dim3((N + 31) / 32, (N + 31) / 32, BH), dim3(32, 8), 0, st>>>((const __nv_bfloat16*)in, (__nv_bfloat16*)out, N);
    return TRI_OK;
}

tri_status sm100_bias_planes(const void* in, float* nat, float* tr, int BH, int N, float f, cudaStream_t st) {
    ProfScope ps("bias_planes_kernel", st);
    bias_planes_kernel<<<dim3((N + 31) / 32, (N + 31) / 32, BH), dim3(32, 8), 0, st>>>((const __nv_bfloat16*)in, nat, tr, N, f);
    return TRI_OK;
}

tri_status sm100_pack_mask(const Problem& p, const unsigned char* mask, void* bits, cudaStream_t st) {
    ProfScope ps("pack_mask_kernel", st);
    pack_mask_kernel<<<dim3(((p.N + 63) / 64 + 3) / 4, p.R, p.B), 128, 0, st>>>(mask, (unsigned long long*)bits, p);
    return TRI_OK;
}

int sm100_sm_count() { return sm_count(); }

// N <= 8192: the fused dQ + dBias stage covers 2048 keys per launch (one cluster rank per two 64-key tiles, <= 16 ranks)
// and runs ceil(N / 2048) key passes; its partial dBias planes (8 x B x H x N^2 fp32) set the practical limit.  N % 8 == 0: the
// bias planes are read by TMA (16-byte row pitch in bf16).  N need not be a multiple of the 64 / 128-position tiles: TMA
// zero-fills what lies beyond N, the packed mask hides keys >= N, stores of queries / keys >= N are predicated off.
bool sm100_supported(const Problem& p, tri_dtype dt) {
    return dt == TRI_BF16 && p.d == 32 && p.N % 8 == 0 && p.N >= 128 && p.N <= 8192 && p.R >= 1 &&
           (p.R == p.N || p.variant == TRI_STARTING);
}

// The forward alone has no cluster in it: its key loop is as long as N wants (long-sequence inference).  16384 keeps
// every item count and TMA coordinate far inside 31 bits.
bool sm100_fwd_supported(const Problem& p, tri_dtype dt) {
    return dt == TRI_BF16 && p.d == 32 && p.N % 8 == 0 && p.N >= 128 && p.N <= 16384 && p.R >= 1 &&
           (p.R == p.N || p.variant == TRI_STARTING);
}

// the kernels need the packed mask words when the caller passed a mask or when the last 64-key tile is partial
bool sm100_needs_maskbits(const Problem& p, const unsigned char* mask) { return mask != nullptr || p.N % 64 != 0; }

size_t sm100_maskbits_bytes(const Problem& p) { return align_up((size_t)p.B * p.R * ((p.N + 63) / 64) * 8, 256); }

size_t sm100_fwd_workspace(const Problem& p) {
    return sm100_maskbits_bytes(p) + align_up((size_t)p.B * p.H * p.N * p.N * 4, 256);  // + log2e * bias[q][k], fp32
}

tri_status sm100_fwd(const Problem& p, const void* Q, const void* K, const void* V, const void* G, const void* bias,
                     const unsigned char* mask, void* O, float* LSE, void* ws, cudaStream_t st) {
    void* maskbits = nullptr;
    if (sm100_needs_maskbits(p, mask)) {
        maskbits = ws;
        tri_status s = sm100_pack_mask(p, mask, maskbits, st);
        if (s != TRI_OK) return s;
        TRI_LAUNCH_CHECK("pack_mask_kernel");
    }
    // log2e * bias as fp32 planes in [q][k] order (the ending-node variant reads bias[b,h,k,q]: transposed here)
    float* biasL = (float*)((char*)ws + sm100_maskbits_bytes(p));
    {
        const bool tr = p.variant == TRI_ENDING;
        tri_status s = sm100_bias_planes(bias, tr ? nullptr : biasL, tr ? biasL : nullptr, p.B * p.H, p.N, kLog2e, st);
        if (s != TRI_OK) return s;
        TRI_LAUNCH_CHECK("bias_planes_kernel");
    }
    CUtensorMap tQ, tK, tV, tB;
    if (!make_tmap_u(&tQ, Q, p.B, p.N, p.H, p.d, p.variant, BQ, p.R) || !make_tmap_u(&tK, K, p.B, p.N, p.H, p.d, p.variant, BK, p.R) ||
        !make_tmap_u(&tV, V, p.B, p.N, p.H, p.d, p.variant, BK, p.R) || !make_tmap_plane_f32(&tB, biasL, p.B * p.H, p.N, BQ))
        return cuda_fail(cudaErrorUnknown, "cuTensorMapEncodeTiled");
    // the opt-in shared-memory size is a per-device function attribute: set it on every launch (cheap, thread-safe)
    auto kern = p.N % 128 == 0 ? sm100_fwd_kernel<true> : sm100_fwd_kernel<false>;
    TRI_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, FwdSmem::total));
    const long long items = (long long)p.B * p.H * ((p.N + BQ - 1) / BQ) * ((p.R + NG - 1) / NG);
    const int grid = (int)(items < sm_count() ? items : sm_count());
    {
        ProfScope ps("sm100_fwd_kernel", st);
        kern<<<grid, FWD_THREADS, FwdSmem::total, st>>>(tQ, tK, tV, tB, p, (const __nv_bfloat16*)G, (const unsigned long long*)maskbits,
                                                        (__nv_bfloat16*)O, LSE, (int)items);
    }
    TRI_LAUNCH_CHECK("sm100_fwd_kernel");
    return TRI_OK;
}

}  // namespace tri

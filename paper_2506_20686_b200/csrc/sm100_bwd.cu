// bf16 backward on tcgen05 / TMEM / TMA (sm_100a).  Listing 2, Table I, gate from the task
// statement.  P is recomputed from the saved LSE; nothing of size N^3 is stored.
//
//   pre      D = rowsum(dO . O), dG = dO . O . (1 - sigmoid G), dA = dO . sigmoid G (bf16, workspace)
//   dkdv     key-stationary (thread = key): S^T = K Q^T, dP^T = V dA^T (SS), P^T, dS^T -> bf16 -> TMEM,
//            dV += P^T dA, dK += dS^T Q (TS, B operand MN-major)
//   dq       query-stationary (thread = query): S, dP (SS), dS -> TMEM, dQ += dS K (TS)
//   dbias    tile-stationary: one CTA owns a 128x128 tile of dBias in registers and streams over ALL broadcast
//            rows in ascending order (S, dP double-buffered in TMEM) -- deterministic, replaces the paper's
//            tl.atomic_add; workspace stays O(N^2 H d).
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

// ------------------------------------------------------------------------------------------------------------
// dq: CTA = (b, row group of R_, h, 128-query block); loop over 64-key tiles (outer) and the R_ rows (inner).
// ------------------------------------------------------------------------------------------------------------
template <int R_>
struct DqSmem {
    static constexpr int qa_off = 0;                          // R_ x (Q, dA) 128x32
    static constexpr int kv_off = qa_off + R_ * 2 * T128;     // 2 stages x (K, V) 64x32
    static constexpr int bias_off = kv_off + 2 * 2 * T64;     // [128 q][64 k] bf16, SWIZZLE_128B
    static constexpr int mask_off = bias_off + 16384;         // 2 x 64 floats
    static constexpr int bar_off = mask_off + 2 * 64 * 4;
    static constexpr int total = bar_off + 64 + 1024;
};

template <int R_>
__global__ void __launch_bounds__(256, 2) sm100_dq_kernel(const __grid_constant__ CUtensorMap tmQ128,
                                                       const __grid_constant__ CUtensorMap tmA128,
                                                       const __grid_constant__ CUtensorMap tmK64,
                                                       const __grid_constant__ CUtensorMap tmV64,
                                                       const __grid_constant__ CUtensorMap tmBiasQK, Problem p,
                                                       const unsigned char* __restrict__ mask,
                                                       const float* __restrict__ LSE, const float* __restrict__ Dws,
                                                       __nv_bfloat16* __restrict__ dQ) {
    using L = DqSmem<R_>;
    constexpr int TCOLS = (128 + 32 * R_) <= 256 ? 256 : 512;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    uint8_t* sQA = smem + L::qa_off;
    uint8_t* sKV = smem + L::kv_off;
    uint8_t* sBias = smem + L::bias_off;
    float* sMask = (float*)(smem + L::mask_off);
    uint64_t* bars = (uint64_t*)(smem + L::bar_off);
    uint64_t* bar_qa = bars + 0;
    uint64_t* bar_kv = bars + 1;  // [2]
    uint64_t* bar_bias = bars + 3;
    uint64_t* bar_mma = bars + 4;
    uint32_t* tmem_slot = (uint32_t*)(bars + 5);

    // 256 threads: a query row (TMEM lane) is shared by two threads, warps w and w+4, 32 key columns each
    const int tid = threadIdx.x, warp = tid >> 5, chalf = warp >> 2;
    const int row = (warp & 3) * 32 + (tid & 31);
    const int NQB = p.N / 128, NKT = p.N / 64, NG = p.N / R_;
    int idx = blockIdx.x;
    const int qb = idx % NQB; idx /= NQB;
    const int h = idx % p.H; idx /= p.H;
    const int g = idx % NG;
    const int b = idx / NG;
    const int r0 = g * R_, q0 = qb * 128, bh = b * p.H + h;

    if (tid == 0) {
        prefetch_tmap(&tmQ128); prefetch_tmap(&tmA128); prefetch_tmap(&tmK64); prefetch_tmap(&tmV64); prefetch_tmap(&tmBiasQK);
        mbar_init(bar_qa, 1); mbar_init(bar_kv, 1); mbar_init(bar_kv + 1, 1); mbar_init(bar_bias, 1); mbar_init(bar_mma, 1);
        fence_barrier_init();
    }
    if (warp == 0) tmem_alloc<TCOLS>(tmem_slot);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    const uint32_t lane_off = (uint32_t)((warp & 3) * 32) << 16;
    const uint32_t tS = tmem, tDP = tmem + 64;
    const int T = NKT * R_;

    auto load_kv = [&](int t) {
        const int kt = t / R_, r = t % R_, st = t & 1;
        mbar_expect_tx(bar_kv + st, 2 * T64);
        tma_load_5d(sKV + st * 2 * T64, &tmK64, bar_kv + st, 0, kt * 64, r0 + r, h, b);
        tma_load_5d(sKV + st * 2 * T64 + T64, &tmV64, bar_kv + st, 0, kt * 64, r0 + r, h, b);
    };
    if (tid == 0) {
        mbar_expect_tx(bar_qa, R_ * 2 * T128);
        for (int r = 0; r < R_; ++r) {
            tma_load_5d(sQA + r * 2 * T128, &tmQ128, bar_qa, 0, q0, r0 + r, h, b);
            tma_load_5d(sQA + r * 2 * T128 + T128, &tmA128, bar_qa, 0, q0, r0 + r, h, b);
        }
        load_kv(0);
        mbar_expect_tx(bar_bias, 16384);
        tma_load_3d(sBias, &tmBiasQK, bar_bias, 0, q0, bh);
    }
    auto mask_val = [&](int t) -> float {
        const int kt = t / R_, r = t % R_;
        const unsigned char mk = mask[(long long)b * p.N * p.N + (long long)(r0 + r) * p.mR + (long long)(kt * 64 + (tid & 63)) * p.mK];
        return mk ? 0.0f : -INFINITY;
    };
    int anymask = 0;
    if (mask) {
        const float mv = mask_val(0);
        if (tid < 64) sMask[tid] = mv;
        anymask = __syncthreads_or(mv != 0.0f);
    }
    float nl[R_], dd[R_];
#pragma unroll
    for (int r = 0; r < R_; ++r) {
        const long long o = (long long)b * p.N * p.H * p.N + (long long)h * p.N + (long long)(r0 + r) * p.lR + (long long)(q0 + row) * p.lQ;
        const float l = __ldg(LSE + o);
        nl[r] = l == -INFINITY ? -INFINITY : -l * kLog2e;
        dd[r] = __ldg(Dws + o);
    }

    constexpr uint32_t idescS = make_idesc(128, 64, false, false);
    constexpr uint32_t idescO = make_idesc(128, DH, false, true);
    const float scale = rsqrtf((float)DH);
    const uint64_t scale2 = pack2(scale, scale), l2e2 = pack2(kLog2e, kLog2e);

    for (int kt = 0; kt < NKT; ++kt) {
#pragma unroll
        for (int r = 0; r < R_; ++r) {
            const int t = kt * R_ + r, st = t & 1;
            if (warp == 0) {  // warp-uniform so the descriptors stay in uniform registers; one elected lane issues
                if (t == 0) mbar_wait(bar_qa, 0);
                mbar_wait(bar_kv + st, (t >> 1) & 1);
                tc_fence_after();
                const uint64_t dq = make_desc_sw64(smem_u32(sQA + r * 2 * T128));
                const uint64_t da = make_desc_sw64(smem_u32(sQA + r * 2 * T128 + T128));
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
            }
            float mnext = 0.0f;
            if (mask && t + 1 < T) mnext = mask_val(t + 1);
            mbar_wait(bar_mma, t & 1);
            tc_fence_after();
            if (tid == 32 && t + 1 < T) load_kv(t + 1);  // warp 1 issues the TMA loads, warp 0 the MMAs
            if (r == 0) mbar_wait(bar_bias, kt & 1);
            const float* mrow = sMask + st * 64;
            {
                const int c32 = chalf;
                uint32_t sraw[32], dpraw[32];
                tmem_ld32(tS + lane_off + c32 * 32, sraw);
                tmem_ld32(tDP + lane_off + c32 * 32, dpraw);
                uint4 bv[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) bv[j] = lds128(sBias + row * 128 + (((c32 * 4 + j) ^ (row & 7)) << 4));
                tmem_ld_wait();
                uint32_t ds[16];
                if (anymask) {
#pragma unroll
                    for (int c4 = 0; c4 < 8; ++c4) {
                        const float4 mv = lds128f(mrow + c32 * 32 + c4 * 4);
                        sraw[c4 * 4] = __float_as_uint(__uint_as_float(sraw[c4 * 4]) + mv.x);  // -inf survives the scale
                        sraw[c4 * 4 + 1] = __float_as_uint(__uint_as_float(sraw[c4 * 4 + 1]) + mv.y);
                        sraw[c4 * 4 + 2] = __float_as_uint(__uint_as_float(sraw[c4 * 4 + 2]) + mv.z);
                        sraw[c4 * 4 + 3] = __float_as_uint(__uint_as_float(sraw[c4 * 4 + 3]) + mv.w);
                    }
                }
                const uint64_t nl2 = pack2(nl[r], nl[r]), nd2 = pack2(-dd[r], -dd[r]);
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
                tmem_st16(tDP + lane_off + c32 * 32, ds);
            }
            if (mask && t + 1 < T && tid < 64) sMask[((t + 1) & 1) * 64 + tid] = mnext;
            tmem_st_wait();
            tc_fence_before();
            if (mask) anymask = __syncthreads_or(mnext != 0.0f); else __syncthreads();
            if (warp == 0) {
                tc_fence_after();
                const uint64_t dk = make_desc_sw64(smem_u32(sKV + st * 2 * T64));
                if (elect_one()) {
#pragma unroll
                    for (int ks = 0; ks < 4; ++ks)
                        mma_ts(tmem + 128 + r * 32, tDP + (ks >> 1) * 32 + (ks & 1) * 8, dk + (uint64_t)ks * 64, idescO,
                               (kt > 0 || ks > 0) ? 1u : 0u);
                    if (r == R_ - 1 && kt + 1 < NKT) {
                        mbar_expect_tx(bar_bias, 16384);
                        tma_load_3d(sBias, &tmBiasQK, bar_bias, (kt + 1) * 64, q0, bh);
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
    for (int r = chalf * (R_ / 2); r < (chalf + 1) * (R_ / 2); ++r) {
        uint32_t v[32];
        tmem_ld32(tmem + lane_off + 128 + r * 32, v);
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
    if (warp == 0) tmem_dealloc<TCOLS>(tmem);
}

// ------------------------------------------------------------------------------------------------------------
// dbias: CTA = (b, h, 128-query tile, 128-key tile), 256 threads: warp w owns TMEM lanes 32*(w&3).. (queries) and
// key columns 64*(w>>2)..+63.  Streams over all N broadcast rows r in ascending order; dBias tile in registers.
// ------------------------------------------------------------------------------------------------------------
struct DbiasSmem {
    static constexpr int NST = 3;
    static constexpr int op_off = 0;                         // NST stages x (Q, dA, K, V) 128x32
    static constexpr int bias_off = op_off + NST * 4 * T128; // 2 x [128 q][64 k] bf16, SWIZZLE_128B
    static constexpr int mask_off = bias_off + 32768;        // 2 x 128 floats
    static constexpr int bar_off = mask_off + 2 * 128 * 4 + 16;  // + two any-flags
    static constexpr int total = bar_off + 128 + 1024;
};

__global__ void __launch_bounds__(288, 1) sm100_dbias_kernel(const __grid_constant__ CUtensorMap tmQ128,
                                                          const __grid_constant__ CUtensorMap tmA128,
                                                          const __grid_constant__ CUtensorMap tmK128,
                                                          const __grid_constant__ CUtensorMap tmV128,
                                                          const __grid_constant__ CUtensorMap tmBiasQK, Problem p,
                                                          const unsigned char* __restrict__ mask,
                                                          const float* __restrict__ LSE, const float* __restrict__ Dws,
                                                          float* __restrict__ dBias, float* __restrict__ planes, int G) {
    using L = DbiasSmem;
    constexpr int NST = L::NST;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    uint8_t* sOp = smem + L::op_off;
    uint8_t* sBias = smem + L::bias_off;
    float* sMask = (float*)(smem + L::mask_off);  // [2][128] floats, then [2] any-flags
    int* sAny = (int*)(sMask + 256);
    uint64_t* bars = (uint64_t*)(smem + L::bar_off);
    uint64_t* bar_full = bars + 0;  // [3] TMA ring
    uint64_t* bar_mma = bars + 3;   // [2] S, dP of a row ready
    uint64_t* bar_bias = bars + 5;
    uint64_t* bar_cons = bars + 6;  // [2] all 8 compute warps have S, dP of the row in registers (buffer free)
    uint32_t* tmem_slot = (uint32_t*)(bars + 8);

    // warps 0-7: compute (TMEM lane quarter = warp & 3, key-column half = warp >> 2); warp 8: TMA + MMA issue + mask staging
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int half = (warp >> 2) & 1, qrow = (warp & 3) * 32 + lane;
    const int NT = p.N / 128;
    int idx = blockIdx.x;
    const int kt = idx % NT; idx /= NT;
    const int qt = idx % NT; idx /= NT;
    const int bh = idx % (p.B * p.H);
    const int gi = idx / (p.B * p.H);  // which slice of the broadcast-row axis (G > 1 only to fill the SMs)
    const int b = bh / p.H, h = bh % p.H;
    const int q0 = qt * 128, k0 = kt * 128;
    const int N = p.N;
    const int rows_per = (N + G - 1) / G, rb = gi * rows_per;
    const int NR = min(rows_per, N - rb);  // this CTA sums rows rb .. rb+NR-1 in ascending order (r below is local)

    if (tid == 0) {
        prefetch_tmap(&tmQ128); prefetch_tmap(&tmA128); prefetch_tmap(&tmK128); prefetch_tmap(&tmV128); prefetch_tmap(&tmBiasQK);
        for (int i = 0; i < 8; ++i) mbar_init(bars + i, (i >= 6) ? 8 : 1);
        fence_barrier_init();
    }
    if (warp == 0) tmem_alloc<512>(tmem_slot);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    const uint32_t lane_off = (uint32_t)((warp & 3) * 32) << 16;
    const float scale = rsqrtf((float)DH);
    uint64_t acc2[32];  // dBias tile: my 64 columns as fp32 pairs
#pragma unroll
    for (int c = 0; c < 32; ++c) acc2[c] = pack2(0.0f, 0.0f);

    if (warp == 8) {
        // =========================== issuer warp (warp-uniform; one elected lane issues TMA / MMA) ===========================
        auto load_ops = [&](int r) {
            const int s = r % NST;
            uint8_t* base = sOp + s * 4 * T128;
            mbar_expect_tx(bar_full + s, 4 * T128);
            tma_load_5d(base, &tmQ128, bar_full + s, 0, q0, rb + r, h, b);
            tma_load_5d(base + T128, &tmA128, bar_full + s, 0, q0, rb + r, h, b);
            tma_load_5d(base + 2 * T128, &tmK128, bar_full + s, 0, k0, rb + r, h, b);
            tma_load_5d(base + 3 * T128, &tmV128, bar_full + s, 0, k0, rb + r, h, b);
        };
        constexpr uint32_t idescS = make_idesc(128, 128, false, false);
        if (elect_one()) {
            for (int r = 0; r < NST && r < NR; ++r) load_ops(r);
            mbar_expect_tx(bar_bias, 32768);
            tma_load_3d(sBias, &tmBiasQK, bar_bias, k0, q0, bh);
            tma_load_3d(sBias + 16384, &tmBiasQK, bar_bias, k0 + 64, q0, bh);
        }
        __syncwarp();
        for (int r = 0; r < NR; ++r) {
            const int s = r % NST, j = r & 1;
            if (r >= 2) mbar_wait(bar_cons + j, ((r - 2) >> 1) & 1);  // row r-2 left TMEM buffer j (and mask slot j)
            if (mask) {  // keep flags of the 128 keys of this tile in row rb+r -> additive 0 / -inf, plus an any-flag
                int any = 0;
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    const int k = lane * 4 + i;
                    const unsigned char mk = mask[(long long)b * N * N + (long long)(rb + r) * p.mR + (long long)(k0 + k) * p.mK];
                    sMask[j * 128 + k] = mk ? 0.0f : -INFINITY;
                    any |= !mk;
                }
                any = __any_sync(0xffffffffu, any);
                if (lane == 0) sAny[j] = any;
                __syncwarp();
            }
            mbar_wait(bar_full + s, (r / NST) & 1);
            tc_fence_after();
            uint8_t* base = sOp + s * 4 * T128;
            const uint64_t dq = make_desc_sw64(smem_u32(base)), da = make_desc_sw64(smem_u32(base + T128));
            const uint64_t dk = make_desc_sw64(smem_u32(base + 2 * T128)), dv = make_desc_sw64(smem_u32(base + 3 * T128));
            const uint32_t tS = tmem + j * 256, tDP = tS + 128;
            if (elect_one()) {
                mma_ss(tS, dq, dk, idescS, 0);
                mma_ss(tS, dq + 2, dk + 2, idescS, 1);
                mma_ss(tDP, da, dv, idescS, 0);
                mma_ss(tDP, da + 2, dv + 2, idescS, 1);
                mma_commit(bar_mma + j);
            }
            __syncwarp();
            if (r >= 1 && r - 1 + NST < NR) {  // MMAs of row r-1 done -> its ring slot is free
                mbar_wait(bar_mma + ((r - 1) & 1), ((r - 1) >> 1) & 1);
                if (elect_one()) load_ops(r - 1 + NST);
                __syncwarp();
            }
        }
    } else {
        // =========================== compute warps ===========================
        auto lse_off = [&](int r) -> long long {
            return (long long)b * N * p.H * N + (long long)h * N + (long long)(rb + r) * p.lR + (long long)(q0 + qrow) * p.lQ;
        };
        float lse_n = __ldg(LSE + lse_off(0)), dd_n = __ldg(Dws + lse_off(0));
        const uint64_t scale2 = pack2(scale, scale), l2e2 = pack2(kLog2e, kLog2e);
        mbar_wait(bar_bias, 0);
        for (int r = 0; r < NR; ++r) {
            const int j = r & 1;
            const float nl = lse_n == -INFINITY ? -INFINITY : -lse_n * kLog2e, dd = dd_n;
            const uint64_t nl2 = pack2(nl, nl), nd2 = pack2(-dd, -dd);
            if (r + 1 < NR) {
                lse_n = __ldg(LSE + lse_off(r + 1));
                dd_n = __ldg(Dws + lse_off(r + 1));
            }
            mbar_wait(bar_mma + j, (r >> 1) & 1);
            tc_fence_after();
            const int anymask = mask ? sAny[j] : 0;
            const uint32_t tS = tmem + j * 256 + half * 64, tDP = tS + 128;
            const float* mrow = sMask + j * 128 + half * 64;
#pragma unroll
            for (int c32 = 0; c32 < 2; ++c32) {
                uint32_t sraw[32], dpraw[32];
                tmem_ld32(tS + lane_off + c32 * 32, sraw);
                tmem_ld32(tDP + lane_off + c32 * 32, dpraw);
                uint4 bv[4];
#pragma unroll
                for (int jj = 0; jj < 4; ++jj)
                    bv[jj] = lds128(sBias + half * 16384 + qrow * 128 + (((c32 * 4 + jj) ^ (qrow & 7)) << 4));
                tmem_ld_wait();
                if (anymask) {
#pragma unroll
                    for (int c4 = 0; c4 < 8; ++c4) {
                        const float4 mv = lds128f(mrow + c32 * 32 + c4 * 4);
                        sraw[c4 * 4] = __float_as_uint(__uint_as_float(sraw[c4 * 4]) + mv.x);
                        sraw[c4 * 4 + 1] = __float_as_uint(__uint_as_float(sraw[c4 * 4 + 1]) + mv.y);
                        sraw[c4 * 4 + 2] = __float_as_uint(__uint_as_float(sraw[c4 * 4 + 2]) + mv.z);
                        sraw[c4 * 4 + 3] = __float_as_uint(__uint_as_float(sraw[c4 * 4 + 3]) + mv.w);
                    }
                }
                if (c32 == 1) {  // my last read of TMEM buffer j and of mask slot j: hand the buffer back to the issuer
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) mbar_arrive(bar_cons + j);
                }
#pragma unroll
                for (int jj = 0; jj < 4; ++jj) {
                    const uint32_t w[4] = {bv[jj].x, bv[jj].y, bv[jj].z, bv[jj].w};
#pragma unroll
                    for (int e = 0; e < 4; ++e) {
                        const int c = jj * 8 + e * 2, k2 = (c32 * 32 + c) >> 1;
                        const uint64_t x2 = fma2(pack2(__uint_as_float(sraw[c]), __uint_as_float(sraw[c + 1])), scale2,
                                                 pack2(bf16_lo(w[e]), bf16_hi(w[e])));
                        float a0, a1;
                        unpack2(fma2(x2, l2e2, nl2), a0, a1);
                        acc2[k2] = fma2(pack2(ex2(a0), ex2(a1)), add2(pack2(__uint_as_float(dpraw[c]), __uint_as_float(dpraw[c + 1])), nd2), acc2[k2]);
                    }
                }
            }
        }
    }
    if (warp < 8) {
    float acc[64];
#pragma unroll
    for (int c = 0; c < 32; ++c) unpack2(acc2[c], acc[2 * c], acc[2 * c + 1]);
    if (G > 1) {  // level-1 partial plane [gi][bh][q][k]; sm100_dbias_reduce_kernel adds the planes in ascending order
        float* out = planes + ((long long)gi * p.B * p.H + bh) * N * N + (long long)(q0 + qrow) * N + k0 + half * 64;
#pragma unroll
        for (int c = 0; c < 64; c += 4) *(float4*)(out + c) = make_float4(acc[c], acc[c + 1], acc[c + 2], acc[c + 3]);
    } else {
        float* out = dBias + (long long)bh * N * N + (long long)(q0 + qrow) * p.bQ + (long long)(k0 + half * 64) * p.bK;
        if (p.bK == 1) {
#pragma unroll
            for (int c = 0; c < 64; c += 4) *(float4*)(out + c) = make_float4(acc[c], acc[c + 1], acc[c + 2], acc[c + 3]);
        } else {
#pragma unroll
            for (int c = 0; c < 64; ++c) out[(long long)c * p.bK] = acc[c];
        }
    }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc<512>(tmem);
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
    int G;   // row slices of the tile-stationary kernel (dqdb, or the dbias fallback)
    int C;   // cluster size of the fused dQ + dBias kernel (0: not covered, use dq + dbias)
};
// Split the broadcast-row axis of the tile-stationary dBias kernel over G CTAs per tile when the tile grid alone
// cannot fill the 148 SMs (1 CTA/SM): pick G in 1..8 minimising waves * rows-per-CTA.
int dbias_split(const Problem& p) {
    const long long tiles = (long long)p.B * p.H * (p.N / 128) * (p.N / 128);
    int best = 1;
    double best_cost = 1e30;
    for (int G = 1; G <= 8; ++G) {
        if (p.N % G) continue;
        const double waves = (double)((tiles * G + 147) / 148);
        const double cost = waves * (p.N / G + 24);  // + per-CTA prologue/drain in row units
        if (cost < best_cost * 0.97) { best_cost = cost; best = G; }
    }
    return best;
}
BwdWs bwd_ws_layout(const Problem& p) {
    BwdWs w;
    size_t o = 0;
    w.d_off = o; o += align_up((size_t)p.B * p.N * p.H * p.N * sizeof(float), 256);
    w.da_off = o; o += align_up((size_t)p.B * p.N * p.H * p.N * p.d * 2, 256);
    w.biast_off = o; o += align_up((size_t)p.B * p.H * p.N * p.N * 2, 256);
    w.biasl_off = o; o += align_up((size_t)p.B * p.H * p.N * p.N * 4, 256);
    w.mask_off = o; o += sm100_maskbits_bytes(p);
    w.C = sm100_dqdb_cluster(p.N);
    w.G = dbias_split(p);                         // the fallback pair's split
    const int gmax = w.C ? kDqdbMaxSplit : w.G;   // the fused kernel picks its split (<= kDqdbMaxSplit) at launch
    w.planes_off = o;
    if (gmax > 1) o += align_up((size_t)gmax * p.B * p.H * p.N * p.N * sizeof(float), 256);
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
    constexpr int RKV = 2, RQ = 4;
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
    const void* bias_qk = p.variant == TRI_STARTING ? bias : biasT;  // [q][k]
    const void* bias_kq = p.variant == TRI_STARTING ? biasT : bias;  // [k][q]

    CUtensorMap tQ64, tA64, tK64, tV64, tQ128, tA128, tK128, tV128, tBqk, tBkq;
    bool ok = make_tmap_u(&tQ64, Q, p.B, p.N, p.H, p.d, p.variant, 64) && make_tmap_u(&tA64, dA, p.B, p.N, p.H, p.d, p.variant, 64) &&
              make_tmap_u(&tK64, K, p.B, p.N, p.H, p.d, p.variant, 64) && make_tmap_u(&tV64, V, p.B, p.N, p.H, p.d, p.variant, 64) &&
              make_tmap_u(&tQ128, Q, p.B, p.N, p.H, p.d, p.variant, 128) && make_tmap_u(&tA128, dA, p.B, p.N, p.H, p.d, p.variant, 128) &&
              make_tmap_u(&tK128, K, p.B, p.N, p.H, p.d, p.variant, 128) && make_tmap_u(&tV128, V, p.B, p.N, p.H, p.d, p.variant, 128) &&
              make_tmap_plane(&tBqk, bias_qk, p.B * p.H, p.N, 128) && make_tmap_plane(&tBkq, bias_kq, p.B * p.H, p.N, 128);
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
    float* planes = (float*)((char*)ws + w.planes_off);
    int Gs = w.G, C2 = 0, grid2 = 0;
    if (w.C && sm100_dqdb_plan(p, &C2, &Gs, &grid2)) {
        // stage 2, fused: dQ and dBias from one recomputation of P / dS (cluster over the key tiles of a query block)
        unsigned long long* maskbits = nullptr;
        if (mask) {
            maskbits = (unsigned long long*)((char*)ws + w.mask_off);
            if ((s = sm100_pack_mask(p, mask, maskbits, st)) != TRI_OK) return s;
            TRI_LAUNCH_CHECK("pack_mask_kernel");
        }
        float* biasL = (float*)((char*)ws + w.biasl_off);
        const bool tr = p.variant == TRI_ENDING;
        if ((s = sm100_bias_planes(bias, tr ? nullptr : biasL, tr ? biasL : nullptr, p.B * p.H, p.N, kLog2e, st)) != TRI_OK) return s;
        TRI_LAUNCH_CHECK("bias_planes_kernel");
        if ((s = sm100_dqdb_launch(p, C2, Gs, grid2, Q, dA, K, V, biasL, maskbits, LSE, Dws, dQ, dBias, planes, st)) != TRI_OK) return s;
    } else {
        Gs = dbias_split(p);
        if ((s = set_smem(sm100_dq_kernel<RQ>, DqSmem<RQ>::total)) != TRI_OK) return s;
        if ((s = set_smem(sm100_dbias_kernel, DbiasSmem::total)) != TRI_OK) return s;
        {
            ProfScope ps("sm100_dq_kernel", st);
            const unsigned grid = (unsigned)((long long)p.B * (p.N / RQ) * p.H * (p.N / 128));
            sm100_dq_kernel<RQ><<<grid, 256, DqSmem<RQ>::total, st>>>(tQ128, tA128, tK64, tV64, tBqk, p, mask, LSE, Dws,
                                                                     (__nv_bfloat16*)dQ);
        }
        TRI_LAUNCH_CHECK("sm100_dq_kernel");
        {
            ProfScope ps("sm100_dbias_kernel", st);
            const unsigned grid = (unsigned)((long long)p.B * p.H * (p.N / 128) * (p.N / 128) * Gs);
            sm100_dbias_kernel<<<grid, 288, DbiasSmem::total, st>>>(tQ128, tA128, tK128, tV128, tBqk, p, mask, LSE, Dws, dBias,
                                                                    planes, Gs);
        }
        TRI_LAUNCH_CHECK("sm100_dbias_kernel");
    }
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

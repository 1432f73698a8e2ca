// bf16 forward on tcgen05 / TMEM / TMA (sm_100a): flash-style online softmax, the [B,N,H,N,N] map never leaves
// the SM (Listing 1, Sec. IV-A; gate, mask and 1/sqrt(d) from the task statement).
//
// One CTA (128 threads = 128 query rows, one TMEM lane each) owns a 128-query block of R_ broadcast rows of one
// (b,h) and walks the key blocks kb = 0..N/128-1 in the OUTER loop and its R_ rows in the INNER loop, so one
// 128x128 bias tile (TMA, SWIZZLE_128B) serves R_ score tiles ("on-the-fly broadcasting").  Per tile:
//   S = Q_r K_r^T        tcgen05.mma SS, M=128 N=128 K=2x16, operands TMA-staged (SWIZZLE_64B, K-major)
//   x = scale*S + bias (+ -inf mask); online max / sum; p = exp2((x - m) log2e)
//   P -> bf16 -> TMEM (aliases S);  O_r += P V_r   tcgen05.mma TS, M=128 N=32 K=8x16, V MN-major
// Epilogue: O = sigmoid(G) * O_r / l, LSE = m + ln l.
#include <stdlib.h>

#include "sm100_common.cuh"
#include "tri_common.cuh"

namespace tri {
using namespace sm100;

namespace {

constexpr int BQ = 128, BK = 128, DH = 32;
constexpr int TILE_BYTES = BQ * DH * 2;  // 8 KB: one 128 x 32 bf16 tile
constexpr float kLazy = 5.0f;            // lazy-rescale threshold on the running max (natural-log units)

template <int R_>
struct FwdSmem {
    static constexpr int q_off = 0;
    static constexpr int kv_off = q_off + R_ * TILE_BYTES;       // 2 stages x (K, V)
    static constexpr int bias_off = kv_off + 4 * TILE_BYTES;     // 2 x 16 KB (key halves), SWIZZLE_128B
    static constexpr int mask_off = bias_off + 2 * 16384;        // 2 x 128 floats
    static constexpr int bar_off = mask_off + 2 * BK * 4;        // mbarriers
    static constexpr int total = bar_off + 64 + 1024;            // + alignment slack
};

template <int R_>
constexpr int tmem_cols() { return (128 + 32 * R_) <= 256 ? 256 : 512; }

template <int R_>
__global__ void __launch_bounds__(128) sm100_fwd_kernel(const __grid_constant__ CUtensorMap tmQ,
                                                        const __grid_constant__ CUtensorMap tmK,
                                                        const __grid_constant__ CUtensorMap tmV,
                                                        const __grid_constant__ CUtensorMap tmBias, Problem p,
                                                        const __nv_bfloat16* __restrict__ G,
                                                        const unsigned char* __restrict__ mask,
                                                        __nv_bfloat16* __restrict__ O, float* __restrict__ LSE) {
    using L = FwdSmem<R_>;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = (uint8_t*)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
    uint8_t* sQ = smem + L::q_off;
    uint8_t* sKV = smem + L::kv_off;
    uint8_t* sBias = smem + L::bias_off;
    float* sMask = (float*)(smem + L::mask_off);
    uint64_t* bars = (uint64_t*)(smem + L::bar_off);
    uint64_t* bar_q = bars + 0;
    uint64_t* bar_kv = bars + 1;  // [2]
    uint64_t* bar_bias = bars + 3;
    uint64_t* bar_mma = bars + 4;
    uint32_t* tmem_slot = (uint32_t*)(bars + 5);

    const int tid = threadIdx.x, warp = tid >> 5;
    const int NQB = p.N / BQ, NKB = p.N / BK, NG = p.N / R_;
    int idx = blockIdx.x;
    const int qb = idx % NQB; idx /= NQB;
    const int h = idx % p.H; idx /= p.H;
    const int g = idx % NG;
    const int b = idx / NG;
    const int r0 = g * R_, q0 = qb * BQ;
    const int bh = b * p.H + h;

    if (tid == 0) {
        prefetch_tmap(&tmQ); prefetch_tmap(&tmK); prefetch_tmap(&tmV); prefetch_tmap(&tmBias);
        mbar_init(bar_q, 1); mbar_init(bar_kv, 1); mbar_init(bar_kv + 1, 1); mbar_init(bar_bias, 1); mbar_init(bar_mma, 1);
        fence_barrier_init();
    }
    if (warp == 0) tmem_alloc<tmem_cols<R_>()>(tmem_slot);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    const uint32_t tS = tmem;                                  // S: columns [0,128); P (bf16 pairs): [0,64)
    const uint32_t lane_off = (uint32_t)(warp * 32) << 16;      // this warp's TMEM lane quarter
    const int T = NKB * R_;

    auto load_kv = [&](int t) {
        const int kb = t / R_, r = t % R_, st = t & 1;
        mbar_expect_tx(bar_kv + st, 2 * TILE_BYTES);
        tma_load_5d(sKV + st * 2 * TILE_BYTES, &tmK, bar_kv + st, 0, kb * BK, r0 + r, h, b);
        tma_load_5d(sKV + st * 2 * TILE_BYTES + TILE_BYTES, &tmV, bar_kv + st, 0, kb * BK, r0 + r, h, b);
    };
    auto load_bias = [&](int kb) {
        mbar_expect_tx(bar_bias, 2 * 16384);
        tma_load_3d(sBias, &tmBias, bar_bias, kb * BK, q0, bh);
        tma_load_3d(sBias + 16384, &tmBias, bar_bias, kb * BK + 64, q0, bh);
    };
    if (tid == 0) {
        mbar_expect_tx(bar_q, R_ * TILE_BYTES);
        for (int r = 0; r < R_; ++r) tma_load_5d(sQ + r * TILE_BYTES, &tmQ, bar_q, 0, q0, r0 + r, h, b);
        load_kv(0);
        load_bias(0);
    }
    // mask for tile t: keep flag of key (kb*128 + tid) in row r0 + r
    auto mask_val = [&](int t) -> float {
        const int kb = t / R_, r = t % R_;
        const unsigned char mk = mask[(long long)b * p.N * p.N + (long long)(r0 + r) * p.mR + (long long)(kb * BK + tid) * p.mK];
        return mk ? 0.0f : -INFINITY;
    };
    int anymask = 0;
    if (mask) {
        const float mv = mask_val(0);
        sMask[tid] = mv;
        anymask = __syncthreads_or(mv != 0.0f);
    }

    constexpr uint32_t idescS = make_idesc(128, 128, false, false);
    constexpr uint32_t idescO = make_idesc(128, DH, false, true);
    const float scale = rsqrtf((float)DH);
    const uint64_t scale2 = pack2(scale, scale);
    float m_run[R_], l_run[R_];
#pragma unroll
    for (int r = 0; r < R_; ++r) { m_run[r] = -INFINITY; l_run[r] = 0.0f; }

    for (int kb = 0; kb < NKB; ++kb) {
#pragma unroll
        for (int r = 0; r < R_; ++r) {
            const int t = kb * R_ + r, st = t & 1;
            if (warp == 0) {  // warp-uniform so the descriptors stay in uniform registers; one elected lane issues
                if (t == 0) mbar_wait(bar_q, 0);
                mbar_wait(bar_kv + st, (t >> 1) & 1);
                tc_fence_after();
                const uint64_t dq = make_desc_sw64(smem_u32(sQ + r * TILE_BYTES));
                const uint64_t dk = make_desc_sw64(smem_u32(sKV + st * 2 * TILE_BYTES));
                if (elect_one()) {
                    mma_ss(tS, dq, dk, idescS, 0);
                    mma_ss(tS, dq + 2, dk + 2, idescS, 1);
                    mma_commit(bar_mma);
                }
                __syncwarp();
            }
            float mnext = 0.0f;
            if (mask && t + 1 < T) mnext = mask_val(t + 1);
            mbar_wait(bar_mma, t & 1);
            tc_fence_after();
            if (tid == 32 && t + 1 < T) load_kv(t + 1);  // (warp 1: warp 0 carries the MMA issue) stage (t+1)&1 was last read by tile t-1
            if (r == 0) mbar_wait(bar_bias, kb & 1);

            // ---- scores of my query row: x = scale*S + bias (+ mask) ---------------------------------------
            float x[BK];
            float mx = -INFINITY;
#pragma unroll
            for (int c32 = 0; c32 < 4; ++c32) {
                uint32_t raw[32];
                tmem_ld32(tS + lane_off + c32 * 32, raw);
                const uint8_t* brow = sBias + (c32 >> 1) * 16384 + tid * 128;
                uint4 bv[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const int c = (c32 & 1) * 4 + j;
                    bv[j] = lds128(brow + ((c ^ (tid & 7)) << 4));
                }
                tmem_ld_wait();
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const uint32_t w[4] = {bv[j].x, bv[j].y, bv[j].z, bv[j].w};
#pragma unroll
                    for (int e = 0; e < 4; ++e) {
                        const int col = c32 * 32 + j * 8 + e * 2;
                        unpack2(fma2(pack2(__uint_as_float(raw[j * 8 + e * 2]), __uint_as_float(raw[j * 8 + e * 2 + 1])), scale2,
                                     pack2(bf16_lo(w[e]), bf16_hi(w[e]))), x[col], x[col + 1]);
                    }
                }
            }
            if (anymask) {
                const float4* mrow = (const float4*)(sMask + st * BK);
#pragma unroll
                for (int c4 = 0; c4 < BK / 4; ++c4) {
                    const float4 mv = lds128f(mrow + c4);
                    x[c4 * 4] += mv.x; x[c4 * 4 + 1] += mv.y; x[c4 * 4 + 2] += mv.z; x[c4 * 4 + 3] += mv.w;
                }
            }
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
            const float m_old = m_run[r];
            const bool bump = mx > m_old + kLazy;
            const float m_new = bump ? mx : m_old;
            const float m_safe = (m_new == -INFINITY) ? 0.0f : m_new;
            const float alpha = bump ? ex2((m_old - m_safe) * kLog2e) : 1.0f;
            const float mneg = -m_safe * kLog2e;
            const uint64_t l2e2 = pack2(kLog2e, kLog2e), mneg2 = pack2(mneg, mneg);
            uint64_t lacc4[4] = {pack2(0.0f, 0.0f), pack2(0.0f, 0.0f), pack2(0.0f, 0.0f), pack2(0.0f, 0.0f)};  // 4 chains (ILP)
#pragma unroll
            for (int c16 = 0; c16 < BK / 32; ++c16) {  // 32 keys -> 16 packed columns per store
                uint32_t pk[16];
#pragma unroll
                for (int e = 0; e < 16; ++e) {
                    float a0, a1;
                    unpack2(fma2(pack2(x[c16 * 32 + 2 * e], x[c16 * 32 + 2 * e + 1]), l2e2, mneg2), a0, a1);
                    const float p0 = ex2(a0), p1 = ex2(a1);
                    lacc4[e & 3] = add2(lacc4[e & 3], pack2(p0, p1));
                    pk[e] = pack_bf16(p0, p1);
                }
                tmem_st16(tS + lane_off + c16 * 16, pk);
            }
            float l0, l1;
            unpack2(add2(add2(lacc4[0], lacc4[1]), add2(lacc4[2], lacc4[3])), l0, l1);
            const float lsum = l0 + l1;
            l_run[r] = l_run[r] * alpha + lsum;
            m_run[r] = m_new;
            if (kb > 0 && __any_sync(0xffffffffu, bump)) {  // rescale the accumulator O_r
                uint32_t o[32];
                tmem_ld32(tmem + lane_off + 128 + r * 32, o);
                tmem_ld_wait();
#pragma unroll
                for (int c = 0; c < 32; ++c) o[c] = __float_as_uint(__uint_as_float(o[c]) * alpha);
                tmem_st32(tmem + lane_off + 128 + r * 32, o);
            }
            if (mask && t + 1 < T) sMask[((t + 1) & 1) * BK + tid] = mnext;
            tmem_st_wait();
            tc_fence_before();
            if (mask) anymask = __syncthreads_or(mnext != 0.0f); else __syncthreads();
            if (warp == 0) {
                tc_fence_after();
                const uint64_t dv = make_desc_sw64(smem_u32(sKV + st * 2 * TILE_BYTES + TILE_BYTES));
                if (elect_one()) {
#pragma unroll
                    for (int ks = 0; ks < BK / 16; ++ks)
                        mma_ts(tmem + 128 + r * 32, tS + ks * 8, dv + (uint64_t)ks * 64, idescO, (kb > 0 || ks > 0) ? 1u : 0u);
                    if (r == R_ - 1 && kb + 1 < NKB) load_bias(kb + 1);  // every thread is past its bias reads
                }
                __syncwarp();
            }
        }
    }
    if (tid == 0) mma_commit(bar_mma);
    mbar_wait(bar_mma, T & 1);
    tc_fence_after();

    // ---- epilogue: O = sigmoid(G) * O_r / l ; LSE = m + ln l -------------------------------------------
#pragma unroll
    for (int r = 0; r < R_; ++r) {
        uint32_t o[32];
        tmem_ld32(tmem + lane_off + 128 + r * 32, o);
        const long long off = (long long)b * p.sB + (long long)h * p.sH + (long long)(r0 + r) * p.sSlice + (long long)(q0 + tid) * p.sPos;
        const uint4* gp = (const uint4*)(G + off);
        uint4 gv[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) gv[j] = __ldg(gp + j);
        tmem_ld_wait();
        const float l = l_run[r];
        const float inv = l > 0.0f ? 1.0f / l : 0.0f;
        uint4 ov[4];
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
            ov[j] = make_uint4(ow[0], ow[1], ow[2], ow[3]);
        }
        uint4* op = (uint4*)(O + off);
#pragma unroll
        for (int j = 0; j < 4; ++j) op[j] = ov[j];
        const long long loff = (long long)b * p.N * p.H * p.N + (long long)h * p.N + (long long)(r0 + r) * p.lR + (long long)(q0 + tid) * p.lQ;
        LSE[loff] = l > 0.0f ? m_run[r] + __logf(l) : -INFINITY;
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc<tmem_cols<R_>()>(tmem);
}

// bf16 plane transpose out[bh][j][i] = in[bh][i][j]  (bias for the ending-node variant: bias[b,h,k,i] -> [q=i][k])
__global__ void transpose_bf16_kernel(const __nv_bfloat16* __restrict__ in, __nv_bfloat16* __restrict__ out, int N) {
    __shared__ __nv_bfloat16 tile[32][33];
    const long long plane = (long long)blockIdx.z * N * N;
    const int x = blockIdx.x * 32 + threadIdx.x, y0 = blockIdx.y * 32;
    for (int j = threadIdx.y; j < 32; j += 8) tile[j][threadIdx.x] = in[plane + (long long)(y0 + j) * N + x];
    __syncthreads();
    const int xo = blockIdx.y * 32 + threadIdx.x, yo0 = blockIdx.x * 32;
    for (int j = threadIdx.y; j < 32; j += 8) out[plane + (long long)(yo0 + j) * N + xo] = tile[threadIdx.x][j];
}

}  // namespace

tri_status sm100_transpose_planes(const void* in, void* out, int BH, int N, cudaStream_t st) {
    ProfScope ps("transpose_bf16_kernel", st);
    transpose_bf16_kernel<<<dim3(N / 32, N / 32, BH), dim3(32, 8), 0, st>>>((const __nv_bfloat16*)in, (__nv_bfloat16*)out, N);
    return TRI_OK;
}

bool sm100_supported(const Problem& p, tri_dtype dt) { return dt == TRI_BF16 && p.d == 32 && p.N % 128 == 0; }

size_t sm100_fwd_workspace(const Problem& p) {
    return p.variant == TRI_ENDING ? align_up((size_t)p.B * p.H * p.N * p.N * 2, 256) : 0;
}

template <int R_>
static tri_status launch_fwd(const Problem& p, const CUtensorMap& tQ, const CUtensorMap& tK, const CUtensorMap& tV,
                             const CUtensorMap& tB, const void* G, const unsigned char* mask, void* O, float* LSE,
                             cudaStream_t st) {
    auto kern = sm100_fwd_kernel<R_>;
    const int smem = FwdSmem<R_>::total;
    // the opt-in shared-memory size is a per-device function attribute: set it on every launch (cheap, thread-safe)
    TRI_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    const unsigned grid = (unsigned)((long long)p.B * (p.N / R_) * p.H * (p.N / BQ));
    {
        ProfScope ps("sm100_fwd_kernel", st);
        kern<<<grid, 128, smem, st>>>(tQ, tK, tV, tB, p, (const __nv_bfloat16*)G, mask, (__nv_bfloat16*)O, LSE);
    }
    TRI_LAUNCH_CHECK("sm100_fwd_kernel");
    return TRI_OK;
}

tri_status sm100_fwd(const Problem& p, const void* Q, const void* K, const void* V, const void* G, const void* bias,
                     const unsigned char* mask, void* O, float* LSE, void* ws, cudaStream_t st) {
    const void* bias_qk = bias;
    if (p.variant == TRI_ENDING) {
        tri_status s = sm100_transpose_planes(bias, ws, p.B * p.H, p.N, st);
        if (s != TRI_OK) return s;
        TRI_LAUNCH_CHECK("sm100_transpose_bf16");
        bias_qk = ws;
    }
    CUtensorMap tQ, tK, tV, tB;
    if (!make_tmap_u(&tQ, Q, p.B, p.N, p.H, p.d, p.variant, BQ) || !make_tmap_u(&tK, K, p.B, p.N, p.H, p.d, p.variant, BK) ||
        !make_tmap_u(&tV, V, p.B, p.N, p.H, p.d, p.variant, BK) || !make_tmap_plane(&tB, bias_qk, p.B * p.H, p.N, BQ))
        return cuda_fail(cudaErrorUnknown, "cuTensorMapEncodeTiled");
    // Default: this file's kernel (2 CTAs/SM, 1.82 ms at cfg4).  TRI_FWD_WS=1 selects the warp-specialised kernel of
    // sm100_fwd3.cu (1 CTA/SM, softmax warpgroups + issuer warps, setmaxnreg; 1.92 ms at cfg4), kept for A/B.
    static const bool ws_kernel = getenv("TRI_FWD_WS") != nullptr;
    if (ws_kernel) return sm100_fwd3_launch(p, tQ, tK, tV, tB, G, mask, O, LSE, st);
    return launch_fwd<4>(p, tQ, tK, tV, tB, G, mask, O, LSE, st);
}

}  // namespace tri

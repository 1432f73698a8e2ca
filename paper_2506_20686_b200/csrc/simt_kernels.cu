// fp32 CUDA-core kernels for triangle attention (any N, d in {16,32,64}, f32 or bf16 storage).
//
// This is the path for dtype f32 (the 1e-4 tolerance excludes TF32 tensor cores, A14) and
// for bf16 shapes the tcgen05 kernels do not cover (N % 8 != 0, N < 128 or d != 32).  Same structure as
// the paper's kernels: flash-style online-softmax forward (Listing 1), backward =
// preprocess D + key-stationary dK/dV + query-stationary dQ;
// dBias is a third, tile-stationary kernel that sums dS over the broadcast axis in ascending order
// (deterministic; replaces the paper's atomic_add).  All arithmetic fp32, expf/logf.
#include <math.h>

#include "tri_common.cuh"

namespace tri {
namespace {

template <typename T> __device__ __forceinline__ float ldf(const T* p);
template <> __device__ __forceinline__ float ldf<float>(const float* p) { return *p; }
template <> __device__ __forceinline__ float ldf<__nv_bfloat16>(const __nv_bfloat16* p) { return __bfloat162float(*p); }
template <typename T> __device__ __forceinline__ void stf(T* p, float v);
template <> __device__ __forceinline__ void stf<float>(float* p, float v) { *p = v; }
template <> __device__ __forceinline__ void stf<__nv_bfloat16>(__nv_bfloat16* p, float v) { *p = __float2bfloat16_rn(v); }

__device__ __forceinline__ float sigmoidf_(float x) { return 1.0f / (1.0f + expf(-x)); }

struct SliceIdx { int b, r, h; long long base; long long lse_base; };
__device__ __forceinline__ SliceIdx decode_slice(const Problem& p, int slice) {
    SliceIdx s;
    s.h = slice % p.H;
    s.r = (slice / p.H) % p.N;
    s.b = slice / (p.H * p.N);
    s.base = s.b * p.sB + s.h * p.sH + s.r * p.sSlice;
    s.lse_base = (long long)s.b * p.N * p.H * p.N + (long long)s.h * p.N + s.r * p.lR;
    return s;
}

// Stage a [ROWS x COLS] tile of bias (rows = queries, cols = keys) into smem, reading along the
// contiguous global dimension.  LD = leading dimension of the smem tile.
template <typename T, int ROWS, int COLS, int LD, int NT>
__device__ __forceinline__ void load_bias_tile(const Problem& p, const T* biasbh, int q0, int k0, float* Bs) {
    for (int idx = threadIdx.x; idx < ROWS * COLS; idx += NT) {
        int qq, kk;
        if (p.bK == 1) { qq = idx / COLS; kk = idx % COLS; } else { qq = idx % ROWS; kk = idx / ROWS; }
        int q = q0 + qq, k = k0 + kk;
        Bs[qq * LD + kk] = (q < p.N && k < p.N) ? ldf(biasbh + (long long)q * p.bQ + (long long)k * p.bK) : 0.0f;
    }
}

// ---------------------------------------------------------------------------------------------
// Forward: one thread per query, K/V chunks staged in shared memory, online softmax.
// ---------------------------------------------------------------------------------------------
template <typename T, int D>
__global__ void __launch_bounds__(64) simt_fwd_kernel(Problem p, const T* __restrict__ Q, const T* __restrict__ K,
                                                      const T* __restrict__ V, const T* __restrict__ G,
                                                      const T* __restrict__ bias, const unsigned char* __restrict__ mask,
                                                      T* __restrict__ O, float* __restrict__ LSE) {
    constexpr int QB = 64, KC = 32;
    __shared__ float Ks[KC][D];
    __shared__ float Vs[KC][D];
    __shared__ float Bs[QB * (KC + 1)];
    __shared__ unsigned char keep[KC];
    const SliceIdx sl = decode_slice(p, blockIdx.x);
    const int q0 = blockIdx.y * QB, q = q0 + threadIdx.x;
    const bool qvalid = q < p.N;
    const float scale = 1.0f / sqrtf((float)D);
    float qreg[D], o[D];
#pragma unroll
    for (int c = 0; c < D; ++c) { qreg[c] = qvalid ? ldf(Q + sl.base + (long long)q * p.sPos + c) : 0.0f; o[c] = 0.0f; }
    float m = -INFINITY, l = 0.0f;
    const T* biasbh = bias + ((long long)sl.b * p.H + sl.h) * p.N * p.N;
    for (int k0 = 0; k0 < p.N; k0 += KC) {
        __syncthreads();
        for (int idx = threadIdx.x; idx < KC * D; idx += QB) {
            int kk = idx / D, c = idx % D, k = k0 + kk;
            Ks[kk][c] = k < p.N ? ldf(K + sl.base + (long long)k * p.sPos + c) : 0.0f;
            Vs[kk][c] = k < p.N ? ldf(V + sl.base + (long long)k * p.sPos + c) : 0.0f;
        }
        if (threadIdx.x < KC) {
            int k = k0 + threadIdx.x;
            keep[threadIdx.x] = (k < p.N) && (!mask || mask[(long long)sl.b * p.N * p.N + (long long)sl.r * p.mR + (long long)k * p.mK]);
        }
        load_bias_tile<T, QB, KC, KC + 1, QB>(p, biasbh, q0, k0, Bs);
        __syncthreads();
        float s[KC];
        float cmax = -INFINITY;
#pragma unroll
        for (int kk = 0; kk < KC; ++kk) {
            float dot = 0.0f;
#pragma unroll
            for (int c = 0; c < D; ++c) dot = fmaf(qreg[c], Ks[kk][c], dot);
            s[kk] = keep[kk] ? fmaf(dot, scale, Bs[threadIdx.x * (KC + 1) + kk]) : -INFINITY;
            cmax = fmaxf(cmax, s[kk]);
        }
        const float mnew = fmaxf(m, cmax);
        if (mnew != -INFINITY) {  // P:L170-177 (mij, alpha, li update) with the -inf guard (A6)
            const float alpha = expf(m - mnew);
            l *= alpha;
#pragma unroll
            for (int c = 0; c < D; ++c) o[c] *= alpha;
#pragma unroll
            for (int kk = 0; kk < KC; ++kk) {
                const float pk = expf(s[kk] - mnew);
                l += pk;
#pragma unroll
                for (int c = 0; c < D; ++c) o[c] = fmaf(pk, Vs[kk][c], o[c]);
            }
            m = mnew;
        }
    }
    if (qvalid) {
        const float inv = l > 0.0f ? 1.0f / l : 0.0f;
        const long long off = sl.base + (long long)q * p.sPos;
#pragma unroll
        for (int c = 0; c < D; ++c) stf(O + off + c, o[c] * inv * sigmoidf_(ldf(G + off + c)));
        LSE[sl.lse_base + (long long)q * p.lQ] = l > 0.0f ? m + logf(l) : -INFINITY;
    }
}

// ---------------------------------------------------------------------------------------------
// Backward preprocess: D = rowsum(dO (.) O), dG = dO (.) O (.) (1 - sigmoid(G))   (A3)
// ---------------------------------------------------------------------------------------------
template <typename T, int D>
__global__ void simt_preprocess_kernel(long long rows, const T* __restrict__ dO, const T* __restrict__ O,
                                       const T* __restrict__ G, T* __restrict__ dG, float* __restrict__ Dws) {
    long long row = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (row >= rows) return;
    float acc = 0.0f;
#pragma unroll
    for (int c = 0; c < D; ++c) {
        const float x = ldf(dO + row * D + c) * ldf(O + row * D + c);
        acc += x;
        stf(dG + row * D + c, x * (1.0f - sigmoidf_(ldf(G + row * D + c))));
    }
    Dws[row] = acc;
}

__device__ __forceinline__ float prob(float s, float lse) {
    return (s == -INFINITY || lse == -INFINITY) ? 0.0f : expf(s - lse);
}

// ---------------------------------------------------------------------------------------------
// Backward stage 2a: dQ, one thread per query (P:L465-491 without the dBias atomics).
// ---------------------------------------------------------------------------------------------
template <typename T, int D>
__global__ void __launch_bounds__(64) simt_dq_kernel(Problem p, const T* __restrict__ dO, const T* __restrict__ Q,
                                                     const T* __restrict__ K, const T* __restrict__ V,
                                                     const T* __restrict__ G, const T* __restrict__ bias,
                                                     const unsigned char* __restrict__ mask, const float* __restrict__ LSE,
                                                     const float* __restrict__ Dws, T* __restrict__ dQ) {
    constexpr int QB = 64, KC = 32;
    __shared__ float Ks[KC][D];
    __shared__ float Vs[KC][D];
    __shared__ float Bs[QB * (KC + 1)];
    __shared__ unsigned char keep[KC];
    const SliceIdx sl = decode_slice(p, blockIdx.x);
    const int q0 = blockIdx.y * QB, q = q0 + threadIdx.x;
    const bool qvalid = q < p.N;
    const float scale = 1.0f / sqrtf((float)D);
    float qreg[D], da[D], dq[D];
    const long long off = sl.base + (long long)q * p.sPos;
#pragma unroll
    for (int c = 0; c < D; ++c) {
        qreg[c] = qvalid ? ldf(Q + off + c) : 0.0f;
        da[c] = qvalid ? ldf(dO + off + c) * sigmoidf_(ldf(G + off + c)) : 0.0f;
        dq[c] = 0.0f;
    }
    const float lse = qvalid ? LSE[sl.lse_base + (long long)q * p.lQ] : -INFINITY;
    const float Dq = qvalid ? Dws[sl.lse_base + (long long)q * p.lQ] : 0.0f;
    const T* biasbh = bias + ((long long)sl.b * p.H + sl.h) * p.N * p.N;
    for (int k0 = 0; k0 < p.N; k0 += KC) {
        __syncthreads();
        for (int idx = threadIdx.x; idx < KC * D; idx += QB) {
            int kk = idx / D, c = idx % D, k = k0 + kk;
            Ks[kk][c] = k < p.N ? ldf(K + sl.base + (long long)k * p.sPos + c) : 0.0f;
            Vs[kk][c] = k < p.N ? ldf(V + sl.base + (long long)k * p.sPos + c) : 0.0f;
        }
        if (threadIdx.x < KC) {
            int k = k0 + threadIdx.x;
            keep[threadIdx.x] = (k < p.N) && (!mask || mask[(long long)sl.b * p.N * p.N + (long long)sl.r * p.mR + (long long)k * p.mK]);
        }
        load_bias_tile<T, QB, KC, KC + 1, QB>(p, biasbh, q0, k0, Bs);
        __syncthreads();
#pragma unroll 4
        for (int kk = 0; kk < KC; ++kk) {
            float dot = 0.0f, dp = 0.0f;
#pragma unroll
            for (int c = 0; c < D; ++c) { dot = fmaf(qreg[c], Ks[kk][c], dot); dp = fmaf(da[c], Vs[kk][c], dp); }
            const float s = keep[kk] ? fmaf(dot, scale, Bs[threadIdx.x * (KC + 1) + kk]) : -INFINITY;
            const float ds = prob(s, lse) * (dp - Dq);
#pragma unroll
            for (int c = 0; c < D; ++c) dq[c] = fmaf(ds, Ks[kk][c], dq[c]);
        }
    }
    if (qvalid) {
#pragma unroll
        for (int c = 0; c < D; ++c) stf(dQ + off + c, dq[c] * scale);
    }
}

// ---------------------------------------------------------------------------------------------
// Backward stage 1: dK, dV, one thread per key, query chunks staged in smem.
// ---------------------------------------------------------------------------------------------
template <typename T, int D>
__global__ void __launch_bounds__(64) simt_dkdv_kernel(Problem p, const T* __restrict__ dO, const T* __restrict__ Q,
                                                       const T* __restrict__ K, const T* __restrict__ V,
                                                       const T* __restrict__ G, const T* __restrict__ bias,
                                                       const unsigned char* __restrict__ mask, const float* __restrict__ LSE,
                                                       const float* __restrict__ Dws, T* __restrict__ dK, T* __restrict__ dV) {
    constexpr int KB = 64, QC = 32;
    __shared__ float Qs[QC][D];
    __shared__ float As[QC][D];
    __shared__ float Bs[QC * (KB + 1)];
    __shared__ float lse_s[QC], D_s[QC];
    const SliceIdx sl = decode_slice(p, blockIdx.x);
    const int k0 = blockIdx.y * KB, k = k0 + threadIdx.x;
    const bool kvalid = k < p.N;
    const float scale = 1.0f / sqrtf((float)D);
    const bool kkeep = kvalid && (!mask || mask[(long long)sl.b * p.N * p.N + (long long)sl.r * p.mR + (long long)k * p.mK]);
    float kreg[D], vreg[D], dk[D], dv[D];
    const long long off = sl.base + (long long)k * p.sPos;
#pragma unroll
    for (int c = 0; c < D; ++c) {
        kreg[c] = kvalid ? ldf(K + off + c) : 0.0f;
        vreg[c] = kvalid ? ldf(V + off + c) : 0.0f;
        dk[c] = 0.0f; dv[c] = 0.0f;
    }
    const T* biasbh = bias + ((long long)sl.b * p.H + sl.h) * p.N * p.N;
    for (int q0 = 0; q0 < p.N; q0 += QC) {
        __syncthreads();
        for (int idx = threadIdx.x; idx < QC * D; idx += KB) {
            int qq = idx / D, c = idx % D, q = q0 + qq;
            const long long o2 = sl.base + (long long)q * p.sPos + c;
            Qs[qq][c] = q < p.N ? ldf(Q + o2) : 0.0f;
            As[qq][c] = q < p.N ? ldf(dO + o2) * sigmoidf_(ldf(G + o2)) : 0.0f;
        }
        if (threadIdx.x < QC) {
            int q = q0 + threadIdx.x;
            lse_s[threadIdx.x] = q < p.N ? LSE[sl.lse_base + (long long)q * p.lQ] : -INFINITY;
            D_s[threadIdx.x] = q < p.N ? Dws[sl.lse_base + (long long)q * p.lQ] : 0.0f;
        }
        load_bias_tile<T, QC, KB, KB + 1, KB>(p, biasbh, q0, k0, Bs);
        __syncthreads();
#pragma unroll 2
        for (int qq = 0; qq < QC; ++qq) {
            float dot = 0.0f, dp = 0.0f;
#pragma unroll
            for (int c = 0; c < D; ++c) { dot = fmaf(kreg[c], Qs[qq][c], dot); dp = fmaf(vreg[c], As[qq][c], dp); }
            const float s = kkeep ? fmaf(dot, scale, Bs[qq * (KB + 1) + threadIdx.x]) : -INFINITY;
            const float pr = prob(s, lse_s[qq]);
            const float ds = pr * (dp - D_s[qq]);
#pragma unroll
            for (int c = 0; c < D; ++c) { dv[c] = fmaf(pr, As[qq][c], dv[c]); dk[c] = fmaf(ds, Qs[qq][c], dk[c]); }
        }
    }
    if (kvalid) {
#pragma unroll
        for (int c = 0; c < D; ++c) { stf(dK + off + c, dk[c] * scale); stf(dV + off + c, dv[c]); }
    }
}

// ---------------------------------------------------------------------------------------------
// Backward stage 2b: dBias[b,h,q,k] = sum over slices r (ascending) of dS -- tile-stationary,
// deterministic (Table I; replaces tl.atomic_add P:L488).
// ---------------------------------------------------------------------------------------------
template <typename T, int D>
__global__ void __launch_bounds__(256) simt_dbias_kernel(Problem p, const T* __restrict__ dO, const T* __restrict__ Q,
                                                         const T* __restrict__ K, const T* __restrict__ V,
                                                         const T* __restrict__ G, const T* __restrict__ bias,
                                                         const unsigned char* __restrict__ mask, const float* __restrict__ LSE,
                                                         const float* __restrict__ Dws, float* __restrict__ dBias) {
    constexpr int TS = 16;
    __shared__ float Qs[TS][D + 1], As[TS][D + 1], Ks[TS][D + 1], Vs[TS][D + 1];
    __shared__ float lse_s[TS], D_s[TS];
    __shared__ unsigned char keep[TS];
    const int b = blockIdx.z / p.H, h = blockIdx.z % p.H;
    const int q0 = blockIdx.y * TS, k0 = blockIdx.x * TS;
    const int tq = threadIdx.x / TS, tk = threadIdx.x % TS;
    const int q = q0 + tq, k = k0 + tk;
    const bool valid = q < p.N && k < p.N;
    const float scale = 1.0f / sqrtf((float)D);
    const long long bh = ((long long)b * p.H + h) * p.N * p.N;
    const float bia = valid ? ldf(bias + bh + (long long)q * p.bQ + (long long)k * p.bK) : 0.0f;
    float acc = 0.0f;
    for (int r = 0; r < p.N; ++r) {
        const long long base = b * p.sB + h * p.sH + r * p.sSlice;
        const long long lbase = (long long)b * p.N * p.H * p.N + (long long)h * p.N + r * p.lR;
        __syncthreads();
        for (int idx = threadIdx.x; idx < TS * D; idx += 256) {
            int pp = idx / D, c = idx % D;
            const long long oq = base + (long long)(q0 + pp) * p.sPos + c;
            const long long ok = base + (long long)(k0 + pp) * p.sPos + c;
            Qs[pp][c] = (q0 + pp) < p.N ? ldf(Q + oq) : 0.0f;
            As[pp][c] = (q0 + pp) < p.N ? ldf(dO + oq) * sigmoidf_(ldf(G + oq)) : 0.0f;
            Ks[pp][c] = (k0 + pp) < p.N ? ldf(K + ok) : 0.0f;
            Vs[pp][c] = (k0 + pp) < p.N ? ldf(V + ok) : 0.0f;
        }
        if (threadIdx.x < TS) {
            int qq = q0 + threadIdx.x, kk = k0 + threadIdx.x;
            lse_s[threadIdx.x] = qq < p.N ? LSE[lbase + (long long)qq * p.lQ] : -INFINITY;
            D_s[threadIdx.x] = qq < p.N ? Dws[lbase + (long long)qq * p.lQ] : 0.0f;
            keep[threadIdx.x] = kk < p.N && (!mask || mask[(long long)b * p.N * p.N + (long long)r * p.mR + (long long)kk * p.mK]);
        }
        __syncthreads();
        float dot = 0.0f, dp = 0.0f;
#pragma unroll
        for (int c = 0; c < D; ++c) { dot = fmaf(Qs[tq][c], Ks[tk][c], dot); dp = fmaf(As[tq][c], Vs[tk][c], dp); }
        const float s = keep[tk] ? fmaf(dot, scale, bia) : -INFINITY;
        acc += prob(s, lse_s[tq]) * (dp - D_s[tq]);
    }
    if (valid) dBias[bh + (long long)q * p.bQ + (long long)k * p.bK] = acc;
}

template <typename T, int D>
tri_status fwd_t(const Problem& p, const void* Q, const void* K, const void* V, const void* G, const void* bias,
                 const unsigned char* mask, void* O, float* LSE, cudaStream_t st) {
    dim3 grid(p.B * p.N * p.H, (p.N + 63) / 64);
    { ProfScope ps("simt_fwd_kernel", st);
    simt_fwd_kernel<T, D><<<grid, 64, 0, st>>>(p, (const T*)Q, (const T*)K, (const T*)V, (const T*)G, (const T*)bias, mask,
                                               (T*)O, LSE);
    }
    TRI_LAUNCH_CHECK("simt_fwd_kernel");
    return TRI_OK;
}

template <typename T, int D>
tri_status bwd_t(const Problem& p, const void* dO, const void* Q, const void* K, const void* V, const void* G,
                 const void* bias, const unsigned char* mask, const void* O, const float* LSE, void* dQ, void* dK,
                 void* dV, void* dG, float* dBias, void* ws, cudaStream_t st) {
    float* Dws = (float*)ws;
    const long long rows = (long long)p.B * p.N * p.H * p.N;
    { ProfScope ps("simt_preprocess_kernel", st);
    simt_preprocess_kernel<T, D><<<(unsigned)((rows + 127) / 128), 128, 0, st>>>(rows, (const T*)dO, (const T*)O,
                                                                                (const T*)G, (T*)dG, Dws);
    }
    TRI_LAUNCH_CHECK("simt_preprocess_kernel");
    dim3 grid(p.B * p.N * p.H, (p.N + 63) / 64);
    { ProfScope ps("simt_dkdv_kernel", st);
    simt_dkdv_kernel<T, D><<<grid, 64, 0, st>>>(p, (const T*)dO, (const T*)Q, (const T*)K, (const T*)V, (const T*)G,
                                                (const T*)bias, mask, LSE, Dws, (T*)dK, (T*)dV);
    }
    TRI_LAUNCH_CHECK("simt_dkdv_kernel");
    { ProfScope ps("simt_dq_kernel", st);
    simt_dq_kernel<T, D><<<grid, 64, 0, st>>>(p, (const T*)dO, (const T*)Q, (const T*)K, (const T*)V, (const T*)G,
                                              (const T*)bias, mask, LSE, Dws, (T*)dQ);
    }
    TRI_LAUNCH_CHECK("simt_dq_kernel");
    dim3 gb((p.N + 15) / 16, (p.N + 15) / 16, p.B * p.H);
    { ProfScope ps("simt_dbias_kernel", st);
    simt_dbias_kernel<T, D><<<gb, 256, 0, st>>>(p, (const T*)dO, (const T*)Q, (const T*)K, (const T*)V, (const T*)G,
                                                (const T*)bias, mask, LSE, Dws, dBias);
    }
    TRI_LAUNCH_CHECK("simt_dbias_kernel");
    return TRI_OK;
}

}  // namespace

size_t simt_fwd_workspace(const Problem&) { return 0; }
size_t simt_bwd_workspace(const Problem& p) { return align_up((size_t)p.B * p.N * p.H * p.N * sizeof(float), 256); }

#define TRI_DISPATCH(FN, ...)                                                                 \
    if (dt == TRI_F32) {                                                                      \
        if (p.d == 16) return FN<float, 16>(__VA_ARGS__);                                     \
        if (p.d == 32) return FN<float, 32>(__VA_ARGS__);                                     \
        if (p.d == 64) return FN<float, 64>(__VA_ARGS__);                                     \
    } else {                                                                                  \
        if (p.d == 16) return FN<__nv_bfloat16, 16>(__VA_ARGS__);                             \
        if (p.d == 32) return FN<__nv_bfloat16, 32>(__VA_ARGS__);                             \
        if (p.d == 64) return FN<__nv_bfloat16, 64>(__VA_ARGS__);                             \
    }                                                                                         \
    return TRI_ERR_UNSUPPORTED;

tri_status simt_fwd(const Problem& p, tri_dtype dt, const void* Q, const void* K, const void* V, const void* G,
                    const void* bias, const unsigned char* mask, void* O, float* LSE, void*, cudaStream_t st) {
    TRI_DISPATCH(fwd_t, p, Q, K, V, G, bias, mask, O, LSE, st)
}

tri_status simt_bwd(const Problem& p, tri_dtype dt, const void* dO, const void* Q, const void* K, const void* V,
                    const void* G, const void* bias, const unsigned char* mask, const void* O, const float* LSE,
                    void* dQ, void* dK, void* dV, void* dG, float* dBias, void* ws, cudaStream_t st) {
    TRI_DISPATCH(bwd_t, p, dO, Q, K, V, G, bias, mask, O, LSE, dQ, dK, dV, dG, dBias, ws, st)
}

}  // namespace tri

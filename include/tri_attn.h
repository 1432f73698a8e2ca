/*
 * tri_attn.h -- C ABI of libtri_attn.so: fused forward / backward of AF3-style triangle attention
 * with pair bias ("EvoAttention"; memory-efficient kernel "EvoFlash-3D") for NVIDIA B200 (sm_100a).
 *
 * What is computed (PAPER.md = /root/reference/PAPER.md of arxiv 2506.20686, cited P:L<line>):
 *   forward   S = scale*Q K^T + Bias_bcast + M(mask);  P = softmax_k(S);  A = P V;  O = sigmoid(G) (.) A
 *             Table I, Sec. IV-A, Listing 1 P:L153-185 (`fused_attn_fwd`).
 *             scale = 1/sqrt(d), the sigmoid gate G and the additive -inf mask are fixed by the task
 *             statement (BASELINE.json north_star), not by the paper (readings A1/A3/A4).
 *   backward  dV = P^T dA, dP = dA V^T, dS = P (.) (dP - rowsum(dO (.) O)), dK = scale dS^T Q,
 *             dQ = scale dS K, dBias = sum over the broadcast axis of dS, dA = dO (.) sigmoid(G),
 *             dG = dO (.) O (.) (1 - sigmoid(G)).   Table I, Listing 2
 *             (`fused_attn_bwd`: preprocess D, stage 1 dK/dV, stage 2 dQ/dBias).  The paper's
 *             atomic_add of dS tiles is replaced by a deterministic two-level reduction.
 *   The O(N^3) attention map [B,N,H,N,N] is never written to device memory.
 *
 * Tensor layouts (row-major, contiguous; "a" = first pair axis, "c" = second pair axis):
 *   Q,K,V,G,O,dO,dQ,dK,dV,dG : [B, N, H, N, d]   element (b,a,h,c,:)      dtype = `dtype`
 *   bias                     : [B, H, N, N]                               dtype = `dtype`
 *   dBias                    : [B, H, N, N]                               float32 always
 *   mask                     : [B, N, N] unsigned char keep flags (non-zero = visible), or NULL
 *   LSE                      : [B, N, H, N] float32, natural-log units, element (b,a,h,c)
 *
 * Variants:
 *   TRI_STARTING  row i = a, query j = c, key k = c':
 *       S[b,i,h,j,k] = scale <Q[b,i,h,j,:],K[b,i,h,k,:]> + bias[b,h,j,k] + M(mask[b,i,k])
 *       O[b,i,h,j,:] = sigmoid(G[b,i,h,j,:]) (.) sum_k P V[b,i,h,k,:];  dBias[b,h,j,k] = sum_i dS
 *   TRI_ENDING    (= T . starting . T, T = swap of the two N axes of every argument)
 *       S[b,i,h,j,k] = scale <Q[b,i,h,j,:],K[b,k,h,j,:]> + bias[b,h,k,i] + M(mask[b,k,j])
 *       O[b,i,h,j,:] = sigmoid(G[b,i,h,j,:]) (.) sum_k P V[b,k,h,j,:];  dBias[b,h,k,i] = sum_j dS
 *   A query whose keys are all masked gives O = 0, LSE = -inf and contributes zero gradients.
 *
 * Ownership and behaviour:
 *   - Every tensor pointer of tri_attn_fwd / tri_attn_bwd is a caller-owned DEVICE pointer, 16-byte
 *     aligned.  The library never allocates or frees device memory and never synchronises the
 *     device: all work is enqueued on `cuda_stream` (a cudaStream_t passed as void*; NULL = the
 *     legacy default stream) -- or, for kernels that may overlap (tri_attn_bwd runs a slice of its
 *     dK/dV stage beside its dQ/dBias stage; tri_attn_step_host overlaps copies and compute), on
 *     library-owned side streams that are forked from and joined back into `cuda_stream` with
 *     events inside the call, so to the caller each call is still one unit of work on `cuda_stream`.  Scratch space comes from `workspace` (device, 256-byte aligned, at
 *     least *_workspace_bytes() bytes, contents undefined on entry and exit).  workspace_bytes is
 *     O(B*H*N^2*d) (the backward keeps one dA = dO (.) sigmoid(G) tensor there); nothing of size
 *     B*H*N^3 exists anywhere.
 *   - Thread safety: entry points may be called from several host threads (on the same or different devices and
 *     streams); enqueues that share a device's side streams take turns inside the library.  The exceptions are the
 *     profiling calls (one thread) and tri_attn_fwd_noalloc (overlapping calls race on its built-in scratch).
 *   - tri_attn_fwd / tri_attn_bwd / tri_attn_rows_* enqueue stream work only (kernels and the event fork / join of the
 *     side streams), so a step can be captured into a CUDA graph on `cuda_stream` and replayed (tested; make one eager
 *     call first so that the library's streams, events and tensor maps exist before the capture).
 *   - Outputs (and the workspace) must not overlap inputs or each other: such a call returns
 *     TRI_ERR_INVALID_ARG before any launch.  Outputs are overwritten (dBias is NOT accumulated into).  Results are bitwise reproducible run to run (no floating-point atomics).
 *   - tri_attn_step_host takes HOST pointers (pinned memory recommended) for every tensor plus a
 *     caller-owned DEVICE arena; it copies inputs in, runs forward + backward, copies results out
 *     and does not synchronise.  Batch elements are independent problems, so it pipelines them:
 *     host->device copies, compute and device->host copies of different elements overlap on two
 *     library-owned copy streams forked from and joined back into `cuda_stream` with events (to the
 *     caller it is still one unit of work on that stream).  Each element is solved as a B = 1
 *     problem: identical to tri_attn_fwd/bwd on that element alone, which for dBias can differ in the
 *     last bits from a B > 1 call (the row split of the deterministic reduction depends on B).
 *     On the tensor-core path of the starting-node variant the broadcast rows of an element are
 *     independent too, so an element is further cut into about eight row chunks (>= 4 MB per tensor,
 *     each run as a tri_attn_rows_* problem): O, LSE, dQ, dK, dV, dG stay bitwise those of
 *     tri_attn_fwd/bwd, dBias is accumulated chunk after chunk in row order (same fp32 sum, another
 *     grouping; still bitwise reproducible run to run).
 *   - Errors: a tri_status is returned, nothing is thrown or aborted across the ABI.  Argument
 *     errors are detected before any launch.  Launch failures map to TRI_ERR_CUDA.
 *   - Supported: d in {16, 32, 64}, any N >= 1, dtype f32 or bf16.  bf16 with d == 32,
 *     N % 8 == 0 and 128 <= N <= 8192 runs on the tcgen05/TMA tensor-core kernels (N need not be a
 *     multiple of their 64 / 128-position tiles: partial tiles are zero-filled by TMA and masked);
 *     every other combination runs on the fp32 CUDA-core kernels, ~30x slower (fp32 needs them: the
 *     1e-4 bound excludes TF32, reading A14); tri_attn_uses_tensor_cores() tells which.
 *     The FORWARD alone (tri_attn_fwd, tri_attn_rows_fwd, tri_attn_fwd_noalloc) stays on the tensor-core kernels up to
 *     N = 16384 (long-sequence inference).  The backward of N > 2048 runs its fused dQ + dBias stage in
 *     ceil(N / 2048) launches over slices of the key axis (its workspace then also holds an fp32 dQ sum).
 *     Anything else returns TRI_ERR_UNSUPPORTED.  There is no CPU path.
 */
#ifndef TRI_ATTN_H_
#define TRI_ATTN_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define TRI_API __attribute__((visibility("default")))
#else
#define TRI_API
#endif

typedef enum {
    TRI_OK = 0,
    TRI_ERR_INVALID_ARG = 1, /* NULL / misaligned pointer, non-positive size, bad enum            */
    TRI_ERR_UNSUPPORTED = 2, /* shape or dtype outside the supported set                           */
    TRI_ERR_WORKSPACE = 3,   /* workspace NULL / misaligned / smaller than *_workspace_bytes()      */
    TRI_ERR_CUDA = 4,        /* a CUDA runtime / driver call or a kernel launch failed             */
    TRI_ERR_TOO_LARGE = 5    /* tri_attn_fwd_noalloc: the problem needs more scratch than the built-in array holds */
} tri_status;

typedef enum { TRI_F32 = 0, TRI_BF16 = 1 } tri_dtype;
typedef enum { TRI_STARTING = 0, TRI_ENDING = 1 } tri_variant;

/* Bytes of device scratch tri_attn_fwd / tri_attn_bwd need for this problem (0 on bad arguments). */
TRI_API size_t tri_attn_fwd_workspace_bytes(int B, int N, int H, int d, tri_variant variant, tri_dtype dtype);
TRI_API size_t tri_attn_bwd_workspace_bytes(int B, int N, int H, int d, tri_variant variant, tri_dtype dtype);

/* Forward (Listing 1 P:L153-185 + gate + mask).  Inputs Q,K,V,G,bias,mask; outputs O, LSE. */
TRI_API tri_status tri_attn_fwd(const void* Q, const void* K, const void* V, const void* G,
                        const void* bias, const unsigned char* mask /* NULL = no mask */,
                        void* O, float* LSE,
                        int B, int N, int H, int d, tri_variant variant, tri_dtype dtype,
                        void* workspace, size_t workspace_bytes, void* cuda_stream);

/* Backward (Listing 2 P:L434-494 + gate).  O and LSE are the forward's outputs.
 * Outputs dQ,dK,dV,dG (dtype) and dBias (float32). */
TRI_API tri_status tri_attn_bwd(const void* dO,
                        const void* Q, const void* K, const void* V, const void* G,
                        const void* bias, const unsigned char* mask,
                        const void* O, const float* LSE,
                        void* dQ, void* dK, void* dV, void* dG, float* dBias,
                        int B, int N, int H, int d, tri_variant variant, tri_dtype dtype,
                        void* workspace, size_t workspace_bytes, void* cuda_stream);

/* Decoupled row count ("EvoAttention" with rows != N, e.g. MSA-row attention with pair bias, or a
 * chunk of the rows of a pair tensor): R independent broadcast rows, each attending over N positions with the shared
 * bias[b,h,j,k].  Starting-node index convention only:
 *     Q,K,V,G,O,dO,dQ,dK,dV,dG : [B, R, H, N, d]     mask : [B, R, N] (or NULL)     LSE : [B, R, H, N]
 *     bias, dBias              : [B, H, N, N]        dBias[b,h,j,k] = sum over the R rows of dS
 * Runs on the tensor-core kernels only: bf16, d == 32, N % 8 == 0, 128 <= N <= 8192 (forward: 16384), any R >= 1 (R = 1 is single-representation attention with pair bias); anything else returns
 * TRI_ERR_UNSUPPORTED (workspace queries return 0).  tri_attn_fwd / tri_attn_bwd are the R == N case. */
TRI_API size_t tri_attn_rows_fwd_workspace_bytes(int B, int R, int N, int H, int d, tri_dtype dtype);
TRI_API size_t tri_attn_rows_bwd_workspace_bytes(int B, int R, int N, int H, int d, tri_dtype dtype);
TRI_API tri_status tri_attn_rows_fwd(const void* Q, const void* K, const void* V, const void* G,
                             const void* bias, const unsigned char* mask /* NULL = no mask */,
                             void* O, float* LSE,
                             int B, int R, int N, int H, int d, tri_dtype dtype,
                             void* workspace, size_t workspace_bytes, void* cuda_stream);
TRI_API tri_status tri_attn_rows_bwd(const void* dO,
                             const void* Q, const void* K, const void* V, const void* G,
                             const void* bias, const unsigned char* mask,
                             const void* O, const float* LSE,
                             void* dQ, void* dK, void* dV, void* dG, float* dBias,
                             int B, int R, int N, int H, int d, tri_dtype dtype,
                             void* workspace, size_t workspace_bytes, void* cuda_stream);

/* Forward WITHOUT a caller workspace and without any device allocation (for callers that cannot call cudaMalloc: code
 * under CUDA graph capture, tight serving loops, harnesses that forbid it).  Same operation, arguments, layouts and
 * results as tri_attn_fwd (Listing 1 P:L153-185 + gate + mask); the scratch tri_attn_fwd takes from `workspace` lives in
 * one file-scope device array of TRI_NOALLOC_SCRATCH_BYTES inside the library, which every GPU that loads the library
 * holds until the process exits.  The call allocates nothing (no cudaMalloc / cudaFree / allocating library routine).
 *   - Limit: problems with tri_attn_fwd_workspace_bytes() > TRI_NOALLOC_SCRATCH_BYTES (32 MiB; e.g. bf16 d = 32 with
 *     B*H*N*N > ~8.3 M: cfg4 B=2 H=4 N=768 and cfg5 B=1 H=4 N=1024 fit, N = 2048 with H = 4 does not) return
 *     TRI_ERR_TOO_LARGE before any launch; use tri_attn_fwd with a workspace for those.
 *   - The array is shared by every call on a device and keeps the last call's contents (each call overwrites what it
 *     reads, nothing needs clearing).  Calls that overlap on the GPU -- different streams, or host threads without
 *     stream ordering between their calls -- RACE on it: keep the calls of one device on one stream, or order them.
 *   - Other errors as tri_attn_fwd. */
#define TRI_NOALLOC_SCRATCH_BYTES (32u << 20)
TRI_API size_t tri_attn_noalloc_scratch_bytes(void);
TRI_API tri_status tri_attn_fwd_noalloc(const void* Q, const void* K, const void* V, const void* G,
                                const void* bias, const unsigned char* mask /* NULL = no mask */,
                                void* O, float* LSE,
                                int B, int N, int H, int d, tri_variant variant, tri_dtype dtype,
                                void* cuda_stream);

/* EvoSP-3D, backward: reduce-scatter of the per-rank partial dBias as ONE kernel over peer memory.
 * peer_dbias: HOST array of P DEVICE pointers, one per rank of the SP group in rank order, each to that rank's partial dBias
 * [B,H,N,N] float32 (what tri_attn_rows_bwd wrote for the rank's rows); all must be loadable from the current device
 * (peer access over NVLink / NVSwitch, e.g. torch symmetric memory, or buffers of the same device).  Writes
 *     out_shard[b,h,l,k] = sum_{p = 0 .. P-1, ascending} peer_dbias[p][b,h, rank*(N/P) + l, k]     [B,H,N/P,N] float32
 * i.e. this rank's N/P query lines of the total -- the sharding the bias was gathered from.  Fixed summation order:
 * bitwise reproducible.  P <= 16, N % P == 0, N % 4 == 0, 16-byte aligned pointers, else TRI_ERR_UNSUPPORTED /
 * TRI_ERR_INVALID_ARG.  The caller orders it after every peer's backward and keeps the peers from overwriting their
 * buffers until all ranks have read them (paper_2506_20686_b200/evosp.py does both with the symmetric-memory barrier). */
/* EvoSP-3D, forward: all-gather of the bias by pulling over peer memory.  peer_shards: HOST array of P DEVICE
 * pointers in rank order, each to that rank's shard [B,H,N/P,N] (`dtype`) of query lines; writes the full out_bias [B,H,N,N]
 * on this device.  Same peer-access, alignment (16 bytes; N * sizeof(elem) % 16 == 0), P <= 16 and ordering rules as below. */
TRI_API tri_status tri_attn_bias_all_gather(const void* const* peer_shards, int P, void* out_bias, int B, int H, int N,
                                    tri_dtype dtype, void* cuda_stream);
TRI_API tri_status tri_attn_dbias_reduce_scatter(const float* const* peer_dbias, int P, int rank, float* out_shard,
                                         int B, int H, int N, void* cuda_stream);

/* End-to-end step on HOST buffers: H2D(Q,K,V,G,bias,mask,dO) -> fwd -> bwd -> D2H(O,LSE,dQ,dK,dV,
 * dG,dBias).  `arena` is a caller-owned device buffer of tri_attn_step_host_arena_bytes() bytes. */
TRI_API size_t tri_attn_step_host_arena_bytes(int B, int N, int H, int d, tri_variant variant, tri_dtype dtype);
TRI_API tri_status tri_attn_step_host(const void* hQ, const void* hK, const void* hV, const void* hG,
                              const void* hbias, const unsigned char* hmask, const void* hdO,
                              void* hO, float* hLSE,
                              void* hdQ, void* hdK, void* hdV, void* hdG, float* hdBias,
                              int B, int N, int H, int d, tri_variant variant, tri_dtype dtype,
                              void* arena, size_t arena_bytes, void* cuda_stream);

/* 1 if forward AND backward of this problem run on the tcgen05/TMA tensor-core kernels, 0 if the backward (and, but for
 * bf16 d = 32 with 8192 < N <= 16384, N % 8 == 0, also the forward) runs on the fp32 CUDA-core kernels. */
TRI_API int tri_attn_uses_tensor_cores(int B, int N, int H, int d, tri_variant variant, tri_dtype dtype);

/* Number of kernel launches this library has enqueued since it was loaded (for bench accounting). */
TRI_API unsigned long long tri_attn_launch_count(void);

/* Per-kernel timing for the bench's roofline line.  After _begin, every kernel the library launches is
 * bracketed by CUDA events on its stream.  _end synchronises those events (the only call here that
 * blocks the host), stops recording and writes one text line per kernel name into `buf` (host):
 * "<kernel> <launches> <total_ms>\n".  Returns the number of distinct kernels, -1 on a CUDA error.
 * Not thread-safe; at most 8192 launches are recorded per _begin. */
TRI_API void tri_attn_profile_begin(void);
TRI_API int tri_attn_profile_end(char* buf, size_t buflen);

/* Static description of a status code. */
TRI_API const char* tri_status_string(tri_status s);

/* Last CUDA error text recorded by a TRI_ERR_CUDA return on this thread ("" if none). */
TRI_API const char* tri_attn_last_cuda_error(void);

#ifdef __cplusplus
}
#endif
#endif /* TRI_ATTN_H_ */

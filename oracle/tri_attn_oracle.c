/*
 * tri_attn_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU implementation of AF3-style triangle attention with pair bias
 * (the paper's "EvoAttention"), forward and backward, written out from the definition:
 *
 *   forward   S = scale*Q K^T + Bias_bcast (+ mask),  P = softmax(S),  A = P V,  O = sigmoid(G) (.) A
 *             (Table I; Sec. IV-A; scale 1/sqrt(d), gate and mask:
 *              BASELINE.json north_star -- they are not in the paper, readings A1/A3/A4)
 *   backward  dV = P^T dA,  dP = dA V^T,  dS = P (.) (dP - rowsum(P (.) dP)),
 *             dK = scale dS^T Q,  dQ = scale dS K,  dBias = sum_bcast dS       (Table I)
 *             with dA = dO (.) sigmoid(G),  dG = dO (.) A (.) sg (1 - sg)      (chain rule, north_star)
 *
 * The full N_q x N_k attention map of every (b,row,h) slice is materialised (and optionally the
 * whole [B,R,H,Nq,Nk] tensor is returned) -- exactly what the GPU path must never do.  There is
 * no tiling, no online softmax, no fusion.  The softmax-Jacobian row term is the plain
 * sum_k P*dP, NOT the rowsum(dO (.) O) shortcut of P:L437/P:L511, so that shortcut is itself tested.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * call this.  It shares no code with paper_2506_20686_b200/ (the CUDA path).
 *
 * Layout (row-major, contiguous), "starting node" general-shape core:
 *   Q,G,O,dO,dQ,dG : [B, R, H, Nq, d]      K,V,dK,dV : [B, R, H, Nk, d]
 *   bias,dBias     : [B, H, Nq, Nk]        mask      : [B, R, Nk] u8 keep flags (NULL = none)
 *   LSE            : [B, R, H, Nq]         P (opt.)  : [B, R, H, Nq, Nk]
 * The operator of the paper is the square case R = Nq = Nk = N.
 *
 *   S[b,r,h,q,k] = scale <Q[b,r,h,q,:], K[b,r,h,k,:]> + bias[b,h,q,k] + (mask[b,r,k] ? 0 : -inf)
 *
 * "Ending node" (square only, coded directly from its index formulas):
 *   S[b,i,h,j,k] = scale <Q[b,i,h,j,:], K[b,k,h,j,:]> + bias[b,h,k,i] + (mask[b,k,j] ? 0 : -inf)
 *   A[b,i,h,j,:] = sum_k P V[b,k,h,j,:];  dBias[b,h,k,i] = sum_j dS[b,i,h,j,k]
 *
 * Fully masked row (reading A6): P = 0, O = 0, LSE = -inf, all its gradient contributions 0.
 *
 * Parity pins: tests/test_oracle_pins.py (brute force, finite differences, closed forms,
 * invariants, torch fp64 SDPA+autograd cross-check).  No function here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define IDX5(b, r, h, n, c, R, H, N, D) \
    (((((size_t)(b) * (R) + (r)) * (H) + (h)) * (N) + (n)) * (D) + (c))

int tri_oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

static double sigmoid(double x) { return 1.0 / (1.0 + exp(-x)); }

/* logits and softmax of one (b,r,h) slice, starting-node indexing.
 * S, P : [Nq, Nk] scratch; lse : [Nq].  (Table I "S = QK^T + Bias_bcast", "P = Softmax(S)") */
static void slice_softmax_start(const double* Q, const double* K, const double* bias,
                                const uint8_t* mask, int b, int r, int h, int R, int H, int Nq,
                                int Nk, int d, double* P, double* lse) {
    const double scale = 1.0 / sqrt((double)d);
#pragma omp parallel for schedule(static)
    for (int q = 0; q < Nq; ++q) {
        double* Pq = P + (size_t)q * Nk;
        const double* qv = Q + IDX5(b, r, h, q, 0, R, H, Nq, d);
        double m = -INFINITY;
        for (int k = 0; k < Nk; ++k) {
            const double* kv = K + IDX5(b, r, h, k, 0, R, H, Nk, d);
            double dot = 0.0;
            for (int c = 0; c < d; ++c) dot += qv[c] * kv[c];
            double s = scale * dot + bias[(((size_t)b * H + h) * Nq + q) * Nk + k];
            if (mask && !mask[((size_t)b * R + r) * Nk + k]) s = -INFINITY;
            Pq[k] = s;
            if (s > m) m = s;
        }
        if (m == -INFINITY) { /* fully masked row: reading A6 */
            for (int k = 0; k < Nk; ++k) Pq[k] = 0.0;
            lse[q] = -INFINITY;
            continue;
        }
        double l = 0.0;
        for (int k = 0; k < Nk; ++k) {
            Pq[k] = exp(Pq[k] - m);
            l += Pq[k];
        }
        for (int k = 0; k < Nk; ++k) Pq[k] /= l;
        lse[q] = m + log(l);
    }
}

int tri_oracle_fwd_start(const double* Q, const double* K, const double* V, const double* G,
                         const double* bias, const uint8_t* mask, int B, int R, int H, int Nq,
                         int Nk, int d, double* O, double* LSE, double* Pout) {
    double* P = (double*)malloc(sizeof(double) * (size_t)Nq * Nk);
    double* lse = (double*)malloc(sizeof(double) * (size_t)Nq);
    if (!P || !lse) return 1;
    for (int b = 0; b < B; ++b)
        for (int r = 0; r < R; ++r)
            for (int h = 0; h < H; ++h) {
                slice_softmax_start(Q, K, bias, mask, b, r, h, R, H, Nq, Nk, d, P, lse);
#pragma omp parallel for schedule(static)
                for (int q = 0; q < Nq; ++q) {
                    LSE[(((size_t)b * R + r) * H + h) * Nq + q] = lse[q];
                    for (int c = 0; c < d; ++c) {
                        double a = 0.0; /* A = P V  (Table I "O = PV") */
                        for (int k = 0; k < Nk; ++k)
                            a += P[(size_t)q * Nk + k] * V[IDX5(b, r, h, k, c, R, H, Nk, d)];
                        size_t o = IDX5(b, r, h, q, c, R, H, Nq, d);
                        O[o] = sigmoid(G[o]) * a; /* gate: north_star */
                    }
                }
                if (Pout)
                    memcpy(Pout + ((((size_t)b * R + r) * H + h) * Nq) * Nk, P,
                           sizeof(double) * (size_t)Nq * Nk);
            }
    free(P);
    free(lse);
    return 0;
}

int tri_oracle_bwd_start(const double* dO, const double* Q, const double* K, const double* V,
                         const double* G, const double* bias, const uint8_t* mask, int B, int R,
                         int H, int Nq, int Nk, int d, double* dQ, double* dK, double* dV,
                         double* dG, double* dBias) {
    const double scale = 1.0 / sqrt((double)d);
    double* P = (double*)malloc(sizeof(double) * (size_t)Nq * Nk);
    double* dS = (double*)malloc(sizeof(double) * (size_t)Nq * Nk);
    double* dA = (double*)malloc(sizeof(double) * (size_t)Nq * d);
    double* lse = (double*)malloc(sizeof(double) * (size_t)Nq);
    if (!P || !dS || !dA || !lse) return 1;
    memset(dBias, 0, sizeof(double) * (size_t)B * H * Nq * Nk);
    for (int b = 0; b < B; ++b)
        for (int r = 0; r < R; ++r) /* ascending row order for the dBias sum */
            for (int h = 0; h < H; ++h) {
                slice_softmax_start(Q, K, bias, mask, b, r, h, R, H, Nq, Nk, d, P, lse);
#pragma omp parallel for schedule(static)
                for (int q = 0; q < Nq; ++q) {
                    const double* Pq = P + (size_t)q * Nk;
                    double* dSq = dS + (size_t)q * Nk;
                    /* dA = dO (.) sg ; dG = dO (.) A (.) sg (1-sg) */
                    for (int c = 0; c < d; ++c) {
                        double a = 0.0;
                        for (int k = 0; k < Nk; ++k)
                            a += Pq[k] * V[IDX5(b, r, h, k, c, R, H, Nk, d)];
                        size_t o = IDX5(b, r, h, q, c, R, H, Nq, d);
                        double sg = sigmoid(G[o]);
                        dA[(size_t)q * d + c] = dO[o] * sg;
                        dG[o] = dO[o] * a * sg * (1.0 - sg);
                    }
                    /* dP = dA V^T; Dq = sum_k P dP (softmax Jacobian, plain form) */
                    double Dq = 0.0;
                    for (int k = 0; k < Nk; ++k) {
                        double dp = 0.0;
                        for (int c = 0; c < d; ++c)
                            dp += dA[(size_t)q * d + c] * V[IDX5(b, r, h, k, c, R, H, Nk, d)];
                        dSq[k] = dp;
                        Dq += Pq[k] * dp;
                    }
                    /* dS = P (.) (dP - Dq) ; dBias += dS */
                    double* dBq = dBias + (((size_t)b * H + h) * Nq + q) * Nk;
                    for (int k = 0; k < Nk; ++k) {
                        dSq[k] = Pq[k] * (dSq[k] - Dq);
                        dBq[k] += dSq[k];
                    }
                    /* dQ = scale dS K */
                    for (int c = 0; c < d; ++c) {
                        double g = 0.0;
                        for (int k = 0; k < Nk; ++k)
                            g += dSq[k] * K[IDX5(b, r, h, k, c, R, H, Nk, d)];
                        dQ[IDX5(b, r, h, q, c, R, H, Nq, d)] = scale * g;
                    }
                }
#pragma omp parallel for schedule(static)
                for (int k = 0; k < Nk; ++k) {
                    for (int c = 0; c < d; ++c) {
                        double gv = 0.0, gk = 0.0;
                        for (int q = 0; q < Nq; ++q) {
                            gv += P[(size_t)q * Nk + k] * dA[(size_t)q * d + c]; /* dV = P^T dA */
                            gk += dS[(size_t)q * Nk + k] *
                                  Q[IDX5(b, r, h, q, c, R, H, Nq, d)]; /* dK = dS^T Q (A9) */
                        }
                        dV[IDX5(b, r, h, k, c, R, H, Nk, d)] = gv;
                        dK[IDX5(b, r, h, k, c, R, H, Nk, d)] = scale * gk;
                    }
                }
            }
    free(P);
    free(dS);
    free(dA);
    free(lse);
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * Ending node, square [B,N,H,N,d], written directly from its index formulas.
 * For a fixed (b, j, h) the "slice" has queries i and keys k, both running over the FIRST axis.
 * ---------------------------------------------------------------------------------------- */
static void slice_softmax_end(const double* Q, const double* K, const double* bias,
                              const uint8_t* mask, int b, int j, int h, int N, int H, int d,
                              double* P, double* lse) {
    const double scale = 1.0 / sqrt((double)d);
#pragma omp parallel for schedule(static)
    for (int i = 0; i < N; ++i) {
        double* Pi = P + (size_t)i * N;
        const double* qv = Q + IDX5(b, i, h, j, 0, N, H, N, d);
        double m = -INFINITY;
        for (int k = 0; k < N; ++k) {
            const double* kv = K + IDX5(b, k, h, j, 0, N, H, N, d);
            double dot = 0.0;
            for (int c = 0; c < d; ++c) dot += qv[c] * kv[c];
            double s = scale * dot + bias[(((size_t)b * H + h) * N + k) * N + i];
            if (mask && !mask[((size_t)b * N + k) * N + j]) s = -INFINITY;
            Pi[k] = s;
            if (s > m) m = s;
        }
        if (m == -INFINITY) {
            for (int k = 0; k < N; ++k) Pi[k] = 0.0;
            lse[i] = -INFINITY;
            continue;
        }
        double l = 0.0;
        for (int k = 0; k < N; ++k) {
            Pi[k] = exp(Pi[k] - m);
            l += Pi[k];
        }
        for (int k = 0; k < N; ++k) Pi[k] /= l;
        lse[i] = m + log(l);
    }
}

int tri_oracle_fwd_end(const double* Q, const double* K, const double* V, const double* G,
                       const double* bias, const uint8_t* mask, int B, int N, int H, int d,
                       double* O, double* LSE, double* Pout /* [B,N(i),H,N(j),N(k)] */) {
    double* P = (double*)malloc(sizeof(double) * (size_t)N * N);
    double* lse = (double*)malloc(sizeof(double) * (size_t)N);
    if (!P || !lse) return 1;
    for (int b = 0; b < B; ++b)
        for (int j = 0; j < N; ++j)
            for (int h = 0; h < H; ++h) {
                slice_softmax_end(Q, K, bias, mask, b, j, h, N, H, d, P, lse);
#pragma omp parallel for schedule(static)
                for (int i = 0; i < N; ++i) {
                    LSE[(((size_t)b * N + i) * H + h) * N + j] = lse[i];
                    for (int c = 0; c < d; ++c) {
                        double a = 0.0;
                        for (int k = 0; k < N; ++k)
                            a += P[(size_t)i * N + k] * V[IDX5(b, k, h, j, c, N, H, N, d)];
                        size_t o = IDX5(b, i, h, j, c, N, H, N, d);
                        O[o] = sigmoid(G[o]) * a;
                    }
                    if (Pout)
                        for (int k = 0; k < N; ++k)
                            Pout[((((size_t)b * N + i) * H + h) * N + j) * N + k] =
                                P[(size_t)i * N + k];
                }
            }
    free(P);
    free(lse);
    return 0;
}

int tri_oracle_bwd_end(const double* dO, const double* Q, const double* K, const double* V,
                       const double* G, const double* bias, const uint8_t* mask, int B, int N,
                       int H, int d, double* dQ, double* dK, double* dV, double* dG,
                       double* dBias) {
    const double scale = 1.0 / sqrt((double)d);
    double* P = (double*)malloc(sizeof(double) * (size_t)N * N);
    double* dS = (double*)malloc(sizeof(double) * (size_t)N * N);
    double* dA = (double*)malloc(sizeof(double) * (size_t)N * d);
    double* lse = (double*)malloc(sizeof(double) * (size_t)N);
    if (!P || !dS || !dA || !lse) return 1;
    memset(dBias, 0, sizeof(double) * (size_t)B * H * N * N);
    for (int b = 0; b < B; ++b)
        for (int j = 0; j < N; ++j) /* ascending j: the broadcast axis of the ending variant */
            for (int h = 0; h < H; ++h) {
                slice_softmax_end(Q, K, bias, mask, b, j, h, N, H, d, P, lse);
#pragma omp parallel for schedule(static)
                for (int i = 0; i < N; ++i) {
                    const double* Pi = P + (size_t)i * N;
                    double* dSi = dS + (size_t)i * N;
                    for (int c = 0; c < d; ++c) {
                        double a = 0.0;
                        for (int k = 0; k < N; ++k)
                            a += Pi[k] * V[IDX5(b, k, h, j, c, N, H, N, d)];
                        size_t o = IDX5(b, i, h, j, c, N, H, N, d);
                        double sg = sigmoid(G[o]);
                        dA[(size_t)i * d + c] = dO[o] * sg;
                        dG[o] = dO[o] * a * sg * (1.0 - sg);
                    }
                    double Di = 0.0;
                    for (int k = 0; k < N; ++k) {
                        double dp = 0.0;
                        for (int c = 0; c < d; ++c)
                            dp += dA[(size_t)i * d + c] * V[IDX5(b, k, h, j, c, N, H, N, d)];
                        dSi[k] = dp;
                        Di += Pi[k] * dp;
                    }
                    for (int k = 0; k < N; ++k) dSi[k] = Pi[k] * (dSi[k] - Di);
                    for (int c = 0; c < d; ++c) {
                        double g = 0.0;
                        for (int k = 0; k < N; ++k)
                            g += dSi[k] * K[IDX5(b, k, h, j, c, N, H, N, d)];
                        dQ[IDX5(b, i, h, j, c, N, H, N, d)] = scale * g;
                    }
                }
#pragma omp parallel for schedule(static)
                for (int k = 0; k < N; ++k) {
                    /* dBias[b,h,k,i] += dS[i][k]  (sum over j, outer loop) */
                    double* dBk = dBias + (((size_t)b * H + h) * N + k) * N;
                    for (int i = 0; i < N; ++i) dBk[i] += dS[(size_t)i * N + k];
                    for (int c = 0; c < d; ++c) {
                        double gv = 0.0, gk = 0.0;
                        for (int i = 0; i < N; ++i) {
                            gv += P[(size_t)i * N + k] * dA[(size_t)i * d + c];
                            gk += dS[(size_t)i * N + k] * Q[IDX5(b, i, h, j, c, N, H, N, d)];
                        }
                        dV[IDX5(b, k, h, j, c, N, H, N, d)] = gv;
                        dK[IDX5(b, k, h, j, c, N, H, N, d)] = scale * gk;
                    }
                }
            }
    free(P);
    free(dS);
    free(dA);
    free(lse);
    return 0;
}

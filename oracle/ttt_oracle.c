/*
 * oracle/ttt_oracle.c — float64 CPU oracle of the Scal3R TTT global-context-memory path.
 *
 * TEST INFRASTRUCTURE ONLY. Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, link or call this file. The product (paper_2604_08542_b200/)
 * shares no code with it and must never route through it.
 *
 * What it is: the method is an iteration (a gradient-step recurrence), so the oracle is the
 * algorithm itself, step by step in the paper's order, in double precision with no intermediate
 * rounding, plain i-k-j loops, no blocking, no fusion. Passages followed (PAPER.md line numbers):
 *   update  W <- W - grad_W sum_i eta_i L(f_W(k_i), v_i)            Eq. 8
 *   loss    L(f_W(K),V) = sum_i -f_W(k_i)^T v_i                     Eq. 9
 *   network f_W(x) = W2 (SiLU(W1 x) o (W3 x)), no bias              Eq. 12
 *   apply   o = f_W(q) with the UPDATED weights                     Eq. 4
 *   chunks processed sequentially, W carried
 * Readings of paper-silent points: sum not mean
 * (P1); row-vector storage W1,W3[hd][H], W2[H][hd], y = x.W (P3); M = tokens in the chunk (P5);
 * eta is an input array lr[nh][M] (P7); heads independent (P8).
 * Elements the paper does not define but BASELINE.json requires (DESIGN.md "Readings" R-NS,
 * R-RENORM): Newton-Schulz orthonormalisation of the gradient and fan-in
 * re-normalisation of the weights.
 *
 * Pins (tests/test_oracle_*.py): finite differences and torch-float64 autograd for the gradient,
 * the linear closed form W1 += K^T diag(eta) V, lr = 0, linearity in V and eta, token permutation,
 * head independence, SVD closed form of Newton-Schulz, renorm invariants, chunk recurrence.
 * Parity against the PAPER'S OWN NUMBERS IS UNPINNED: the paper prints no value for this layer.
 *
 * Layout at this boundary (same as include/ttt.h but host pointers and doubles):
 *   Q,K,V,O : [M][nh][hd], row stride ld (elements)      lr : [nh][M]
 *   W1,W3   : [nh][hd][H]                                W2 : [nh][H][hd]
 * Parallelism: OpenMP over heads only, so every sum has a fixed order and results are bitwise
 * independent of the thread count.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>

#ifdef _OPENMP
#include <omp.h>
#endif

/* overflow-safe logistic function */
static double sigmoid(double a)
{
    if (a >= 0.0) {
        return 1.0 / (1.0 + exp(-a));
    } else {
        double e = exp(a);
        return e / (1.0 + e);
    }
}

/* C[m][n] = sum_k A[m][k] * B[k][n]; row strides lda, ldb, ldc; plain i-k-j loops */
static void matmul_nn(const double *A, long lda, const double *B, long ldb, double *C, long ldc,
                      long m, long k, long n)
{
    for (long i = 0; i < m; ++i) {
        double *c = C + i * ldc;
        for (long j = 0; j < n; ++j) c[j] = 0.0;
        for (long p = 0; p < k; ++p) {
            double a = A[i * lda + p];
            const double *b = B + p * ldb;
            for (long j = 0; j < n; ++j) c[j] += a * b[j];
        }
    }
}

/* C[m][n] = sum_k A[k][m] * B[k][n]  (A^T B), contraction over the leading (row) index */
static void matmul_tn(const double *A, long lda, const double *B, long ldb, double *C, long ldc,
                      long m, long k, long n)
{
    for (long i = 0; i < m; ++i)
        for (long j = 0; j < n; ++j) C[i * ldc + j] = 0.0;
    for (long p = 0; p < k; ++p) {
        const double *a = A + p * lda;
        const double *b = B + p * ldb;
        for (long i = 0; i < m; ++i) {
            double av = a[i];
            double *c = C + i * ldc;
            for (long j = 0; j < n; ++j) c[j] += av * b[j];
        }
    }
}

/* C[m][n] = sum_k A[m][k] * B[n][k]  (A B^T) */
static void matmul_nt(const double *A, long lda, const double *B, long ldb, double *C, long ldc,
                      long m, long k, long n)
{
    for (long i = 0; i < m; ++i)
        for (long j = 0; j < n; ++j) {
            double acc = 0.0;
            for (long p = 0; p < k; ++p) acc += A[i * lda + p] * B[j * ldb + p];
            C[i * ldc + j] = acc;
        }
}

/* ------------------------------------------------------------------------------------------ */
/* One head.                                                                                  */
/* ------------------------------------------------------------------------------------------ */

/* apply (Eq. 4 with Eq. 12):  O = (SiLU(X W1) o (X W3)) W2.   linear mode: O = X W1. */
static void head_apply(const double *X, long ldx, long M, int hd, int H,
                       const double *W1, const double *W2, const double *W3,
                       int linear, double *O, long ldo)
{
    if (linear) {                       /* f_W(x) = x W1 with W1 [hd][H], H == hd */
        matmul_nn(X, ldx, W1, H, O, ldo, M, hd, H);
        return;
    }
    double *A = (double *)malloc(sizeof(double) * (size_t)M * H);
    double *B = (double *)malloc(sizeof(double) * (size_t)M * H);
    matmul_nn(X, ldx, W1, H, A, H, M, hd, H);            /* W1 x */
    matmul_nn(X, ldx, W3, H, B, H, M, hd, H);            /* W3 x */
    for (long i = 0; i < M * (long)H; ++i)               /* SiLU(W1 x) o (W3 x) */
        A[i] = A[i] * sigmoid(A[i]) * B[i];
    matmul_nn(A, H, W2, hd, O, ldo, M, H, hd);           /* W2 ( . ) */
    free(A);
    free(B);
}

/* gradient of  l(W) = sum_i eta_i * ( - f_W(k_i)^T v_i )   (the quantity Eq. 8 differentiates,
 * with Eq. 9 as L) at the CURRENT W, all M tokens of the chunk as one update unit.
 * Returns l(W).  G1,G3 [hd][H], G2 [H][hd]. */
static double head_grad(const double *K, const double *V, long ld, const double *eta, long M,
                        int hd, int H, const double *W1, const double *W2, const double *W3,
                        int linear, double *G1, double *G2, double *G3)
{
    size_t MH = (size_t)M * H;
    double *dY = (double *)malloc(sizeof(double) * (size_t)M * hd);
    /* dl/df_W(k_i) = -eta_i v_i   (dot-product loss: independent of f_W(k_i)) */
    for (long i = 0; i < M; ++i)
        for (int j = 0; j < hd; ++j) dY[i * hd + j] = -eta[i] * V[i * ld + j];

    double loss = 0.0;
    if (linear) {
        /* f_W(x) = x W1:  G1 = K^T dY ; loss = sum (K W1) o dY */
        double *F = (double *)malloc(sizeof(double) * (size_t)M * H);
        matmul_nn(K, ld, W1, H, F, H, M, hd, H);
        for (size_t i = 0; i < (size_t)M * H; ++i) loss += F[i] * dY[i];
        matmul_tn(K, ld, dY, hd, G1, H, hd, M, H);
        memset(G2, 0, sizeof(double) * (size_t)H * hd);
        memset(G3, 0, sizeof(double) * (size_t)hd * H);
        free(F);
        free(dY);
        return loss;
    }

    double *A = (double *)malloc(sizeof(double) * MH);
    double *B = (double *)malloc(sizeof(double) * MH);
    double *Hd = (double *)malloc(sizeof(double) * MH);
    double *dHd = (double *)malloc(sizeof(double) * MH);
    double *dA = (double *)malloc(sizeof(double) * MH);
    double *dB = (double *)malloc(sizeof(double) * MH);

    matmul_nn(K, ld, W1, H, A, H, M, hd, H);             /* A = K W1 */
    matmul_nn(K, ld, W3, H, B, H, M, hd, H);             /* B = K W3 */
    matmul_nt(dY, hd, W2, hd, dHd, H, M, hd, H);         /* dHd = dY W2^T */
    for (size_t i = 0; i < MH; ++i) {
        double a = A[i], b = B[i];
        double s = sigmoid(a);
        double S = a * s;                                /* SiLU(a) */
        Hd[i] = S * b;                                   /* hidden activation */
        dB[i] = dHd[i] * S;                              /* d/dB of S o B */
        dA[i] = dHd[i] * b * (s * (1.0 + a * (1.0 - s)));/* SiLU'(a) = s (1 + a (1 - s)) */
        loss += Hd[i] * dHd[i];                          /* = sum_i -eta_i f_W(k_i)^T v_i */
    }
    matmul_tn(K, ld, dA, H, G1, H, hd, M, H);            /* G1 = K^T dA  */
    matmul_tn(K, ld, dB, H, G3, H, hd, M, H);            /* G3 = K^T dB  */
    matmul_tn(Hd, H, dY, hd, G2, hd, H, M, hd);          /* G2 = Hd^T dY */

    free(A); free(B); free(Hd); free(dHd); free(dA); free(dB); free(dY);
    return loss;
}

/* Newton-Schulz orthonormalisation (reading R-NS; not in PAPER.md).
 * G [r][c] row-major, in place. If r > c the iteration runs on G^T (Gram matrix min x min) and the
 * result is transposed back. X0 = G/(||G||_F + 1e-7); n times: A = X X^T; B = b A + c A A;
 * X = a X + B X, (a,b,c) = (3.4445, -4.7750, 2.0315). */
static void newton_schulz(double *G, int r, int c, int iters)
{
    const double ca = 3.4445, cb = -4.7750, cc = 2.0315;
    int tr = r > c;
    int p = tr ? c : r;      /* small side */
    int q = tr ? r : c;      /* large side */
    double *X = (double *)malloc(sizeof(double) * (size_t)p * q);
    double *Xn = (double *)malloc(sizeof(double) * (size_t)p * q);
    double *A = (double *)malloc(sizeof(double) * (size_t)p * p);
    double *B = (double *)malloc(sizeof(double) * (size_t)p * p);
    double fro = 0.0;
    for (long i = 0; i < (long)r * c; ++i) fro += G[i] * G[i];
    fro = sqrt(fro) + 1e-7;
    for (int i = 0; i < r; ++i)
        for (int j = 0; j < c; ++j) {
            double x = G[(long)i * c + j] / fro;
            if (tr) X[(long)j * q + i] = x; else X[(long)i * q + j] = x;
        }
    for (int it = 0; it < iters; ++it) {
        matmul_nt(X, q, X, q, A, p, p, q, p);            /* A = X X^T      */
        matmul_nn(A, p, A, p, B, p, p, p, p);            /* A A            */
        for (long i = 0; i < (long)p * p; ++i) B[i] = cb * A[i] + cc * B[i];
        matmul_nn(B, p, X, q, Xn, q, p, p, q);           /* B X            */
        for (long i = 0; i < (long)p * q; ++i) X[i] = ca * X[i] + Xn[i];
    }
    for (int i = 0; i < r; ++i)
        for (int j = 0; j < c; ++j)
            G[(long)i * c + j] = tr ? X[(long)j * q + i] : X[(long)i * q + j];
    free(X); free(Xn); free(A); free(B);
}

/* column 2-norms of W [r][c] */
static void col_norms(const double *W, int r, int c, double *n)
{
    for (int j = 0; j < c; ++j) {
        double acc = 0.0;
        for (int i = 0; i < r; ++i) acc += W[(long)i * c + j] * W[(long)i * c + j];
        n[j] = sqrt(acc);
    }
}

/* re-normalisation (reading R-RENORM): W[:,j] *= n0[j] / (||W[:,j]|| + 1e-5) */
static void renorm_cols(double *W, int r, int c, const double *n0)
{
    for (int j = 0; j < c; ++j) {
        double acc = 0.0;
        for (int i = 0; i < r; ++i) acc += W[(long)i * c + j] * W[(long)i * c + j];
        double f = n0[j] / (sqrt(acc) + 1e-5);
        for (int i = 0; i < r; ++i) W[(long)i * c + j] *= f;
    }
}

/* ------------------------------------------------------------------------------------------ */
/* Exported entry points (all heads; OpenMP over heads).                                      */
/* ------------------------------------------------------------------------------------------ */

/* n0_1,n0_3 [nh][H], n0_2 [nh][hd] = column norms of the current weights (called at init) */
void ttt_oracle_col_norms(const double *W1, const double *W2, const double *W3, int nh, int hd,
                          int H, double *n0_1, double *n0_2, double *n0_3)
{
    for (int h = 0; h < nh; ++h) {
        col_norms(W1 + (size_t)h * hd * H, hd, H, n0_1 + (size_t)h * H);
        col_norms(W3 + (size_t)h * hd * H, hd, H, n0_3 + (size_t)h * H);
        col_norms(W2 + (size_t)h * H * hd, H, hd, n0_2 + (size_t)h * hd);
    }
}

/* gradients only (no state change): G1,G3 [nh][hd][H], G2 [nh][H][hd], loss [nh] */
void ttt_oracle_grad(const double *K, const double *V, const double *lr, long M, long ld,
                     int nh, int hd, int H, int linear,
                     const double *W1, const double *W2, const double *W3,
                     double *G1, double *G2, double *G3, double *loss)
{
#pragma omp parallel for schedule(dynamic, 1)
    for (int h = 0; h < nh; ++h) {
        size_t o13 = (size_t)h * hd * H, o2 = (size_t)h * H * hd;
        loss[h] = head_grad(K + (size_t)h * hd, V + (size_t)h * hd, ld, lr + (size_t)h * M, M,
                            hd, H, W1 + o13, W2 + o2, W3 + o13, linear,
                            G1 + o13, G2 + o2, G3 + o13);
    }
}

/* Newton-Schulz on a batch of n matrices [r][c], in place */
void ttt_oracle_newton_schulz(double *G, int n, int r, int c, int iters)
{
#pragma omp parallel for schedule(dynamic, 1)
    for (int i = 0; i < n; ++i) newton_schulz(G + (size_t)i * r * c, r, c, iters);
}

/* weight commit: W_j <- W_j - G_j (simultaneously), then optional re-normalisation */
void ttt_oracle_commit(double *W1, double *W2, double *W3,
                       const double *G1, const double *G2, const double *G3,
                       int nh, int hd, int H, int renorm,
                       const double *n0_1, const double *n0_2, const double *n0_3)
{
    size_t n = (size_t)nh * hd * H;
    for (size_t i = 0; i < n; ++i) W1[i] -= G1[i];
    for (size_t i = 0; i < n; ++i) W2[i] -= G2[i];
    for (size_t i = 0; i < n; ++i) W3[i] -= G3[i];
    if (renorm) {
        for (int h = 0; h < nh; ++h) {
            renorm_cols(W1 + (size_t)h * hd * H, hd, H, n0_1 + (size_t)h * H);
            renorm_cols(W3 + (size_t)h * hd * H, hd, H, n0_3 + (size_t)h * H);
            renorm_cols(W2 + (size_t)h * H * hd, H, hd, n0_2 + (size_t)h * hd);
        }
    }
}

/* update = Eq. 8: gradient at the pre-update W -> [NS] -> commit -> [renorm]; loss [nh] out */
void ttt_oracle_update(const double *K, const double *V, const double *lr, long M, long ld,
                       int nh, int hd, int H, int linear, int ns_iters, int renorm,
                       double *W1, double *W2, double *W3,
                       const double *n0_1, const double *n0_2, const double *n0_3, double *loss)
{
    size_t n = (size_t)nh * hd * H;
    double *G1 = (double *)malloc(sizeof(double) * n);
    double *G2 = (double *)malloc(sizeof(double) * n);
    double *G3 = (double *)malloc(sizeof(double) * n);
    ttt_oracle_grad(K, V, lr, M, ld, nh, hd, H, linear, W1, W2, W3, G1, G2, G3, loss);
    if (ns_iters > 0) {
        ttt_oracle_newton_schulz(G1, nh, hd, H, ns_iters);
        if (!linear) {
            ttt_oracle_newton_schulz(G2, nh, H, hd, ns_iters);
            ttt_oracle_newton_schulz(G3, nh, hd, H, ns_iters);
        }
    }
    ttt_oracle_commit(W1, W2, W3, G1, G2, G3, nh, hd, H, renorm, n0_1, n0_2, n0_3);
    free(G1); free(G2); free(G3);
}

/* apply = Eq. 4 with the current weights */
void ttt_oracle_apply(const double *Q, long M, long ld, int nh, int hd, int H, int linear,
                      const double *W1, const double *W2, const double *W3, double *O, long ldo)
{
#pragma omp parallel for schedule(dynamic, 1)
    for (int h = 0; h < nh; ++h) {
        size_t o13 = (size_t)h * hd * H, o2 = (size_t)h * H * hd;
        head_apply(Q + (size_t)h * hd, ld, M, hd, H, W1 + o13, W2 + o2, W3 + o13, linear,
                   O + (size_t)h * hd, ldo);
    }
}

/* chunk step = update ; apply */
void ttt_oracle_chunk_step(const double *Q, const double *K, const double *V, const double *lr,
                           long M, long ld, int nh, int hd, int H, int linear, int ns_iters,
                           int renorm, double *W1, double *W2, double *W3,
                           const double *n0_1, const double *n0_2, const double *n0_3,
                           double *O, long ldo, double *loss)
{
    ttt_oracle_update(K, V, lr, M, ld, nh, hd, H, linear, ns_iters, renorm, W1, W2, W3,
                      n0_1, n0_2, n0_3, loss);
    ttt_oracle_apply(Q, M, ld, nh, hd, H, linear, W1, W2, W3, O, ldo);
}

int ttt_oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/*
 * tnrd_oracle_bwd.c -- CPU ORACLE for the BACKWARD pass of a TNRD stage.  TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, double-precision transcription of the gradient formulas of the supplement of
 *   Chen, Yu, Pock, arXiv 1503.05768 ("Notes on diffusion networks", Sec. 2):
 *     dl/dlambda  Supp. Eq. 7      dl/dk_i   Supp. Eq. 10
 *     dl/dw_i     Supp. Eq. 19      du_{t+1}/du_t   PAPER.md:612-616 (used in Supp. Eq. 21)
 * for the stage  u_t = u - ( sum_i kbar_i * phi_i(k_i * u~) + lambda (u - f) )  exactly as the forward
 * oracle (tnrd_oracle.c, steps O1-O5, boundary reading A) computes it:  u~ = E u is the mirror extension
 * by 2r (O1), K_i the valid convolution (O2), Kbar_i the valid correlation (O4), so that
 *     u_t = u - sum_i Kbar_i phi_i(K_i E u) - lambda (u - f)          on H x W  (the crop is built in).
 * Every matrix-transpose of the paper (K^T, Kbar^T, P_T^T, U^T, V^T) is written here as the literal adjoint
 * loop of the corresponding forward loop of tnrd_oracle.c (same index expressions, "+=" on the other side),
 * so that it can be checked against that file by eye.  Every intermediate image is materialised.
 *
 * Same rules as tnrd_oracle.c: only tests/, __graft_entry__.smoke() and bench.py's cpu legs may use it; it
 * shares nothing with paper_1503_05768_b200/csrc.
 *
 * Readings:
 *   BR1  sign of dl/dlambda: Supp. Eq. 6 prints du_t/dlambda = (u - f)^T; from Supp. Eq. 4 it is -(u - f)^T
 *        (u_t = u - (... + lambda (u - f))).  The sign of Eq. 4 is taken: dl/dlambda = -<u - f, e>.
 *   BR2  phi': the printed formula is garbled (gamma used as a precision, wrong index); the
 *        derivative of phi_g as defined at PAPER.md:553 is used:
 *        phi'(z) = -sum_j w_j (z - mu_j) / gamma^2 * exp(-(z - mu_j)^2 / (2 gamma^2)).
 *   BR3  e = dl/du_t is an argument on H x W (the paper's e = T^T (T u_t - u_gt) lives on the padded image
 *        and is zero outside the crop; with the crop built into the stage it is u_t - u_gt on H x W).
 *   BR4  gradients of parameters are summed over the images of a batch (Supp. Eq. 3: the loss is a sum over
 *        samples); dl/du is per image.
 *
 * Pins (tests/test_oracle_bwd.py, "-m 'not gpu'"): BP1 adjoint identities of each transposed loop against the
 * pinned forward loops; BP2 closed form of phi' for one non-zero weight; BP3 central finite differences of
 * the PINNED forward oracle (loss 1/2 ||u_t - u_gt||^2) for every gradient; BP4 dense-matrix Jacobian on tiny
 * images; BP5 degenerate parameters; BP6 T-stage back-propagation against finite differences of oracle_diffuse.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>

#define ORACLE_OK 0
#define ORACLE_ERR_ARG (-1)
#define ORACLE_ERR_MEM (-2)

/* forward loops of tnrd_oracle.c (linked into the same shared object) */
int oracle_mirror(int q, int n);
void oracle_pad(const double *u, int H, int W, int p, int symmetric, double *up);
void oracle_conv_valid(const double *in, int Hin, int Win, const double *k, int K, double *out);
void oracle_corr_valid(const double *in, int Hin, int Win, const double *k, int K, double *out);
void oracle_phi(const double *z, size_t n, const double *w, const double *mu, int M, double gamma, double *v);
int oracle_stage(const double *f, const double *u_in, int B, int H, int W, int N_k, int K, const double *filters_t,
                 const double *rbf_w_t, const double *rbf_mu, int M, double gamma, double lambda_t, double *u_out,
                 int mode);

/* Adjoint of oracle_pad (symmetric): u[m(sy)][m(sx)] += up[y][x].  This is P^T. */
void oracle_pad_T(const double *up, int H, int W, int p, double *u)
{
    const int Hp = H + 2 * p, Wp = W + 2 * p;
    memset(u, 0, sizeof(double) * (size_t)H * W);
    for (int y = 0; y < Hp; ++y)
        for (int x = 0; x < Wp; ++x) {
            const int sy = y - p, sx = x - p;
            u[(size_t)oracle_mirror(sy, H) * W + oracle_mirror(sx, W)] += up[(size_t)y * Wp + x];
        }
}

/* Adjoint of oracle_conv_valid (K_i^T): in[y + (K-1) - a][x + (K-1) - b] += k[a][b] * out[y][x]. */
void oracle_conv_valid_T(const double *out, int Hin, int Win, const double *k, int K, double *in)
{
    const int Ho = Hin - K + 1, Wo = Win - K + 1;
    memset(in, 0, sizeof(double) * (size_t)Hin * Win);
    for (int y = 0; y < Ho; ++y)
        for (int x = 0; x < Wo; ++x)
            for (int a = 0; a < K; ++a)
                for (int b = 0; b < K; ++b)
                    in[(size_t)(y + (K - 1) - a) * Win + (x + (K - 1) - b)] += k[a * K + b] * out[(size_t)y * Wo + x];
}

/* Adjoint of oracle_corr_valid (Kbar_i^T, "careful boundary handling"):
 * in[y + a][x + b] += k[a][b] * out[y][x]. */
void oracle_corr_valid_T(const double *out, int Hin, int Win, const double *k, int K, double *in)
{
    const int Ho = Hin - K + 1, Wo = Win - K + 1;
    memset(in, 0, sizeof(double) * (size_t)Hin * Win);
    for (int y = 0; y < Ho; ++y)
        for (int x = 0; x < Wo; ++x)
            for (int a = 0; a < K; ++a)
                for (int b = 0; b < K; ++b)
                    in[(size_t)(y + a) * Win + (x + b)] += k[a * K + b] * out[(size_t)y * Wo + x];
}

/* phi'(z), reading BR2 (derivative of PAPER.md:553). */
double oracle_dphi1(double z, const double *w, const double *mu, int M, double gamma)
{
    double acc = 0.0;
    for (int j = 0; j < M; ++j) {
        const double d = z - mu[j];
        acc += -w[j] * d / (gamma * gamma) * exp(-(d * d) / (2.0 * gamma * gamma));
    }
    return acc;
}

void oracle_dphi(const double *z, size_t n, const double *w, const double *mu, int M, double gamma, double *dv)
{
#pragma omp parallel for schedule(static)
    for (long long p = 0; p < (long long)n; ++p) dv[p] = oracle_dphi1(z[p], w, mu, M, gamma);
}

/* Backward pass of one stage for ONE image.  Any of g_u, g_k, g_w, g_lambda may be NULL (skipped).
 * g_k [N_k][K][K], g_w [N_k][M] and g_lambda[1] are ACCUMULATED into (the caller zeroes them), g_u is written. */
static int stage_backward_one(const double *f, const double *u, const double *e, int H, int W, int N_k, int K,
                              const double *filters, const double *rbf_w, const double *rbf_mu, int M, double gamma,
                              double lambda, double *g_u, double *g_k, double *g_w, double *g_lambda)
{
    const int r = (K - 1) / 2;
    const int Hu = H + 4 * r, Wu = W + 4 * r, Hz = H + 2 * r, Wz = W + 2 * r;
    const size_t nu = (size_t)Hu * Wu, nz = (size_t)Hz * Wz, n = (size_t)H * W;
    double *ue = (double *)malloc(sizeof(double) * nu);  /* u~ = E u */
    double *z = (double *)malloc(sizeof(double) * nz);   /* K_i u~ */
    double *v = (double *)malloc(sizeof(double) * nz);   /* phi_i(z) */
    double *dv = (double *)malloc(sizeof(double) * nz);  /* Lambda_i = diag(phi_i'(z)) */
    double *q = (double *)malloc(sizeof(double) * nz);   /* Kbar_i^T e */
    double *pq = (double *)malloc(sizeof(double) * nz);  /* Lambda_i Kbar_i^T e */
    double *gi = (double *)malloc(sizeof(double) * nu);  /* K_i^T Lambda_i Kbar_i^T e */
    double *ge = (double *)calloc(nu, sizeof(double));   /* sum over i */
    double *gu = (double *)malloc(sizeof(double) * n);
    if (!ue || !z || !v || !dv || !q || !pq || !gi || !ge || !gu) {
        free(ue); free(z); free(v); free(dv); free(q); free(pq); free(gi); free(ge); free(gu);
        return ORACLE_ERR_MEM;
    }
    oracle_pad(u, H, W, 2 * r, 1, ue);                                                   /* O1 */
    for (int i = 0; i < N_k; ++i) {
        const double *k = filters + (size_t)i * K * K;
        const double *w = rbf_w + (size_t)i * M;
        oracle_conv_valid(ue, Hu, Wu, k, K, z);                                           /* O2: z = K_i u~ */
        oracle_corr_valid_T(e, Hz, Wz, k, K, q);                                          /* q = Kbar_i^T e */
        if (g_w) {
            /* Supp. Eq. 19: dl/dw_i = -G^T Kbar_i^T e,  G[p][j] = exp(-(z_p - mu_j)^2 / (2 gamma^2))  (Eq. 17) */
            for (int j = 0; j < M; ++j) {
                double acc = 0.0;
                for (size_t p = 0; p < nz; ++p) {
                    const double d = z[p] - rbf_mu[j];
                    acc += exp(-(d * d) / (2.0 * gamma * gamma)) * q[p];
                }
                g_w[(size_t)i * M + j] += -acc;
            }
        }
        oracle_dphi(z, nz, w, rbf_mu, M, gamma, dv);                                      /* Lambda_i */
        for (size_t p = 0; p < nz; ++p) pq[p] = dv[p] * q[p];
        if (g_k) {
            /* Supp. Eq. 10: dl/dk_i = -(P_inv^T V^T + U^T Lambda Kbar_i^T) e.
             * first term: s[y][x] = sum_{a,b} k[a][b] v[y + a][x + b]  (O4)  =>  d s[y][x] / d k[a][b] = v[y + a][x + b]
             * second term: z[Y][X] = sum_{a,b} k[a][b] u~[Y + K-1 - a][X + K-1 - b]  (O2)
             *              =>  d z[Y][X] / d k[a][b] = u~[Y + K-1 - a][X + K-1 - b]                                  */
            oracle_phi(z, nz, w, rbf_mu, M, gamma, v);                                    /* O3 */
            for (int a = 0; a < K; ++a)
                for (int b = 0; b < K; ++b) {
                    double t1 = 0.0, t2 = 0.0;
                    for (int y = 0; y < H; ++y)
                        for (int x = 0; x < W; ++x) t1 += e[(size_t)y * W + x] * v[(size_t)(y + a) * Wz + (x + b)];
                    for (int Y = 0; Y < Hz; ++Y)
                        for (int X = 0; X < Wz; ++X)
                            t2 += ue[(size_t)(Y + (K - 1) - a) * Wu + (X + (K - 1) - b)] * pq[(size_t)Y * Wz + X];
                    g_k[(size_t)i * K * K + a * K + b] += -(t1 + t2);
                }
        }
        if (g_u) {
            oracle_conv_valid_T(pq, Hu, Wu, k, K, gi);                                    /* K_i^T Lambda_i Kbar_i^T e */
            for (size_t p = 0; p < nu; ++p) ge[p] += gi[p];
        }
    }
    if (g_u) {
        /* PAPER.md:612-616:  (du_t/du_{t-1})^T e = P^T ( (1 - lambda) e~ - sum_i K_i^T Lambda_i Kbar_i^T e ),
         * where the identity term acts on the un-extended u: (1 - lambda) e on H x W. */
        oracle_pad_T(ge, H, W, 2 * r, gu);
        for (size_t p = 0; p < n; ++p) g_u[p] = (1.0 - lambda) * e[p] - gu[p];
    }
    if (g_lambda) {
        double acc = 0.0;                                                                 /* Supp. Eq. 7, reading BR1 */
        for (size_t p = 0; p < n; ++p) acc += (u[p] - f[p]) * e[p];
        g_lambda[0] += -acc;
    }
    free(ue); free(z); free(v); free(dv); free(q); free(pq); free(gi); free(ge); free(gu);
    return ORACLE_OK;
}

/* Backward pass of one stage on a batch.  g_u [B][H][W] written; g_k [N_k][K][K], g_w [N_k][M], g_lambda [1] are
 * zeroed here and summed over the batch (reading BR4).  Any of them may be NULL. */
int oracle_stage_backward(const double *f, const double *u_in, const double *e, int B, int H, int W, int N_k, int K,
                          const double *filters_t, const double *rbf_w_t, const double *rbf_mu, int M, double gamma,
                          double lambda_t, double *g_u, double *g_k, double *g_w, double *g_lambda)
{
    if (!f || !u_in || !e || !filters_t || !rbf_w_t || !rbf_mu) return ORACLE_ERR_ARG;
    if (B < 1 || H < K - 1 || W < K - 1 || N_k < 1 || M < 1 || K < 1 || !(K & 1) || !(gamma > 0.0)) return ORACLE_ERR_ARG;
    if (g_k) memset(g_k, 0, sizeof(double) * (size_t)N_k * K * K);
    if (g_w) memset(g_w, 0, sizeof(double) * (size_t)N_k * M);
    if (g_lambda) g_lambda[0] = 0.0;
    for (int b = 0; b < B; ++b) {
        const size_t off = (size_t)b * H * W;
        int rc = stage_backward_one(f + off, u_in + off, e + off, H, W, N_k, K, filters_t, rbf_w_t, rbf_mu, M, gamma,
                                    lambda_t, g_u ? g_u + off : NULL, g_k, g_w, g_lambda);
        if (rc != ORACLE_OK) return rc;
    }
    return ORACLE_OK;
}

/* Back-propagation through T stages (joint training, Supp. Eq. 20-21).
 * Runs the forward stages from u0 keeping every iterate, then the backward recurrence from e_T = dl/du_T:
 *     e_{t-1} = (du_t/du_{t-1})^T e_t,   dl/dTheta_t from (u_{t-1}, e_t)   (Supp. Eq. 5 with e = dl/du_t).
 * u_T [B][H][W] (may be NULL) receives the forward result; e_T is read AFTER the forward pass through the
 * callback-free convention: if u_gt != NULL then e_T = u_T - u_gt (loss 1/2 ||u_T - u_gt||^2, Supp. Eq. 3 / 20),
 * else e_T is taken from e_T_in.  g_k [T][N_k][K][K], g_w [T][N_k][M], g_lambda [T], g_u0 [B][H][W]. */
int oracle_diffuse_backward(const double *f, const double *u0, const double *u_gt, const double *e_T_in, int B, int H,
                            int W, int T, int N_k, int K, const double *filters, const double *rbf_w,
                            const double *rbf_mu, int M, double gamma, const double *lambda, double *u_T, double *g_u0,
                            double *g_k, double *g_w, double *g_lambda)
{
    if (!f || !u0 || T < 1 || (!u_gt && !e_T_in)) return ORACLE_ERR_ARG;
    const size_t n = (size_t)B * H * W;
    double *us = (double *)malloc(sizeof(double) * n * (size_t)(T + 1));
    double *e = (double *)malloc(sizeof(double) * n);
    double *e2 = (double *)malloc(sizeof(double) * n);
    if (!us || !e || !e2) { free(us); free(e); free(e2); return ORACLE_ERR_MEM; }
    memcpy(us, u0, sizeof(double) * n);
    int rc = ORACLE_OK;
    for (int t = 0; t < T && rc == ORACLE_OK; ++t)
        rc = oracle_stage(f, us + (size_t)t * n, B, H, W, N_k, K, filters + (size_t)t * N_k * K * K,
                          rbf_w + (size_t)t * N_k * M, rbf_mu, M, gamma, lambda[t], us + (size_t)(t + 1) * n, 0);
    if (rc == ORACLE_OK) {
        const double *uT = us + (size_t)T * n;
        if (u_T) memcpy(u_T, uT, sizeof(double) * n);
        for (size_t p = 0; p < n; ++p) e[p] = u_gt ? uT[p] - u_gt[p] : e_T_in[p];
        for (int t = T - 1; t >= 0 && rc == ORACLE_OK; --t) {
            rc = oracle_stage_backward(f, us + (size_t)t * n, e, B, H, W, N_k, K, filters + (size_t)t * N_k * K * K,
                                       rbf_w + (size_t)t * N_k * M, rbf_mu, M, gamma, lambda[t], e2,
                                       g_k ? g_k + (size_t)t * N_k * K * K : NULL,
                                       g_w ? g_w + (size_t)t * N_k * M : NULL, g_lambda ? g_lambda + t : NULL);
            double *tmp = e; e = e2; e2 = tmp;
        }
        if (rc == ORACLE_OK && g_u0) memcpy(g_u0, e, sizeof(double) * n);
    }
    free(us); free(e); free(e2);
    return rc;
}

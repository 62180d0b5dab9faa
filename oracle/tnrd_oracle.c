/*
 * tnrd_oracle.c -- CPU ORACLE for the TNRD inference hot path.  TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, double-precision transcription of the stage update of
 *   Chen, Yu, Pock, "On learning optimized reaction diffusion processes for effective
 *   image restoration" (arXiv 1503.05768), Main Eq. 7 with the boundary
 *   handling of Supp. Sec. 1:
 *
 *     u_t = u_{t-1} - ( sum_i  kbar_i^t * phi_i^t( k_i^t * u_{t-1} )  +  lambda^t (u_{t-1} - f) )
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may build, link or call this file.  It shares no code, header, table or helper with the
 * CUDA library (paper_1503_05768_b200/csrc) and neither includes the other.
 *
 * The method is its own definition, so the oracle follows it step by step (O1..O6 below,
 * DESIGN.md "Readings"), every intermediate image materialised, no tiling, no fusion, no
 * lookup table, no truncation of the 63-term sum, libm exp(), IEEE double, no -ffast-math.
 * The only concession to run time is an OpenMP "parallel for" over rows of an image; it
 * does not change the order of any floating-point sum.
 *
 * Pins (tests/test_oracle_pins.py, all "-m 'not gpu'"): P1 delta response, P2 constant
 * image invariant, P3 closed form of phi for one non-zero weight, P4 adjoint identity under
 * zero padding, P5 finite-difference of the FoE energy (erf closed form), P6 linear-phi
 * special case against scipy.signal, P7 dense-matrix brute force on 8x8, P8 literal
 * pad-omega/crop procedure for several omega, P9 flip/transpose equivariance, P12 degenerate
 * parameters, P13 interior shift-equivariance; PT1-PT3 (tests/test_oracle_triangle.py) the triangular basis against
 * numpy.interp, its partition of unity and closed forms.  Absolute end-to-end values for the
 * BASELINE.json configs are "parity unpinned by the paper" (no printed example, no weights).
 *
 * Layouts: images row-major [B][H][W] (x fastest); filters [N_k][K][K] with k[a][b],
 * a = row, b = column; rbf_w [N_k][M]; rbf_mu [M].
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_OK 0
#define ORACLE_ERR_ARG (-1)
#define ORACLE_ERR_MEM (-2)

/* mode of boundary handling */
#define ORACLE_SYMMETRIC_2R 0 /* reading A (default): mirror-extend u by 2r, two valid convolutions, crop */
#define ORACLE_ZERO_SAME 1    /* Main Eq. 2 with K^T under zero padding; used by pins P1, P4, P5 only */

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_set_num_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* O1 mirror map (PAPER.md:383 "pad ... with mirror reflections of itself"; :387 "symmetric
 * boundary condition").  Half-sample symmetric, edge pixel repeated:  ... b a | a b ...
 * valid for -n <= q < 2n. */
int oracle_mirror(int q, int n)
{
    if (q < 0) return -1 - q;
    if (q >= n) return 2 * n - 1 - q;
    return q;
}

/* Extend an H x W image by p pixels on every side.  symmetric != 0: mirror map; else zeros.
 * up has (H+2p) x (W+2p) elements. */
void oracle_pad(const double *u, int H, int W, int p, int symmetric, double *up)
{
    const int Hp = H + 2 * p, Wp = W + 2 * p;
    for (int y = 0; y < Hp; ++y) {
        for (int x = 0; x < Wp; ++x) {
            const int sy = y - p, sx = x - p;
            double val;
            if (symmetric) {
                val = u[(size_t)oracle_mirror(sy, H) * W + oracle_mirror(sx, W)];
            } else {
                val = (sy >= 0 && sy < H && sx >= 0 && sx < W) ? u[(size_t)sy * W + sx] : 0.0;
            }
            up[(size_t)y * Wp + x] = val;
        }
    }
}

/* O2 forward filter: TRUE 2-D convolution (kernel flipped), "valid" extent (PAPER.md:70,
 * "K_i u <=> k_i * u").  in is Hin x Win, out is (Hin-K+1) x (Win-K+1):
 *   out[y][x] = sum_{a,b} k[a][b] * in[y + (K-1) - a][x + (K-1) - b]                    */
void oracle_conv_valid(const double *in, int Hin, int Win, const double *k, int K, double *out)
{
    const int Ho = Hin - K + 1, Wo = Win - K + 1;
#pragma omp parallel for schedule(static)
    for (int y = 0; y < Ho; ++y) {
        for (int x = 0; x < Wo; ++x) {
            double acc = 0.0;
            for (int a = 0; a < K; ++a)
                for (int b = 0; b < K; ++b)
                    acc += k[a * K + b] * in[(size_t)(y + (K - 1) - a) * Win + (x + (K - 1) - b)];
            out[(size_t)y * Wo + x] = acc;
        }
    }
}

/* O4 transposed filter: convolution with kbar = rot180(k), i.e. correlation
 * with k, "valid" extent:
 *   out[y][x] = sum_{a,b} k[a][b] * in[y + a][x + b]                                    */
void oracle_corr_valid(const double *in, int Hin, int Win, const double *k, int K, double *out)
{
    const int Ho = Hin - K + 1, Wo = Win - K + 1;
#pragma omp parallel for schedule(static)
    for (int y = 0; y < Ho; ++y) {
        for (int x = 0; x < Wo; ++x) {
            double acc = 0.0;
            for (int a = 0; a < K; ++a)
                for (int b = 0; b < K; ++b)
                    acc += k[a * K + b] * in[(size_t)(y + a) * Win + (x + b)];
            out[(size_t)y * Wo + x] = acc;
        }
    }
}

/* Radial basis of the influence functions: 0 = Gaussian phi_g (the paper's results, default),
 * 1 = triangular-shaped phi_t.  A process-wide switch of the ORACLE (tests set it around a call and restore it); it
 * selects which of the two printed formulas oracle_phi1 evaluates, nothing else. */
static int g_basis = 0;
void oracle_set_basis(int basis) { g_basis = basis ? 1 : 0; }
int oracle_get_basis(void) { return g_basis; }

/* O3 influence function, RBF mixture (Eq. 6):  phi(z) = sum_{j=1..M} w_j varphi(|z - mu_j| / gamma)
 *   Gaussian   (:553)  varphi_g = exp( -(z - mu_j)^2 / (2 gamma^2) )
 *   triangular (:557)  varphi_t = 1 - |z - mu_j| / gamma  if |z - mu_j| <= gamma,  0 otherwise                        */
double oracle_phi1(double z, const double *w, const double *mu, int M, double gamma)
{
    double acc = 0.0;
    for (int j = 0; j < M; ++j) {
        const double d = z - mu[j];
        if (g_basis == 0) {
            acc += w[j] * exp(-(d * d) / (2.0 * gamma * gamma));
        } else {
            const double ad = fabs(d);
            if (ad <= gamma) acc += w[j] * (1.0 - ad / gamma);
        }
    }
    return acc;
}

void oracle_phi(const double *z, size_t n, const double *w, const double *mu, int M, double gamma,
                double *v)
{
#pragma omp parallel for schedule(static)
    for (long long p = 0; p < (long long)n; ++p) v[p] = oracle_phi1(z[p], w, mu, M, gamma);
}

/* One stage for one image (O1..O5). */
static int stage_one(const double *f, const double *u, int H, int W, int N_k, int K,
                     const double *filters, const double *rbf_w, const double *rbf_mu, int M,
                     double gamma, double lambda, double *u_out, int mode)
{
    const int r = (K - 1) / 2;
    int Hu, Wu, Hz, Wz; /* extended u; z and v maps */
    if (mode == ORACLE_SYMMETRIC_2R) {
        Hu = H + 4 * r; Wu = W + 4 * r; Hz = H + 2 * r; Wz = W + 2 * r;
    } else {
        Hu = H + 2 * r; Wu = W + 2 * r; Hz = H; Wz = W;
    }
    const int Hv = H + 2 * r, Wv = W + 2 * r; /* v as seen by the transposed filter */
    double *ue = (double *)malloc(sizeof(double) * (size_t)Hu * Wu);
    double *z = (double *)malloc(sizeof(double) * (size_t)Hz * Wz);
    double *v = (double *)malloc(sizeof(double) * (size_t)Hz * Wz);
    double *ve = (double *)malloc(sizeof(double) * (size_t)Hv * Wv);
    double *si = (double *)malloc(sizeof(double) * (size_t)H * W);
    double *s = (double *)calloc((size_t)H * W, sizeof(double));
    if (!ue || !z || !v || !ve || !si || !s) {
        free(ue); free(z); free(v); free(ve); free(si); free(s);
        return ORACLE_ERR_MEM;
    }
    /* O1 */
    if (mode == ORACLE_SYMMETRIC_2R) oracle_pad(u, H, W, 2 * r, 1, ue);
    else oracle_pad(u, H, W, r, 0, ue);

    for (int i = 0; i < N_k; ++i) {
        const double *k = filters + (size_t)i * K * K;
        oracle_conv_valid(ue, Hu, Wu, k, K, z);                              /* O2 */
        oracle_phi(z, (size_t)Hz * Wz, rbf_w + (size_t)i * M, rbf_mu, M, gamma, v); /* O3 */
        const double *vin = v;
        if (mode == ORACLE_ZERO_SAME) { /* v = 0 outside the image: this is K_i^T v */
            oracle_pad(v, H, W, r, 0, ve);
            vin = ve;
        }
        oracle_corr_valid(vin, Hv, Wv, k, K, si);                            /* O4 */
        for (size_t p = 0; p < (size_t)H * W; ++p) s[p] += si[p];            /* sum over i */
    }
    /* O5 */
    for (size_t p = 0; p < (size_t)H * W; ++p) u_out[p] = u[p] - (s[p] + lambda * (u[p] - f[p]));

    free(ue); free(z); free(v); free(ve); free(si); free(s);
    return ORACLE_OK;
}

static int check_shape(int B, int H, int W, int N_k, int K, int M)
{
    if (B < 1 || H < 1 || W < 1 || N_k < 1 || M < 1) return ORACLE_ERR_ARG;
    if (K < 1 || (K % 2) == 0) return ORACLE_ERR_ARG;
    if (H < K - 1 || W < K - 1) return ORACLE_ERR_ARG; /* mirror source must exist: min(H,W) >= 2r */
    return ORACLE_OK;
}

/* One stage on a batch.  u_out must not alias u_in or f. */
int oracle_stage(const double *f, const double *u_in, int B, int H, int W, int N_k, int K,
                 const double *filters_t, const double *rbf_w_t, const double *rbf_mu, int M,
                 double gamma, double lambda_t, double *u_out, int mode)
{
    if (!f || !u_in || !filters_t || !rbf_w_t || !rbf_mu || !u_out) return ORACLE_ERR_ARG;
    if (check_shape(B, H, W, N_k, K, M) != ORACLE_OK || !(gamma > 0.0)) return ORACLE_ERR_ARG;
    for (int b = 0; b < B; ++b) {
        const size_t off = (size_t)b * H * W;
        int rc = stage_one(f + off, u_in + off, H, W, N_k, K, filters_t, rbf_w_t, rbf_mu, M, gamma,
                           lambda_t, u_out + off, mode);
        if (rc != ORACLE_OK) return rc;
    }
    return ORACLE_OK;
}

/* O6: T stages with per-stage parameters Theta_t.  T = 0 copies u0. */
int oracle_diffuse(const double *f, const double *u0, int B, int H, int W, int T, int N_k, int K,
                   const double *filters, const double *rbf_w, const double *rbf_mu, int M,
                   double gamma, const double *lambda, double *out, int mode)
{
    if (!f || !u0 || !out || T < 0) return ORACLE_ERR_ARG;
    if (T > 0 && (!filters || !rbf_w || !rbf_mu || !lambda)) return ORACLE_ERR_ARG;
    if (check_shape(B, H, W, N_k, K, M) != ORACLE_OK || !(gamma > 0.0)) return ORACLE_ERR_ARG;
    const size_t n = (size_t)B * H * W;
    double *cur = (double *)malloc(sizeof(double) * n);
    double *nxt = (double *)malloc(sizeof(double) * n);
    if (!cur || !nxt) { free(cur); free(nxt); return ORACLE_ERR_MEM; }
    memcpy(cur, u0, sizeof(double) * n);
    for (int t = 0; t < T; ++t) {
        int rc = oracle_stage(f, cur, B, H, W, N_k, K, filters + (size_t)t * N_k * K * K,
                              rbf_w + (size_t)t * N_k * M, rbf_mu, M, gamma, lambda[t], nxt, mode);
        if (rc != ORACLE_OK) { free(cur); free(nxt); return rc; }
        double *tmp = cur; cur = nxt; nxt = tmp;
    }
    memcpy(out, cur, sizeof(double) * n);
    free(cur); free(nxt);
    return ORACLE_OK;
}

/* =====================================================================================================
 * JPEG-deblocking stage (Main Eq. 9; Supp. Eq. 26-29):
 *     y = u_{t-1} - sum_i kbar_i * phi_i(k_i * u_{t-1})      (diffusion term only, no reaction term)
 *     z = D y            D = orthonormal 2-D DCT-II of every 8x8 block ("D^T D = D D^T = I")
 *     v = eta(z)         point-wise projection onto the box [a_p, b_p] (QCS, Supp. Eq. 26)
 *     u_t = D^T v
 * Coefficient (p, q) of block (by, bx) is stored at pixel position (8 by + p, 8 bx + q); a, b use the same
 * layout.  H and W must be multiples of 8.  The paper pads by omega = 8: a whole block, so the
 * block grid of the padded image coincides with the image's own and, with re-padding every stage
 * (u_tp = P_T u_t), the centre H x W result is exactly the above with the diffusion term of O1-O4
 * (reading D1).
 * Pins (tests/test_oracle_deblock.py): D against scipy.fft.dctn(norm="ortho"), orthogonality / Parseval,
 * closed forms (constant block, single cosine), projection properties, reduction to the pinned denoising
 * stage when the box is infinite.
 * ===================================================================================================== */

/* 2-D DCT-II (inverse != 0: DCT-III, its transpose) of every 8x8 block, by the definition:
 *   c[p][q] = alpha_p alpha_q sum_{y,x} in[y][x] cos(pi (2y+1) p / 16) cos(pi (2x+1) q / 16),
 *   alpha_0 = sqrt(1/8), alpha_p = sqrt(2/8).                                                          */
int oracle_block_dct8(const double *in, int H, int W, int inverse, double *out)
{
    if (!in || !out || H < 8 || W < 8 || (H % 8) || (W % 8)) return ORACLE_ERR_ARG;
    const double pi = 3.14159265358979323846;
    double cs[8][8]; /* cs[p][y] = alpha_p cos(pi (2y+1) p / 16) */
    for (int p = 0; p < 8; ++p)
        for (int y = 0; y < 8; ++y)
            cs[p][y] = (p == 0 ? sqrt(1.0 / 8.0) : sqrt(2.0 / 8.0)) * cos(pi * (2.0 * y + 1.0) * p / 16.0);
#pragma omp parallel for schedule(static)
    for (int by = 0; by < H / 8; ++by) {
        for (int bx = 0; bx < W / 8; ++bx) {
            const double *src = in + (size_t)(8 * by) * W + 8 * bx;
            double *dst = out + (size_t)(8 * by) * W + 8 * bx;
            double tmp[8][8];
            for (int p = 0; p < 8; ++p)
                for (int q = 0; q < 8; ++q) {
                    double acc = 0.0;
                    for (int y = 0; y < 8; ++y)
                        for (int x = 0; x < 8; ++x) {
                            const double basis = inverse ? cs[y][p] * cs[x][q] : cs[p][y] * cs[q][x];
                            acc += src[(size_t)y * W + x] * basis;
                        }
                    tmp[p][q] = acc;
                }
            for (int p = 0; p < 8; ++p)
                for (int q = 0; q < 8; ++q) dst[(size_t)p * W + q] = tmp[p][q];
        }
    }
    return ORACLE_OK;
}

/* u = D^T eta(D y): projection of one image onto the QCS in the DCT domain (Supp. Eq. 26-27). */
int oracle_qcs_project(const double *y, int H, int W, const double *lo, const double *hi, double *u)
{
    if (!y || !lo || !hi || !u) return ORACLE_ERR_ARG;
    const size_t n = (size_t)H * W;
    double *z = (double *)malloc(sizeof(double) * n);
    if (!z) return ORACLE_ERR_MEM;
    int rc = oracle_block_dct8(y, H, W, 0, z);
    if (rc == ORACLE_OK) {
        for (size_t p = 0; p < n; ++p) { /* eta, Supp. Eq. 26 */
            if (z[p] > hi[p]) z[p] = hi[p];
            else if (z[p] < lo[p]) z[p] = lo[p];
        }
        rc = oracle_block_dct8(z, H, W, 1, u);
    }
    free(z);
    return rc;
}

/* One deblocking stage on a batch (Supp. Eq. 29).  lo / hi are [B][H][W]. */
int oracle_deblock_stage(const double *u_in, int B, int H, int W, int N_k, int K, const double *filters_t,
                         const double *rbf_w_t, const double *rbf_mu, int M, double gamma, const double *lo,
                         const double *hi, double *u_out)
{
    if (!u_in || !lo || !hi || !u_out) return ORACLE_ERR_ARG;
    if ((H % 8) || (W % 8)) return ORACLE_ERR_ARG;
    const size_t n = (size_t)H * W;
    double *y = (double *)malloc(sizeof(double) * n);
    if (!y) return ORACLE_ERR_MEM;
    int rc = ORACLE_OK;
    for (int b = 0; b < B && rc == ORACLE_OK; ++b) {
        /* y = u - sum_i kbar_i * phi_i(k_i * u): the denoising stage with lambda = 0 (f is then irrelevant) */
        rc = oracle_stage(u_in + b * n, u_in + b * n, 1, H, W, N_k, K, filters_t, rbf_w_t, rbf_mu, M, gamma, 0.0, y,
                          ORACLE_SYMMETRIC_2R);
        if (rc == ORACLE_OK) rc = oracle_qcs_project(y, H, W, lo + b * n, hi + b * n, u_out + b * n);
    }
    free(y);
    return rc;
}

/* T deblocking stages with per-stage parameters Theta_t = {phi_i^t, k_i^t}. */
int oracle_deblock_diffuse(const double *u0, int B, int H, int W, int T, int N_k, int K, const double *filters,
                           const double *rbf_w, const double *rbf_mu, int M, double gamma, const double *lo,
                           const double *hi, double *out)
{
    if (!u0 || !out || T < 0) return ORACLE_ERR_ARG;
    const size_t n = (size_t)B * H * W;
    double *cur = (double *)malloc(sizeof(double) * n);
    double *nxt = (double *)malloc(sizeof(double) * n);
    if (!cur || !nxt) { free(cur); free(nxt); return ORACLE_ERR_MEM; }
    memcpy(cur, u0, sizeof(double) * n);
    int rc = ORACLE_OK;
    for (int t = 0; t < T && rc == ORACLE_OK; ++t) {
        rc = oracle_deblock_stage(cur, B, H, W, N_k, K, filters + (size_t)t * N_k * K * K,
                                  rbf_w + (size_t)t * N_k * M, rbf_mu, M, gamma, lo, hi, nxt);
        double *tmp = cur; cur = nxt; nxt = tmp;
    }
    if (rc == ORACLE_OK) memcpy(out, cur, sizeof(double) * n);
    free(cur); free(nxt);
    return rc;
}

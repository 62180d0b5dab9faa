// tnrd_bwd.cu -- backward pass of one TNRD stage (Supp. Sec. 2).
//
// For the stage  u_t = u - sum_i Kbar_i phi_i(K_i E u) - lambda (u - f)  (E = mirror extension by 2r, K_i valid
// convolution, Kbar_i valid correlation; the forward kernel of tnrd_fused.cu) and e = dl/du_t on H x W:
//   g_u      = (1 - lambda) e - E^T sum_i K_i^T Lambda_i Kbar_i^T e        PAPER.md:612-616 (Supp. Eq. 21)
//   g_w[i,j] = - sum_p exp(-(z_ip - mu_j)^2 / 2 gamma^2) (Kbar_i^T e)_p      Supp. Eq. 19
//   g_k[i]   = -(P_inv^T V^T + U^T Lambda_i Kbar_i^T) e                      Supp. Eq. 10
//   g_lambda = -<u - f, e>                                                    Supp. Eq. 7 with the sign of Eq. 4
// with z_i = K_i E u, Lambda_i = diag(phi_i'(z_i)), V = phi_i(z_i).
//
// Kernel 1, stage_bwd_kernel: the same fused tile structure as the forward kernel.  One CTA owns a tile of the
// EXTENDED output domain [-2r, H+2r) x [-2r, W+2r) (K_i^T reaches 2r beyond the image; E^T folds that rim back).
// Per filter i (streamed): z' = k'_i * u~ and q' = k'_i * e0 (e0 = e, zero outside the image: Kbar_i^T e is a true
// convolution of the zero-extended e) in registers on the tile + r ring; the 63 exponentials E_j are evaluated ONCE
// and feed  V = sum_j w'_j E_j  (phi, for g_k),  U = sum_j w'_j mu'_j E_j  (A = z' V - U = sum_j w'_j d'_j E_j is phi')
// and the g_w sums  sum_p E_j q'_p
// (reduced over the warp with a halving butterfly, then one shared-memory reduction per centre);
// P = -2 ln2 A q' (= Lambda_i Kbar_i^T e / s) goes to a double-buffered shared map, the k'_i taps are applied to the
// map of filter i-1 (K_i^T is a correlation with k_i) into per-thread accumulators.  Epilogue: the accumulators go to
// shared memory, every image pixel of the tile adds up its mirror pre-images (E^T) and g_u is written.
// When g_k is wanted, P and V of the owned pixels are also written to HBM maps [B][N_k][H+2r][W+2r] for kernel 2.
// Partial sums of g_w / g_lambda go to per-CTA slots and are added in fixed order by reduce_partials_kernel
// (deterministic, no float atomics in global memory).
//
// Kernel 2, wgrad_kernel: g_k from the maps -- per (tile, filter) 2 x ks^2 lag products
//   t1[a][b] = sum_{y,x} e[y][x] V[y+a][x+b],   t2[a][b] = sum_{Y,X} u~[Y+K-1-a][X+K-1-b] P[Y][X]
// accumulated in registers (ks^2 accumulators per thread), reduced per CTA, summed by reduce_partials_kernel.
#include <cstdio>
#include <cstdlib>

#include "tnrd_device.cuh"
#include "tnrd_internal.h"

namespace tnrd {

namespace {

template <int KS>
struct BCfg {
    static constexpr int R = (KS - 1) / 2;
    static constexpr int RW = 64, RH = 64, NT = 256;    // phi area (tile + r ring) <= 64 x 64, 256 threads
    static constexpr int TMAX = RW - 2 * R;             // largest output tile
    static constexpr int US = RW + 8;                   // u / e tile row stride
    static constexpr int UH = RH + 2 * R;               // u / e tile rows
    static constexpr int VS = RW;
    static constexpr int VPLANE = RH * RW + 16;
    static constexpr int TS = prm_ts(KS);
    static constexpr int PRM = prm_stride(KS);
    static constexpr int NB = (RW / 4) * (RH / 2) / NT; // 2 blocks of 4x2 pixels per thread
    static constexpr int NG = TNRD_MP / 8;
    // dynamic shared memory: u tile, e tile, two P maps, four staged records
    static constexpr size_t SMEM = sizeof(float) * (2 * (size_t)UH * US + 2 * (size_t)VPLANE + 4 * (size_t)PRM);
};

// 8 RBF terms (7 in the last step) for the 8 responses of a block.  z = z' (scaled responses), qm = q' of the pixels
// this tile owns (0 elsewhere).  Accumulates V = sum_j w'_j E_j (phi) and U = sum_j w'_j mu'_j E_j -- the caller forms
// sum_j w'_j (z' - mu'_j) E_j (phi') as z' V - U, one packed instruction per term less than accumulating it directly; the
// cancellation costs log2(|z'| / |z' - mu'_j|) < 5 bits where a term is not negligible -- and, per term, S[m] = sum over
// the 8 pixels of E q'.
template <int NTERM, bool WANT_W>
__device__ __forceinline__ void phi_bwd_step(const float* __restrict__ mw, const float2 (&z)[4], const float2 (&qm)[4],
                                             float2 (&U)[4], float2 (&V)[4], float (&S)[8])
{
    float c[16];
    lds_vec(mw, c);
#pragma unroll
    for (int m = 0; m < 8; ++m) {
        if (m >= NTERM) { S[m] = 0.f; continue; }
        float2 s2 = make_float2(0.f, 0.f);
        const float wmu = -c[2 * m] * c[2 * m + 1];           // c = (-mu', w')
#pragma unroll
        for (int p = 0; p < 4; ++p) {
            const float2 d = __fadd2_rn(z[p], make_float2(c[2 * m], c[2 * m]));
            const float2 t = __fmul2_rn(d, d);
            const float2 e = make_float2(ex2_neg(t.x), ex2_neg(t.y));
            V[p] = __ffma2_rn(e, make_float2(c[2 * m + 1], c[2 * m + 1]), V[p]);
            U[p] = __ffma2_rn(e, make_float2(wmu, wmu), U[p]);
            if (WANT_W) s2 = __ffma2_rn(e, qm[p], s2);
        }
        S[m] = s2.x + s2.y;
    }
}

// Sum S[0..7] over the 32 lanes of the warp with a halving butterfly (4 + 2 + 1 + 1 + 1 shuffles instead of 40):
// afterwards lane l holds the warp total of term (l >> 2) & 7 ... returned value; lanes with (l & 3) == 0 publish it.
__device__ __forceinline__ float warp_reduce8(const float (&S)[8], int lane)
{
    float a[4], b[2], c;
    const bool h4 = lane & 16, h3 = lane & 8, h2 = lane & 4;
#pragma unroll
    for (int m = 0; m < 4; ++m) {     // keep terms 0..3 (lanes < 16) or 4..7, hand the other half over
        const float keep = h4 ? S[m + 4] : S[m], give = h4 ? S[m] : S[m + 4];
        a[m] = keep + __shfl_xor_sync(0xffffffffu, give, 16);
    }
#pragma unroll
    for (int m = 0; m < 2; ++m) {
        const float keep = h3 ? a[m + 2] : a[m], give = h3 ? a[m] : a[m + 2];
        b[m] = keep + __shfl_xor_sync(0xffffffffu, give, 8);
    }
    {
        const float keep = h2 ? b[1] : b[0], give = h2 ? b[0] : b[1];
        c = keep + __shfl_xor_sync(0xffffffffu, give, 4);
    }
    c += __shfl_xor_sync(0xffffffffu, c, 2);
    c += __shfl_xor_sync(0xffffffffu, c, 1);
    return c;     // term index of this lane: 4 * bit4 + 2 * bit3 + bit2
}

// order-preserving map float <-> uint32 (warp-wide min / max by redux.sync)
__device__ __forceinline__ unsigned f2ord(float x)
{
    const unsigned b = __float_as_uint(x);
    return b ^ ((unsigned)((int)b >> 31) | 0x80000000u);
}
__device__ __forceinline__ float ord2f(unsigned o) { return __uint_as_float(o ^ (((o >> 31) - 1u) | 0x80000000u)); }

// origin (extended coordinate, >= -2r) of tile t of n over an axis of `len` image pixels
__device__ __forceinline__ int tile_origin(int t, int n, int len, int R) { return (int)((long long)t * (len + 4 * R) / n) - 2 * R; }

template <int KS, bool WANT_W, bool WANT_K>
__global__ void __launch_bounds__(BCfg<KS>::NT, 2)
stage_bwd_kernel(BwdArgs a, int ntx, int nty)
{
    using C = BCfg<KS>;
    constexpr int R = C::R, TS = C::TS, KKP = prm_kkp(KS), NT = C::NT;
    extern __shared__ __align__(16) float smem[];
    float* us = smem;                              // [UH][US]  u~ on the tile + 2r
    float* es = us + C::UH * C::US;                // [UH][US]  e0 (zero outside the image) on the tile + 2r
    float* vs = es + C::UH * C::US;                // [2][VPLANE]  P maps of filters i and i-1
    float* ps = vs + 2 * C::VPLANE;                // [4][PRM]  staged records
    __shared__ float gws[2][NT / 32][64];          // per-warp g_w sums of filters i and i-1
    __shared__ float red[NT / 32];
    __shared__ float crange[2 * BCfg<KS>::NG];     // smallest / largest scaled centre of every step of 8 terms

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    int t = blockIdx.x;
    const int tx = t % ntx; t /= ntx;
    const int ty = t % nty; t /= nty;
    const int img = t;
    const int OX0 = tile_origin(tx, ntx, a.W, R), OY0 = tile_origin(ty, nty, a.H, R);    // extended coordinates
    const int tw = tile_origin(tx + 1, ntx, a.W, R) - OX0, th = tile_origin(ty + 1, nty, a.H, R) - OY0;
    const size_t plane = (size_t)a.H * a.W;
    const float* __restrict__ u_img = a.u + img * plane;
    const float* __restrict__ e_img = a.e + img * plane;
    const int N_k = a.N_k;

    const int nbx = (tw + 2 * R + 3) >> 2, nby = (th + 2 * R + 1) >> 1;   // phi area = tile + r ring
    const int nbxo = (tw + 3) >> 2, nbyo = (th + 1) >> 1;                  // output tile
    const int nrounds = (nbx * nby + NT - 1) / NT;

    // ---- u~ (mirror map) and e0 (zero extension) on the tile + 2r --------------------------------------------------
    {
        const int nr = min(C::UH, 2 * nby + 2 * R), nc = min(C::US, 4 * nbx + 2 * R + 4);
        for (int uy = warp; uy < nr; uy += NT / 32) {
            const int Y = OY0 - 2 * R + uy;
            const bool yin = Y >= 0 && Y < a.H;
            const size_t ro = (size_t)mirror_clamp(Y, a.H) * a.W;
#pragma unroll
            for (int q = 0; q < (C::US + 31) / 32; ++q) {
                const int ux = lane + 32 * q;
                if (ux < nc) {
                    const int X = OX0 - 2 * R + ux;
                    cp_async4(us + uy * C::US + ux, u_img + ro + mirror_clamp(X, a.W));     // asynchronous copies
                    if (yin && X >= 0 && X < a.W) cp_async4(es + uy * C::US + ux, e_img + ro + X);
                    else es[uy * C::US + ux] = 0.0f;
                }
            }
        }
    }
    for (int idx = tid; idx < 2 * C::PRM; idx += NT)
        if (idx < N_k * C::PRM) ps[idx] = __ldg(a.prm + idx);
    for (int idx = tid; idx < 2 * (NT / 32) * 64; idx += NT) (&gws[0][0][0])[idx] = 0.0f;
    if (tid < C::NG) {      // the centres are the same for every filter: record 0 holds (-mu'_j, w'_j) pairs
        float lo = __int_as_float(0x7f800000), hi = __int_as_float(0xff800000);
        for (int m = 0; m < 8 && 8 * tid + m < TNRD_M; ++m) {
            const float mu = -__ldg(a.prm + KKP + 2 * (8 * tid + m));
            lo = fminf(lo, mu); hi = fmaxf(hi, mu);
        }
        crange[2 * tid] = lo; crange[2 * tid + 1] = hi;
    }

    int uoff[C::NB], voff[C::NB], coff[C::NB];
    unsigned own[C::NB];            // bit (4 j + p): pixel (row j, column p) of phi block n belongs to this tile
#pragma unroll
    for (int n = 0; n < C::NB; ++n) {
        const int blk = tid + n * NT;
        const int by = blk / nbx, bx = blk - by * nbx;
        uoff[n] = (by < nby) ? (2 * by) * C::US + 4 * bx : -1;
        voff[n] = (2 * by) * C::VS + 4 * bx;
        unsigned m = 0;
#pragma unroll
        for (int j = 0; j < 2; ++j)
#pragma unroll
            for (int p = 0; p < 4; ++p) {
                const int ly = 2 * by + j - R, lx = 4 * bx + p - R;          // output-tile coordinates
                if (ly >= 0 && ly < th && lx >= 0 && lx < tw) m |= 1u << (4 * j + p);
            }
        own[n] = m;
        const int cy = blk / nbxo, cx = blk - cy * nbxo;
        coff[n] = (cy < nbyo) ? (2 * cy) * C::VS + 4 * cx : -1;
    }
    float2 acc[C::NB][4];
#pragma unroll
    for (int n = 0; n < C::NB; ++n)
#pragma unroll
        for (int p = 0; p < 4; ++p) acc[n][p] = make_float2(0.f, 0.f);

    cp_async_wait_all();
    __syncthreads();

    // prologue: z' and q' of filter 0 on this thread's first block
    float2 zc[4] = {{0.f, 0.f}, {0.f, 0.f}, {0.f, 0.f}, {0.f, 0.f}};
    float2 qc[4] = {{0.f, 0.f}, {0.f, 0.f}, {0.f, 0.f}, {0.f, 0.f}};
    if (uoff[0] >= 0) {
#pragma unroll
        for (int wr = 0; wr <= KS; ++wr) {
            rowstep<KS, false>(us + uoff[0] + wr * C::US, ps + (KS - wr) * TS, zc);
            rowstep<KS, false>(es + uoff[0] + wr * C::US, ps + (KS - wr) * TS, qc);
        }
    }
    const size_t Hz = a.H + 2 * R, Wz = a.W + 2 * R;

    for (int i = 0; i < N_k; ++i) {
        if (i + 2 < N_k) {
            const float* src = a.prm + (size_t)(i + 2) * C::PRM;
            float* dst = ps + ((i + 2) & 3) * C::PRM;
            for (int idx = tid; idx < C::PRM; idx += NT) dst[idx] = __ldg(src + idx);
        }
        if (WANT_W && i > 0 && tid < 64) {     // flush the g_w sums of filter i-1 (complete since the last barrier)
            float s = 0.f;
#pragma unroll
            for (int wq = 0; wq < NT / 32; ++wq) { s += gws[(i + 1) & 1][wq][tid]; gws[(i + 1) & 1][wq][tid] = 0.f; }
            a.part_w[((size_t)blockIdx.x * N_k + (i - 1)) * 64 + tid] = s;
        }
        const float* rec = ps + (i & 3) * C::PRM;
        const float* recn = ps + ((i + 1) & 3) * C::PRM;
        const float* recp = ps + ((i + 3) & 3) * C::PRM;
        float* vcur = vs + (i & 1) * C::VPLANE;
        const float* vprev = vs + ((i + 1) & 1) * C::VPLANE;
        float* gw_slot = &gws[i & 1][warp][0];
#pragma unroll
        for (int n = 0; n < C::NB; ++n) {
            if (n >= nrounds) break;
            const bool last = (n == nrounds - 1);
            const int un = last ? uoff[0] : uoff[(n + 1) % C::NB];
            const bool hasB = uoff[n] >= 0;
            const bool hasN = un >= 0 && (!last || i + 1 < N_k);
            const bool hasC = i > 0 && coff[n] >= 0;
            const bool warpB = __any_sync(0xffffffffu, hasB);
            const float* tapsN = last ? recn : rec;
            const float* uwn = us + (un >= 0 ? un : 0);
            const float* ewn = es + (un >= 0 ? un : 0);
            const float* vw = vprev + (coff[n] >= 0 ? coff[n] : 0);
            float2 U[4] = {{0.f, 0.f}, {0.f, 0.f}, {0.f, 0.f}, {0.f, 0.f}};
            float2 V[4] = {{0.f, 0.f}, {0.f, 0.f}, {0.f, 0.f}, {0.f, 0.f}};
            float2 zn[4] = {{0.f, 0.f}, {0.f, 0.f}, {0.f, 0.f}, {0.f, 0.f}};
            float2 qn[4] = {{0.f, 0.f}, {0.f, 0.f}, {0.f, 0.f}, {0.f, 0.f}};
            float2 qm[4];
#pragma unroll
            for (int p = 0; p < 4; ++p)
                qm[p] = make_float2((own[n] >> p) & 1 ? qc[p].x : 0.f, (own[n] >> (4 + p)) & 1 ? qc[p].y : 0.f);
            // A step of 8 terms whose centres are all farther than D from every response of the warp contributes exact
            // zeros to A, V and the g_w sums (2^{-d^2} has flushed to zero): skipped, as the forward kernels skip dead
            // groups.  The warp's response range by redux over an order-preserving integer map; a NaN response keeps
            // every step live (max.NaN makes the upper end NaN and both tests false).
            float wlo, whi;
            {
                float zlo, zhi, t0, t1;
                asm("min.NaN.f32 %0, %1, %2;" : "=f"(t0) : "f"(fminf(zc[0].x, zc[0].y)), "f"(fminf(zc[1].x, zc[1].y)));
                asm("min.NaN.f32 %0, %1, %2;" : "=f"(t1) : "f"(fminf(zc[2].x, zc[2].y)), "f"(fminf(zc[3].x, zc[3].y)));
                asm("min.NaN.f32 %0, %1, %2;" : "=f"(zlo) : "f"(t0), "f"(t1));
                asm("max.NaN.f32 %0, %1, %2;" : "=f"(t0) : "f"(zc[0].x), "f"(zc[0].y));
                asm("max.NaN.f32 %0, %1, %2;" : "=f"(t1) : "f"(zc[1].x), "f"(zc[1].y));
                asm("max.NaN.f32 %0, %1, %2;" : "=f"(zhi) : "f"(t0), "f"(t1));
                asm("max.NaN.f32 %0, %1, %2;" : "=f"(t0) : "f"(zc[2].x), "f"(zc[2].y));
                asm("max.NaN.f32 %0, %1, %2;" : "=f"(t1) : "f"(zc[3].x), "f"(zc[3].y));
                asm("max.NaN.f32 %0, %1, %2;" : "=f"(zhi) : "f"(zhi), "f"(t0));
                asm("max.NaN.f32 %0, %1, %2;" : "=f"(zhi) : "f"(zhi), "f"(t1));
                if (!hasB) { zlo = __int_as_float(0x7f800000); zhi = __int_as_float(0xff800000); }
                wlo = ord2f(__reduce_min_sync(0xffffffffu, f2ord(zlo)));
                whi = ord2f(__reduce_max_sync(0xffffffffu, f2ord(zhi)));
            }
#pragma unroll 1
            for (int g = 0; g < C::NG; ++g) {
                float S[8];
                const float cmin = crange[2 * g], cmax = crange[2 * g + 1];
                const bool live = !((wlo - cmax > TNRD_FCLAMP && whi == whi) || cmin - whi > TNRD_FCLAMP);
                if (hasB && live) {
                    if (g < C::NG - 1) phi_bwd_step<8, WANT_W>(rec + KKP + 16 * g, zc, qm, U, V, S);
                    else phi_bwd_step<TNRD_M - 8 * (C::NG - 1), WANT_W>(rec + KKP + 16 * g, zc, qm, U, V, S);
                } else {
#pragma unroll
                    for (int m = 0; m < 8; ++m) S[m] = 0.f;
                }
                if (WANT_W && warpB && live) {
                    const float tot = warp_reduce8(S, lane);
                    if ((lane & 3) == 0) gw_slot[8 * g + (lane >> 2)] += tot;
                }
                if (g <= KS) {
                    if (hasN) {
                        rowstep<KS, false>(uwn + g * C::US, tapsN + (KS - g) * TS, zn);
                        rowstep<KS, false>(ewn + g * C::US, tapsN + (KS - g) * TS, qn);
                    }
                    if (hasC) rowstep<KS, true>(vw + g * C::VS, recp + g * TS, acc[n]);
                }
                if (KS + 1 > C::NG && g + C::NG <= KS) {
                    const int g2 = g + C::NG;
                    if (hasN) {
                        rowstep<KS, false>(uwn + g2 * C::US, tapsN + (KS - g2) * TS, zn);
                        rowstep<KS, false>(ewn + g2 * C::US, tapsN + (KS - g2) * TS, qn);
                    }
                    if (hasC) rowstep<KS, true>(vw + g2 * C::VS, recp + g2 * TS, acc[n]);
                }
            }
            if (hasB) {
                // P = Lambda_i Kbar_i^T e / s = -(A / gamma^2) (q' / s) / s = -2 ln2 A q'   (s^2 gamma^2 = log2(e) / 2)
                constexpr float C0 = -1.3862943611198906f;
                float2 P[4];
#pragma unroll
                for (int p = 0; p < 4; ++p) {
                    const float2 A = make_float2(fmaf(zc[p].x, V[p].x, -U[p].x), fmaf(zc[p].y, V[p].y, -U[p].y));   // phi' terms
                    P[p] = make_float2(C0 * A.x * qc[p].x, C0 * A.y * qc[p].y);
                }
                *reinterpret_cast<float4*>(vcur + voff[n]) = make_float4(P[0].x, P[1].x, P[2].x, P[3].x);
                *reinterpret_cast<float4*>(vcur + voff[n] + C::VS) = make_float4(P[0].y, P[1].y, P[2].y, P[3].y);
                if (WANT_K && own[n]) {     // owned pixels go to the HBM maps of kernel 2 (phi-region coordinates)
                    const int by = voff[n] / C::VS, bx = voff[n] - by * C::VS;      // phi-area-local block origin
                    const size_t mb = ((size_t)img * N_k + i) * Hz * Wz;
#pragma unroll
                    for (int j = 0; j < 2; ++j)
#pragma unroll
                        for (int p = 0; p < 4; ++p)
                            if ((own[n] >> (4 * j + p)) & 1) {
                                const int Yp = OY0 + by + j, Xp = OX0 + bx + p;     // = extended coordinate + r
                                if (Yp >= 0 && Yp < (int)Hz && Xp >= 0 && Xp < (int)Wz) {
                                    a.pmap[mb + (size_t)Yp * Wz + Xp] = j ? P[p].y : P[p].x;
                                    a.vmap[mb + (size_t)Yp * Wz + Xp] = j ? V[p].y : V[p].x;
                                }
                            }
                }
            }
#pragma unroll
            for (int p = 0; p < 4; ++p) { zc[p] = zn[p]; qc[p] = qn[p]; }
        }
        __syncthreads();
    }

    // ---- K_i^T of the last filter; flush its g_w sums -------------------------------------------------------------
    {
        const float* recp = ps + ((N_k - 1) & 3) * C::PRM;
        const float* vprev = vs + ((N_k - 1) & 1) * C::VPLANE;
#pragma unroll
        for (int n = 0; n < C::NB; ++n) {
            if (coff[n] < 0) continue;
#pragma unroll
            for (int wr = 0; wr <= KS; ++wr) rowstep<KS, true>(vprev + coff[n] + wr * C::VS, recp + wr * TS, acc[n]);
        }
        if (WANT_W && tid < 64) {
            float s = 0.f;
#pragma unroll
            for (int wq = 0; wq < NT / 32; ++wq) s += gws[(N_k - 1) & 1][wq][tid];
            a.part_w[((size_t)blockIdx.x * N_k + (N_k - 1)) * 64 + tid] = s;
        }
    }
    __syncthreads();        // every warp is done reading the P maps: plane 0 now receives the accumulators

    // ---- E^T: fold the 2r rim back onto the image (adjoint of the mirror map), g_u, g_lambda ---------------------
    float* G = vs;          // [RH][RW], output-tile coordinates
#pragma unroll
    for (int n = 0; n < C::NB; ++n) {
        if (coff[n] < 0) continue;
        *reinterpret_cast<float4*>(G + coff[n]) = make_float4(acc[n][0].y, acc[n][1].y, acc[n][2].y, acc[n][3].y);
        *reinterpret_cast<float4*>(G + coff[n] + C::VS) = make_float4(acc[n][0].x, acc[n][1].x, acc[n][2].x, acc[n][3].x);
    }
    __syncthreads();
    const float lambda = a.lambda_ptr ? __ldg(a.lambda_ptr) : a.lambda_val;
    const float* __restrict__ f_img = a.f + img * plane;
    float gl = 0.f;
    for (int idx = tid; idx < th * tw; idx += NT) {
        const int oy = idx / tw, ox = idx - oy * tw;
        const int y = OY0 + oy, x = OX0 + ox;
        if (y < 0 || y >= a.H || x < 0 || x >= a.W) continue;       // the rim itself owns nothing
        // pre-images of y under the mirror map inside [-2r, H + 2r): y, -1 - y (if y < 2r), 2H - 1 - y (if y >= H - 2r)
        int ys[3], xs[3], ny = 1, nx = 1;
        ys[0] = oy; xs[0] = ox;
        if (y < 2 * R) ys[ny++] = -1 - y - OY0;
        if (y >= a.H - 2 * R) ys[ny++] = 2 * a.H - 1 - y - OY0;
        if (x < 2 * R) xs[nx++] = -1 - x - OX0;
        if (x >= a.W - 2 * R) xs[nx++] = 2 * a.W - 1 - x - OX0;
        float s = 0.f;
        for (int p = 0; p < ny; ++p)
            for (int q = 0; q < nx; ++q) s += G[ys[p] * C::VS + xs[q]];
        const float ee = es[(oy + 2 * R) * C::US + ox + 2 * R];
        const size_t gidx = (size_t)y * a.W + x;
        if (a.g_u) a.g_u[img * plane + gidx] = (1.0f - lambda) * ee - s;
        gl += (us[(oy + 2 * R) * C::US + ox + 2 * R] - __ldg(f_img + gidx)) * ee;
    }
    if (a.part_l) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) gl += __shfl_xor_sync(0xffffffffu, gl, o);
        if (lane == 0) red[warp] = gl;
        __syncthreads();
        if (tid == 0) {
            float s = 0.f;
#pragma unroll
            for (int wq = 0; wq < NT / 32; ++wq) s += red[wq];
            a.part_l[blockIdx.x] = s;
        }
    }
}

// ---- kernel 2: g_k from the P / V maps ------------------------------------------------------------------------------
// Both terms of Supp. Eq. 10 are sums over the phi-region pixels (Y, X) (image coordinates, -r <= Y < H + r):
//   t2[a][b] = sum P_i[Y][X] u~(Y - a + r, X - b + r),   t1[a][b] = sum V_i[Y][X] e0(Y - a + r, X - b + r)
// (u~ mirror-extended, e0 zero-extended; the second is  sum_{y,x} e[y][x] V[y+a-r][x+b-r]  re-indexed by the V pixel).
// CTA (i, g) owns filter i and the tiles g, g + G, ... of 64 x 32 phi pixels: the ks^2 accumulators of a thread live
// across all its tiles and are reduced once.  A thread takes a 4 x 2 pixel block of each tile.
template <int KS>
struct WCfg {
    static constexpr int R = (KS - 1) / 2, TW = 64, TH = 32, NT = 256;
    static constexpr int SW = TW + KS - 1, SS = ((SW + 3) / 4) * 4 + 4, SH = TH + KS - 1;   // source tile (u~, e0)
    static constexpr int KK = KS * KS;
};

template <int KS>
__global__ void __launch_bounds__(WCfg<KS>::NT, KS <= 7 ? 2 : 1)
wgrad_kernel(BwdArgs a, int ntx, int nty, int G, float* __restrict__ part_k)
{
    using C = WCfg<KS>;
    constexpr int R = C::R, NT = C::NT, KK = C::KK, NV = (4 + KS - 1 + 3) / 4;
    __shared__ __align__(16) float us[C::SH * C::SS];
    __shared__ __align__(16) float es[C::SH * C::SS];
    __shared__ float redk[NT / 32][KK];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int i = blockIdx.x, g = blockIdx.y;
    const int Hz = a.H + 2 * R, Wz = a.W + 2 * R;
    const size_t plane = (size_t)a.H * a.W;
    const int bx4 = 4 * (tid & 15), by2 = 2 * (tid >> 4);      // this thread's block inside a tile

    float acc[KK];
#pragma unroll
    for (int q = 0; q < KK; ++q) acc[q] = 0.f;

    const int ntiles = ntx * nty * a.B;
    for (int tile = g; tile < ntiles; tile += G) {
        int t = tile;
        const int tx = t % ntx; t /= ntx;
        const int ty = t % nty; t /= nty;
        const int img = t;
        const int PX0 = tx * C::TW, PY0 = ty * C::TH;          // phi-region index of the tile origin (= image coord + r)
        const float* __restrict__ u_img = a.u + img * plane;
        const float* __restrict__ e_img = a.e + img * plane;
        // this thread's P and V values (zero outside the phi region): issued first, consumed after the source fill
        float P[2][4], V[2][4];
        const size_t mb = ((size_t)img * a.N_k + i) * (size_t)Hz * Wz;
#pragma unroll
        for (int j = 0; j < 2; ++j)
#pragma unroll
            for (int p = 0; p < 4; ++p) {
                const int Y = PY0 + by2 + j, X = PX0 + bx4 + p;
                const bool ok = Y < Hz && X < Wz;
                P[j][p] = ok ? __ldg(a.pmap + mb + (size_t)Y * Wz + X) : 0.f;
                V[j][p] = ok ? __ldg(a.vmap + mb + (size_t)Y * Wz + X) : 0.f;
            }
        // source pixel of phi index (Y, X) and lag (a, b): image coordinate (Y - r) - a + r = Y - a  ->  rows PY0 - (KS-1) ..
        // all loads of the fill are issued before the first store (a rolled loop would serialise on the load latency).
        // A warp takes rows sy = warp, warp + 8, ..., a lane columns sx = lane, lane + 32, ...: the mirror map and the
        // range tests of a column are computed once per tile and those of a row once per row, not once per element
        // (the per-element index arithmetic was what bound this kernel: ALU pipe 46 %, FMA pipe 37 %).
        constexpr int NCOL = (C::SW + 31) / 32, NROW = (C::SH + NT / 32 - 1) / (NT / 32);
        int xm[NCOL];
        unsigned xfl = 0;               // bit c: column inside the extended image, bit 8 + c: inside the image
#pragma unroll
        for (int c = 0; c < NCOL; ++c) {
            const int sx = lane + 32 * c, x = PX0 - (KS - 1) + sx;
            if (sx < C::SW && x >= -2 * R && x < a.W + 2 * R) xfl |= 1u << c;
            if (sx < C::SW && x >= 0 && x < a.W) xfl |= 1u << (8 + c);
            xm[c] = mirror_clamp(x, a.W);
        }
        float fu[NROW][NCOL], fe[NROW][NCOL];
#pragma unroll
        for (int q = 0; q < NROW; ++q) {
            const int sy = warp + q * (NT / 32), y = PY0 - (KS - 1) + sy;
            const bool yext = sy < C::SH && y >= -2 * R && y < a.H + 2 * R, yin = sy < C::SH && y >= 0 && y < a.H;
            const float* urow = u_img + (size_t)mirror_clamp(y, a.H) * a.W;
            const float* erow = e_img + (size_t)(yin ? y : 0) * a.W + (PX0 - (KS - 1) + lane);
#pragma unroll
            for (int c = 0; c < NCOL; ++c) {
                fu[q][c] = (yext && ((xfl >> c) & 1)) ? __ldg(urow + xm[c]) : 0.f;
                fe[q][c] = (yin && ((xfl >> (8 + c)) & 1)) ? __ldg(erow + 32 * c) : 0.f;
            }
        }
        __syncthreads();                                        // the previous tile's source is no longer read
#pragma unroll
        for (int q = 0; q < NROW; ++q) {
            const int sy = warp + q * (NT / 32);
#pragma unroll
            for (int c = 0; c < NCOL; ++c) {
                const int sx = lane + 32 * c;
                if (sy < C::SH && sx < C::SW) { us[sy * C::SS + sx] = fu[q][c]; es[sy * C::SS + sx] = fe[q][c]; }
            }
        }
        __syncthreads();
        // window rows wr = 0..KS: source row sy = by2 + wr serves lag a = j + (KS-1) - wr of block row j
#pragma unroll
        for (int wr = 0; wr <= KS; ++wr) {
            float ur[NV * 4], er[NV * 4];
            lds_vec(us + (by2 + wr) * C::SS + bx4, ur);
            lds_vec(es + (by2 + wr) * C::SS + bx4, er);
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                const int la = j + (KS - 1) - wr;
                if (la < 0 || la >= KS) continue;
#pragma unroll
                for (int b = 0; b < KS; ++b)
#pragma unroll
                    for (int p = 0; p < 4; ++p) {
                        // source column: phi X = PX0 + bx4 + p, lag b -> tile column bx4 + p - b + (KS-1)
                        acc[la * KS + b] = fmaf(P[j][p], ur[p - b + KS - 1], acc[la * KS + b]);
                        acc[la * KS + b] = fmaf(V[j][p], er[p - b + KS - 1], acc[la * KS + b]);
                    }
            }
        }
    }
    // ---- reduce the ks^2 sums over the CTA (fixed order) and store this CTA's partial ------------------------------
#pragma unroll
    for (int q = 0; q < KK; ++q) {
        float v = acc[q];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) redk[warp][q] = v;
    }
    __syncthreads();
    if (tid < KK) {
        float s = 0.f;
#pragma unroll
        for (int wq = 0; wq < NT / 32; ++wq) s += redk[wq][tid];
        part_k[((size_t)g * a.N_k + i) * KK + tid] = s;
    }
}

// ---- final sums in fixed order --------------------------------------------------------------------------------------
// g_w[i][j] = -(1/s) sum_cta part_w[cta][i][j];  g_k[i][q] = -s sum_g part_k[g][i][q];  g_lambda = -sum_cta part_l[cta]
__global__ void __launch_bounds__(256) reduce_partials_kernel(const float* __restrict__ part_w, int n_cta,
                                                              const float* __restrict__ part_k, int G,
                                                              const float* __restrict__ part_l, int N_k, int KK, float s,
                                                              float* __restrict__ g_w, float* __restrict__ g_k,
                                                              float* __restrict__ g_lambda)
{
    // 32 outputs x 8 slices per block: slice y adds the partials c = y, y + 8, ... in that order, the slices are added in
    // the order 0..7 (a fixed order: deterministic).  One thread per output took 140 us for 1296 partials.
    __shared__ float sl[8][33];
    const int idx = blockIdx.x * 32 + threadIdx.x, y = threadIdx.y;
    const int nw = N_k * 64, nk = N_k * KK;
    float acc = 0.f;
    if (idx < nw) {
        if (g_w && (idx & 63) < TNRD_M)
            for (int c = y; c < n_cta; c += 8) acc += __ldg(part_w + (size_t)c * nw + idx);
    } else if (idx < nw + nk) {
        if (g_k)
            for (int c = y; c < G; c += 8) acc += __ldg(part_k + (size_t)c * nk + (idx - nw));
    } else if (idx == nw + nk && g_lambda) {
        for (int c = y; c < n_cta; c += 8) acc += __ldg(part_l + c);
    }
    sl[y][threadIdx.x] = acc;
    __syncthreads();
    if (y != 0) return;
    float tot = 0.f;
#pragma unroll
    for (int q = 0; q < 8; ++q) tot += sl[q][threadIdx.x];
    if (idx < nw) {
        if (g_w && (idx & 63) < TNRD_M) g_w[(idx >> 6) * TNRD_M + (idx & 63)] = -tot / s;
    } else if (idx < nw + nk) {
        if (g_k) g_k[idx - nw] = -tot * s;
    } else if (idx == nw + nk && g_lambda) {
        g_lambda[0] = -tot;
    }
}

__global__ void sub_kernel(const float* __restrict__ x, const float* __restrict__ y, float* __restrict__ out, size_t n)
{
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
        out[i] = x[i] - y[i];
}

template <int KS, bool WANT_W, bool WANT_K>
cudaError_t launch_bwd_cfg(const BwdArgs& a, const BwdPlan& pl, cudaStream_t st)
{
    using C = BCfg<KS>;
    // the opt-in is an attribute of the CURRENT device's copy of the kernel: set at every launch (cheap), so that a
    // process that uses several devices works on each of them
    cudaError_t e = cudaFuncSetAttribute(stage_bwd_kernel<KS, WANT_W, WANT_K>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM);
    if (e != cudaSuccess) return e;
    stage_bwd_kernel<KS, WANT_W, WANT_K><<<(unsigned)pl.n_cta, C::NT, C::SMEM, st>>>(a, pl.ntx, pl.nty);
    return cudaGetLastError();
}

// `what`: 1 = the stage kernel, 2 = the lag-product kernel (g_k from the maps the stage kernel wrote), 3 = both in turn
template <int KS>
cudaError_t launch_bwd_ks(const BwdArgs& a, const BwdPlan& pl, float* part_k, int what, cudaStream_t st,
                          unsigned long long* launches)
{
    const bool want_w = a.part_w != nullptr, want_k = a.pmap != nullptr;
    cudaError_t e = cudaSuccess;
    if (what & 1) {
        if (want_k) e = launch_bwd_cfg<KS, true, true>(a, pl, st);          // g_k is only asked for together with g_w
        else if (want_w) e = launch_bwd_cfg<KS, true, false>(a, pl, st);
        else e = launch_bwd_cfg<KS, false, false>(a, pl, st);
        ++*launches;
    }
    if (e != cudaSuccess || !want_k || !(what & 2)) return e;
    wgrad_kernel<KS><<<dim3((unsigned)a.N_k, (unsigned)pl.G), WCfg<KS>::NT, 0, st>>>(a, pl.wtx, pl.wty, pl.G, part_k);
    ++*launches;
    return cudaGetLastError();
}

}  // namespace

BwdPlan plan_stage_bwd(int B, int H, int W, int N_k, int ksize, int num_sms)
{
    const int R = (ksize - 1) / 2, tmax = 64 - 2 * R;
    BwdPlan p;
    p.ntx = (W + 4 * R + tmax - 1) / tmax;
    p.nty = (H + 4 * R + tmax - 1) / tmax;
    p.n_cta = (long long)p.ntx * p.nty * B;
    p.wtx = (W + 2 * R + 63) / 64;               // wgrad tiles of 64 x 32 phi pixels
    p.wty = (H + 2 * R + 31) / 32;
    const long long wt = (long long)p.wtx * p.wty * B;
    // wgrad: N_k x G CTAs, each walking over its share of the tiles (a CTA lasts as long as its share).  G such that the
    // CTAs fill whole waves of the resident slots (2 CTAs per SM, 1 for 9x9): 13 CTAs per filter for 48 filters were 624
    // CTAs on 296 slots, 2.1 waves of work in the time of 3.
    const long long slots = (long long)(ksize <= 7 ? 2 : 1) * num_sms;
    long long G = 1;
    double best = -1.0;
    for (long long w = 12; w >= 1; --w) {      // many short CTAs rather than few long ones: they fill the gaps other kernels leave
        long long g = slots * w / N_k;
        if (g < 1) g = 1;
        if (g > wt) g = wt;
        const long long ctas = g * N_k, waves = (ctas + slots - 1) / slots;
        // the tiles of a filter are dealt out in turn: a CTA takes ceil(wt / g) tiles at most
        const double eff = (double)wt / (double)(((wt + g - 1) / g) * g) * (double)ctas / (double)(waves * slots);
        if (eff > best + 1e-9) { best = eff; G = g; }
    }
    p.G = (int)G;
    return p;
}

cudaError_t launch_stage_bwd(const BwdArgs& a, const BwdPlan& pl, float* part_k, int what, cudaStream_t st,
                             unsigned long long* launches)
{
    if (pl.n_cta > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    switch (a.ksize) {
        case 3: return launch_bwd_ks<3>(a, pl, part_k, what, st, launches);
        case 5: return launch_bwd_ks<5>(a, pl, part_k, what, st, launches);
        case 7: return launch_bwd_ks<7>(a, pl, part_k, what, st, launches);
        case 9: return launch_bwd_ks<9>(a, pl, part_k, what, st, launches);
        default: return cudaErrorInvalidValue;
    }
}

cudaError_t launch_reduce_partials(const float* part_w, long long n_cta, const float* part_k, int G, const float* part_l,
                                   int N_k, int ksize, float s, float* g_w, float* g_k, float* g_lambda, cudaStream_t st,
                                   unsigned long long* launches)
{
    const int total = N_k * 64 + N_k * ksize * ksize + 1;
    reduce_partials_kernel<<<(total + 31) / 32, dim3(32, 8), 0, st>>>(part_w, (int)n_cta, part_k, G, part_l, N_k,
                                                                      ksize * ksize, s, g_w, g_k, g_lambda);
    ++*launches;
    return cudaGetLastError();
}

cudaError_t launch_sub(const float* x, const float* y, float* out, size_t n, cudaStream_t st, unsigned long long* launches)
{
    const unsigned grid = (unsigned)((n + 255) / 256 < 4096 ? (n + 255) / 256 : 4096);
    sub_kernel<<<grid, 256, 0, st>>>(x, y, out, n);
    ++*launches;
    return cudaGetLastError();
}

}  // namespace tnrd

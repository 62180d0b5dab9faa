// tnrd_fused.cu -- the fused stage kernel (rows a1-a4 of the hot path in one pass) and the update kernel (a5).
//
//   u_t = u - ( sum_i kbar_i * phi_i(k_i * u~) + lambda (u - f) )          Main Eq. 7
//
// stage_fused_kernel: one CTA owns one tile of tw x th pixels of the phi region (the image plus its r ring) of one
// image; tiles PARTITION that region, so no influence value is computed twice:
//   a1  the u tile with its r halo is gathered through the mirror index map into shared
//       memory -- the padded image is never materialised;
//   then, one filter i at a time (streamed, so that only two influence maps live on chip):
//   a2  z' = k'_i * u~ on the tile, in registers, 4x2 pixels per unit of work,
//   a3  v = phi_i(z'): all 63 Gaussians, one MUFU.EX2 each (ex2.approx.ftz) -- or the windowed / table evaluator --
//       in registers, written once to a double-buffered shared-memory map whose ring outside the tile is zero,
//   a4  the rot180 taps of filter i-1 are applied to the map finished in the previous iteration, over the tile AND its
//       r ring (the pixels this tile's values reach), and summed into per-thread accumulators that live across the
//       whole filter loop; at the end the CTA stores these partial sums (64 KB).
// One __syncthreads() per filter.  stage_update_kernel (a5): u_t = u - (sum of the partial sums of the <= 2 x 2 tiles
// -- times the chunks of a split filter bank -- that reach the pixel + lambda (u - f)), point-wise, fixed order.
// HBM traffic: 4 B read + ~4.5 B written per pixel-stage by the tile kernel, ~16.5 B by the update kernel.
//
// This is the TILE kernel (tnrd_set_kernel(2)): both filterings on the FP32 FMA pipe.  It serves the shapes the
// tensor-core stage kernel (tnrd_tc.cu) does not take: 3x3 and 9x9 banks, more than 48 filters, the direct / windowed /
// table evaluators, and images too small to fill that kernel's 128-lane strips.  With the default factorised evaluator
// it is bound by the FMA pipe (8544 FMA-pipe operations per pixel-stage for 48 x 7x7), with the direct evaluator
// (TNRD_PHI_DENSE) by the XU pipe (3024 ex2).  Two things keep the pipes fed (profiles/r01_*.md):
//   * software pipelining inside a thread: the 63-term phi loop of block n is interleaved, row-step by row-step, with
//     the forward filter of the NEXT block (a2) and the transposed filter of block n for the previous filter (a4), so
//     every warp always carries a mix of MUFU and FMA work instead of all warps of a CTA filtering in lock-step;
//   * packed fp32x2 arithmetic (FADD2 / FMUL2 / FFMA2, sm_100): the two output rows of a 4x2 block form the two
//     halves of one register pair, which halves the issue slots of everything that is not a MUFU.
#include <cstdio>
#include <cstdlib>

#include "tnrd_internal.h"
#include "tnrd_device.cuh"

#define TNRD_FACT_NP 2   // pairs of responses per factorised-phi step

namespace tnrd {

namespace {

// Geometry of one CTA (all in "phi coordinates": index 0 = image coordinate -r; the phi region is (H+2r) x (W+2r)).
// The CTA owns a tile of tw x th phi pixels at (X0, Y0) -- tiles PARTITION the phi region, nothing is computed twice --
// and produces the partial transposed-filter sums of those pixels on the output area
//   columns [X0 - r, X0 + tw + r)
//   rows    [Y0 - r, Y0 + th + r),
// at most RW x RH pixels, i.e. tw <= RW - 2r, th <= RH - 2r.  Shared memory:
//   us   u tile, origin (Y0 - r, X0 - r) in phi coordinates = (Y0 - 2r, X0 - 2r) in image coordinates
//   vs   two influence maps, origin (Y0 - 2r, X0 - 8): the tile's own values surrounded by a ring of zeros, so that
//        the transposed filter can run over the whole output area (window row oy + a, column ox + b + 8 - 2r: the row
//        is read from the 16-byte aligned column of the output block and the window starts SHIFT = 8 - 2r into it)
template <int KS, int RW, int RH, int NT, int MINB = 1>
struct Cfg {
    static constexpr int R = (KS - 1) / 2;
    static constexpr int TWMAX = RW - 2 * R, THMAX = RH - 2 * R;   // largest tile
    static constexpr int US = RW + 8;                   // u tile row stride (floats)
    static constexpr int UH = RH + 2;                   // u tile rows (th + 2r + 1 window rows)
    static constexpr int VS = RW + 8;                   // phi map row stride
    static constexpr int VH = RH + 2 * R;               // phi map rows
    static constexpr int VPLANE = VH * VS;              // one phi map
    static constexpr int SHIFT = 8 - 2 * R;             // column shift of the transposed-filter window (see above)
    static constexpr int CTA_FLOATS = RW * RH;          // partial sums of one CTA (row-major over the output area)
    static constexpr int TS = prm_ts(KS);               // floats per row of tap pairs
    static constexpr int PRM = prm_stride(KS);          // floats per staged record
    static constexpr int NB = ((RW / 4) * (RH / 2) + NT - 1) / NT;  // 4x2 work blocks per thread (max)
    static constexpr int NG = TNRD_MP / 8;              // phi steps of 8 terms
    static constexpr size_t SMEM = sizeof(float) * ((size_t)UH * US + 2 * (size_t)VPLANE + 4 * (size_t)PRM);
};

// NTERM (8, or 7 in the last step: 63 = 7 * 8 + 7) RBF terms for the 8 responses of a block: 4 x LDS.128 of
// (-mu', w') pairs, then per term and response pair FADD2, FMUL2, 2 x MUFU.EX2, FFMA2
template <int NTERM>
__device__ __forceinline__ void phi_step(const float* __restrict__ mw, const float2 (&z)[4], float2 (&v)[4])
{
    float c[16];
    lds_vec(mw, c);
#pragma unroll
    for (int m = 0; m < NTERM; ++m)
#pragma unroll
        for (int p = 0; p < 4; ++p) {
            const float2 d = __fadd2_rn(z[p], make_float2(c[2 * m], c[2 * m]));
            const float2 t = __fmul2_rn(d, d);
            const float2 e = make_float2(ex2_neg(t.x), ex2_neg(t.y));
            v[p] = __ffma2_rn(e, make_float2(c[2 * m + 1], c[2 * m + 1]), v[p]);
        }
}

// ---- windowed phi evaluator (PHI = 1) -------------------------------------------------------------------------------
// With equidistant centres (spacing delta' in scaled units) and gamma <= delta, every centre farther than 6.5 gamma from
// a response z contributes less than e^{-21.1} = 6.7e-10 of its weight -- below fp32 rounding of the sum.  Each response
// therefore evaluates only the 14 consecutive centres j0 .. j0+13 (j0 even) that contain [jc-6, jc+6], jc = nearest
// centre: 14 MUFU.EX2 instead of 63, weights gathered per lane (8-byte loads) from the plain w' row of the staged record.
// win_setup: per response the offset d = z' - mu'_{j0} and the byte offset of w'_{j0} inside the record.
__device__ __forceinline__ void win_setup1(float z, float inv_delta, float mu0, float delta, float& d, int& wofs)
{
    const float tq = (z - mu0) * inv_delta;
    int jc = __float2int_rn(fminf(fmaxf(tq, 0.0f), 62.0f));
    int j0 = min(max(jc - 6, 0) & ~1, 50);
    d = (z - mu0) - (float)j0 * delta;
    wofs = j0 * 4;
}

// one step = two consecutive centres (2g, 2g+1 of the window) for the 8 responses of a block; dd is advanced by the
// caller.  wsec = shared-memory byte address of w'_{i,0} + 8 g.
__device__ __forceinline__ void phi_win_step(unsigned wsec, const int (&wofs)[4][2], float delta, float2 (&dd)[4],
                                             float2 (&v)[4])
{
#pragma unroll
    for (int p = 0; p < 4; ++p) {
        float2 wa, wb;
        asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(wa.x), "=f"(wa.y) : "r"(wsec + wofs[p][0]));
        asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(wb.x), "=f"(wb.y) : "r"(wsec + wofs[p][1]));
        const float2 d0 = dd[p];
        const float2 d1 = __fadd2_rn(d0, make_float2(-delta, -delta));
        const float2 t0 = __fmul2_rn(d0, d0), t1 = __fmul2_rn(d1, d1);
        const float2 e0 = make_float2(ex2_neg(t0.x), ex2_neg(t0.y));
        const float2 e1 = make_float2(ex2_neg(t1.x), ex2_neg(t1.y));
        v[p] = __ffma2_rn(e0, make_float2(wa.x, wb.x), v[p]);
        v[p] = __ffma2_rn(e1, make_float2(wa.y, wb.y), v[p]);
        dd[p] = __fadd2_rn(d1, make_float2(-delta, -delta));
    }
}

// ---- factorised phi evaluator (PHI = 3) -----------------------------------------------------------------------------
// All 63 Gaussians, but 3 ex2 per GROUP of 2S+1 = 13 neighbouring centres instead of one per centre (tnrd_internal.h,
// "fact"): with d = z' - mu'_a (a = the group's middle centre), g = 2^{-d^2}, rho = 2^{kappa d},
//   sum_{j=-S..S} w'_{a+j} 2^{-(d - j delta')^2} = g * ( sum_{j>=0} c_j rho^j + sum_{j<0} c_j rho^j ),
// the two sums by Horner's rule in rho and 1/rho.  Per response and group: FADD, 2 FMNMX (clamp), 2 FMUL, 3 MUFU.EX2,
// 2S + 1 FFMA -- 15 ex2 and 80 FMA-pipe operations per response where the direct form needs 63 and 189.
// fact_pairs: pairs P0, P0+1 of the block (two packed responses each) for one group record.
__device__ __forceinline__ float fclamp_nan(float x, float lim)          // NaN stays NaN (as in the direct evaluator)
{
    float y;
    asm("min.NaN.f32 %0, %1, %2;" : "=f"(y) : "f"(x), "f"(lim));
    asm("max.NaN.f32 %0, %0, %1;" : "+f"(y) : "f"(-lim));
    return y;
}
__device__ __forceinline__ float ex2_pos(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
// true if some response of some lane of the warp lies inside the clamp of the group anchored at -c0 (NaNs count as live)
__device__ __forceinline__ bool fact_group_live(const float2 (&z)[4], float c0, float dmax, bool hasB)
{
    bool l = false;
#pragma unroll
    for (int p = 0; p < 4; ++p) l = l || !(fabsf(z[p].x + c0) >= dmax) || !(fabsf(z[p].y + c0) >= dmax);
    return __any_sync(0xffffffffu, hasB && l);
}
template <int NP> struct FactStateN { float2 g[NP], rho[NP], rhoi[NP]; };
using FactState = FactStateN<TNRD_FACT_NP>;   // of two pairs of responses: 2^{-d^2}, 2^{kappa d}, 2^{-kappa d}

// first half of a group for pairs P0, P0+1: the clamped distances to the anchor and the three exponentials of each response
template <int P0>
__device__ __forceinline__ void fact_exp(const float (&c)[TNRD_FSTRIDE], float kappa, float dmax, const float2 (&z)[4],
                                         FactState& s)
{
    constexpr int NP = TNRD_FACT_NP;
#pragma unroll
    for (int p = 0; p < NP; ++p) {
        float2 d = __fadd2_rn(z[P0 + p], make_float2(c[0], c[0]));
        d = make_float2(fclamp_nan(d.x, dmax), fclamp_nan(d.y, dmax));
        const float2 t = __fmul2_rn(d, d);
        const float2 e = __fmul2_rn(d, make_float2(kappa, kappa));
        s.g[p] = make_float2(ex2_neg(t.x), ex2_neg(t.y));
        s.rho[p] = make_float2(ex2_pos(e.x), ex2_pos(e.y));
        s.rhoi[p] = make_float2(ex2_neg(e.x), ex2_neg(e.y));
    }
}
// second half: the two Horner polynomials and the sum into v
template <int P0>
__device__ __forceinline__ void fact_poly(const float (&c)[TNRD_FSTRIDE], const FactState& s, float2 (&v)[4])
{
    constexpr int S = TNRD_FS, NP = TNRD_FACT_NP;
    float2 h[NP], hl[NP];
#pragma unroll
    for (int p = 0; p < NP; ++p) {
        h[p] = __ffma2_rn(make_float2(c[1], c[1]), s.rho[p], make_float2(c[2], c[2]));               // c_S rho + c_{S-1}
        hl[p] = __ffma2_rn(make_float2(c[S + 2], c[S + 2]), s.rhoi[p], make_float2(c[S + 3], c[S + 3]));
    }
#pragma unroll
    for (int q = 2; q <= S; ++q)                                             // c_{S-2} .. c_0
#pragma unroll
        for (int p = 0; p < NP; ++p) h[p] = __ffma2_rn(h[p], s.rho[p], make_float2(c[1 + q], c[1 + q]));
#pragma unroll
    for (int q = 2; q < S; ++q)                                              // c_{-S+2} .. c_{-1}
#pragma unroll
        for (int p = 0; p < NP; ++p) hl[p] = __ffma2_rn(hl[p], s.rhoi[p], make_float2(c[S + 2 + q], c[S + 2 + q]));
#pragma unroll
    for (int p = 0; p < NP; ++p) {
        h[p] = __ffma2_rn(hl[p], s.rhoi[p], h[p]);
        v[P0 + p] = __ffma2_rn(s.g[p], h[p], v[P0 + p]);
    }
}

// A group whose Gaussian factor has flushed to zero for EVERY response of the warp is skipped (fact_group_live): its
// contribution is an exact 0 either way, so the result is bit-identical; the run time then depends on the responses
// (bench.py reports the executed next to the defined phi work).
// One block of the software pipeline with the factorised evaluator: phi of the block's 8 responses (TNRD_FG groups, two
// pairs of responses at a time) with the KS + 1 window rows of both filterings riding along -- rows 1 .. KS-1 two per
// group in the first (KS-1)/2 groups, the one-sided rows 0 and KS (rowstep_half) in the last group.  A window row of the
// forward filter sits between the exponentials of a pair and their polynomials: its FMAs cover the MUFU latency.
template <int KS, class C>
__device__ __forceinline__ void fact_block(const float* __restrict__ frec, float kappa, float dmax, const float2 (&zc)[4],
                                           float2 (&v)[4], const float* __restrict__ uwn, const float* __restrict__ tapsN,
                                           float2 (&zn)[4], const float* __restrict__ vw, const float* __restrict__ recp,
                                           float2 (&acc)[4], bool hasB_, bool hasN, bool hasC)
{
    constexpr int TS = C::TS, NGR = (KS - 1) / 2;
    static_assert(NGR <= TNRD_FG - 1, "not enough phi groups for the window rows");
    float fc[TNRD_FSTRIDE];
    FactState st;
    lds_vec(frec, fc);
#pragma unroll
    for (int g = 0; g < NGR; ++g) {
        const bool hasB = fact_group_live(zc, fc[0], dmax, hasB_);
        if (hasB) fact_exp<0>(fc, kappa, dmax, zc, st);
        if (hasN) rowstep<KS, false>(uwn + (2 * g + 1) * C::US, tapsN + (KS - 2 * g - 1) * TS, zn);
        if (hasB) fact_poly<0>(fc, st, v);
        if (hasC) rowstep<KS, true, C::SHIFT>(vw + (2 * g + 1) * C::VS, recp + (2 * g + 1) * TS, acc);
        if (hasB) fact_exp<2>(fc, kappa, dmax, zc, st);
        if (hasN) rowstep<KS, false>(uwn + (2 * g + 2) * C::US, tapsN + (KS - 2 * g - 2) * TS, zn);
        if (hasB) fact_poly<2>(fc, st, v);
        if (hasC) rowstep<KS, true, C::SHIFT>(vw + (2 * g + 2) * C::VS, recp + (2 * g + 2) * TS, acc);
        lds_vec(frec + (g + 1) * TNRD_FSTRIDE, fc);
    }
#pragma unroll 1
    for (int g = NGR; g < TNRD_FG - 1; ++g) {
        const bool hasB = fact_group_live(zc, fc[0], dmax, hasB_);
        if (hasB) {
            fact_exp<0>(fc, kappa, dmax, zc, st);
            fact_poly<0>(fc, st, v);
            fact_exp<2>(fc, kappa, dmax, zc, st);
            fact_poly<2>(fc, st, v);
        }
        lds_vec(frec + (g + 1) * TNRD_FSTRIDE, fc);
    }
    const bool hasB = fact_group_live(zc, fc[0], dmax, hasB_);
    if (hasB) fact_exp<0>(fc, kappa, dmax, zc, st);
    if (hasN) rowstep_half<KS, false, 0, 0>(uwn, tapsN + KS * TS, zn);                            // window row 0
    if (hasB) fact_poly<0>(fc, st, v);
    if (hasC) rowstep_half<KS, true, C::SHIFT, 1>(vw, recp, acc);
    if (hasB) fact_exp<2>(fc, kappa, dmax, zc, st);
    if (hasN) rowstep_half<KS, false, 0, 1>(uwn + KS * C::US, tapsN, zn);                         // window row KS
    if (hasB) fact_poly<2>(fc, st, v);
    if (hasC) rowstep_half<KS, true, C::SHIFT, 0>(vw + KS * C::VS, recp + KS * TS, acc);
}

template <int KS, int RW, int RH, int NT, int MINB, int PHI>
__global__ void __launch_bounds__(NT, MINB)
stage_fused_kernel(StageArgs a, int tw_nom, int th_nom, int ntx, int nty, int n_full, int nsplit,
                   float* __restrict__ part)
{
    using C = Cfg<KS, RW, RH, NT, MINB>;
    constexpr int R = C::R, TS = C::TS, KKP = prm_kkp(KS);
    extern __shared__ __align__(16) float smem[];
    float* us = smem;                              // [UH][US]   u tile with r halo
    float* vs = us + C::UH * C::US;                // [2][VPLANE] influence maps of filters i and i-1 (zero ring)
    float* ps = vs + 2 * C::VPLANE;                // [4][PRM]   staged records of filters i-1 .. i+2

    const int tid = threadIdx.x;
    // CTAs 0 .. n_full-1 take a whole tile each; the tiles after that are split over nsplit CTAs, each with a contiguous
    // chunk of the filter bank (small images: n_full = 0; large ones: only the tiles of the last, partly filled wave)
    const int split_r = (int)blockIdx.x - n_full;
    const int parts = split_r < 0 ? 1 : nsplit, chunk = split_r < 0 ? 0 : split_r % nsplit;
    int t = split_r < 0 ? (int)blockIdx.x : n_full + split_r / nsplit;   // tile
    const int tx = t % ntx; t /= ntx;
    const int ty = t % nty; t /= nty;
    const int img = t;
    const int X0 = tx * tw_nom, Y0 = ty * th_nom;  // phi coordinates of the tile origin
    const int tw = min(tw_nom, a.W + 2 * R - X0), th = min(th_nom, a.H + 2 * R - Y0);   // ragged last tiles
    const float* __restrict__ u_img = a.u_in + (size_t)img * a.H * a.W;
    const int f0 = chunk * a.N_k / parts;
    const int N_k = (chunk + 1) * a.N_k / parts - f0;                       // filters f0 .. f0 + N_k - 1
    // The windowed evaluator runs only if the staging kernel found the centres equidistant; when it is selected both
    // kernels are launched and the one that does not apply returns at once (no host synchronisation needed).
    float w_inv_delta = 0.f, w_mu0 = 0.f, w_delta = 0.f;
    if (PHI == 1) {
        if (__ldg(a.prm + prm_hdr(KS) + 3) == 0.0f) return;
        w_inv_delta = __ldg(a.prm + prm_hdr(KS) + 0);
        w_mu0 = __ldg(a.prm + prm_hdr(KS) + 1);
        w_delta = __ldg(a.prm + prm_hdr(KS) + 2);
    } else if (PHI == 0 && a.dense_is_fallback) {
        if (__ldg(a.prm + prm_hdr(KS) + 3) != 0.0f) return;
    }
    // factorised evaluator: applies when the staging kernel said so, else this kernel evaluates the direct form
    constexpr bool DIRECT = PHI == 0 || PHI == 3;
    float f_kappa = 0.f, f_dmax = 0.f;
    bool fact = false;
    if (PHI == 3) {
        f_kappa = __ldg(a.prm + prm_hdr(KS) + 4);
        f_dmax = __ldg(a.prm + prm_hdr(KS) + 5);
        fact = __ldg(a.prm + prm_hdr(KS) + 6) != 0.0f;
    }
    // piecewise-linear table evaluator (PHI = 2; tnrd_table.cu): t = a z' + b in node units
    float t_a = 0.f, t_b = 0.f, t_max = 0.f;
    if (PHI == 2) { t_a = __ldg(a.tabhdr); t_b = __ldg(a.tabhdr + 1); t_max = __ldg(a.tabhdr + 2); }

    // ---- work decomposition: 4x2 pixel blocks, NB per thread ----------------------------------------------
    const int nbx = (tw + 3) >> 2, nby = (th + 1) >> 1;                         // phi blocks: the tile itself
    const int nbxo = (tw + 2 * R + 3) >> 2, nbyo = (th + 2 * R + 1) >> 1;       // output blocks: tile + ring
    const int nrounds = (nbxo * nbyo + NT - 1) / NT; // rounds of blocks this tile needs (<= NB): the software pipeline
                                                     // wraps from the last USED round to block 0 of the next filter

    // ---- a1: gather the u tile through the mirror map (only the rows / columns some block will read) -----
    {
        const int nr = min(C::UH, 2 * nby + 2 * R), nc = min(C::US, 4 * nbx + 2 * R + 4);
        for (int idx = tid; idx < 2 * C::VPLANE / 4; idx += NT)               // zero ring of both maps
            reinterpret_cast<float4*>(vs)[idx] = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll 2
        for (int uy = tid >> 5; uy < nr; uy += NT / 32) {
            const float* __restrict__ grow = u_img + (size_t)mirror_clamp(Y0 - 2 * R + uy, a.H) * a.W;
#pragma unroll
            for (int q = 0; q < (C::US + 31) / 32; ++q) {          // asynchronous copies: every row of the tile is in flight at once
                const int ux = (tid & 31) + 32 * q;
                if (ux < nc) cp_async4(us + uy * C::US + ux, grow + mirror_clamp(X0 - 2 * R + ux, a.W));
            }
        }
    }
    for (int idx = tid; idx < 2 * C::PRM / 4; idx += NT)                                // records 0 and 1
        if (4 * idx < N_k * C::PRM) cp_async16(ps + 4 * idx, a.prm + (size_t)f0 * C::PRM + 4 * idx);

    int uoff[C::NB], voff[C::NB], coff[C::NB];   // block origins in us / a phi map (phi side) / a phi map (output side)
    unsigned own = 0;                            // bit 8 n + 4 j + p: pixel (row j, column p) of phi block n is in the tile
#pragma unroll
    for (int n = 0; n < C::NB; ++n) {
        const int blk = tid + n * NT;
        const int by = blk / nbx, bx = blk - by * nbx;
        uoff[n] = (by < nby) ? (2 * by) * C::US + 4 * bx : -1;
        voff[n] = (2 * by + 2 * R) * C::VS + 4 * bx + 8;
#pragma unroll
        for (int j = 0; j < 2; ++j)
#pragma unroll
            for (int p = 0; p < 4; ++p)
                if (2 * by + j < th && 4 * bx + p < tw) own |= 1u << (8 * n + 4 * j + p);
        const int cy = blk / nbxo, cx = blk - cy * nbxo;
        coff[n] = (cy < nbyo) ? (2 * cy) * C::VS + 4 * cx : -1;
    }
    float2 acc[C::NB][4];                          // (row 1, row 0) of the transposed-filter sum, per block column
#pragma unroll
    for (int n = 0; n < C::NB; ++n)
#pragma unroll
        for (int p = 0; p < 4; ++p) acc[n][p] = make_float2(0.f, 0.f);

    cp_async_wait_all();                           // the u tile and the first records have landed
    __syncthreads();

    // prologue: responses of filter 0 on this thread's first block
    float2 zc[4] = {{0.f, 0.f}, {0.f, 0.f}, {0.f, 0.f}, {0.f, 0.f}};
    if (uoff[0] >= 0) {
#pragma unroll
        for (int wr = 0; wr <= KS; ++wr) rowstep<KS, false>(us + uoff[0] + wr * C::US, ps + (KS - wr) * TS, zc);
    }

    // ---- filter loop ------------------------------------------------------------------------------------------
    for (int i = 0; i < N_k; ++i) {
        if (i + 2 < N_k) {                                    // stage record i+2 (read from iteration i+1 on)
            const float* src = a.prm + (size_t)(f0 + i + 2) * C::PRM;
            float* dst = ps + ((i + 2) & 3) * C::PRM;
            for (int idx = tid; idx < C::PRM / 4; idx += NT) cp_async16(dst + 4 * idx, src + 4 * idx);
        }
        const float* rec = ps + (i & 3) * C::PRM;             // filter i: phi pairs, a2 of blocks 1..NB-1
        const float* recn = ps + ((i + 1) & 3) * C::PRM;      // filter i+1: a2 of block 0
        const float* recp = ps + ((i + 3) & 3) * C::PRM;      // filter i-1: a4
        float* vcur = vs + (i & 1) * C::VPLANE;
        const float* vprev = vs + ((i + 1) & 1) * C::VPLANE;
#pragma unroll
        for (int n = 0; n < C::NB; ++n) {
            if (n >= nrounds) break;
            const bool last = (n == nrounds - 1);
            const int un = last ? uoff[0] : uoff[(n + 1) % C::NB];
            const bool hasB = uoff[n] >= 0;                               // phi of block n
            const bool hasN = un >= 0 && (!last || i + 1 < N_k);          // forward filter of the next block
            const bool hasC = i > 0 && coff[n] >= 0;                      // transposed filter of output block n
            const float* tapsN = last ? recn : rec;
            const float* uwn = us + (un >= 0 ? un : 0);
            const float* vw = vprev + (coff[n] >= 0 ? coff[n] : 0);
            float2 v[4] = {{0.f, 0.f}, {0.f, 0.f}, {0.f, 0.f}, {0.f, 0.f}};
            float2 zn[4] = {{0.f, 0.f}, {0.f, 0.f}, {0.f, 0.f}, {0.f, 0.f}};
            float2 dd[4];
            int wofs[4][2];
            unsigned wsec = 0;
            float2 te[4][2];                       // PHI = 2: table entries (value, slope) of the 8 responses ...
            float2 tf[4];                          // ... and the positions inside their table cells
            if (PHI == 2 && hasB) {                // the gathers are issued here and used after the row-steps below
                const float2* __restrict__ tabi = reinterpret_cast<const float2*>(a.tab) + (size_t)(f0 + i) * TNRD_TAB_NODES;
#pragma unroll
                for (int p = 0; p < 4; ++p) {
                    const float tx_ = fminf(fmaxf(fmaf(zc[p].x, t_a, t_b), 0.0f), t_max);
                    const float ty_ = fminf(fmaxf(fmaf(zc[p].y, t_a, t_b), 0.0f), t_max);
                    const int jx = min((int)tx_, (int)t_max - 1), jy = min((int)ty_, (int)t_max - 1);
                    tf[p] = make_float2(tx_ - (float)jx, ty_ - (float)jy);
                    te[p][0] = __ldg(tabi + jx);
                    te[p][1] = __ldg(tabi + jy);
                }
            }
            if (PHI == 1) {
#pragma unroll
                for (int p = 0; p < 4; ++p) {
                    win_setup1(zc[p].x, w_inv_delta, w_mu0, w_delta, dd[p].x, wofs[p][0]);
                    win_setup1(zc[p].y, w_inv_delta, w_mu0, w_delta, dd[p].y, wofs[p][1]);
                }
                wsec = (unsigned)__cvta_generic_to_shared(rec + prm_wplain(KS));
            }
            if (PHI == 3 && fact) {
                const float* frec = rec + prm_fact(KS);
                    fact_block<KS, C>(frec, f_kappa, f_dmax, zc, v, uwn, tapsN, zn, vw, recp, acc[n], hasB, hasN, hasC);
            } else {
#pragma unroll (DIRECT ? 1 : 2)
            for (int g = 0; g < C::NG - 1; ++g) {
                if (hasB) {
                    if (PHI == 1) phi_win_step(wsec + 8 * g, wofs, w_delta, dd, v);
                    else if (DIRECT) phi_step<8>(rec + KKP + 16 * g, zc, v);
                }
                if (g <= KS) {
                    if (hasN) rowstep<KS, false>(uwn + g * C::US, tapsN + (KS - g) * TS, zn);
                    if (hasC) rowstep<KS, true, C::SHIFT>(vw + g * C::VS, recp + g * TS, acc[n]);
                }
                if (KS + 1 > C::NG && g + C::NG <= KS) {      // ksize 9: ten row-steps in eight phi steps
                    const int g2 = g + C::NG;
                    if (hasN) rowstep<KS, false>(uwn + g2 * C::US, tapsN + (KS - g2) * TS, zn);
                    if (hasC) rowstep<KS, true, C::SHIFT>(vw + g2 * C::VS, recp + g2 * TS, acc[n]);
                }
            }
            {   // last step: the remaining 63 - 56 = 7 terms (dense); the window's 14 centres are done after 7 steps
                constexpr int g = C::NG - 1;
                if (hasB) {
                    if (DIRECT) phi_step<TNRD_M - 8 * g>(rec + KKP + 16 * g, zc, v);
                }
                if (g <= KS) {
                    if (hasN) rowstep<KS, false>(uwn + g * C::US, tapsN + (KS - g) * TS, zn);
                    if (hasC) rowstep<KS, true, C::SHIFT>(vw + g * C::VS, recp + g * TS, acc[n]);
                }
            }
            }
            if (PHI == 2 && hasB) {
#pragma unroll
                for (int p = 0; p < 4; ++p)
                    v[p] = make_float2(fmaf(tf[p].x, te[p][0].y, te[p][0].x), fmaf(tf[p].y, te[p][1].y, te[p][1].x));
            }
            if (hasB) {     // pixels of a ragged block that lie outside the tile belong to the neighbour: keep the ring zero
                const unsigned m = own >> (8 * n);
                *reinterpret_cast<float4*>(vcur + voff[n]) = make_float4(
                    m & 1 ? v[0].x : 0.f, m & 2 ? v[1].x : 0.f, m & 4 ? v[2].x : 0.f, m & 8 ? v[3].x : 0.f);
                *reinterpret_cast<float4*>(vcur + voff[n] + C::VS) = make_float4(
                    m & 16 ? v[0].y : 0.f, m & 32 ? v[1].y : 0.f, m & 64 ? v[2].y : 0.f, m & 128 ? v[3].y : 0.f);
            }
#pragma unroll
            for (int p = 0; p < 4; ++p) zc[p] = zn[p];
        }
        cp_async_wait_all();                                  // record i+2 has landed
        __syncthreads();
    }

    // ---- a4 of the last filter --------------------------------------------------------------------------------
    {
        const float* recp = ps + ((N_k - 1) & 3) * C::PRM;
        const float* vprev = vs + ((N_k - 1) & 1) * C::VPLANE;
#pragma unroll
        for (int n = 0; n < C::NB; ++n) {
            if (coff[n] < 0) continue;
#pragma unroll
            for (int wr = 0; wr <= KS; ++wr)
                rowstep<KS, true, C::SHIFT>(vprev + coff[n] + wr * C::VS, recp + wr * TS, acc[n]);
        }
    }

    // ---- the partial sums of this CTA (its tile, its chunk of the filter bank) go to scratch, row-major over the
    // output area: pixel (oy, ox) at oy * RW + ox.  stage_update_kernel adds the partial sums of every CTA that reaches a
    // pixel in fixed order and applies the reaction term (a5).
    float* mine = part + (size_t)blockIdx.x * C::CTA_FLOATS;            // slot = CTA index
#pragma unroll
    for (int n = 0; n < C::NB; ++n) {
        if (coff[n] < 0) continue;
        const int oy = coff[n] / C::VS, ox = coff[n] - oy * C::VS;
        float* d = mine + oy * RW + ox;
        __stcg(reinterpret_cast<float4*>(d), make_float4(acc[n][0].y, acc[n][1].y, acc[n][2].y, acc[n][3].y));
        __stcg(reinterpret_cast<float4*>(d + RW), make_float4(acc[n][0].x, acc[n][1].x, acc[n][2].x, acc[n][3].x));
    }
}

// a5: u_t = u - (s + lambda (u - f)), s = sum of the partial sums of the (at most 2 x 2) tiles whose output
// area holds the pixel, times the nsplit chunks of the filter bank, added in a fixed order (deterministic).
// grid (ceil(W / (128 PX)), rows of the batch over y and z), 128 threads, PX consecutive pixels per thread: the kernel is
// bound by the latency of its 4-byte reads, so large images take PX = 4 (more loads in flight per thread) and small ones
// PX = 1 (more threads).
template <int PX>
__global__ void __launch_bounds__(128)
stage_update_kernel(StageArgs a, const float* __restrict__ part, int tw, int th, int ntx, int nty, int n_full, int nsplit,
                    int cta_floats, int rw, int R)
{
    const long long row = (long long)blockIdx.z * 65535 + blockIdx.y;            // row of the whole batch
    const int x0 = (blockIdx.x * 128 + threadIdx.x) * PX;
    if (x0 >= a.W || row >= (long long)a.B * a.H) return;
    const int img = (int)(row / a.H), y = (int)(row - (long long)img * a.H);
    const size_t idx0 = (size_t)row * a.W + x0;
    const int yp = y + R;                                                        // phi coordinates
    const int tylo = y / th, tyhi = min(nty - 1, (yp + R) / th);
    float uu[PX], ff[PX], s[PX];
#pragma unroll
    for (int q = 0; q < PX; ++q) {
        const bool ok = x0 + q < a.W;
        uu[q] = ok ? a.u_in[idx0 + q] : 0.f;     // plain loads: u_out may be u_in (and f, deblocking) -- in place
        ff[q] = ok ? a.f[idx0 + q] : 0.f;
        s[q] = 0.f;
    }
    for (int ty = tylo; ty <= tyhi; ++ty) {
        const int oy = yp - (ty * th - R);
#pragma unroll
        for (int q = 0; q < PX; ++q) {
            const int x = x0 + q, xp = x + R;
            if (x >= a.W) continue;
            const int txlo = x / tw, txhi = min(ntx - 1, (xp + R) / tw);
            for (int tx = txlo; tx <= txhi; ++tx) {
                const int ox = xp - (tx * tw - R);
                const long long tile = ((long long)img * nty + ty) * ntx + tx;       // slots are in CTA order
                const long long slot = tile < n_full ? tile : n_full + (tile - n_full) * nsplit;
                const int cnt = tile < n_full ? 1 : nsplit;
                const float* p = part + (size_t)slot * cta_floats + oy * rw + ox;
#pragma unroll 4
                for (int c = 0; c < cnt; ++c) s[q] += __ldcg(p + (size_t)c * cta_floats);
            }
        }
    }
    const float lambda = a.lambda_ptr ? __ldg(a.lambda_ptr) : a.lambda_val;
#pragma unroll
    for (int q = 0; q < PX; ++q)
        if (x0 + q < a.W) a.u_out[idx0 + q] = uu[q] - (s[q] + lambda * (uu[q] - ff[q]));
}

// ---- host side: tile plan and launch ------------------------------------------------------------------------------
struct Plan {
    int ntx, nty, tw, th, nsplit;
    long long n_full; // tiles taken by one CTA each (the rest are split over nsplit CTAs)
    double cost;      // estimated time of the launch in (thread-rounds x filters) per SM (see plan_tiles)
    long long work;   // phi blocks of one CTA (critical path; tie-break)
};

inline int env_int(const char* name)
{
    const char* e = getenv(name);
    return e ? atoi(e) : 0;
}
// TNRD_TILE=<id> / TNRD_SPLIT=<n> (environment, read at every plan) force a kernel configuration / a filter split;
// tuning and test knobs, not part of the ABI.
inline int forced_tile() { return env_int("TNRD_TILE"); }
inline int forced_split() { return env_int("TNRD_SPLIT"); }

// Tile plan for one kernel configuration.  An SM's time is (CTAs per SM) x (filters per CTA x time of one filter + a
// per-CTA constant), both from a model fitted on B200 (see below).  Try the fewest equal tiles that cover the phi region and a few more in each direction; when the tiles of
// the whole batch do not fill the GPU (small images), also try splitting the filter bank of a tile over nsplit CTAs --
// every split pays the per-CTA constant again.  Keep the cheapest.
template <int KS, int RW, int RH, int NT, int MINB>
Plan plan_tiles(const StageArgs& a, int num_sms)
{
    using C = Cfg<KS, RW, RH, NT, MINB>;
    constexpr int R = (KS - 1) / 2;
    const int Wz = a.W + 2 * R, Hz = a.H + 2 * R;
    Plan best{0, 0, 0, 0, 1, 0, -1.0, 0};
    // Time of one filter on one CTA with a tw x th tile, in microseconds, for the default (factorised) evaluator.  The CTA
    // works in rounds of NT blocks; a round in which w warps have phi work takes 2.85 + 0.105 w us (the instruction stream
    // of one block, ~1200 mostly dependent instructions, sets the floor; more warps only fill its gaps), a round with
    // transposed-filter work only 1.5 us, plus 1.0 us per filter that does not overlap (barrier, pipeline restart); a tile
    // of a single round runs 2.8 + 0.18 w.  A CTA costs filters x this + 6 to 17 us (tile gather, fill / drain, stores:
    // cta_const).  Fitted on one-wave launches of 12 x 12 tiles of 28 .. 122 pixels (B200, 48 and 24 filters 7x7); two
    // co-resident CTAs of 256 threads share the sub-partitions, hence the factor on w.
    auto per_filter = [&](int tw, int th) {
        const long long bphi = (long long)((tw + 3) / 4) * ((th + 1) / 2);
        const long long bout = (long long)((tw + 2 * R + 3) / 4) * ((th + 2 * R + 1) / 2);
        const double share = MINB * NT / 512.0;
        if (bout <= NT) return 2.8 + 0.18 * share * (double)((bphi + 31) / 32);
        double pf = 1.0;
        for (long long done = 0; done < bout; done += NT) {
            const long long inr = bphi - done < 0 ? 0 : (bphi - done > NT ? NT : bphi - done);
            const long long wr = (inr + 31) / 32;                      // warps with phi work in this round
            pf += wr > 0 ? 2.85 + 0.105 * share * (double)wr : 1.5;
        }
        return pf;
    };
    auto cta_const = [&](int tw, int th) {
        return 6.2 + (double)((tw + 2 * R + 3) / 4) * ((th + 2 * R + 1) / 2) / 190.0;
    };
    const int ntx0 = (Wz + C::TWMAX - 1) / C::TWMAX, nty0 = (Hz + C::THMAX - 1) / C::THMAX;
    const int fx = env_int("TNRD_NTX"), fy = env_int("TNRD_NTY");       // tuning knobs: force the tile counts
    for (int dx = 0; dx < 3; ++dx)
        for (int dy = 0; dy < 3; ++dy) {
            int ntx = ntx0 + dx, nty = nty0 + dy;
            if (fx >= ntx0 && fy >= nty0) { ntx = fx; nty = fy; }
            if (ntx > Wz || nty > Hz) continue;
            const int tw = (Wz + ntx - 1) / ntx, th = (Hz + nty - 1) / nty;
            if ((long long)(ntx - 1) * tw >= Wz || (long long)(nty - 1) * th >= Hz) continue;   // an empty last tile
            const long long bphi = (long long)((tw + 3) / 4) * ((th + 1) / 2);
            const double pf = per_filter(tw, th), cc = cta_const(tw, th);
            const long long tiles = (long long)ntx * nty * a.B;
            int smax = 1;
            if (tiles < (long long)num_sms * MINB) smax = a.N_k < 32 ? a.N_k : 32;
            int slo = 1;
            if (forced_split() > 0) slo = smax = forced_split() < a.N_k ? forced_split() : a.N_k;
            for (int sp = slo; sp <= smax; ++sp) {
                const int nf = (a.N_k + sp - 1) / sp;                      // filters of the largest chunk
                if (sp > slo && (a.N_k + sp - 2) / (sp - 1) == nf) continue; // same chunk as sp - 1: only more CTAs
                const long long ctas = tiles * sp;
                const double cost = (double)((ctas + num_sms - 1) / num_sms) * (pf * nf + cc);
                if (best.cost < 0 || cost < best.cost || (cost == best.cost && bphi < best.work))
                    best = Plan{ntx, nty, tw, th, sp, 0, cost, bphi};
            }
            if (!(MINB == 1 && smax == 1 && forced_split() <= 0 && tiles > num_sms)) continue;
            // large images: whole waves of one CTA per tile, and the tiles of the last, partly filled wave split over
            // sp CTAs each so that the tail costs a fraction of a wave (MINB = 1 only: one CTA per SM at a time)
            const long long full = tiles / num_sms * num_sms, rem = tiles - full;
            auto tail_of = [&](double pf_tile, int& sp_best) {
                double t = rem ? pf_tile * a.N_k + cc : 0.0;
                sp_best = 1;
                for (int sp = 2; rem && sp <= (a.N_k < 16 ? a.N_k : 16); ++sp) {
                    const double c = (double)((rem * sp + num_sms - 1) / num_sms) * (pf_tile * ((a.N_k + sp - 1) / sp) + cc);
                    if (c < t) { t = c; sp_best = sp; }
                }
                return t;
            };
            int sp_eq = 1;
            const double cost_eq = (double)(full / num_sms) * (pf * a.N_k + cc) + tail_of(pf, sp_eq);
            if (sp_eq > 1 && cost_eq < best.cost) best = Plan{ntx, nty, tw, th, sp_eq, full, cost_eq, bphi};
            // many waves: tiles of the LARGEST size with a ragged last row / column do the same phi work per CTA on more
            // pixels (a 122 x 122 tile costs what a 121 x 121 one does); CTAs then differ in length, which only many
            // waves average out -- cost = total work / SMs
            if (tiles >= 4LL * num_sms && fx < ntx0) {
                const int twm = C::TWMAX < Wz ? C::TWMAX : Wz, thm = C::THMAX < Hz ? C::THMAX : Hz;
                const int nx = (Wz + twm - 1) / twm, ny = (Hz + thm - 1) / thm;
                if (nx == ntx && ny == nty && (twm != tw || thm != th)) {
                    const int twr = Wz - (nx - 1) * twm, thr = Hz - (ny - 1) * thm;
                    const double c_ff = per_filter(twm, thm) * a.N_k + cta_const(twm, thm),
                                 c_rf = per_filter(twr, thm) * a.N_k + cta_const(twr, thm),
                                 c_fr = per_filter(twm, thr) * a.N_k + cta_const(twm, thr),
                                 c_rr = per_filter(twr, thr) * a.N_k + cta_const(twr, thr);
                    const double total = a.B * ((double)(nx - 1) * (ny - 1) * c_ff + (double)(ny - 1) * c_rf
                                                + (double)(nx - 1) * c_fr + c_rr);
                    int sp_rg = 1;
                    const double tail = tail_of(per_filter(twm, thr), sp_rg);      // the last tiles are bottom-row tiles
                    const double cost_rg = total * ((double)full / tiles) / num_sms + tail;
                    if (cost_rg < best.cost)
                        best = Plan{nx, ny, twm, thm, sp_rg > 1 ? sp_rg : 1, sp_rg > 1 ? full : 0, cost_rg, bphi};
                }
            }
        }
    return best;
}

template <int KS, int RW, int RH, int NT, int MINB, int PHI>
cudaError_t launch_cfg(const StageArgs& a, const FusedPlan& pl, float* part, cudaStream_t st)
{
    using C = Cfg<KS, RW, RH, NT, MINB>;
    // the opt-in is an attribute of the CURRENT device's copy of the kernel: set at every launch (cheap), so that a
    // process that uses several devices works on each of them
    cudaError_t e = cudaFuncSetAttribute(stage_fused_kernel<KS, RW, RH, NT, MINB, PHI>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM);
    if (e != cudaSuccess) return e;
    const long long tiles = (long long)pl.ntx * pl.nty * a.B;
    const long long grid = pl.n_full + (tiles - pl.n_full) * pl.nsplit;
    if (grid > 0x7fffffffLL || pl.n_full > tiles || !part) return cudaErrorInvalidConfiguration;
    stage_fused_kernel<KS, RW, RH, NT, MINB, PHI><<<(unsigned)grid, NT, C::SMEM, st>>>(
        a, pl.tw, pl.th, pl.ntx, pl.nty, (int)pl.n_full, pl.nsplit, part);
    return cudaGetLastError();
}

template <int KS>
FusedPlan plan_ks(const StageArgs& a, int num_sms)
{
    // 1: 128x128 output area, 512 threads, 1 CTA/SM; 2: 64x32, 256 threads, 2 CTAs/SM (small images);
    // 3: 64x64, 256 threads, 2 CTAs/SM.  Cheapest estimated plan wins; ties go to the shorter CTA.
    const Plan p[3] = {plan_tiles<KS, 128, 128, 512, 1>(a, num_sms), plan_tiles<KS, 64, 32, 256, 2>(a, num_sms),
                       plan_tiles<KS, 64, 64, 256, 2>(a, num_sms)};
    const int per_cta[3] = {Cfg<KS, 128, 128, 512, 1>::CTA_FLOATS, Cfg<KS, 64, 32, 256, 2>::CTA_FLOATS,
                            Cfg<KS, 64, 64, 256, 2>::CTA_FLOATS};
    int id = forced_tile();
    if (id < 1 || id > 3) {
        id = 1;
        if (p[2].cost < p[id - 1].cost || (p[2].cost == p[id - 1].cost && p[2].work < p[id - 1].work)) id = 3;
        if (p[1].cost < p[id - 1].cost || (p[1].cost == p[id - 1].cost && p[1].work < p[id - 1].work)) id = 2;
    }
    const Plan& b = p[id - 1];
    if (env_int("TNRD_DEBUG_PLAN"))
        fprintf(stderr, "tnrd plan: %dx%dx%d ks %d N_k %d -> cfg %d, %d x %d tiles of %d x %d, %lld whole + split %d, cost %.0f\n",
                a.B, a.H, a.W, KS, a.N_k, id, b.ntx, b.nty, b.tw, b.th, b.n_full, b.nsplit, b.cost);
    FusedPlan fp{id, b.ntx, b.nty, b.tw, b.th, b.nsplit, b.n_full, per_cta[id - 1], 0};
    const long long tiles = (long long)b.ntx * b.nty * a.B;
    fp.part_floats = (size_t)(b.n_full + (tiles - b.n_full) * b.nsplit) * per_cta[id - 1];
    return fp;
}

template <int KS, int PHI>
cudaError_t launch_ks(const StageArgs& a, const FusedPlan& pl, float* part, cudaStream_t st)
{
    switch (pl.cfg) {
        case 1: return launch_cfg<KS, 128, 128, 512, 1, PHI>(a, pl, part, st);
        case 2: return launch_cfg<KS, 64, 32, 256, 2, PHI>(a, pl, part, st);
        case 3: return launch_cfg<KS, 64, 64, 256, 2, PHI>(a, pl, part, st);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace

cudaError_t fused_init() { return cudaSuccess; }

FusedPlan plan_stage_fused(const StageArgs& a, int num_sms)
{
    switch (a.ksize) {
        case 3: return plan_ks<3>(a, num_sms);
        case 5: return plan_ks<5>(a, num_sms);
        case 7: return plan_ks<7>(a, num_sms);
        default: return plan_ks<9>(a, num_sms);
    }
}

template <int PHI>
cudaError_t launch_phi(const StageArgs& a, const FusedPlan& pl, float* part, cudaStream_t st)
{
    switch (a.ksize) {
        case 3: return launch_ks<3, PHI>(a, pl, part, st);
        case 5: return launch_ks<5, PHI>(a, pl, part, st);
        case 7: return launch_ks<7, PHI>(a, pl, part, st);
        case 9: return launch_ks<9, PHI>(a, pl, part, st);
        default: return cudaErrorInvalidValue;
    }
}

cudaError_t launch_stage_fused(const StageArgs& a_in, const FusedPlan& pl, float* part, int phi_mode, cudaStream_t st,
                               unsigned long long* launches)
{
    StageArgs a = a_in;
    a.dense_is_fallback = (phi_mode == 1);
    cudaError_t e;
    if (phi_mode == 3) {            // factorised dense evaluator (the kernel falls back to the direct form by itself)
        e = launch_phi<3>(a, pl, part, st);
        ++*launches;
    } else if (phi_mode == 2) {            // piecewise-linear table evaluator (always applicable)
        if (!a.tab || !a.tabhdr) return cudaErrorInvalidValue;
        e = launch_phi<2>(a, pl, part, st);
        ++*launches;
    } else {
        if (phi_mode == 1) {        // windowed evaluator; exits at once when the centres are not equidistant ...
            e = launch_phi<1>(a, pl, part, st);
            ++*launches;
            if (e != cudaSuccess) return e;
        }
        e = launch_phi<0>(a, pl, part, st);   // ... in which case this dense launch does the work (else it exits)
        ++*launches;
    }
    if (e != cudaSuccess) return e;
    const long long rows = (long long)a.B * a.H;
    const int rw = pl.cfg == 1 ? 128 : 64, R = (a.ksize - 1) / 2;
    const dim3 gy((unsigned)(rows < 65535 ? rows : 65535), (unsigned)((rows + 65534) / 65535));
    if (rows * a.W >= (1LL << 22))
        stage_update_kernel<4><<<dim3((unsigned)((a.W + 511) / 512), gy.x, gy.y), 128, 0, st>>>(
            a, part, pl.tw, pl.th, pl.ntx, pl.nty, (int)pl.n_full, pl.nsplit, pl.cta_floats, rw, R);
    else
        stage_update_kernel<1><<<dim3((unsigned)((a.W + 127) / 128), gy.x, gy.y), 128, 0, st>>>(
            a, part, pl.tw, pl.th, pl.ntx, pl.nty, (int)pl.n_full, pl.nsplit, pl.cta_floats, rw, R);
    ++*launches;
    return cudaGetLastError();
}

}  // namespace tnrd

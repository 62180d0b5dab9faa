// tnrd_small.cu -- the small-image path: ALL T stages of an image that fits a thread-block
// cluster in ONE launch, parameter staging included.
//
//   u_t = u_{t-1} - ( sum_i kbar_i * phi_i(k_i * u~_{t-1}) + lambda_t (u_{t-1} - f) ),  t = 1..T     Main Eq. 7
//   "5 stages are typically enough", jointly trained models must run all T
//
// A 64 x 64 image is 2 us of arithmetic per stage; launched stage by stage (staging kernel + T x (tile kernel + update
// kernel)) it costs 39 us per call, almost all of it launch latency and dependent DRAM / L2 round trips
// (profiles/r02_small_banks_ncu.md).  Here one cluster of 8 or 16 CTAs owns one image: CTA r owns a band of rows, every
// stage it
//   - derives the scaled taps and factorised-phi records from the caller's raw parameters in shared memory (what
//     prep_params_kernel does for the other kernels; of all T stages before the first one when they fit),
//   - gathers its band of u_{t-1} with a 2r halo through the mirror map from global memory / L2,
//   - computes responses and influence values of the band + r ring in registers, one warp per (filter, 128 pixels), four
//     pixels per thread with packed arithmetic (the evaluator of the tensor-core kernel), into one shared-memory map per
//     filter, then -- after ONE __syncthreads -- the transposed bank: a thread takes 4 output rows of one column and a
//     residue class of the filters (uniform tap loads, conflict-free map reads), the classes' partial sums meet in shared
//     memory and are added in a fixed order,
//   - writes its rows of u_t with the reaction term, and
//   - meets the other CTAs at a cluster barrier (release / acquire): their halo rows of u_t are then visible.
// The r rows above and below a band are recomputed (no partial sums in global memory).  Iterates alternate between `out`
// and one ping-pong plane.  No atomics; results are deterministic.
// Where the time of a 64 x 64, T = 2 call goes (clock64 trace, 16 CTAs): 28.3 k clocks = 14.4 us: first loads and the
// equidistance test 2.6 k, parameters 3.9 k (every CTA derives all of them), then per stage phi 5.7 k (FMA-pipe bound:
// half of a band's phi rows are the recomputed ring), transposed bank 2.0 k, update 1.0 k, cluster barrier 1.3 k, tile
// load 1.6 k.
#include <cooperative_groups.h>
#include <cstdio>

#include "tnrd_internal.h"
#include "tnrd_device.cuh"

namespace cg = cooperative_groups;

namespace tnrd {

namespace {

constexpr int SM_CS = 8;        // CTAs per cluster = row bands per image (16 for images of 32 rows and more)
constexpr int SM_NT = 1024;     // threads per CTA (64 registers each)
constexpr int SM_REC = TNRD_FG * TNRD_FSTRIDE;   // floats per filter: factorised records (or w' of the direct form)

struct SmallArgs {
    const float* f;
    const float* u0;
    float* out;
    float* pp;                  // ping-pong plane [B][H][W] (unused when T == 1)
    const float* filters;       // [T][N_k][ks][ks]
    const float* rbf_w;         // [T][N_k][63]
    const float* rbf_mu;        // [63]
    const float* lambda;        // [T] device, or null -> lambda_val (tnrd_stage)
    float lambda_val;
    float gamma;
    int B, H, W, T, N_k;
    int rpc;                    // rows per CTA
    int force_direct;           // phi mode 0
    int all_stages;             // 1: the parameters of all T stages are staged at once (they fit shared memory)
};

__device__ __forceinline__ float ex2a(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// Four responses per thread (two packed pairs): the form the tensor-core kernel uses (tc_phi_fact in tnrd_tc.cu) -- packed
// FMAs, the group range from per-lane integer bounds (olo = -(D + ganch) ginv, ohi = (D - ganch) ginv), four independent
// Horner chains per thread instead of one.  One warp item is then (filter, 128 pixels): a band of a 64 x 64 image is ONE
// item per warp, where single responses took four dependent rounds.
template <int NP>     // NP = 2: four responses; NP = 1: two (the last, nearly empty chunk of a band)
__device__ __forceinline__ void small_phi_fact4(const float* __restrict__ rec, float kappa, float olo, float ohi, float ginv,
                                                const float2 (&z)[NP], float2 (&v)[NP])
{
    constexpr int S = TNRD_FS, GC = TNRD_FG / 2;
    float zlo, zhi;
    asm("min.NaN.f32 %0, %1, %2;" : "=f"(zlo) : "f"(z[0].x), "f"(z[0].y));
    asm("max.NaN.f32 %0, %1, %2;" : "=f"(zhi) : "f"(z[0].x), "f"(z[0].y));
    if (NP == 2) {
        float t0, t1;
        asm("min.NaN.f32 %0, %1, %2;" : "=f"(t0) : "f"(z[NP - 1].x), "f"(z[NP - 1].y));
        asm("max.NaN.f32 %0, %1, %2;" : "=f"(t1) : "f"(z[NP - 1].x), "f"(z[NP - 1].y));
        asm("min.NaN.f32 %0, %1, %2;" : "=f"(zlo) : "f"(zlo), "f"(t0));
        asm("max.NaN.f32 %0, %1, %2;" : "=f"(zhi) : "f"(zhi), "f"(t1));
    }
    // clamped BEFORE the conversion (infinite responses must not overflow the + 1); NaN -> -8 resp. +8: every group live
    const float xl = fminf(fmaxf(fmaf(zlo, ginv, olo), -8.0f), 8.0f);
    const float xh = fmaxf(fminf(fmaf(zhi, ginv, ohi), 8.0f), -8.0f);
    const int g0 = max(0, __reduce_min_sync(0xffffffffu, __float2int_rd(xl)) + 1);
    const int g1 = min(TNRD_FG - 1, __reduce_max_sync(0xffffffffu, __float2int_ru(xh)) - 1);
    if (g0 > g1) return;
    float2 rho0[NP], rhoi0[NP];
    {
        const float c0 = rec[GC * TNRD_FSTRIDE];
#pragma unroll
        for (int p = 0; p < NP; ++p) {
            const float2 e = __fmul2_rn(__fadd2_rn(z[p], make_float2(c0, c0)), make_float2(kappa, kappa));
            rho0[p] = make_float2(ex2a(e.x), ex2a(e.y));
            rhoi0[p] = make_float2(ex2a(-e.x), ex2a(-e.y));
        }
    }
#pragma unroll 1
    for (int g = g0; g <= g1; ++g) {
        float c[TNRD_FSTRIDE];
        lds_vec(rec + g * TNRD_FSTRIDE, c);
        float2 gg[NP], rho[NP], rhoi[NP], h[NP], hl[NP];
#pragma unroll
        for (int p = 0; p < NP; ++p) {
            const float2 d = __fadd2_rn(z[p], make_float2(c[0], c[0]));
            const float2 t = __fmul2_rn(d, d);
            gg[p] = make_float2(ex2a(-t.x), ex2a(-t.y));
            rho[p] = make_float2(__saturatef(rho0[p].x * c[14]), __saturatef(rho0[p].y * c[14]));
            rhoi[p] = make_float2(__saturatef(rhoi0[p].x * c[15]), __saturatef(rhoi0[p].y * c[15]));
            h[p] = __ffma2_rn(make_float2(c[1], c[1]), rho[p], make_float2(c[2], c[2]));
            hl[p] = __ffma2_rn(make_float2(c[S + 2], c[S + 2]), rhoi[p], make_float2(c[S + 3], c[S + 3]));
        }
#pragma unroll
        for (int q = 2; q <= S; ++q)
#pragma unroll
            for (int p = 0; p < NP; ++p) h[p] = __ffma2_rn(h[p], rho[p], make_float2(c[1 + q], c[1 + q]));
#pragma unroll
        for (int q = 2; q < S; ++q)
#pragma unroll
            for (int p = 0; p < NP; ++p) hl[p] = __ffma2_rn(hl[p], rhoi[p], make_float2(c[S + 2 + q], c[S + 2 + q]));
#pragma unroll
        for (int p = 0; p < NP; ++p) {
            h[p] = make_float2(fmaf(hl[p].x, rhoi[p].x, h[p].x), fmaf(hl[p].y, rhoi[p].y, h[p].y));
            v[p] = make_float2(fmaf(gg[p].x, h[p].x, v[p].x), fmaf(gg[p].y, h[p].y, v[p].y));
        }
    }
}

// direct form, four responses: w' of the filter in rec[0..62], -mu' in mun[0..62]
template <int N>
__device__ __forceinline__ void small_phi_direct4(const float* __restrict__ rec, const float* __restrict__ mun,
                                                  const float (&z)[N], float (&v)[N])
{
#pragma unroll
    for (int k = 0; k < N; ++k) v[k] = 0.0f;
#pragma unroll 3
    for (int j = 0; j < TNRD_M; ++j) {
        const float m = mun[j], w = rec[j];
#pragma unroll
        for (int k = 0; k < N; ++k) {
            const float d = z[k] + m;
            v[k] = fmaf(ex2a(-d * d), w, v[k]);
        }
    }
}

// a2 + a3 for N (4 or 2) pixels p0 + 32 j of one filter: responses by the true convolution k[a][b] u[y + r - a][x + r - b]
// (PAPER.md:70), influence values by the factorised or the direct form, stored to the filter's map.  A pixel index beyond
// the band is clamped to the band's last pixel (computed, not stored), so it never widens the warp's response range.
template <int KS, int N>
__device__ __forceinline__ void small_item(const float* __restrict__ tp, const float* __restrict__ us, const int* __restrict__ poff,
                                           int p0, int npx_phi, int UW, bool fact, const float* __restrict__ rec,
                                           const float* __restrict__ mun, float kappa, float olo, float ohi, float ginv,
                                           float* __restrict__ vmap)
{
    const float* uw[N];
#pragma unroll
    for (int j = 0; j < N; ++j) uw[j] = us + poff[min(p0 + 32 * j, npx_phi - 1)];   // window of phi pixel p
    float zz[N];
#pragma unroll
    for (int j = 0; j < N; ++j) zz[j] = 0.0f;
#pragma unroll
    for (int ka = 0; ka < KS; ++ka)
#pragma unroll
        for (int kb = 0; kb < KS; ++kb) {
            const float tap = tp[ka * KS + kb];
#pragma unroll
            for (int j = 0; j < N; ++j) zz[j] = fmaf(tap, uw[j][(KS - 1 - ka) * UW + (KS - 1 - kb)], zz[j]);
        }
    float vv[N];
    if (fact) {
        float2 z2[N / 2], v2[N / 2];
#pragma unroll
        for (int p = 0; p < N / 2; ++p) { z2[p] = make_float2(zz[2 * p], zz[2 * p + 1]); v2[p] = make_float2(0.0f, 0.0f); }
        small_phi_fact4<N / 2>(rec, kappa, olo, ohi, ginv, z2, v2);
#pragma unroll
        for (int p = 0; p < N / 2; ++p) { vv[2 * p] = v2[p].x; vv[2 * p + 1] = v2[p].y; }
    } else {
        small_phi_direct4<N>(rec, mun, zz, vv);
    }
#pragma unroll
    for (int j = 0; j < N; ++j)
        if (p0 + 32 * j < npx_phi) vmap[p0 + 32 * j] = vv[j];
}

// a4: the filters are summed in `parts` residue classes by different threads (more threads busy on a small band); as many
// as one pass of the CTA's threads over (part, group of 4 rows, 32-column block) allows, and 16 KB of partial sums
__host__ __device__ inline int small_parts(int N_k, int rpc, int W)
{
    const int per_part = ((rpc + 3) / 4) * ((W + 31) & ~31);
    int n = N_k < 8 ? N_k : 8;
    while (n > 1 && (n * per_part > SM_NT || n * rpc * W > 4096)) --n;
    return n;
}

template <int KS>
__global__ void __launch_bounds__(SM_NT, 1) small_diffuse_kernel(SmallArgs a)
{
    constexpr int R = (KS - 1) / 2, KK = KS * KS;
    extern __shared__ __align__(16) float sm[];
    cg::cluster_group cluster = cg::this_cluster();
    const int rank = (int)cluster.block_rank(), img = blockIdx.y, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int H = a.H, W = a.W;
    const int row0 = min(H, rank * a.rpc), row1 = min(H, row0 + a.rpc), nrow = row1 - row0;       // this CTA's band
    const int UW = W + 4 * R, UH = a.rpc + 4 * R;          // u tile (origin: image (row0 - 2r, -2r))
    const int VW = W + 2 * R, VH = a.rpc + 2 * R;          // influence maps (origin: image (row0 - r, -r))
    float* us = sm;                                        // [UH][UW]
    float* vs = us + ((UH * UW + 3) & ~3);                 // [N_k][vplane]
    const int vplane = (VH * VW + 3) & ~3;
    const int tstride = (a.N_k * KK + 3) & ~3;             // floats of one stage's taps
    const int nst = a.all_stages ? a.T : 1;                // parameter sets resident at once
    float* taps = vs + (size_t)a.N_k * vplane;             // [nst][N_k][KK] scaled taps k' = s k
    float* recs = taps + (size_t)nst * tstride;            // [nst][N_k][SM_REC]
    float* mun = recs + (size_t)nst * a.N_k * SM_REC;      // [64] -mu'_j (direct form)
    int* poff = reinterpret_cast<int*>(mun + 64);          // [VH * VW] offset of an influence pixel's window in the u tile
    float* psum = reinterpret_cast<float*>(poff + ((VH * VW + 3) & ~3));   // [parts][rows of the band][W] partial sums of a4
    __shared__ int s_okf;

    // Programmatic dependent launch: let the next kernel of the stream (typically the next call of this one) be
    // scheduled now -- it waits below, like this one, before it touches global memory -- so that its launch latency and
    // cluster set-up overlap this kernel's run instead of following it.  The wait returns once the previous kernel of
    // the stream has completed and its writes are visible: stream order is kept.
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");

    // ---- loads nothing depends on yet, issued before the first barrier (one L2 round trip instead of three in a row):
    // f of this thread's output pixel (the same in every stage) and this thread's first element of the u_0 tile
    const size_t plane = (size_t)H * W;
    const float* f_img = a.f + (size_t)img * plane;
    const int npx_out = nrow * W;
    const int Wp = (W + 31) & ~31;                         // a4: a warp's lanes are 32 columns of one (part, row group)
    const int nsp = small_parts(a.N_k, a.rpc, W);          // a4: parts (residue classes of the filters) summed separately
    const bool one_iter = npx_out <= SM_NT;                // a5: every thread has at most one output pixel
    float f_pre = 0.0f, u_pre = 0.0f;
    if (one_iter && tid < npx_out) f_pre = __ldg(f_img + (size_t)row0 * W + tid);
    if (nrow > 0 && tid < (nrow + 4 * R) * UW) {
        const int uy = tid / UW, ux = tid - uy * UW;
        u_pre = __ldcg(a.u0 + (size_t)img * plane + (size_t)mirror_clamp(row0 - 2 * R + uy, H) * W + mirror_clamp(ux - 2 * R, W));
    }
    const float s = sqrtf(1.4426950408889634f / (2.0f * a.gamma * a.gamma));
    const float mu0 = __ldg(a.rbf_mu), delta = (__ldg(a.rbf_mu + TNRD_M - 1) - mu0) / (float)(TNRD_M - 1);
    const float ds = s * delta, kappa = 2.0f * ds, dmax = TNRD_FCLAMP;
    // the factorisation applies to centres that are equidistant to rounding and widths in its range (same rule as
    // prep_params_kernel); otherwise the direct form
    if (tid < 32) {
        // both centres of this lane loaded before anything is tested: one round trip together with mu0 and mu62 above
        const int j1 = min(tid + 32, TNRD_M - 1);
        const float m0 = __ldg(a.rbf_mu + tid), m1 = __ldg(a.rbf_mu + j1);
        const float tol = 1.5e-7f * (fabsf(mu0) + 62.0f * delta);
        bool ok = delta > 0.0f && !a.force_direct;
        ok = ok && fabsf(m0 - fmaf((float)tid, delta, mu0)) <= tol && fabsf(m1 - fmaf((float)j1, delta, mu0)) <= tol;
        const float reach = dmax - (float)TNRD_FS * ds;
        float emax = 0.0f;
        for (int j = 1; j <= TNRD_FS; ++j) emax = fmaxf(emax, (float)j * kappa * dmax - (float)(j * j) * ds * ds);
        ok = ok && reach > 0.0f && reach * reach >= 30.0f && emax <= 92.0f;
        ok = __all_sync(0xffffffffu, ok);
        if (tid == 0) s_okf = ok ? 1 : 0;
    }
    if (tid < 64) mun[tid] = tid < TNRD_M ? -s * __ldg(a.rbf_mu + tid) : 0.0f;
    for (int p = tid; p < VH * VW; p += SM_NT) poff[p] = (p / VW) * UW + (p % VW);
    __syncthreads();
    const bool fact = s_okf != 0;
    const float ganch = s * mu0 + (float)TNRD_FS * ds, ginv = 1.0f / ((float)TNRD_FM * ds);
    const float lR = kappa * dmax;                         // log2 of the cap R of rho
    const float olo = -(dmax + ganch) * ginv, ohi = (dmax - ganch) * ginv;     // small_phi_fact4: group range of a response

    const int npx_phi = (nrow > 0 ? (nrow + 2 * R) : 0) * VW;      // influence values of this band, per filter
    const int nchunk = (npx_phi + 127) >> 7;                       // ... in chunks of 128 (four per thread)
    for (int t = 1; t <= a.T; ++t) {
        const float* src = (t == 1) ? a.u0 : (((a.T - t + 1) & 1) ? a.pp : a.out);
        float* dst = ((a.T - t) & 1) ? a.pp : a.out;
        src += (size_t)img * plane;
        dst += (size_t)img * plane;
        // ---- a1: the band of u_{t-1} with its 2r halo, through the mirror map (issued first: the longest latency) ----
        if (nrow > 0)
            for (int i = tid; i < (nrow + 4 * R) * UW; i += SM_NT) {
                const int uy = i / UW, ux = i - uy * UW;
                us[i] = (t == 1 && i == tid) ? u_pre
                                             : __ldcg(src + (size_t)mirror_clamp(row0 - 2 * R + uy, H) * W + mirror_clamp(ux - 2 * R, W));
            }
        // ---- parameters: of every stage before the first one when they fit shared memory, else of stage t ----
        if (t == 1 || !a.all_stages) {
            // one flat index over (stage, filter, entry): the loads of all resident stages are in flight together
            const int ts0 = a.all_stages ? 0 : t - 1, nts = a.all_stages ? a.T : 1;
            const int ntap = a.N_k * KK, nrec = a.N_k * SM_REC;
            const float* kt = a.filters + (size_t)ts0 * ntap;
            const float* wt = a.rbf_w + (size_t)ts0 * a.N_k * TNRD_M;
            const float tap0 = tid < nts * ntap ? __ldg(kt + tid) : 0.0f;          // used after the records below
            // two entries per thread and pass, both loads issued before either value is finished (a band of a 64 x 64
            // image has 1280 entries for two stages: one round trip instead of two)
            for (int i0 = tid; i0 < nts * nrec; i0 += 2 * SM_NT) {
                float wv[2] = {0.0f, 0.0f}, scale[2] = {0.0f, 0.0f}, val[2] = {0.0f, 0.0f};
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const int i = i0 + e * SM_NT;
                    if (i >= nts * nrec) continue;
                    const int ts = i / nrec, ir = i - ts * nrec, fi = ir / SM_REC, o = ir - fi * SM_REC;
                    const float* wf = wt + ((size_t)ts * a.N_k + fi) * TNRD_M;
                    if (!fact) {
                        if (o < TNRD_M) { wv[e] = __ldg(wf + o); scale[e] = 1.0f; }
                    } else {
                        const int g = o / TNRD_FSTRIDE, q = o - g * TNRD_FSTRIDE, anchor = g * TNRD_FM + TNRD_FS;
                        if (q == 0) val[e] = -s * (mu0 + (float)anchor * delta);
                        else if (q <= TNRD_FM) {
                            const int j = q <= TNRD_FS + 1 ? TNRD_FS + 1 - q : q - 2 * TNRD_FS - 2;     // S .. 0, then -S .. -1
                            const int c = anchor + j;
                            if (c >= 0 && c < TNRD_M) {
                                wv[e] = __ldg(wf + c);
                                scale[e] = exp2f(-(float)(j * j) * ds * ds + (float)abs(j) * lR);
                            }
                        } else if (q >= TNRD_FSTRIDE - 2) {
                            const int mid = (TNRD_FG / 2) * TNRD_FM + TNRD_FS;
                            const float ex = -2.0f * ds * ds * (float)(anchor - mid);
                            val[e] = exp2f((q == TNRD_FSTRIDE - 2 ? ex : -ex) - lR);
                        }
                    }
                }
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const int i = i0 + e * SM_NT;
                    if (i >= nts * nrec) continue;
                    const int ts = i / nrec, ir = i - ts * nrec;
                    recs[(size_t)ts * nrec + ir] = scale[e] != 0.0f ? wv[e] / s * scale[e] : val[e];
                }
            }
            for (int i = tid; i < nts * ntap; i += SM_NT) {
                const int ts = i / ntap;
                taps[(size_t)ts * tstride + (i - ts * ntap)] = s * (i == tid ? tap0 : __ldg(kt + i));
            }
        }
        const float* taps_t = taps + (size_t)(a.all_stages ? t - 1 : 0) * tstride;
        const float* recs_t = recs + (size_t)(a.all_stages ? t - 1 : 0) * a.N_k * SM_REC;
        __syncthreads();
        // ---- a2 + a3: every (filter, chunk of 128 influence pixels) is one warp's item, four pixels per thread
        // (p0 + 32 j): responses and influence values in registers, written to the filter's map.  No synchronisation
        // between filters.  A pixel index beyond the band is clamped to the band's last pixel (computed, not stored), so
        // it never widens the warp's response range.
        for (int it = warp; it < a.N_k * nchunk; it += SM_NT / 32) {
            const int i = it / nchunk, c0 = (it - i * nchunk) * 128, p0 = c0 + lane;
            float* vmap = vs + (size_t)i * vplane;
            if (c0 + 64 < npx_phi)      // warp-uniform: the last chunk of a band may need its first two pixels per thread only
                small_item<KS, 4>(taps_t + i * KK, us, poff, p0, npx_phi, UW, fact, recs_t + i * SM_REC, mun, kappa, olo, ohi, ginv, vmap);
            else
                small_item<KS, 2>(taps_t + i * KK, us, poff, p0, npx_phi, UW, fact, recs_t + i * SM_REC, mun, kappa, olo, ohi, ginv, vmap);
        }
        __syncthreads();
        // ---- a4: the transposed bank.  One thread takes (part, group of 4 output rows, column) and sums the filters of its
        // part (a residue class of the filters) into four accumulators: the lanes of a warp are 32 neighbouring columns of
        // ONE filter at a time, so the taps are uniform loads and the influence values consecutive words (no bank conflicts;
        // the rows shared by neighbouring output rows are loaded once).  Partial sums go to shared memory ----
        const float lambda = a.lambda ? __ldg(a.lambda + (t - 1)) : a.lambda_val;
        const int nrg = (nrow + 3) >> 2;
        for (int item = tid; item < nsp * nrg * Wp; item += SM_NT) {
            const int part = item / (nrg * Wp), rem = item - part * (nrg * Wp), rg = rem / Wp, x = rem - rg * Wp;
            if (x >= W) continue;
            float acc[4] = {0.0f, 0.0f, 0.0f, 0.0f};
            for (int i = part; i < a.N_k; i += nsp) {
                const float* tp = taps_t + i * KK;
                const float* vw = vs + (size_t)i * vplane + (4 * rg) * VW + x;      // phi pixel (4 rg + r + a, x + b)
#pragma unroll
                for (int rr = 0; rr < KS + 3; ++rr) {               // phi row rr of the group feeds output rows rr - ka
                    if (4 * rg + rr >= nrow + 2 * R) break;
                    float vv[KS];
#pragma unroll
                    for (int kb = 0; kb < KS; ++kb) vv[kb] = vw[rr * VW + kb];
#pragma unroll
                    for (int r = 0; r < 4; ++r) {
                        const int ka = rr - r;
                        if (ka >= 0 && ka < KS) {
#pragma unroll
                            for (int kb = 0; kb < KS; ++kb) acc[r] = fmaf(tp[ka * KS + kb], vv[kb], acc[r]);
                        }
                    }
                }
            }
#pragma unroll
            for (int r = 0; r < 4; ++r)
                if (4 * rg + r < nrow) psum[(size_t)part * npx_out + (4 * rg + r) * W + x] = acc[r];
        }
        __syncthreads();
        // ---- a5: the parts added in a fixed order, reaction term, update of this band ----
        for (int q = tid; q < npx_out; q += SM_NT) {
            const int oy = q / W, ox = q - oy * W;                   // output pixel = image (row0 + oy, ox)
            float sacc = psum[q];
            for (int part = 1; part < nsp; ++part) sacc += psum[(size_t)part * npx_out + q];
            const float uu = us[(oy + 2 * R) * UW + ox + 2 * R];
            const float ff = one_iter ? f_pre : __ldg(f_img + (size_t)(row0 + oy) * W + ox);
            __stcg(dst + (size_t)(row0 + oy) * W + ox, uu - (sacc + lambda * (uu - ff)));
        }
        // every CTA's rows of u_t are visible to the whole cluster after this barrier (release / acquire); it also
        // orders this stage's shared-memory reads before the next stage's parameter and tile writes
        cluster.sync();
    }
}

// nst = parameter sets resident at once (T, or 1)
size_t small_smem_bytes(int W, int N_k, int ksize, int rpc, int nst)
{
    const int R = (ksize - 1) / 2, KK = ksize * ksize;
    const size_t us = ((size_t)(rpc + 4 * R) * (W + 4 * R) + 3) & ~(size_t)3;
    const size_t vpx = (size_t)(rpc + 2 * R) * (W + 2 * R), vp = (vpx + 3) & ~(size_t)3;
    const size_t psum = (size_t)small_parts(N_k, rpc, W) * rpc * W;
    return sizeof(float) * (us + (size_t)N_k * vp + (size_t)nst * ((((size_t)N_k * KK + 3) & ~(size_t)3) + (size_t)N_k * SM_REC)
                            + 64 + ((vpx + 3) & ~(size_t)3) + psum);
}

template <int KS>
cudaError_t launch_small_ks(const SmallArgs& a, int cs, size_t smem, cudaStream_t st)
{
    cudaError_t e = cudaFuncSetAttribute(small_diffuse_kernel<KS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    if (cs > 8) {
        e = cudaFuncSetAttribute(small_diffuse_kernel<KS>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
        if (e != cudaSuccess) return e;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)cs, (unsigned)a.B, 1);
    cfg.blockDim = dim3(SM_NT, 1, 1);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[2];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)cs;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;     // see griddepcontrol in the kernel
    attr[1].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 2;
    return cudaLaunchKernelEx(&cfg, small_diffuse_kernel<KS>, a);
}

// cluster size: 16 CTAs (the non-portable maximum) when the image has rows for them, else 8
int small_cluster(int H) { return H >= 32 ? 16 : SM_CS; }

}  // namespace

// The small-image kernel takes images whose row bands fit one CTA each (the u tile and all N_k influence maps of a band
// within 200 KB of shared memory), at most 65535 images, and little enough work that one cluster per image is the right
// granularity.
bool small_supported(int B, int H, int W, int N_k, int ksize)
{
    if (B > 65535 || (long long)B * H * W > 32768) return false;
    const int cs = small_cluster(H), rpc = (H + cs - 1) / cs;
    return small_smem_bytes(W, N_k, ksize, rpc, 1) <= 200 * 1024;
}

cudaError_t launch_small_diffuse(const float* f, const float* u0, float* out, float* pp, const float* filters,
                                 const float* rbf_w, const float* rbf_mu, float gamma, const float* lambda, float lambda_val,
                                 int B, int H, int W, int T, int N_k, int ksize, int force_direct, cudaStream_t st,
                                 unsigned long long* launches)
{
    const int cs = small_cluster(H);
    SmallArgs a{f, u0, out, pp, filters, rbf_w, rbf_mu, lambda, lambda_val, gamma, B, H, W, T, N_k, (H + cs - 1) / cs,
                force_direct, 0};
    a.all_stages = small_smem_bytes(W, N_k, ksize, a.rpc, T) <= 96 * 1024 ? 1 : 0;
    const size_t smem = small_smem_bytes(W, N_k, ksize, a.rpc, a.all_stages ? T : 1);
    cudaError_t e;
    switch (ksize) {
        case 3: e = launch_small_ks<3>(a, cs, smem, st); break;
        case 5: e = launch_small_ks<5>(a, cs, smem, st); break;
        case 7: e = launch_small_ks<7>(a, cs, smem, st); break;
        case 9: e = launch_small_ks<9>(a, cs, smem, st); break;
        default: return cudaErrorInvalidValue;
    }
    ++*launches;
    return e;
}

}  // namespace tnrd

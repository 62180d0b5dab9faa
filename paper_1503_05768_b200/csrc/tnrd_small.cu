// tnrd_small.cu -- the small-image path: ALL T stages of an image that fits a thread-block
// cluster in ONE launch, parameter staging included.
//
//   u_t = u_{t-1} - ( sum_i kbar_i * phi_i(k_i * u~_{t-1}) + lambda_t (u_{t-1} - f) ),  t = 1..T     Main Eq. 7
//   "5 stages are typically enough", jointly trained models must run all T
//
// A 64 x 64 image is 2 us of arithmetic per stage; launched stage by stage (staging kernel + T x (tile kernel + update
// kernel)) it costs 39 us per call, almost all of it launch latency and dependent DRAM / L2 round trips
// (profiles/r02_small_banks_ncu.md).  Here one cluster of 8 CTAs owns one image: CTA r owns a band of rows, every
// stage it
//   - derives the stage's scaled taps and factorised-phi records from the caller's raw parameters in shared memory
//     (what prep_params_kernel does for the other kernels),
//   - gathers its band of u_{t-1} with a 2r halo through the mirror map from global memory / L2,
//   - computes responses and influence values of the band + r ring in registers, one warp per (filter, 32 pixels),
//     into one shared-memory map per filter, then -- after ONE __syncthreads -- the transposed bank summed over all
//     filters per output pixel (split over up to 8 lanes per pixel, folded by shuffles in a fixed order),
//   - writes its rows of u_t with the reaction term, and
//   - meets the other CTAs at a cluster barrier (release / acquire): their halo rows of u_t are then visible.
// The r rows above and below a band are recomputed (no partial sums).  Iterates alternate between `out` and one
// ping-pong plane.  No atomics; results are deterministic.
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

// order-preserving float <-> uint32 map (warp-wide min / max by redux.sync)
__device__ __forceinline__ unsigned s_f2ord(float x)
{
    const unsigned b = __float_as_uint(x);
    return b ^ ((unsigned)((int)b >> 31) | 0x80000000u);
}
__device__ __forceinline__ float s_ord2f(unsigned o) { return __uint_as_float(o ^ (((o >> 31) - 1u) | 0x80000000u)); }

// One response through the factorised influence function (tnrd_internal.h "fact"; the scalar twin of tc_phi_fact in
// tnrd_tc.cu): rec = TNRD_FG group records with the coefficients scaled by R^|j| and K_g, 1/K_g by 1/R, R = 2^{kappa D}.
// Groups out of reach of every response of the warp are skipped (exact zeros).  `active` = this lane has a response.
__device__ __forceinline__ float small_phi_fact(const float* __restrict__ rec, float kappa, float dmax, float ganch, float ginv,
                                                float z, bool active)
{
    constexpr int S = TNRD_FS, GC = TNRD_FG / 2;
    const float zl = active ? z : __int_as_float(0x7f800000), zh = active ? z : __int_as_float(0xff800000);
    const float wlo = s_ord2f(__reduce_min_sync(0xffffffffu, s_f2ord(zl)));
    const float whi = s_ord2f(__reduce_max_sync(0xffffffffu, s_f2ord(zh)));
    int g0 = 0, g1 = TNRD_FG - 1;
    if (!__any_sync(0xffffffffu, active && z != z)) {
        // clamped BEFORE the conversion: an infinite range (no active lane, infinite responses) must not overflow the + 1
        g0 = max(0, __float2int_rd(fminf(fmaxf((wlo - dmax - ganch) * ginv, -8.0f), 8.0f)) + 1);
        g1 = min(TNRD_FG - 1, __float2int_ru(fminf(fmaxf((whi + dmax - ganch) * ginv, -8.0f), 8.0f)) - 1);
    }
    const float e0 = (z + rec[GC * TNRD_FSTRIDE]) * kappa;
    const float rho0 = ex2a(e0), rhoi0 = ex2a(-e0);
    float v = 0.0f;
#pragma unroll 1
    for (int g = g0; g <= g1; ++g) {
        float c[TNRD_FSTRIDE];
        lds_vec(rec + g * TNRD_FSTRIDE, c);
        const float d = z + c[0];
        const float gg = ex2a(-d * d);
        const float x = __saturatef(rho0 * c[14]), xi = __saturatef(rhoi0 * c[15]);
        float h = fmaf(c[1], x, c[2]), hl = fmaf(c[S + 2], xi, c[S + 3]);
#pragma unroll
        for (int q = 2; q <= S; ++q) h = fmaf(h, x, c[1 + q]);
#pragma unroll
        for (int q = 2; q < S; ++q) hl = fmaf(hl, xi, c[S + 2 + q]);
        h = fmaf(hl, xi, h);
        v = fmaf(gg, h, v);
    }
    return v;
}

// direct form: w' of the filter in rec[0..62], -mu' in mun[0..62]
__device__ __forceinline__ float small_phi_direct(const float* __restrict__ rec, const float* __restrict__ mun, float z)
{
    float v = 0.0f;
#pragma unroll 7
    for (int j = 0; j < TNRD_M; ++j) {
        const float d = z + mun[j];
        v = fmaf(ex2a(-d * d), rec[j], v);
    }
    return v;
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
    __shared__ int s_okf;

    const float s = sqrtf(1.4426950408889634f / (2.0f * a.gamma * a.gamma));
    const float mu0 = __ldg(a.rbf_mu), delta = (__ldg(a.rbf_mu + TNRD_M - 1) - mu0) / (float)(TNRD_M - 1);
    const float ds = s * delta, kappa = 2.0f * ds, dmax = TNRD_FCLAMP;
    // the factorisation applies to centres that are equidistant to rounding and widths in its range (same rule as
    // prep_params_kernel); otherwise the direct form
    if (tid < 32) {
        bool ok = delta > 0.0f && !a.force_direct;
        for (int j = tid; j < TNRD_M; j += 32)
            ok = ok && fabsf(__ldg(a.rbf_mu + j) - fmaf((float)j, delta, mu0)) <= 1.5e-7f * (fabsf(mu0) + 62.0f * delta);
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

    const size_t plane = (size_t)H * W;
    const float* f_img = a.f + (size_t)img * plane;
    const int npx_phi = (nrow > 0 ? (nrow + 2 * R) : 0) * VW;      // influence values of this band, per filter
    const int nchunk = (npx_phi + 31) >> 5;                        // ... in warp-sized chunks
    const int npx_out = nrow * W;
    // a4 is split over `nsplit` lanes per output pixel (each a residue class of the filters), folded by xor-shuffles
    int nsplit = 1;
    while (nsplit < 8 && 2 * nsplit <= a.N_k && npx_out * 2 * nsplit <= SM_NT) nsplit *= 2;

    for (int t = 1; t <= a.T; ++t) {
        const float* src = (t == 1) ? a.u0 : (((a.T - t + 1) & 1) ? a.pp : a.out);
        float* dst = ((a.T - t) & 1) ? a.pp : a.out;
        src += (size_t)img * plane;
        dst += (size_t)img * plane;
        // ---- a1: the band of u_{t-1} with its 2r halo, through the mirror map (issued first: the longest latency) ----
        if (nrow > 0)
            for (int i = tid; i < (nrow + 4 * R) * UW; i += SM_NT) {
                const int uy = i / UW, ux = i - uy * UW;
                us[i] = __ldcg(src + (size_t)mirror_clamp(row0 - 2 * R + uy, H) * W + mirror_clamp(ux - 2 * R, W));
            }
        // ---- parameters: of every stage before the first one when they fit shared memory, else of stage t ----
        if (t == 1 || !a.all_stages)
            for (int ts = (a.all_stages ? 0 : t - 1); ts < (a.all_stages ? a.T : t); ++ts) {
                const float* kt = a.filters + (size_t)ts * a.N_k * KK;
                const float* wt = a.rbf_w + (size_t)ts * a.N_k * TNRD_M;
                float* tdst = taps + (size_t)(a.all_stages ? ts : 0) * tstride;
                float* rdst = recs + (size_t)(a.all_stages ? ts : 0) * a.N_k * SM_REC;
                for (int i = tid; i < a.N_k * KK; i += SM_NT) tdst[i] = s * __ldg(kt + i);
                for (int i = tid; i < a.N_k * SM_REC; i += SM_NT) {
                    const int fi = i / SM_REC, o = i - fi * SM_REC;
                    float val = 0.0f;
                    if (!fact) {
                        if (o < TNRD_M) val = __ldg(wt + fi * TNRD_M + o) / s;
                    } else {
                        const int g = o / TNRD_FSTRIDE, q = o - g * TNRD_FSTRIDE, anchor = g * TNRD_FM + TNRD_FS;
                        if (q == 0) val = -s * (mu0 + (float)anchor * delta);
                        else if (q <= TNRD_FM) {
                            const int j = q <= TNRD_FS + 1 ? TNRD_FS + 1 - q : q - 2 * TNRD_FS - 2;     // S .. 0, then -S .. -1
                            const int c = anchor + j;
                            if (c >= 0 && c < TNRD_M)
                                val = __ldg(wt + fi * TNRD_M + c) / s * exp2f(-(float)(j * j) * ds * ds + (float)abs(j) * lR);
                        } else if (q >= TNRD_FSTRIDE - 2) {
                            const int mid = (TNRD_FG / 2) * TNRD_FM + TNRD_FS;
                            const float ex = -2.0f * ds * ds * (float)(anchor - mid);
                            val = exp2f((q == TNRD_FSTRIDE - 2 ? ex : -ex) - lR);
                        }
                    }
                    rdst[i] = val;
                }
            }
        const float* taps_t = taps + (size_t)(a.all_stages ? t - 1 : 0) * tstride;
        const float* recs_t = recs + (size_t)(a.all_stages ? t - 1 : 0) * a.N_k * SM_REC;
        __syncthreads();
        // ---- a2 + a3: every (filter, chunk of 32 influence pixels) is one warp's item: responses and influence values
        // in registers, written to the filter's map.  No synchronisation between filters.
        for (int it = warp; it < a.N_k * nchunk; it += SM_NT / 32) {
            const int i = it / nchunk, p = (it - i * nchunk) * 32 + lane;
            const bool active = p < npx_phi;
            const float* tp = taps_t + i * KK;
            float z = 0.0f;
            if (active) {
                const float* uw = us + poff[p];                    // window of phi pixel p = image (row0 - r + p / VW, p % VW - r)
#pragma unroll
                for (int ka = 0; ka < KS; ++ka)
#pragma unroll
                    for (int kb = 0; kb < KS; ++kb)                // true convolution: k[a][b] u[y + r - a][x + r - b]
                        z = fmaf(tp[ka * KS + kb], uw[(KS - 1 - ka) * UW + (KS - 1 - kb)], z);
            }
            float v;
            if (fact) v = small_phi_fact(recs_t + i * SM_REC, kappa, dmax, ganch, ginv, z, active);
            else v = small_phi_direct(recs_t + i * SM_REC, mun, z);
            if (active) vs[(size_t)i * vplane + p] = v;
        }
        __syncthreads();
        // ---- a4 + a5: transposed bank summed over the filters, reaction term, update of this band ----
        const float lambda = a.lambda ? __ldg(a.lambda + (t - 1)) : a.lambda_val;
        const int per_iter = SM_NT / nsplit;
        for (int q0 = 0; q0 < npx_out; q0 += per_iter) {           // whole warps iterate together (shuffles below)
            const int q = q0 + tid / nsplit, part = tid % nsplit;
            float sacc = 0.0f;
            int oy = 0, ox = 0;
            if (q < npx_out) {
                oy = q / W; ox = q - oy * W;                       // output pixel = image (row0 + oy, ox)
                for (int i = part; i < a.N_k; i += nsplit) {
                    const float* tp = taps_t + i * KK;
                    const float* vw = vs + (size_t)i * vplane + oy * VW + ox;    // phi pixel (oy + a, ox + b)
#pragma unroll
                    for (int ka = 0; ka < KS; ++ka)
#pragma unroll
                        for (int kb = 0; kb < KS; ++kb) sacc = fmaf(tp[ka * KS + kb], vw[ka * VW + kb], sacc);
                }
            }
            for (int m = 1; m < nsplit; m <<= 1) sacc += __shfl_xor_sync(0xffffffffu, sacc, m);    // fixed order
            if (q < npx_out && part == 0) {
                const float uu = us[(oy + 2 * R) * UW + ox + 2 * R];
                const float ff = __ldg(f_img + (size_t)(row0 + oy) * W + ox);
                __stcg(dst + (size_t)(row0 + oy) * W + ox, uu - (sacc + lambda * (uu - ff)));
            }
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
    return sizeof(float) * (us + (size_t)N_k * vp + (size_t)nst * ((((size_t)N_k * KK + 3) & ~(size_t)3) + (size_t)N_k * SM_REC)
                            + 64 + vpx);
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
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)cs;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
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

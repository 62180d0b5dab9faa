// tnrd_microbench.cu -- register-only micro-kernels that measure the roofline denominators of the TNRD path on
// the current device: FP32 FFMA rate, MUFU.EX2 rate, the rate of the phi inner loop (FADD, FMUL, MUFU.EX2,
// FFMA per RBF term; Main Eq. 6) and the warp-level tensor path (mma.sync TF32 / BF16).  Timed with
// CUDA events on the caller's stream.
#include "tnrd_internal.h"
#include <cstring>

namespace tnrd {
namespace {

constexpr int MB_THREADS = 512;
constexpr int MB_ILP = 8;

__device__ __forceinline__ float ex2_approx(float x)
{
    float y;
    asm volatile("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

__global__ void __launch_bounds__(MB_THREADS, 1) mb_ffma(float* out, int iters, float x, float y)
{
    float acc[MB_ILP];
#pragma unroll
    for (int k = 0; k < MB_ILP; ++k) acc[k] = (float)(threadIdx.x + k);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int rep = 0; rep < 16; ++rep)
#pragma unroll
            for (int k = 0; k < MB_ILP; ++k) acc[k] = fmaf(acc[k], x, y);
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < MB_ILP; ++k) s += acc[k];
    if (s == 123.456f) out[0] = s;
}

__global__ void __launch_bounds__(MB_THREADS, 1) mb_mufu(float* out, int iters)
{
    float acc[MB_ILP];
#pragma unroll
    for (int k = 0; k < MB_ILP; ++k) acc[k] = 0.01f * (float)((threadIdx.x + k) & 63);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int rep = 0; rep < 16; ++rep)
#pragma unroll
            for (int k = 0; k < MB_ILP; ++k) acc[k] = ex2_approx(-acc[k]);   // stays in [0.5, 1]
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < MB_ILP; ++k) s += acc[k];
    if (s == 123.456f) out[0] = s;
}

// the phi inner loop exactly as the fused kernel runs it: 8 responses per thread, 64 (mu', w') pairs from
// shared memory (broadcast LDS.64), FADD + FMUL + MUFU.EX2 + FFMA per term
__global__ void __launch_bounds__(MB_THREADS, 1) mb_phi(float* out, int iters)
{
    __shared__ float2 mw[TNRD_MP];
    if (threadIdx.x < TNRD_MP) mw[threadIdx.x] = make_float2(-3.1f + 0.1f * threadIdx.x, 0.01f * threadIdx.x);
    __syncthreads();
    float z[MB_ILP], v[MB_ILP];
#pragma unroll
    for (int k = 0; k < MB_ILP; ++k) { z[k] = 0.003f * (float)((threadIdx.x * 7 + k * 13) & 1023) - 1.5f; v[k] = 0.f; }
    for (int it = 0; it < iters; ++it) {
#pragma unroll 4
        for (int m = 0; m < TNRD_MP; ++m) {
            const float2 c = mw[m];
#pragma unroll
            for (int k = 0; k < MB_ILP; ++k) {
                const float d = z[k] - c.x;
                v[k] = fmaf(ex2_approx(-d * d), c.y, v[k]);
            }
        }
#pragma unroll
        for (int k = 0; k < MB_ILP; ++k) z[k] += 1e-3f;
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < MB_ILP; ++k) s += v[k];
    if (s == 123.456f) out[0] = s;
}

// legacy warp-level tensor path (mma.sync -> HMMA), register-only: TF32 m16n8k8 (BF16 = false) or BF16 m16n8k16, fp32
// accumulation.  The denominator for the filterings as an implicit GEMM.
template <bool BF16>
__global__ void __launch_bounds__(MB_THREADS, 1) mb_mma(float* out, int iters)
{
    float c[MB_ILP][4];
    const unsigned a0 = threadIdx.x, a1 = 3u * threadIdx.x, a2 = 7u, a3 = 9u, b0 = blockIdx.x, b1 = 5u;
#pragma unroll
    for (int k = 0; k < MB_ILP; ++k)
#pragma unroll
        for (int q = 0; q < 4; ++q) c[k][q] = 0.f;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < MB_ILP; ++k) {
            if (BF16)
                asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                             : "+f"(c[k][0]), "+f"(c[k][1]), "+f"(c[k][2]), "+f"(c[k][3])
                             : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
            else
                asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                             : "+f"(c[k][0]), "+f"(c[k][1]), "+f"(c[k][2]), "+f"(c[k][3])
                             : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
        }
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < MB_ILP; ++k)
#pragma unroll
        for (int q = 0; q < 4; ++q) s += c[k][q];
    if (s == 123.456f) out[0] = s;
}


// ---- which = 5: the forward filter bank of the 48 x 7x7 model as an implicit GEMM on the warp-level tensor path ----------
// A prototype of DESIGN.md 11 (iii), not used by the product path: z_n(y, x) = sum_{a,b} K_n[a][b] U[y + 7 - a][x + b] for a
// 128 x 128 tile resident in shared memory.  Per warp M = 16 consecutive pixels of a row, N = 48 filters (6 n-tiles),
// K = 64 slots (slot 16 ks + j: tap row a = 2 ks + (j >= 8), tap column b = j % 8; b = 7 and a = 7 are zero).  The A fragment
// is gathered tap by tap from the fp32 tile (the im2col matrix never exists) and split in registers into BF16 halves
// x = x_hi + x_lo; the filters are split once on the device; three products (hi hi, hi lo, lo hi) accumulate in fp32.
constexpr int FB_NK = 48, FB_TW = 128, FB_TH = 128, FB_UH = FB_TH + 8, FB_US = 148, FB_MT = 2, FB_NKS = 4, FB_NNT = FB_NK / 8;
constexpr int FB_FG = 5, FB_FST = 16;                 // phi groups, coefficient slots per group (which = 6)
constexpr int FB_CSTRIDE = FB_FG * FB_FST + 1;        // float2 per filter pair: odd, so that the four pairs a warp reads hit different banks
constexpr int FB_SNT = 7;                              // n-tiles of the scatter table: 49 taps padded to 56 (which = 7)
constexpr int FB_SMEM = FB_UH * FB_US * 4 + FB_NKS * FB_NNT * 32 * 16 + FB_NK / 2 * FB_CSTRIDE * 8 + 3 * FB_SNT * 32 * 16;
static_assert((FB_NK / 2 * FB_CSTRIDE * 8) % 16 == 0, "the scatter-table fragments must stay 16-byte aligned");

__device__ __forceinline__ float fb_hash(unsigned i)      // [0, 1)
{
    i ^= i >> 16; i *= 0x7feb352du; i ^= i >> 15; i *= 0x846ca68bu; i ^= i >> 16;
    return (float)(i >> 8) * (1.0f / 16777216.0f);
}
__device__ __forceinline__ unsigned fb_pack(float hi, float lo)
{
    unsigned d;
    asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(d) : "f"(hi), "f"(lo));
    return d;
}
__device__ __forceinline__ void fb_split2(float x0, float x1, unsigned& h, unsigned& l)
{
    h = fb_pack(x1, x0);
    l = fb_pack(x1 - __uint_as_float(h & 0xffff0000u), x0 - __uint_as_float(h << 16));
}
__device__ __forceinline__ void fb_mma(float (&c)[4], const unsigned (&a)[4], unsigned b0, unsigned b1)
{
    asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ float fb_tap(const float* kf, int slot, int n)   // B[slot][n]
{
    const int a = 2 * (slot / 16) + ((slot % 16) >= 8), b = slot % 8;
    return (a < 7 && b < 7) ? kf[n * 49 + a * 7 + b] : 0.f;
}

// one CTA: a pseudo-random tile on the 0..255 scale, 48 zero-mean unit-norm filters, and their B fragments
__global__ void __launch_bounds__(512) fb_init(float* U, float* kf, uint4* bfrag, uint4* b2frag)
{
    for (int i = threadIdx.x; i < FB_UH * FB_US; i += 512) U[i] = 255.0f * fb_hash(i);
    if (threadIdx.x < FB_NK) {
        float* k = kf + threadIdx.x * 49;
        float s = 0.f, n2 = 0.f;
        for (int t = 0; t < 49; ++t) { k[t] = fb_hash(100000u + threadIdx.x * 49 + t) - 0.5f; s += k[t]; }
        for (int t = 0; t < 49; ++t) { k[t] -= s / 49.0f; n2 += k[t] * k[t]; }
        for (int t = 0; t < 49; ++t) k[t] *= rsqrtf(n2);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < FB_NKS * FB_NNT * 32; i += 512) {
        const int lane = i & 31, nt = (i >> 5) % FB_NNT, ks = (i >> 5) / FB_NNT, n = 8 * nt + (lane >> 2), c = lane & 3;
        unsigned h[2], l[2];                           // b0: slots 2c, 2c+1; b1: slots 2c+8, 2c+9
        for (int q = 0; q < 2; ++q)
            fb_split2(fb_tap(kf, 16 * ks + 2 * c + 8 * q, n), fb_tap(kf, 16 * ks + 2 * c + 8 * q + 1, n), h[q], l[q]);
        bfrag[i] = make_uint4(h[0], h[1], l[0], l[1]);
    }
    // transposed bank as a scatter table S[px][tap] = sum_f v_f(px) K_f[tap]: B[k = filter 16 s + ..][n = tap 8 nt + g]
    for (int i = threadIdx.x; i < 3 * FB_SNT * 32; i += 512) {
        const int lane = i & 31, nt = (i >> 5) % FB_SNT, s3 = (i >> 5) / FB_SNT, tap = 8 * nt + (lane >> 2), c = lane & 3;
        unsigned h[2], l[2];
        for (int q = 0; q < 2; ++q) {
            const int f = 16 * s3 + 2 * c + 8 * q;
            fb_split2(tap < 49 ? kf[f * 49 + tap] : 0.f, tap < 49 ? kf[(f + 1) * 49 + tap] : 0.f, h[q], l[q]);
        }
        b2frag[i] = make_uint4(h[0], h[1], l[0], l[1]);
    }
}

// check of the scatter table of one CTA's tile against plain fp32 sums (v and S as the check launch wrote them)
__global__ void fb_check_s(const float* __restrict__ v, const float* __restrict__ S, const float* __restrict__ kf, unsigned* maxdiff)
{
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= FB_TH * FB_TW) return;
    float worst = 0.f;
    for (int tap = 0; tap < 49; ++tap) {
        float r = 0.f;
        for (int f = 0; f < FB_NK; ++f) r = fmaf(v[(size_t)p * FB_NK + f], kf[f * 49 + tap], r);
        worst = fmaxf(worst, 1000.0f * fabsf(r - S[(size_t)p * 56 + tap]));     // |S| ~ 1: same 0.05 threshold as z after x 1000
    }
    atomicMax(maxdiff, __float_as_uint(worst));
}

// which = 6: the factorised phi on the accumulator layout -- a register pair holds two ADJACENT FILTERS of one
// pixel, so the Horner coefficients are packed pairs (LDS.64, one per FFMA2 of each of the NZ responses) instead of broadcast
// scalars.  Synthetic coefficients: the instruction stream does not depend on the values.
template <int NZ>
__device__ __forceinline__ void fb_phi_pairs(float2 (&z)[NZ], const float2* __restrict__ cf)
{
    float2 v[NZ];
#pragma unroll
    for (int i = 0; i < NZ; ++i) v[i] = make_float2(0.f, 0.f);
#pragma unroll 1
    for (int gr = 0; gr < FB_FG; ++gr) {
        const float2* c = cf + gr * FB_FST;
        float2 g[NZ], rho[NZ], rhoi[NZ], h[NZ], hl[NZ];
        const float2 c0 = c[0];
#pragma unroll
        for (int i = 0; i < NZ; ++i) {
            float2 d = __ffma2_rn(z[i], make_float2(0.0849f, 0.0849f), c0);
            asm("min.NaN.f32 %0, %0, %1;" : "+f"(d.x) : "f"(11.3f));
            asm("max.NaN.f32 %0, %0, %1;" : "+f"(d.x) : "f"(-11.3f));
            asm("min.NaN.f32 %0, %0, %1;" : "+f"(d.y) : "f"(11.3f));
            asm("max.NaN.f32 %0, %0, %1;" : "+f"(d.y) : "f"(-11.3f));
            const float2 t = __fmul2_rn(d, d), e = __fmul2_rn(d, make_float2(1.698f, 1.698f));
            g[i] = make_float2(ex2_approx(-t.x), ex2_approx(-t.y));
            rho[i] = make_float2(ex2_approx(e.x), ex2_approx(e.y));
            rhoi[i] = make_float2(ex2_approx(-e.x), ex2_approx(-e.y));
        }
        {
            const float2 a = c[1], b = c[2], a2 = c[8], b2 = c[9];
#pragma unroll
            for (int i = 0; i < NZ; ++i) { h[i] = __ffma2_rn(a, rho[i], b); hl[i] = __ffma2_rn(a2, rhoi[i], b2); }
        }
#pragma unroll
        for (int q = 3; q <= 7; ++q) {
            const float2 a = c[q];
#pragma unroll
            for (int i = 0; i < NZ; ++i) h[i] = __ffma2_rn(h[i], rho[i], a);
        }
#pragma unroll
        for (int q = 10; q <= 13; ++q) {
            const float2 a = c[q];
#pragma unroll
            for (int i = 0; i < NZ; ++i) hl[i] = __ffma2_rn(hl[i], rhoi[i], a);
        }
#pragma unroll
        for (int i = 0; i < NZ; ++i) {
            h[i] = __ffma2_rn(hl[i], rhoi[i], h[i]);
            v[i] = __ffma2_rn(g[i], h[i], v[i]);
        }
    }
#pragma unroll
    for (int i = 0; i < NZ; ++i) z[i] = v[i];
}

template <bool CHECK, bool PHI, bool SCATTER>
__global__ void __launch_bounds__(MB_THREADS, 1) fb_fwd(const float* __restrict__ U, const float* __restrict__ kf,
                                                        const uint4* __restrict__ bfrag, const uint4* __restrict__ b2frag,
                                                        float* __restrict__ vout, float* __restrict__ sout,
                                                        float* __restrict__ sink, unsigned* __restrict__ maxdiff, int reps)
{
    extern __shared__ __align__(16) float fb_sm[];
    float* us = fb_sm;                                               // [FB_UH][FB_US]
    uint4* bs = reinterpret_cast<uint4*>(us + FB_UH * FB_US);       // [FB_NKS][FB_NNT][32]
    for (int i = threadIdx.x; i < FB_UH * FB_US; i += MB_THREADS) us[i] = U[i];
    float2* cfs = reinterpret_cast<float2*>(bs + FB_NKS * FB_NNT * 32);   // [FB_NK / 2][FB_CSTRIDE]
    for (int i = threadIdx.x; i < FB_NKS * FB_NNT * 32; i += MB_THREADS) bs[i] = bfrag[i];
    uint4* b2s = reinterpret_cast<uint4*>(cfs + FB_NK / 2 * FB_CSTRIDE);   // [3][FB_SNT][32]
    for (int i = threadIdx.x; i < 3 * FB_SNT * 32; i += MB_THREADS) b2s[i] = b2frag[i];
    for (int i = threadIdx.x; i < FB_NK / 2 * FB_CSTRIDE; i += MB_THREADS)
        cfs[i] = make_float2(0.01f * (float)(i % 13) - 0.05f, 0.02f * (float)(i % 7) - 0.06f);
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, g = lane >> 2, c = lane & 3;
    float total = 0.f;
    for (int rep = 0; rep < reps; ++rep) {
        for (int mt0 = warp * FB_MT; mt0 < FB_TH * (FB_TW / 16); mt0 += (MB_THREADS / 32) * FB_MT) {
            float acc[FB_MT][FB_NNT][4];
#pragma unroll
            for (int m = 0; m < FB_MT; ++m)
#pragma unroll
                for (int n = 0; n < FB_NNT; ++n)
#pragma unroll
                    for (int q = 0; q < 4; ++q) acc[m][n][q] = 0.f;
#pragma unroll
            for (int ks = 0; ks < FB_NKS; ++ks) {
                unsigned ah[FB_MT][4], al[FB_MT][4];
#pragma unroll
                for (int m = 0; m < FB_MT; ++m) {
                    const int mt = mt0 + m, y = mt / (FB_TW / 16), x0 = (mt % (FB_TW / 16)) * 16;
                    const float* p0 = us + max(y + 7 - 2 * ks, 0) * FB_US + x0 + g + 2 * c;      // tap row a = 2 ks
                    const float* p1 = us + max(y + 6 - 2 * ks, 0) * FB_US + x0 + g + 2 * c;      // a = 2 ks + 1 (a = 7: zero taps)
                    fb_split2(p0[0], p0[1], ah[m][0], al[m][0]);     // pixel g,     slots 2c, 2c+1
                    fb_split2(p0[8], p0[9], ah[m][1], al[m][1]);     // pixel g + 8
                    fb_split2(p1[0], p1[1], ah[m][2], al[m][2]);     // pixel g,     slots 2c+8, 2c+9
                    fb_split2(p1[8], p1[9], ah[m][3], al[m][3]);
                }
#pragma unroll
                for (int n = 0; n < FB_NNT; ++n) {
                    const uint4 b = bs[(ks * FB_NNT + n) * 32 + lane];
#pragma unroll
                    for (int m = 0; m < FB_MT; ++m) {
                        fb_mma(acc[m][n], ah[m], b.x, b.y);
                        fb_mma(acc[m][n], ah[m], b.z, b.w);
                        fb_mma(acc[m][n], al[m], b.x, b.y);
                    }
                }
            }
            if (CHECK && mt0 < 8 * MB_THREADS / 32 * FB_MT) {     // self-check against plain fp32 FMAs (first 8 rounds of m-tiles)
                float worst = 0.f;
                for (int m = 0; m < FB_MT; ++m)
                    for (int n = 0; n < FB_NNT; ++n)
                        for (int q = 0; q < 4; ++q) {
                            const int mt = mt0 + m, y = mt / (FB_TW / 16), x = (mt % (FB_TW / 16)) * 16 + g + 8 * (q >> 1);
                            const float* k = kf + (8 * n + 2 * c + (q & 1)) * 49;
                            float z = 0.f;
                            for (int a = 0; a < 7; ++a)
                                for (int b = 0; b < 7; ++b) z = fmaf(k[a * 7 + b], us[(y + 7 - a) * FB_US + x + b], z);
                            float got = 0.f;                              // acc[m][n][q] with run-time indices
#pragma unroll
                            for (int mm = 0; mm < FB_MT; ++mm)
#pragma unroll
                                for (int nn = 0; nn < FB_NNT; ++nn)
#pragma unroll
                                    for (int qq = 0; qq < 4; ++qq)
                                        if (mm == m && nn == n && qq == q) got = acc[mm][nn][qq];
                            worst = fmaxf(worst, fabsf(got - z));
                        }
                atomicMax(maxdiff, __float_as_uint(worst));
            }
            if (PHI) {
#pragma unroll
                for (int n = 0; n < FB_NNT; ++n) {
                    float2 zz[2 * FB_MT];
#pragma unroll
                    for (int m = 0; m < FB_MT; ++m) {
                        zz[2 * m] = make_float2(acc[m][n][0], acc[m][n][1]);
                        zz[2 * m + 1] = make_float2(acc[m][n][2], acc[m][n][3]);
                    }
                    fb_phi_pairs<2 * FB_MT>(zz, cfs + (4 * n + c) * FB_CSTRIDE);
#pragma unroll
                    for (int m = 0; m < FB_MT; ++m) {
                        acc[m][n][0] = zz[2 * m].x; acc[m][n][1] = zz[2 * m].y;
                        acc[m][n][2] = zz[2 * m + 1].x; acc[m][n][3] = zz[2 * m + 1].y;
                    }
                }
            }
            if (SCATTER) {   // S[px][tap] = sum_f v_f(px) K_f[tap]: two n-tiles of accumulators ARE the A fragment of one k-step
#pragma unroll
                for (int m = 0; m < FB_MT; ++m) {
                    if (!PHI) {
#pragma unroll
                        for (int n = 0; n < FB_NNT; ++n)
#pragma unroll
                            for (int q = 0; q < 4; ++q) acc[m][n][q] *= 0.004f;       // stand-in for v on its scale
                    }
                    float S[FB_SNT][4];
#pragma unroll
                    for (int n = 0; n < FB_SNT; ++n)
#pragma unroll
                        for (int q = 0; q < 4; ++q) S[n][q] = 0.f;
#pragma unroll
                    for (int s3 = 0; s3 < 3; ++s3) {
                        unsigned vh[4], vl[4];
                        fb_split2(acc[m][2 * s3][0], acc[m][2 * s3][1], vh[0], vl[0]);
                        fb_split2(acc[m][2 * s3][2], acc[m][2 * s3][3], vh[1], vl[1]);
                        fb_split2(acc[m][2 * s3 + 1][0], acc[m][2 * s3 + 1][1], vh[2], vl[2]);
                        fb_split2(acc[m][2 * s3 + 1][2], acc[m][2 * s3 + 1][3], vh[3], vl[3]);
#pragma unroll
                        for (int n = 0; n < FB_SNT; ++n) {
                            const uint4 b = b2s[(s3 * FB_SNT + n) * 32 + lane];
                            fb_mma(S[n], vh, b.x, b.y);
                            fb_mma(S[n], vh, b.z, b.w);
                            fb_mma(S[n], vl, b.x, b.y);
                        }
                    }
                    if (CHECK) {
                        const int mt = mt0 + m, y = mt / (FB_TW / 16), x0 = (mt % (FB_TW / 16)) * 16;
#pragma unroll
                        for (int n = 0; n < FB_NNT; ++n)
#pragma unroll
                            for (int q = 0; q < 4; ++q)
                                vout[(size_t)(y * FB_TW + x0 + g + 8 * (q >> 1)) * FB_NK + 8 * n + 2 * c + (q & 1)] = acc[m][n][q];
#pragma unroll
                        for (int n = 0; n < FB_SNT; ++n)
#pragma unroll
                            for (int q = 0; q < 4; ++q)
                                sout[(size_t)(y * FB_TW + x0 + g + 8 * (q >> 1)) * 56 + 8 * n + 2 * c + (q & 1)] = S[n][q];
                    }
#pragma unroll
                    for (int n = 0; n < FB_SNT; ++n) total += (S[n][0] + S[n][1]) + (S[n][2] + S[n][3]);
                }
            }
#pragma unroll
            for (int m = 0; m < FB_MT; ++m)
#pragma unroll
                for (int n = 0; n < FB_NNT; ++n) total += (acc[m][n][0] + acc[m][n][1]) + (acc[m][n][2] + acc[m][n][3]);
        }
    }
    if (total == 123.456f) sink[0] = total;
}

cudaError_t run_fwd_bank_probe(int which, double* rate, cudaStream_t st, unsigned long long* launches, int sms)
{
    float *U = nullptr, *kf = nullptr, *sink = nullptr;
    uint4 *bfrag = nullptr, *b2frag = nullptr;
    float *vbuf = nullptr, *sbuf = nullptr;
    unsigned* maxdiff = nullptr;
    cudaError_t e = cudaMalloc(&U, (size_t)FB_UH * FB_US * 4);
    if (e == cudaSuccess) e = cudaMalloc(&kf, FB_NK * 49 * 4);
    if (e == cudaSuccess) e = cudaMalloc(&sink, 4);
    if (e == cudaSuccess) e = cudaMalloc(&bfrag, (size_t)FB_NKS * FB_NNT * 32 * 16);
    if (e == cudaSuccess) e = cudaMalloc(&maxdiff, 4);
    if (e == cudaSuccess) e = cudaMalloc(&b2frag, (size_t)3 * FB_SNT * 32 * 16);
    if (e == cudaSuccess) e = cudaMalloc(&vbuf, (size_t)FB_TH * FB_TW * FB_NK * 4);
    if (e == cudaSuccess) e = cudaMalloc(&sbuf, (size_t)FB_TH * FB_TW * 56 * 4);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(fb_fwd<false, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, FB_SMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(fb_fwd<false, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, FB_SMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(fb_fwd<false, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, FB_SMEM);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(fb_fwd<true, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, FB_SMEM);
    float best_ms = 1e30f;
    unsigned diff_bits = 0;
    if (e == cudaSuccess) {
        cudaEvent_t e0, e1;
        cudaEventCreate(&e0);
        cudaEventCreate(&e1);
        cudaMemsetAsync(maxdiff, 0, 4, st);
        fb_init<<<1, 512, 0, st>>>(U, kf, bfrag, b2frag);
        fb_fwd<true, false, true><<<1, MB_THREADS, FB_SMEM, st>>>(U, kf, bfrag, b2frag, vbuf, sbuf, sink, maxdiff, 1);
        fb_check_s<<<(FB_TH * FB_TW + 255) / 256, 256, 0, st>>>(vbuf, sbuf, kf, maxdiff);
        *launches += 3;
        const int reps = 16;
        for (int rep = 0; rep < 4 && e == cudaSuccess; ++rep) {   // rep 0 = warm-up
            cudaEventRecord(e0, st);
            if (which == 7) fb_fwd<false, true, true><<<sms, MB_THREADS, FB_SMEM, st>>>(U, kf, bfrag, b2frag, vbuf, sbuf, sink, maxdiff, reps);
            else if (which == 6) fb_fwd<false, true, false><<<sms, MB_THREADS, FB_SMEM, st>>>(U, kf, bfrag, b2frag, vbuf, sbuf, sink, maxdiff, reps);
            else fb_fwd<false, false, false><<<sms, MB_THREADS, FB_SMEM, st>>>(U, kf, bfrag, b2frag, vbuf, sbuf, sink, maxdiff, reps);
            ++*launches;
            cudaEventRecord(e1, st);
            e = cudaEventSynchronize(e1);
            float ms = 0.f;
            if (e == cudaSuccess) cudaEventElapsedTime(&ms, e0, e1);
            if (rep > 0 && ms < best_ms) best_ms = ms;
        }
        if (e == cudaSuccess) e = cudaMemcpyAsync(&diff_bits, maxdiff, 4, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        cudaEventDestroy(e0);
        cudaEventDestroy(e1);
        if (e == cudaSuccess) e = cudaGetLastError();
        *rate = (double)sms * reps * FB_TH * FB_TW / ((double)best_ms * 1e-3);      // pixels (48 responses each) per second
    }
    cudaFree(U); cudaFree(kf); cudaFree(sink); cudaFree(bfrag); cudaFree(maxdiff); cudaFree(b2frag); cudaFree(vbuf); cudaFree(sbuf);
    if (e != cudaSuccess) return e;
    float diff;
    memcpy(&diff, &diff_bits, 4);
    // |z| ~ 75 on this input; the split drops x_lo k_lo (~2^-16 relative per product): observed 2e-3, a wrong fragment layout gives ~10
    return (diff == diff && diff < 0.05f) ? cudaSuccess : cudaErrorAssert;
}

}  // namespace

cudaError_t run_microbench(int which, double* rate, cudaStream_t st, unsigned long long* launches)
{
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return e;
    if (which >= 5) return run_fwd_bank_probe(which, rate, st, launches, sms);
    float* d_out = nullptr;
    e = cudaMalloc(&d_out, sizeof(float));
    if (e != cudaSuccess) return e;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int grid = sms * 2;   // 2 waves of 1 CTA/SM x 512 threads
    double ops_per_thread = 0.0;
    float best_ms = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {   // rep 0 = warm-up
        cudaEventRecord(e0, st);
        if (which == 0) {
            const int iters = 4096;
            mb_ffma<<<grid, MB_THREADS, 0, st>>>(d_out, iters, 1.0000001f, 1e-9f);
            ops_per_thread = (double)iters * 16 * MB_ILP;
        } else if (which == 1) {
            const int iters = 1024;
            mb_mufu<<<grid, MB_THREADS, 0, st>>>(d_out, iters);
            ops_per_thread = (double)iters * 16 * MB_ILP;
        } else if (which == 2) {
            const int iters = 256;
            mb_phi<<<grid, MB_THREADS, 0, st>>>(d_out, iters);
            ops_per_thread = (double)iters * TNRD_MP * MB_ILP;
        } else if (which == 3) {
            const int iters = 4096;
            mb_mma<false><<<grid, MB_THREADS, 0, st>>>(d_out, iters);
            ops_per_thread = (double)iters * MB_ILP * (16 * 8 * 8) / 32.0;      // multiply-adds per thread
        } else {
            const int iters = 4096;
            mb_mma<true><<<grid, MB_THREADS, 0, st>>>(d_out, iters);
            ops_per_thread = (double)iters * MB_ILP * (16 * 8 * 16) / 32.0;
        }
        ++*launches;
        cudaEventRecord(e1, st);
        e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) break;
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best_ms) best_ms = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(d_out);
    if (e != cudaSuccess) return e;
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    *rate = ops_per_thread * (double)grid * MB_THREADS / ((double)best_ms * 1e-3);
    return cudaSuccess;
}

}  // namespace tnrd

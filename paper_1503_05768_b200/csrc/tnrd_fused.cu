// tnrd_fused.cu -- the fused per-stage kernel (rows a1-a5 of the hot path in ONE pass; kernel variant 2).
//
//   u_t = u - ( sum_i kbar_i * phi_i(k_i * u~) + lambda (u - f) )          Main Eq. 7
//
// One CTA owns one output tile of tw x th pixels of one image:
//   a1  the u tile with its 2r halo is gathered through the mirror index map into shared
//       memory -- the padded image is never materialised;
//   then, one filter i at a time (streamed, so that only two influence maps live on chip):
//   a2  z' = k'_i * u~ on the (tw+2r) x (th+2r) "phi region", in registers, 4x2 pixels per thread-block-of-work,
//   a3  v = sum_j w'_ij 2^{-(z' - mu'_j)^2}, all 63 terms, one MUFU.EX2 each (ex2.approx.ftz), in registers,
//       written once to a double-buffered shared-memory map,
//   a4  the rot180 taps of filter i-1 are applied to the map finished in the previous iteration and summed into
//       per-thread output accumulators that live across the whole filter loop,
//   a5  epilogue: u_t = u - (s + lambda (u - f)) straight from the shared u tile to global memory.
// One __syncthreads() per filter.  HBM traffic is the algorithmic 12 B per pixel-stage plus the halo re-read.
//
// The path is bound by the XU (MUFU) pipe: 3024 ex2 per pixel-stage for the 48 x 7x7 model against 4704 FFMA of
// filtering; tensor cores are not used.
#include <cstdlib>

#include "tnrd_internal.h"

namespace tnrd {

namespace {

__device__ __forceinline__ float ex2_approx(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

template <int KS, int RW, int RH, int NT, int MINB = 1>
struct Cfg {
    static constexpr int R = (KS - 1) / 2;
    static constexpr int US = RW + 8;                   // u tile row stride (floats)
    static constexpr int UH = RH + 2 * R;               // u tile rows
    static constexpr int VS = RW;                       // phi map row stride
    static constexpr int VPLANE = RH * RW + 16;         // one phi map (+ overrun pad for masked pixels)
    static constexpr int PRM = prm_stride(KS);          // floats per staged record
    static constexpr int NB = ((RW / 4) * (RH / 2) + NT - 1) / NT;  // 4x2 work blocks per thread (max)
    static constexpr size_t SMEM = sizeof(float) * ((size_t)UH * US + 2 * (size_t)VPLANE + 3 * (size_t)PRM);
};

// forward filter (a2): z[j][p] += sum_{a,b} k[a][b] * U[py0 + j + 2r - a][px0 + p + 2r - b]
// `uw` points at U[py0][px0]; `taps` at the staged record (rows of TS floats, but stored densely a*KS+b)
template <int KS, int US>
__device__ __forceinline__ void conv_fwd_block(const float* __restrict__ uw, const float* __restrict__ taps,
                                               float (&z)[2][4])
{
    constexpr int WC = 4 + KS - 1, NV = (WC + 3) / 4;
#pragma unroll
    for (int wr = 0; wr < KS + 1; ++wr) {
        float row[NV * 4];
#pragma unroll
        for (int q = 0; q < NV; ++q) {
            const float4 t = *reinterpret_cast<const float4*>(uw + wr * US + 4 * q);
            row[4 * q + 0] = t.x; row[4 * q + 1] = t.y; row[4 * q + 2] = t.z; row[4 * q + 3] = t.w;
        }
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            const int a = j + (KS - 1) - wr;
            if (a < 0 || a >= KS) continue;
#pragma unroll
            for (int b = 0; b < KS; ++b) {
                const float k = taps[a * KS + b];
#pragma unroll
                for (int p = 0; p < 4; ++p) z[j][p] = fmaf(k, row[p + (KS - 1) - b], z[j][p]);
            }
        }
    }
}

// transposed filter (a4): s[j][p] += sum_{a,b} k[a][b] * V[oy0 + j + a][ox0 + p + b]; `vw` points at V[oy0][ox0]
template <int KS, int VS>
__device__ __forceinline__ void conv_bwd_block(const float* __restrict__ vw, const float* __restrict__ taps,
                                               float (&s)[2][4])
{
    constexpr int WC = 4 + KS - 1, NV = (WC + 3) / 4;
#pragma unroll
    for (int wr = 0; wr < KS + 1; ++wr) {
        float row[NV * 4];
#pragma unroll
        for (int q = 0; q < NV; ++q) {
            const float4 t = *reinterpret_cast<const float4*>(vw + wr * VS + 4 * q);
            row[4 * q + 0] = t.x; row[4 * q + 1] = t.y; row[4 * q + 2] = t.z; row[4 * q + 3] = t.w;
        }
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            const int a = wr - j;
            if (a < 0 || a >= KS) continue;
#pragma unroll
            for (int b = 0; b < KS; ++b) {
                const float k = taps[a * KS + b];
#pragma unroll
                for (int p = 0; p < 4; ++p) s[j][p] = fmaf(k, row[p + b], s[j][p]);
            }
        }
    }
}

// influence function (a3) on 8 responses held in registers; mw = 64 pairs (mu'_j, w'_ij)
__device__ __forceinline__ void phi_block(const float2* __restrict__ mw, const float (&z)[2][4], float (&v)[2][4])
{
#pragma unroll
    for (int j = 0; j < 2; ++j)
#pragma unroll
        for (int p = 0; p < 4; ++p) v[j][p] = 0.0f;
#pragma unroll 4
    for (int m = 0; m < TNRD_MP; ++m) {
        const float2 c = mw[m];
#pragma unroll
        for (int j = 0; j < 2; ++j)
#pragma unroll
            for (int p = 0; p < 4; ++p) {
                const float d = z[j][p] - c.x;
                v[j][p] = fmaf(ex2_approx(-d * d), c.y, v[j][p]);
            }
    }
}

template <int KS, int RW, int RH, int NT, int MINB>
__global__ void __launch_bounds__(NT, MINB)
stage_fused_kernel(StageArgs a, int tw, int th, int ntx, int nty)
{
    using C = Cfg<KS, RW, RH, NT, MINB>;
    constexpr int R = C::R;
    extern __shared__ __align__(16) float smem[];
    float* us = smem;                              // [UH][US]
    float* vs = us + C::UH * C::US;                // [2][VPLANE]
    float* ps = vs + 2 * C::VPLANE;                // [3][PRM]

    const int tid = threadIdx.x;
    int t = blockIdx.x;
    const int tx = t % ntx; t /= ntx;
    const int ty = t % nty; t /= nty;
    const int img = t;
    const int X0 = tx * tw, Y0 = ty * th;          // image coordinates of the output tile origin
    const float* __restrict__ u_img = a.u_in + (size_t)img * a.H * a.W;

    // ---- a1: gather the u tile through the mirror map ----------------------------------------------------
    for (int idx = tid; idx < C::UH * C::US; idx += NT) {
        const int uy = idx / C::US, ux = idx - uy * C::US;
        const int gy = mirror_clamp(Y0 - 2 * R + uy, a.H), gx = mirror_clamp(X0 - 2 * R + ux, a.W);
        us[idx] = __ldg(u_img + (size_t)gy * a.W + gx);
    }
    for (int idx = tid; idx < C::PRM; idx += NT) ps[idx] = __ldg(a.prm + idx);

    // ---- work decomposition: 4x2 pixel blocks, NB per thread ----------------------------------------------
    const int nbx = (tw + 2 * R + 3) >> 2, nby = (th + 2 * R + 1) >> 1;   // phi region
    const int nbxo = (tw + 3) >> 2, nbyo = (th + 1) >> 1;                  // output tile
    int offA[C::NB], offC[C::NB];   // offsets of the block origin (row*stride + col), -1 = no work
#pragma unroll
    for (int n = 0; n < C::NB; ++n) {
        const int blk = tid + n * NT;
        const int by = blk / nbx, bx = blk - by * nbx;
        offA[n] = (by < nby) ? ((2 * by) << 16 | (4 * bx)) : -1;
        const int cy = blk / nbxo, cx = blk - cy * nbxo;
        offC[n] = (cy < nbyo) ? ((2 * cy) << 16 | (4 * cx)) : -1;
    }
    float acc[C::NB][2][4];
#pragma unroll
    for (int n = 0; n < C::NB; ++n)
#pragma unroll
        for (int j = 0; j < 2; ++j)
#pragma unroll
            for (int p = 0; p < 4; ++p) acc[n][j][p] = 0.0f;

    __syncthreads();

    // ---- filter loop: a2 + a3 for filter i, a4 for filter i-1 ---------------------------------------------
    for (int i = 0; i <= a.N_k; ++i) {
        if (i + 1 < a.N_k) {  // stage the next record (triple buffer: i-1 is still read by a4)
            const float* src = a.prm + (size_t)(i + 1) * C::PRM;
            float* dst = ps + ((i + 1) % 3) * C::PRM;
            for (int idx = tid; idx < C::PRM; idx += NT) dst[idx] = __ldg(src + idx);
        }
        if (i < a.N_k) {
            const float* rec = ps + (i % 3) * C::PRM;
            float* vcur = vs + (i & 1) * C::VPLANE;
#pragma unroll 1
            for (int n = 0; n < C::NB; ++n) {
                if (offA[n] < 0) continue;
                const int py = offA[n] >> 16, px = offA[n] & 0xffff;
                float z[2][4] = {{0.f, 0.f, 0.f, 0.f}, {0.f, 0.f, 0.f, 0.f}};
                conv_fwd_block<KS, C::US>(us + py * C::US + px, rec, z);
                float v[2][4];
                phi_block(reinterpret_cast<const float2*>(rec + prm_kkp(KS)), z, v);
                *reinterpret_cast<float4*>(vcur + py * C::VS + px) = make_float4(v[0][0], v[0][1], v[0][2], v[0][3]);
                *reinterpret_cast<float4*>(vcur + (py + 1) * C::VS + px) =
                    make_float4(v[1][0], v[1][1], v[1][2], v[1][3]);
            }
        }
        if (i > 0) {
            const float* rec = ps + ((i - 1) % 3) * C::PRM;
            const float* vprev = vs + ((i - 1) & 1) * C::VPLANE;
#pragma unroll
            for (int n = 0; n < C::NB; ++n) {
                if (offC[n] < 0) continue;
                const int oy = offC[n] >> 16, ox = offC[n] & 0xffff;
                conv_bwd_block<KS, C::VS>(vprev + oy * C::VS + ox, rec, acc[n]);
            }
        }
        __syncthreads();
    }

    // ---- a5: reaction term and update ------------------------------------------------------------------------
    const float lambda = a.lambda_ptr ? __ldg(a.lambda_ptr) : a.lambda_val;
    const float* __restrict__ f_img = a.f + (size_t)img * a.H * a.W;
    float* __restrict__ o_img = a.u_out + (size_t)img * a.H * a.W;
#pragma unroll
    for (int n = 0; n < C::NB; ++n) {
        if (offC[n] < 0) continue;
        const int oy = offC[n] >> 16, ox = offC[n] & 0xffff;
#pragma unroll
        for (int j = 0; j < 2; ++j)
#pragma unroll
            for (int p = 0; p < 4; ++p) {
                const int ly = oy + j, lx = ox + p, gy = Y0 + ly, gx = X0 + lx;
                if (ly < th && lx < tw && gy < a.H && gx < a.W) {
                    const float uu = us[(ly + 2 * R) * C::US + lx + 2 * R];
                    const size_t g = (size_t)gy * a.W + gx;
                    o_img[g] = uu - (acc[n][j][p] + lambda * (uu - __ldg(f_img + g)));
                }
            }
    }
}

// balanced tile edge: the fewest tiles of at most `maxt` that cover n, all of (nearly) equal size
inline void split(int n, int maxt, int* nt, int* tsz)
{
    *nt = (n + maxt - 1) / maxt;
    *tsz = (n + *nt - 1) / *nt;
}

template <int KS, int RW, int RH, int NT, int MINB>
cudaError_t launch_cfg(const StageArgs& a, cudaStream_t st)
{
    using C = Cfg<KS, RW, RH, NT, MINB>;
    static bool attr_done = false;  // per-process; the attribute is per-function and sticky
    if (!attr_done) {
        cudaError_t e = cudaFuncSetAttribute(stage_fused_kernel<KS, RW, RH, NT, MINB>,
                                             cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM);
        if (e != cudaSuccess) return e;
        attr_done = true;
    }
    int ntx, nty, tw, th;
    split(a.W, RW - 2 * C::R, &ntx, &tw);
    split(a.H, RH - 2 * C::R, &nty, &th);
    const long long grid = (long long)ntx * nty * a.B;
    if (grid > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    stage_fused_kernel<KS, RW, RH, NT, MINB><<<(unsigned)grid, NT, C::SMEM, st>>>(a, tw, th, ntx, nty);
    return cudaGetLastError();
}

// TNRD_TILE=<id> (environment, read once) forces a tile configuration; a tuning knob, not part of the ABI.
inline int forced_tile()
{
    static int v = -1;
    if (v < 0) {
        const char* e = getenv("TNRD_TILE");
        v = e ? atoi(e) : 0;
    }
    return v;
}

template <int KS>
cudaError_t launch_ks(const StageArgs& a, int num_sms, cudaStream_t st)
{
    int id = forced_tile();
    if (id == 0) {
        // Large tiles (less halo recompute) when they still fill the machine, small tiles otherwise.
        int ntx, nty, tw, th;
        split(a.W, 128 - (KS - 1), &ntx, &tw);
        split(a.H, 128 - (KS - 1), &nty, &th);
        id = ((long long)ntx * nty * a.B >= 2LL * num_sms) ? 1 : 2;
    }
    switch (id) {
        case 1: return launch_cfg<KS, 128, 128, 512, 1>(a, st);
        case 2: return launch_cfg<KS, 64, 32, 256, 2>(a, st);
        case 3: return launch_cfg<KS, 128, 64, 256, 2>(a, st);
        case 4: return launch_cfg<KS, 64, 128, 256, 2>(a, st);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace

cudaError_t fused_init() { return cudaSuccess; }

cudaError_t launch_stage_fused(const StageArgs& a, int num_sms, cudaStream_t st, unsigned long long* launches)
{
    cudaError_t e;
    switch (a.ksize) {
        case 3: e = launch_ks<3>(a, num_sms, st); break;
        case 5: e = launch_ks<5>(a, num_sms, st); break;
        case 7: e = launch_ks<7>(a, num_sms, st); break;
        case 9: e = launch_ks<9>(a, num_sms, st); break;
        default: return cudaErrorInvalidValue;
    }
    ++*launches;
    return e;
}

}  // namespace tnrd

// tnrd_microbench.cu -- register-only micro-kernels that measure the roofline denominators of the TNRD path on
// the current device: FP32 FFMA rate, MUFU.EX2 rate and the rate of the direct phi inner loop (FADD, FMUL, MUFU.EX2,
// FFMA per RBF term; Main Eq. 6).  Timed with CUDA events on the caller's stream.
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

// FFMA2 (FMA pipe, 2 cycles per warp) and FMNMX (ALU pipe, 2 cycles per warp) interleaved 1:1 on independent registers,
// 6 warps per scheduler.  Pipes that issued side by side would sustain 1.0 warp instructions per clock per scheduler
// (0.5 each), one fully shared dispatch 0.5; B200 measures 0.66: the FMA and ALU pipes overlap only in part.  The
// tensor-core stage kernel runs with FMA-pipe cycles + ALU-pipe cycles = 87 % of the time.
__global__ void __launch_bounds__(768, 1) mb_dispatch(float* out, int iters, float x, float y)
{
    float2 h[4], r[4];
    float m[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        h[k] = make_float2((float)(threadIdx.x + k), 1.0f);
        r[k] = make_float2(x + 1e-7f * (float)threadIdx.x, x);
        m[k] = (float)(threadIdx.x * 3 + k);
    }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int rep = 0; rep < 16; ++rep)
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                h[k] = __ffma2_rn(h[k], r[k], make_float2(y, y));
                m[k] = fminf(m[k], m[(k + 1) & 3]);
                asm volatile("" : "+f"(m[k]));                   // keep every FMNMX
            }
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < 4; ++k) s += h[k].x + h[k].y + m[k];
    if (s == 123.456f) out[0] = s;
}

}  // namespace

cudaError_t run_microbench(int which, double* rate, cudaStream_t st, unsigned long long* launches)
{
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return e;
    if (which < 0 || which > 3) return cudaErrorInvalidValue;
    float* d_out = nullptr;
    e = cudaMalloc(&d_out, sizeof(float));
    if (e != cudaSuccess) return e;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int grid = which == 3 ? sms : sms * 2;   // 2 waves of 1 CTA/SM x 512 threads (the dispatch probe: 1 x 768)
    int threads = MB_THREADS;
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
        } else {
            const int iters = 2048;
            threads = 768;
            mb_dispatch<<<grid, threads, 0, st>>>(d_out, iters, 0.9999f, 1e-9f);
            ops_per_thread = (double)iters * 16 * 4 * 2 / 32.0;     // WARP instructions (FFMA2 + FMNMX) per thread / 32
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
    *rate = ops_per_thread * (double)grid * threads / ((double)best_ms * 1e-3);
    return cudaSuccess;
}

}  // namespace tnrd

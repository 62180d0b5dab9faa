// tnrd_qcs.cu -- the non-smooth part of the JPEG-deblocking stage (Main Eq. 9; Supp. Eq. 26-29):
//     u_t = D^T eta( D y ),   D = orthonormal 2-D DCT-II of every 8x8 block,  eta = clamp to the QCS box [lo, hi].
// y = u_{t-1} - sum_i kbar_i * phi_i(k_i * u_{t-1}) comes from the fused stage kernel run with lambda = 0.
// The step moves 16 B per pixel (y, lo, hi in; u out) against ~64 FMA per pixel: it is HBM-bound and costs < 1 % of
// the stage, so it is a separate, simple kernel: 8 threads per block, row pass / column pass through shared memory.
#include "tnrd_internal.h"

namespace tnrd {
namespace {

// c_dct[p][y] = alpha_p cos(pi (2y+1) p / 16), alpha_0 = sqrt(1/8), alpha_p = sqrt(2/8)  (D^T D = I)
__constant__ float c_dct[64] = {
    3.535533906e-01f, 3.535533906e-01f, 3.535533906e-01f, 3.535533906e-01f, 3.535533906e-01f, 3.535533906e-01f, 3.535533906e-01f, 3.535533906e-01f,
    4.903926402e-01f, 4.157348062e-01f, 2.777851165e-01f, 9.754516101e-02f, -9.754516101e-02f, -2.777851165e-01f, -4.157348062e-01f, -4.903926402e-01f,
    4.619397663e-01f, 1.913417162e-01f, -1.913417162e-01f, -4.619397663e-01f, -4.619397663e-01f, -1.913417162e-01f, 1.913417162e-01f, 4.619397663e-01f,
    4.157348062e-01f, -9.754516101e-02f, -4.903926402e-01f, -2.777851165e-01f, 2.777851165e-01f, 4.903926402e-01f, 9.754516101e-02f, -4.157348062e-01f,
    3.535533906e-01f, -3.535533906e-01f, -3.535533906e-01f, 3.535533906e-01f, 3.535533906e-01f, -3.535533906e-01f, -3.535533906e-01f, 3.535533906e-01f,
    2.777851165e-01f, -4.903926402e-01f, 9.754516101e-02f, 4.157348062e-01f, -4.157348062e-01f, -9.754516101e-02f, 4.903926402e-01f, -2.777851165e-01f,
    1.913417162e-01f, -4.619397663e-01f, 4.619397663e-01f, -1.913417162e-01f, -1.913417162e-01f, 4.619397663e-01f, -4.619397663e-01f, 1.913417162e-01f,
    9.754516101e-02f, -2.777851165e-01f, 4.157348062e-01f, -4.903926402e-01f, 4.903926402e-01f, -4.157348062e-01f, 2.777851165e-01f, -9.754516101e-02f,
};

constexpr int QB = 32;   // 8x8 blocks per CTA (256 threads)

__global__ void __launch_bounds__(QB * 8) qcs_project_kernel(const float* y, const float* __restrict__ lo,
                                                             const float* __restrict__ hi, float* u,
                                                             int H, int W, long long nblk, int vec_ok)
{
    __shared__ float s[QB][8][9];
    const int t = threadIdx.x, lb = t >> 3, r = t & 7;
    const long long blk = (long long)blockIdx.x * QB + lb;
    const bool live = blk < nblk;
    const int bw = W >> 3, bh = H >> 3;
    const long long img = live ? blk / ((long long)bw * bh) : 0;
    const int rem = live ? (int)(blk - img * bw * bh) : 0;
    const int by = rem / bw, bx = rem - by * bw;
    const size_t base = (size_t)img * H * W + (size_t)(8 * by) * W + 8 * bx;   // block origin

    // forward, rows: thread (block, row r)
    float v[8];
    if (live) {
        const float* src = y + base + (size_t)r * W;
        if (vec_ok) {
            const float4 a = *reinterpret_cast<const float4*>(src), b = *reinterpret_cast<const float4*>(src + 4);
            v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w; v[4] = b.x; v[5] = b.y; v[6] = b.z; v[7] = b.w;
        } else {
#pragma unroll
            for (int x = 0; x < 8; ++x) v[x] = src[x];
        }
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            float acc = 0.f;
#pragma unroll
            for (int x = 0; x < 8; ++x) acc = fmaf(c_dct[q * 8 + x], v[x], acc);
            s[lb][r][q] = acc;
        }
    }
    __syncthreads();
    // forward columns, projection (Supp. Eq. 26), inverse columns: thread (block, column q = r)
    if (live) {
        float col[8], c[8];
#pragma unroll
        for (int yy = 0; yy < 8; ++yy) col[yy] = s[lb][yy][r];
#pragma unroll
        for (int p = 0; p < 8; ++p) {
            float acc = 0.f;
#pragma unroll
            for (int yy = 0; yy < 8; ++yy) acc = fmaf(c_dct[p * 8 + yy], col[yy], acc);
            const size_t g = base + (size_t)p * W + r;
            c[p] = fminf(fmaxf(acc, __ldg(lo + g)), __ldg(hi + g));
        }
#pragma unroll
        for (int yy = 0; yy < 8; ++yy) {
            float acc = 0.f;
#pragma unroll
            for (int p = 0; p < 8; ++p) acc = fmaf(c_dct[p * 8 + yy], c[p], acc);
            col[yy] = acc;
        }
#pragma unroll
        for (int yy = 0; yy < 8; ++yy) s[lb][yy][r] = col[yy];   // column r is read and written by this thread only
    }
    __syncthreads();
    // inverse rows: thread (block, row r)
    if (live) {
#pragma unroll
        for (int q = 0; q < 8; ++q) v[q] = s[lb][r][q];
        float o[8];
#pragma unroll
        for (int x = 0; x < 8; ++x) {
            float acc = 0.f;
#pragma unroll
            for (int q = 0; q < 8; ++q) acc = fmaf(c_dct[q * 8 + x], v[q], acc);
            o[x] = acc;
        }
        float* dst = u + base + (size_t)r * W;
        if (vec_ok) {
            *reinterpret_cast<float4*>(dst) = make_float4(o[0], o[1], o[2], o[3]);
            *reinterpret_cast<float4*>(dst + 4) = make_float4(o[4], o[5], o[6], o[7]);
        } else {
#pragma unroll
            for (int x = 0; x < 8; ++x) dst[x] = o[x];
        }
    }
}

}  // namespace

cudaError_t launch_qcs_project(const float* y, const float* lo, const float* hi, float* u, int B, int H, int W,
                               cudaStream_t st, unsigned long long* launches)
{
    const long long nblk = (long long)B * (H / 8) * (W / 8);
    const long long grid = (nblk + QB - 1) / QB;
    if (grid > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    const int vec_ok = ((reinterpret_cast<size_t>(y) | reinterpret_cast<size_t>(u)) & 15) == 0;
    qcs_project_kernel<<<(unsigned)grid, QB * 8, 0, st>>>(y, lo, hi, u, H, W, nblk, vec_ok);
    ++*launches;
    return cudaGetLastError();
}

}  // namespace tnrd

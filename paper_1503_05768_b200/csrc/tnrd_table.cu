// tnrd_table.cu -- piecewise-linear tables of the influence functions.
//
// Two uses of one evaluator (PHI = 2 of the fused stage kernel: one table gather + one FFMA per response):
//   * triangular-shaped radial basis phi_t: with equidistant centres and gamma = spacing, sum_j w_j phi_t
//     IS the linear interpolant of the weights at the centres ("any input z only involves two basis functions",
//     PAPER.md:564) -- a 65-node table (the 63 weights and a zero node on either side), exact;
//   * the authors' own speed-up of the Gaussian basis: "the function values at discrete points are
//     precomputed and stored in a lookup-table, then the function values at point z can be retrieved efficiently using
//     linear interpolation" -- 4096 nodes from 6 gamma below the lowest centre to 6 gamma above the highest (step 0.18 for
//     the configs' centres), every node the full 63-term sum.  An approximation: |error| <= h^2/8 max|phi''| per response.
// A triangular basis that does not meet the exact condition is tabulated on the fine grid as well (then approximate).
//
// Table of filter i: TNRD_TAB_NODES entries (phi(c_m) / s, (phi(c_{m+1}) - phi(c_m)) / s), c_m = c0 + m h.
// Header (device, 4 floats): a = 1 / (s h), b = -c0 / h, tmax = nodes - 1, exact flag; the kernel evaluates
// t = clamp(a z' + b, 0, tmax), j = min(floor(t), nodes - 2), phi / s = entry_j.x + (t - j) entry_j.y.
#include "tnrd_internal.h"

namespace tnrd {

namespace {

__global__ void __launch_bounds__(256)
build_phi_table_kernel(const float* __restrict__ rbf_w, const float* __restrict__ rbf_mu, float gamma, int basis,
                       float2* __restrict__ tab, float* __restrict__ hdr)
{
    const int rec = blockIdx.x;                                   // (stage, filter)
    const int m = blockIdx.y * blockDim.x + threadIdx.x;          // node
    const float s = sqrtf(1.4426950408889634f / (2.0f * gamma * gamma));
    // grid of nodes, from the centres (every thread computes the same few numbers)
    const float mu0 = rbf_mu[0], delta = (rbf_mu[TNRD_M - 1] - mu0) / (float)(TNRD_M - 1);
    float lo = mu0, hi = mu0;
    bool equi = delta > 0.0f;
    for (int j = 0; j < TNRD_M; ++j) {
        const float mj = rbf_mu[j];
        lo = fminf(lo, mj); hi = fmaxf(hi, mj);
        equi = equi && fabsf(mj - fmaf((float)j, delta, mu0)) <= 1.5e-7f * (fabsf(mu0) + 62.0f * delta);
    }
    const bool exact = basis == 1 && equi && fabsf(gamma - delta) <= 1e-5f * delta;
    int nodes;
    float c0, h;
    if (exact) { nodes = TNRD_M + 2; c0 = mu0 - delta; h = delta; }
    else {
        const float reach = basis == 1 ? gamma : 6.0f * gamma;
        nodes = TNRD_TAB_NODES; c0 = lo - reach; h = (hi + reach - c0) / (float)(TNRD_TAB_NODES - 1);
    }
    if (rec == 0 && m == 0) {
        hdr[0] = 1.0f / (s * h); hdr[1] = -c0 / h; hdr[2] = (float)(nodes - 1); hdr[3] = exact ? 1.0f : 0.0f;
    }
    if (m >= TNRD_TAB_NODES) return;
    const float* __restrict__ w = rbf_w + (size_t)rec * TNRD_M;
    float val[2];
#pragma unroll
    for (int q = 0; q < 2; ++q) {                                 // phi at nodes m and m + 1
        const int mm = m + q;
        float acc = 0.0f;
        if (mm < nodes) {
            if (exact) acc = (mm >= 1 && mm <= TNRD_M) ? w[mm - 1] : 0.0f;
            else {
                const float z = c0 + (float)mm * h;
                for (int j = 0; j < TNRD_M; ++j) {
                    const float d = z - rbf_mu[j];
                    if (basis == 1) acc += w[j] * fmaxf(0.0f, 1.0f - fabsf(d) / gamma);
                    else acc += w[j] * expf(-(d * d) / (2.0f * gamma * gamma));
                }
            }
        }
        val[q] = acc;
    }
    float2 e = make_float2(0.0f, 0.0f);
    if (m < nodes) e = make_float2(val[0] / s, m + 1 < nodes ? (val[1] - val[0]) / s : 0.0f);
    tab[(size_t)rec * TNRD_TAB_NODES + m] = e;
}

}  // namespace

cudaError_t launch_build_table(const float* rbf_w, const float* rbf_mu, float gamma, int TN, int basis, float* tab,
                               float* hdr, cudaStream_t st, unsigned long long* launches)
{
    if (TN <= 0) return cudaSuccess;
    build_phi_table_kernel<<<dim3((unsigned)TN, TNRD_TAB_NODES / 256), 256, 0, st>>>(
        rbf_w, rbf_mu, gamma, basis, reinterpret_cast<float2*>(tab), hdr);
    ++*launches;
    return cudaGetLastError();
}

}  // namespace tnrd

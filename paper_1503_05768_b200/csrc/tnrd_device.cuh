// tnrd_device.cuh -- device helpers shared by the stage kernels (forward: tnrd_fused.cu, backward: tnrd_bwd.cu).
#pragma once
#include "tnrd_internal.h"

namespace tnrd {

// 2^{-x}: the negation rides on the MUFU operand
__device__ __forceinline__ float ex2_neg(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(-x));
    return y;
}

// asynchronous global -> shared copies (LDGSTS): no register staging, every copy of a loop is in flight at once
__device__ __forceinline__ void cp_async4(float* smem_dst, const float* gmem_src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::
                 "r"((unsigned)__cvta_generic_to_shared(smem_dst)), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async16(float* smem_dst, const float* gmem_src)      // both 16-byte aligned
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::
                 "r"((unsigned)__cvta_generic_to_shared(smem_dst)), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

template <int N>
__device__ __forceinline__ void lds_vec(const float* __restrict__ p, float (&d)[N])
{
#pragma unroll
    for (int q = 0; q < N / 4; ++q) {
        const float4 t = *reinterpret_cast<const float4*>(p + 4 * q);
        d[4 * q + 0] = t.x; d[4 * q + 1] = t.y; d[4 * q + 2] = t.z; d[4 * q + 3] = t.w;
    }
}

// One window row of either filtering for a 4x2 block.  acc[p] holds the two output rows of column p as one pair;
// trow = row of tap pairs P[rho][b] = (k[rho-1][b], k[rho][b]).  REV = false: forward filter (a2), pair = (row 0,
// row 1), rho = KS - wr, source column p + 2r - b.  REV = true: transposed filter (a4), pair = (row 1, row 0),
// rho = wr, source column p + b.
// SHIFT: extra column offset of the source window (the source row is read from a 16-byte aligned address).
template <int KS, bool REV, int SHIFT = 0>
__device__ __forceinline__ void rowstep(const float* __restrict__ srow, const float* __restrict__ trow,
                                        float2 (&acc)[4])
{
    constexpr int TS = prm_ts(KS), NV = (4 + KS - 1 + SHIFT + 3) / 4;
    float row[NV * 4], kp[TS];
    lds_vec(srow, row);
    lds_vec(trow, kp);
#pragma unroll
    for (int b = 0; b < KS; ++b)
#pragma unroll
        for (int p = 0; p < 4; ++p) {
            const float x = REV ? row[p + b + SHIFT] : row[p + (KS - 1) - b + SHIFT];
            acc[p] = __ffma2_rn(make_float2(kp[2 * b], kp[2 * b + 1]), make_float2(x, x), acc[p]);
        }
}

// The first and the last window row of a filtering touch only ONE of the two output rows (their tap pairs are
// (k[ks-1][b], 0) and (0, k[0][b])): scalar FFMAs on that half, at half the FMA-pipe cycles of the packed form.
// HALF = 0: the .x halves with the first tap of each pair, HALF = 1: the .y halves with the second.
template <int KS, bool REV, int SHIFT, int HALF>
__device__ __forceinline__ void rowstep_half(const float* __restrict__ srow, const float* __restrict__ trow,
                                             float2 (&acc)[4])
{
    constexpr int TS = prm_ts(KS), NV = (4 + KS - 1 + SHIFT + 3) / 4;
    float row[NV * 4], kp[TS];
    lds_vec(srow, row);
    lds_vec(trow, kp);
#pragma unroll
    for (int b = 0; b < KS; ++b)
#pragma unroll
        for (int p = 0; p < 4; ++p) {
            const float x = REV ? row[p + b + SHIFT] : row[p + (KS - 1) - b + SHIFT];
            if (HALF == 0) acc[p].x = fmaf(kp[2 * b], x, acc[p].x);
            else acc[p].y = fmaf(kp[2 * b + 1], x, acc[p].y);
        }
}

}  // namespace tnrd

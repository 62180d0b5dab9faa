// tnrd_tc.cu -- the stage kernel with both filterings on the 5th-generation tensor cores (tcgen05.mma, accumulators
// in tensor memory) and the update fused in: rows a1-a5 of the hot path in ONE pass, u_t written by the same kernel.
//
//   u_t = u - ( sum_i kbar_i * phi_i(k_i * u~) + lambda (u - f) )          Main Eq. 7
//
// The two filterings are the only dense contractions of the path (PAPER.md:70 "K_i u <=> k_i * u", :125 the rot180
// bank, :387-389 the patch-matrix form U k); everything else is the point-wise influence function.
// One CTA owns a column strip of 256 phi columns (128 tensor-memory lanes x 2 pixels) and walks down it two phi rows
// (one "batch" = 512 pixels) at a time:
//
//   a1  loader warps gather u rows through the mirror map into a ring of shared-memory rows,
//       as 16-byte CELLS (row, g) = u~[row][2g .. 2g+3] -- every pixel twice, so that the 4-pixel window of ANY
//       even column starts on a 16-byte boundary -- split x = hi + lo with hi = the top 19 bits (a TF32 number);
//   a2  z = k * u~ as an implicit GEMM with NO im2col: M = 128 lanes (pixel pairs), K = (tap row a, window column
//       c = 0..7) read straight from the cell ring by a K-major, unswizzled shared-memory descriptor whose two 16-byte
//       chunks are the cells g and g + 2 (the window u~[row + a][2g .. 2g+7]), N = (filter i, pixel j of the pair) with
//       the Toeplitz operand B[(a, c)][(i, j)] = k_i[K-1-a][K-1-(c-j)].  Three TF32 products hi*hi + hi*lo + lo*hi with
//       fp32 accumulation in tensor memory: fp32-level accuracy (a single TF32 pass would not hold the tolerance).
//   a3  phi warps read z from tensor memory (tcgen05.ld), evaluate all 63 Gaussians by the factorised form
//       (tnrd_internal.h "fact": 3 ex2 per group of 13 centres, groups that are dead for the whole warp skipped), and
//       write v = phi(z) back IN PLACE as BF16 pairs (hi, lo) (tcgen05.st);
//   a4  the transposed bank as a SCATTER table, A = v straight from tensor memory (no shared-memory round trip):
//       T[lane][(a, xo)] = sum_{i,j} v_i[pixel j of the lane] k_i[a][j + 2r - xo] is what the lane's two pixels add
//       to output row py - a at columns 2g - 2r + xo.  The fold over a happens inside tensor memory (the two rows of
//       a batch accumulate into the same table one 8-column block apart), the fold over neighbouring lanes and over
//       batches in shared memory, in a fixed order (deterministic, no atomics);
//   a5  the thread that completes an output pixel applies the reaction term and writes u_t.
//
// Strips overlap by 2r phi columns and row segments by 2r phi rows (recomputed) so that a CTA completes its own
// outputs: no partial sums in HBM, no second kernel, 12 B of DRAM traffic per pixel-stage.
// When one stage of a call has too few such units to fill the GPU (a single 321x481 image), the filter bank is cut into
// chunks as well (plan_stage_tc): a unit then evaluates only its chunk's filters and writes the partial sum of Eq. 7's
// diffusion term to scratch, and tc_update_kernel adds the chunks in a fixed order and applies the reaction term.
// Warp roles: 24 phi warps (6 per tensor-memory lane quarter, sharing the quarter's filter pairs through a ticket
// counter), 4 drain warps (fold + a5), 1 MMA-issuing warp, 2 loader warps; mbarrier pipelines between them (u row pairs,
// z double-buffered, scatter table).
#include <cuda_bf16.h>
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstdlib>

#include "tnrd_internal.h"
#include "tnrd_device.cuh"

namespace tnrd {

namespace {

#ifndef TNRD_TC_PHI_WARPS
#define TNRD_TC_PHI_WARPS 24
#endif
#ifndef TNRD_TC_LOAD_WARPS
#define TNRD_TC_LOAD_WARPS 2    // one warp delivered a row pair in ~ 6 k clocks: the floor of a batch with few filters (a third: same)
#endif
constexpr int TC_PHI_WARPS = TNRD_TC_PHI_WARPS, TC_LOAD_WARPS = TNRD_TC_LOAD_WARPS;   // phi warps: a multiple of 4 (TC_PHI_WARPS / 4 per lane quarter)
constexpr int TC_DRAIN_WARPS = 4;                               // one per lane quarter, right after the phi warps
constexpr int TC_MMA_WARP = TC_PHI_WARPS + TC_DRAIN_WARPS;      // warp index of the MMA issuer
constexpr int TC_THREADS = (TC_PHI_WARPS + TC_DRAIN_WARPS + 1 + TC_LOAD_WARPS) * 32;
constexpr int TC_CW = 132;                                      // cells per ring row (130 used)
constexpr int TC_CWU = 130;
constexpr int TC_NP = 6;                                        // row pairs in the ring
constexpr int TC_NKP_MAX = 48;                                  // filters (padded to a multiple of 8)
constexpr int TC_TCOL = 8 * TC_NKP_MAX;                         // first tensor-memory column of the scatter table

template <int KS>
struct TcCfg {
    static constexpr int R = (KS - 1) / 2;
    static constexpr int OW = 256 - 2 * R;                      // output columns a strip completes
    static constexpr int NSB = KS + 1;                          // 8-column blocks of one scatter MMA (the last one is padding)
    static constexpr int NSC = 8 * NSB;                         // its N
    static constexpr int XK = R + 1;                            // float2 slots per (block, lane) of the exchange buffer
    static constexpr int PRM = prm_stride(KS);
    // shared memory (bytes)
    static constexpr int SM_UHI = 0;
    static constexpr int U_BYTES = TC_NP * 2 * TC_CW * 16;
    static constexpr int SM_ULO = SM_UHI + U_BYTES;
    static constexpr int SM_BFH = SM_ULO + U_BYTES;
    static constexpr int BF_BYTES = KS * 2 * (2 * TC_NKP_MAX) * 16;
    static constexpr int SM_BFL = SM_BFH + BF_BYTES;
    static constexpr int SM_BS = SM_BFL + BF_BYTES;
    static constexpr int BS_BYTES = TC_NKP_MAX * NSC * 16;
    static constexpr int SM_COEF = SM_BS + BS_BYTES;
    static constexpr int COEF_BYTES = TC_NKP_MAX * TNRD_FG * TNRD_FSTRIDE * 4;
    static constexpr int SM_X = SM_COEF + COEF_BYTES;
    static constexpr int X_BYTES = (KS + 1) * XK * 128 * 8;
    static constexpr int SM_O = SM_X + X_BYTES;
    static constexpr int O_BYTES = 8 * 128 * 8;
    static constexpr int SM_BAR = SM_O + O_BYTES;
    static constexpr int SMEM = SM_BAR + 256;
};

// workspace of one stage (global memory, written by tc_prep_kernel): forward operand hi, lo (TF32), scatter operand
__host__ __device__ constexpr size_t tc_ws_bf_bytes(int ks, int nkp) { return (size_t)ks * 2 * (2 * nkp) * 16; }
__host__ __device__ constexpr size_t tc_ws_bs_bytes(int ks, int nkp) { return (size_t)nkp * (8 * (ks + 1)) * 16; }
__host__ __device__ constexpr size_t tc_ws_stage_bytes(int ks, int nkp) { return 2 * tc_ws_bf_bytes(ks, nkp) + tc_ws_bs_bytes(ks, nkp); }

// ---- PTX wrappers ----------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
// Shared-memory operand descriptor, K-major and unswizzled: 8 rows of a core matrix 16 bytes apart, `sbo` between 8-row
// groups, `lbo` between the two 16-byte K chunks of one MMA.  64 bits: start >> 4 in bits 0-13, lbo >> 4 in 16-29,
// sbo >> 4 in 32-45, version 1 in bit 46 -- kept as two words (umma_desc_lo / umma_desc_hi below).
// instruction descriptor: fp32 accumulate, A and B K-major, fmt 1 = BF16, 2 = TF32
__device__ __forceinline__ uint32_t umma_idesc(int fmt, int M, int N)
{
    return (1u << 4) | ((uint32_t)fmt << 7) | ((uint32_t)fmt << 10) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}
// MMAs with the descriptors as (low, high) words and the accumulate flag as a constant: the issuing thread adds an offset
// to the low word (the 14-bit address field, no carry) instead of building a 64-bit descriptor per instruction.  What is
// left of the issue time is the tensor pipe's: about 73 clocks per forward MMA (M 128, K 8: the A operand is read from
// shared memory) and 240 per scatter MMA (A from tensor memory, every one into the accumulator of the last) -- 42 + nkp
// MMAs per batch, 5 k clocks with 8 filters, which is what a batch of a small filter chunk costs at least.
__device__ __forceinline__ uint32_t umma_desc_lo(uint32_t saddr, uint32_t lbo) { return ((saddr >> 4) & 0x3FFF) | (((lbo >> 4) & 0x3FFF) << 16); }
__device__ __forceinline__ uint32_t umma_desc_hi(uint32_t sbo) { return ((sbo >> 4) & 0x3FFF) | (1u << 14); }
template <bool ACC>
__device__ __forceinline__ void umma_tf32_ss2(uint32_t d, uint32_t a_lo, uint32_t a_hi, uint32_t b_lo, uint32_t b_hi, uint32_t idesc)
{
    asm volatile("{\n\t.reg .b64 da, db;\n\t.reg .pred p;\n\tsetp.ne.b32 p, %6, 0;\n\t"
                 "mov.b64 da, {%1, %2};\n\tmov.b64 db, {%3, %4};\n\t"
                 "tcgen05.mma.cta_group::1.kind::tf32 [%0], da, db, %5, p;\n\t}\n"
                 :: "r"(d), "r"(a_lo), "r"(a_hi), "r"(b_lo), "r"(b_hi), "r"(idesc), "n"(ACC ? 1 : 0) : "memory");
}
template <bool ACC>
__device__ __forceinline__ void umma_bf16_ts2(uint32_t d, uint32_t a_tmem, uint32_t b_lo, uint32_t b_hi, uint32_t idesc)
{
    asm volatile("{\n\t.reg .b64 db;\n\t.reg .pred p;\n\tsetp.ne.b32 p, %5, 0;\n\tmov.b64 db, {%2, %3};\n\t"
                 "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], db, %4, p;\n\t}\n"
                 :: "r"(d), "r"(a_tmem), "r"(b_lo), "r"(b_hi), "r"(idesc), "n"(ACC ? 1 : 0) : "memory");
}
__device__ __forceinline__ void umma_commit(uint64_t* bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" :: "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" :: "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
{
    asm volatile("{\n\t.reg .pred p;\n\tWAIT_%=:\n\t"
                 "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
                 "@p bra DONE_%=;\n\tbra WAIT_%=;\n\tDONE_%=:\n\t}\n" :: "r"(smem_u32(bar)), "r"(parity) : "memory");
}
// The same for the warps that wait most of the time (MMA issuer, loader, drain): a spinning try_wait loop takes issue
// slots from the phi warps on its scheduler (20 % of all issued instructions in a profile), so back off between polls.
#ifndef TNRD_TC_SLEEP_DRAIN
#define TNRD_TC_SLEEP_DRAIN 200      // 200 .. 2000 ns: no difference in the stage time (measured)
#define TNRD_TC_SLEEP_LOAD 200
#define TNRD_TC_SLEEP_MMA 200
#endif
template <unsigned NS>
__device__ __forceinline__ void mbar_wait_idle(uint64_t* bar, uint32_t parity)
{
    for (;;) {
        uint32_t done;
        asm volatile("{\n\t.reg .pred p;\n\t"
                     "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
                     "selp.u32 %0, 1, 0, p;\n\t}\n" : "=r"(done) : "r"(smem_u32(bar)), "r"(parity) : "memory");
        if (done) return;
        __nanosleep(NS);
    }
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tmem_ld4(uint32_t taddr, uint32_t (&r)[4])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(taddr));
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&r)[16])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
                   "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
                 : "r"(taddr));
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_st4(uint32_t taddr, const uint32_t (&r)[4])
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1,%2,%3,%4};"
                 :: "r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]) : "memory");
}
__device__ __forceinline__ void tmem_st_wait() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void bar_drain() { asm volatile("bar.sync 1, %0;" :: "n"(TC_DRAIN_WARPS * 32) : "memory"); }

__device__ __forceinline__ float ex2f(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// Factorised influence function (tnrd_internal.h "fact"; PAPER.md:553 with equidistant centres, :117) of the two
// response pairs z[0], z[1] of one filter; crec = the filter's TNRD_FG group records in shared memory (broadcast
// loads; scaled at kernel start, see there).  Per response: ONE pair rho0 = 2^{kappa d0}, 1/rho0 for the middle
// group; the other groups' rho_g = 2^{kappa d_g} = rho0 K_g with the constants K_g = 2^{kappa (d_g - d0)} staged in
// the group record (anchors are a fixed number of centres apart), capped at R = 2^{kappa D} (beyond |d_g| = D the
// Gaussian factor 2^{-d_g^2} has flushed to zero, so the cap changes no value and keeps rho^S finite): 2 + TNRD_FG
// ex2 per response instead of 3 TNRD_FG.  The shared FMA / ALU dispatch is what binds this kernel, so
// the scaling and the cap are ONE single-cycle instruction per value, x = sat(rho0 K_g / R) (a NaN response is
// flushed to 0 here and comes back through the Gaussian factor).
// A group is skipped when its Gaussian factor is zero for every response of the warp (an exact 0 either way): the
// loop runs over the groups within reach D of the warp's smallest .. largest response (NaN responses keep every
// group live); ganch = mu' of the first group's anchor, ginv = 1 / (anchor spacing).
// The range is taken per lane first -- x = (z -+ D - ganch) * ginv as ONE fused multiply-add with the offsets
// olo = -(D + ganch) ginv, ohi = (D - ganch) ginv, clamped, rounded down / up -- and then reduced over the warp as small
// integers (floor and ceil are monotone: the same range as rounding the warp's extreme responses).  The min / max over a
// lane's four responses propagate NaN, and the order of the two clamps sends a NaN to the full range on either side.
// D leaves a margin (the factor flushes to zero from d^2 = 126 on, D^2 = 127.7), so the rounding of the fused form
// cannot cut a group that still contributes.
__device__ __forceinline__ int tc_phi_fact(const float* __restrict__ crec, float kappa, float olo, float ohi, float ginv,
                                           const float2 (&z)[2], float2 (&v)[2])
{
    constexpr int S = TNRD_FS, GC = TNRD_FG / 2;
    float zlo, zhi, t0, t1;
    asm("min.NaN.f32 %0, %1, %2;" : "=f"(t0) : "f"(z[0].x), "f"(z[0].y));
    asm("min.NaN.f32 %0, %1, %2;" : "=f"(t1) : "f"(z[1].x), "f"(z[1].y));
    asm("min.NaN.f32 %0, %1, %2;" : "=f"(zlo) : "f"(t0), "f"(t1));
    asm("max.NaN.f32 %0, %1, %2;" : "=f"(t0) : "f"(z[0].x), "f"(z[0].y));
    asm("max.NaN.f32 %0, %1, %2;" : "=f"(t1) : "f"(z[1].x), "f"(z[1].y));
    asm("max.NaN.f32 %0, %1, %2;" : "=f"(zhi) : "f"(t0), "f"(t1));
    // clamped BEFORE the conversion (infinite responses must not overflow the + 1); NaN -> -8 resp. +8
    const float xl = fminf(fmaxf(fmaf(zlo, ginv, olo), -8.0f), 8.0f);
    const float xh = fmaxf(fminf(fmaf(zhi, ginv, ohi), 8.0f), -8.0f);
    const int g0 = max(0, __reduce_min_sync(0xffffffffu, __float2int_rd(xl)) + 1);
    const int g1 = min(TNRD_FG - 1, __reduce_max_sync(0xffffffffu, __float2int_ru(xh)) - 1);
    if (g0 > g1) return 0;
    // the shared exponential pair (middle group)
    float2 rho0[2], rhoi0[2];
    {
        const float c0 = crec[GC * TNRD_FSTRIDE];
#pragma unroll
        for (int p = 0; p < 2; ++p) {
            const float2 e = __fmul2_rn(__fadd2_rn(z[p], make_float2(c0, c0)), make_float2(kappa, kappa));
            rho0[p] = make_float2(ex2f(e.x), ex2f(e.y));
            rhoi0[p] = make_float2(ex2f(-e.x), ex2f(-e.y));
        }
    }
#pragma unroll 1
    for (int g = g0; g <= g1; ++g) {
        float c[TNRD_FSTRIDE];
        lds_vec(crec + g * TNRD_FSTRIDE, c);
        float2 gg[2], rho[2], rhoi[2], h[2], hl[2];
#pragma unroll
        for (int p = 0; p < 2; ++p) {
            const float2 d = __fadd2_rn(z[p], make_float2(c[0], c[0]));
            const float2 t = __fmul2_rn(d, d);
            gg[p] = make_float2(ex2f(-t.x), ex2f(-t.y));
            // x = min(rho_g, R) / R, rho_g = rho0 K_g: c[14] = K_g / R, and the saturation to [0, 1] IS the cap
            rho[p] = make_float2(__saturatef(rho0[p].x * c[14]), __saturatef(rho0[p].y * c[14]));
            rhoi[p] = make_float2(__saturatef(rhoi0[p].x * c[15]), __saturatef(rhoi0[p].y * c[15]));
        }
#pragma unroll
        for (int p = 0; p < 2; ++p) {
            h[p] = __ffma2_rn(make_float2(c[1], c[1]), rho[p], make_float2(c[2], c[2]));
            hl[p] = __ffma2_rn(make_float2(c[S + 2], c[S + 2]), rhoi[p], make_float2(c[S + 3], c[S + 3]));
        }
#pragma unroll
        for (int q = 2; q <= S; ++q)
#pragma unroll
            for (int p = 0; p < 2; ++p) h[p] = __ffma2_rn(h[p], rho[p], make_float2(c[1 + q], c[1 + q]));
#pragma unroll
        for (int q = 2; q < S; ++q)
#pragma unroll
            for (int p = 0; p < 2; ++p) hl[p] = __ffma2_rn(hl[p], rhoi[p], make_float2(c[S + 2 + q], c[S + 2 + q]));
#pragma unroll
        for (int p = 0; p < 2; ++p) {
            // three register-pair operands make a packed FMA take 3.3 issue cycles instead of 2: two scalar FMAs here
            h[p] = make_float2(fmaf(hl[p].x, rhoi[p].x, h[p].x), fmaf(hl[p].y, rhoi[p].y, h[p].y));
            v[p] = make_float2(fmaf(gg[p].x, h[p].x, v[p].x), fmaf(gg[p].y, h[p].y, v[p].y));
        }
    }
    return g1 - g0 + 1;
}

// Direct form (one ex2 per Gaussian) for centre sets the factorisation does not cover; (-mu', w') pairs from the
// staged record in global memory (uniform loads).  Rare path.
__device__ __forceinline__ void tc_phi_direct(const float* __restrict__ pairs, const float2 (&z)[2], float2 (&v)[2])
{
#pragma unroll 3
    for (int j = 0; j < TNRD_M; ++j) {
        const float2 mw = __ldg(reinterpret_cast<const float2*>(pairs) + j);
#pragma unroll
        for (int p = 0; p < 2; ++p) {
            const float2 d = __fadd2_rn(z[p], make_float2(mw.x, mw.x));
            const float2 t = __fmul2_rn(d, d);
            v[p] = __ffma2_rn(make_float2(ex2f(-t.x), ex2f(-t.y)), make_float2(mw.y, mw.y), v[p]);
        }
    }
}

// v = (v.x, v.y) -> packed BF16 pairs: hi = (bf16(v.x) | bf16(v.y) << 16), lo = the same of the remainders
__device__ __forceinline__ void split_bf16(float2 v, uint32_t& hi, uint32_t& lo)
{
    asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(hi) : "f"(v.y), "f"(v.x));
    const float hx = __uint_as_float(hi << 16), hy = __uint_as_float(hi & 0xFFFF0000u);
    asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(lo) : "f"(v.y - hy), "f"(v.x - hx));
}

// Host entry point, one image: the input plane is still arriving (copy engine, in blocks of 32 whole rows, so every
// block ends on a 128-byte line and no line is read into L1 before all of it is there) while the first stage runs.
// arrived[1 + b] != 0 once block b is there.  A CTA reads its rows top to bottom, so it checks each block as it enters
// it: waits until the block of row `need - 1` is there and returns the first row of the next block; gives up after
// about two seconds (word 0, reported by the entry point) rather than hang the GPU.
__device__ __forceinline__ int tc_wait_rows(unsigned* arrived, int need, int have)
{
    if (have >= need) return have;
    const int blk = (need - 1) >> 5;
    int spins = 0;
    for (;;) {
        unsigned v;
        asm volatile("ld.acquire.sys.global.u32 %0, [%1];" : "=r"(v) : "l"(arrived + 1 + blk) : "memory");
        if (v) break;
        __nanosleep(500);
        if (++spins > (1 << 22)) { atomicExch(arrived, 1u); break; }
    }
    return (blk + 1) << 5;
}

// One 16-byte cell (row, g) = u~[row][2g .. 2g+3] of the u ring, through the mirror map, split
// x = hi + lo with hi = the top 19 bits (a TF32 number; lo is exact): the four loads ...
__device__ __forceinline__ void tc_cell_load(const float* __restrict__ u_img, int H, int W, int urow, int ucol, float (&v)[4])
{
    const float* __restrict__ grow = u_img + (size_t)mirror_clamp(urow, H) * W;
#pragma unroll
    for (int e = 0; e < 4; ++e) v[e] = __ldg(grow + mirror_clamp(ucol + e, W));
}
// ... and the two stores
__device__ __forceinline__ void tc_cell_store(unsigned char* smem_hi, unsigned char* smem_lo, int cell_byte, const float (&v)[4])
{
    float h[4], l[4];
#pragma unroll
    for (int e = 0; e < 4; ++e) {
        h[e] = __uint_as_float(__float_as_uint(v[e]) & 0xFFFFE000u);
        l[e] = v[e] - h[e];
    }
    *reinterpret_cast<float4*>(smem_hi + cell_byte) = make_float4(h[0], h[1], h[2], h[3]);
    *reinterpret_cast<float4*>(smem_lo + cell_byte) = make_float4(l[0], l[1], l[2], l[3]);
}

// ---- operand staging kernel: Toeplitz operands of both banks from the staged records (scaled taps k' = s k) ------
//   forward  BF[(2a + cc)][n = 2i + j][e]   = k'_i[K-1-a][K-1-(4cc + e - j)]   (TF32 hi / lo)
//   scatter  BS[pass][kp / 8][n = 8 blk + xo][kp % 8],  kp = 4i + 2s + j  (s = 0: the hi half of v, 1: the lo half)
//            = hi(k'_i[blk][j + 2r - xo]) for pass 0;  lo(k') for pass 1, s = 0;  0 for pass 1, s = 1
__global__ void tc_prep_kernel(const float* __restrict__ prm, int T, int N_k, int nkp, int ks, unsigned char* __restrict__ ws)
{
    const int PRM = prm_stride(ks), R = (ks - 1) / 2, NSC = 8 * (ks + 1);
    const size_t bfb = tc_ws_bf_bytes(ks, nkp), stb = tc_ws_stage_bytes(ks, nkp);
    const int n_bf = ks * 2 * 2 * nkp * 4, n_bs = nkp * NSC * 8;
    for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < T * (n_bf + n_bs); idx += gridDim.x * blockDim.x) {
        const int t = idx / (n_bf + n_bs), q = idx - t * (n_bf + n_bs);
        const float* rec = prm + (size_t)t * N_k * PRM;
        unsigned char* wst = ws + (size_t)t * stb;
        if (q < n_bf) {
            const int e = q & 3, n = (q >> 2) % (2 * nkp), kc = (q >> 2) / (2 * nkp);
            const int a = kc >> 1, cc = kc & 1, i = n >> 1, j = n & 1, b = 4 * cc + e - j;
            float v = 0.0f;
            if (i < N_k && b >= 0 && b < ks) v = rec[(size_t)i * PRM + prm_tap(ks, ks - 1 - a, ks - 1 - b)];
            const float h = __uint_as_float(__float_as_uint(v) & 0xFFFFE000u);
            reinterpret_cast<float*>(wst)[q] = h;
            reinterpret_cast<float*>(wst + bfb)[q] = v - h;
        } else {
            const int qq = q - n_bf;
            const int k8 = qq & 7, n = (qq >> 3) % NSC, kc = ((qq >> 3) / NSC) % (nkp / 2), pass = (qq >> 3) / NSC / (nkp / 2);
            const int kp = 8 * kc + k8, i = kp >> 2, s = (kp >> 1) & 1, j = kp & 1, blk = n >> 3, xo = n & 7, b = j + 2 * R - xo;
            float v = 0.0f;
            if (i < N_k && blk < ks && b >= 0 && b < ks) v = rec[(size_t)i * PRM + prm_tap(ks, blk, b)];
            const __nv_bfloat16 h = __float2bfloat16_rn(v);
            const __nv_bfloat16 l = __float2bfloat16_rn(v - __bfloat162float(h));
            reinterpret_cast<__nv_bfloat16*>(wst + 2 * bfb)[qq] = pass == 0 ? h : (s == 0 ? l : __float2bfloat16_rn(0.0f));
        }
    }
}

// ---- the stage kernel ------------------------------------------------------------------------------------------
// grid: one CTA per unit = (image, row segment, strip); the unit completes output rows [ys0, ys1) x columns
// [xs OW, xs OW + OW) from phi rows [ys0, ys1 + 2r) x phi columns [xs OW, xs OW + 256) (phi coordinates = image + r).
template <int KS, bool STATS>
__global__ void __launch_bounds__(TC_THREADS, 1)
stage_tc_kernel(StageArgs a, const unsigned char* __restrict__ ws, int nkp_all, int nxs, int nys, int seg_rows, int nchunk,
                float* __restrict__ part)
{
    using C = TcCfg<KS>;
    constexpr int R = C::R;
    extern __shared__ __align__(1024) unsigned char smem[];
    __shared__ uint32_t tmem_base_s;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + C::SM_BAR);
    uint64_t* pfull = bars;                     // [TC_NP] loader -> MMA: row pair landed
    uint64_t* pempty = bars + TC_NP;            // [TC_NP] MMA -> loader: row pair no longer read
    uint64_t* zfull = bars + 2 * TC_NP;         // [2] forward bank of a batch done
    uint64_t* vdone = zfull + 2;                // [2] phi warps wrote v of a batch
    uint64_t* tfull = vdone + 2;                // scatter table of a batch complete
    uint64_t* tfree = tfull + 1;                // scatter table read out

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    // a unit = (image, filter chunk, row segment, strip).  nchunk > 1 (images too small to fill the GPU otherwise): the CTA
    // takes filters [f0, f0 + nkp) of the bank and stores its partial transposed-bank sums to part[chunk][image][H][W];
    // tc_update_kernel adds the chunks in fixed order and applies the reaction term.
    int unit = blockIdx.x;
    const int xs = unit % nxs; unit /= nxs;
    const int ysg = unit % nys; unit /= nys;
    const int chunk = unit % nchunk; unit /= nchunk;
    const int img = unit;
    const int nkp = nkp_all / nchunk, f0 = chunk * nkp;         // this CTA's filters (a multiple of 8)
    const int X0 = xs * C::OW;                                  // phi column of lane 0, pixel 0 = image column X0 - r
    const int row_hi = a.row_hi > 0 ? a.row_hi : a.H;
    const int ys0 = a.row_lo + ysg * seg_rows, ys1 = min(row_hi, ys0 + seg_rows);
    const int rows_out = ys1 - ys0;
    const int NB = (rows_out + 2 * R - 1) / 2 + 1;              // batches: phi rows ys0 .. ys0 + 2 NB - 1
    const int NPAIRS = NB + R;                                  // u row pairs: u~ rows ys0 .. ys0 + 2 NB + 2r - 1
    const float* __restrict__ u_img = a.u_in + (size_t)img * a.H * a.W;

    // Programmatic dependent launch (launch_tc_ks): the next kernel of the stream may be scheduled as soon as every CTA
    // of this one is running -- its CTAs take SMs as ours leave them and set themselves up -- and this kernel waits for
    // the previous one (complete, writes visible) before it touches anything that kernel may have written: at once when
    // that includes our operands (first stage of a call), else after the set-up.
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    if (a.pdl != 2) asm volatile("griddepcontrol.wait;" ::: "memory");
    // ---- setup: operands and coefficients to shared memory, barriers, tensor memory ----
    {
        // forward operand: cells [2 KS chunks][2 nkp_all columns] -> this CTA's 2 nkp columns, compact
        const size_t bfb = tc_ws_bf_bytes(KS, nkp_all);
        for (int i = tid; i < 2 * KS * 2 * nkp; i += TC_THREADS) {
            const int kc = i / (2 * nkp), n = i - kc * 2 * nkp;
            const size_t src = ((size_t)kc * 2 * nkp_all + 2 * f0 + n) * 4;
            cp_async16(reinterpret_cast<float*>(smem + C::SM_BFH) + 4 * i, reinterpret_cast<const float*>(ws) + src);
            cp_async16(reinterpret_cast<float*>(smem + C::SM_BFL) + 4 * i, reinterpret_cast<const float*>(ws + bfb) + src);
        }
        // scatter operand: cells [2 passes][nkp_all / 2 K chunks][NSC] -> the K chunks of this CTA's filters
        for (int i = tid; i < 2 * (nkp / 2) * C::NSC; i += TC_THREADS) {
            const int pass = i / ((nkp / 2) * C::NSC), r = i - pass * (nkp / 2) * C::NSC;
            const size_t src = ((size_t)(pass * (nkp_all / 2) + f0 / 2) * C::NSC + r) * 4;
            cp_async16(reinterpret_cast<float*>(smem + C::SM_BS) + 4 * i, reinterpret_cast<const float*>(ws + 2 * bfb) + src);
        }
        constexpr int CF = TNRD_FG * TNRD_FSTRIDE;              // coefficient floats per filter
        for (int i = tid; i < nkp * CF / 4; i += TC_THREADS) {
            const int fi = f0 + (4 * i) / CF, o = (4 * i) % CF;
            float* dst = reinterpret_cast<float*>(smem + C::SM_COEF) + 4 * i;
            if (fi < a.N_k) cp_async16(dst, a.prm + (size_t)fi * C::PRM + prm_fact(KS) + o);
            else *reinterpret_cast<float4*>(dst) = make_float4(0.f, 0.f, 0.f, 0.f);
        }
    }
    // The phi warps run Horner's rule in x = min(rho, R) / R with R = 2^{kappa D} (one saturating multiply does the
    // scaling by K_g AND the cap, tc_phi_fact), so the coefficient of rho^j is scaled by R^|j| and K_g, 1/K_g by 1/R.
    // |c_j| R^|j| <= |w'| 2^92 by the staging kernel's range check (tnrd_internal.h "fact").
    const float tc_kappa = __ldg(a.prm + prm_hdr(KS) + 4), tc_dmax = __ldg(a.prm + prm_hdr(KS) + 5);
    if (tid == 0) {
        for (int i = 0; i < TC_NP; ++i) { mbar_init(pfull + i, TC_LOAD_WARPS); mbar_init(pempty + i, 1); }
        for (int i = 0; i < 2; ++i) { mbar_init(zfull + i, 1); mbar_init(vdone + i, TC_PHI_WARPS); }
        mbar_init(tfull, 1);
        mbar_init(tfree, TC_DRAIN_WARPS);
        for (int i = 0; i < 4; ++i) reinterpret_cast<int*>(smem + C::SM_BAR + 192)[i] = 0;      // ticket counters
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == TC_MMA_WARP) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" :: "r"(smem_u32(&tmem_base_s)), "r"(512) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    auto finish_coefs = [&]() {
        cp_async_wait_all();
        {
            constexpr int CF = TNRD_FG * TNRD_FSTRIDE, S = TNRD_FS;
            float* cf = reinterpret_cast<float*>(smem + C::SM_COEF);
            for (int i = tid; i < nkp * CF / 4; i += TC_THREADS) {   // the same 16-byte pieces this thread copied above
                if (f0 + (4 * i) / CF >= a.N_k) continue;
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const int o = (4 * i + e) % TNRD_FSTRIDE;        // slot inside the group record
                    int pw = 0;                                      // power of R
                    if (o >= 1 && o <= S + 1) pw = S + 1 - o;        // c_S .. c_0
                    else if (o >= S + 2 && o <= 2 * S + 1) pw = 2 * S + 2 - o;   // c_-S .. c_-1
                    else if (o >= TNRD_FSTRIDE - 2) pw = -1;         // K_g, 1 / K_g
                    if (pw != 0) cf[4 * i + e] *= exp2f((float)pw * tc_kappa * tc_dmax);
                }
            }
        }
    };
    if (a.pdl == 2) {
        finish_coefs();
        asm volatile("griddepcontrol.wait;" ::: "memory");
    }
    // The first R + 1 row pairs (what the first batch needs) are gathered by ALL threads: left to the loader warp alone
    // they would cost R + 1 round trips to L2 per thread chain before the first MMA can issue.
    if (a.arrived) {       // the first R + 1 pairs: rows ys0 - 2r .. ys0 + 1 (mirrored rows above the image: rows up to 2r)
        if (tid == 0) {
            tc_wait_rows(a.arrived, max(ys0 - 2 * R, 0) + 1, 0);
            tc_wait_rows(a.arrived, min(a.H, max(ys0 + 2, 2 * R + 1)), 0);
        }
        __syncthreads();
    }
    {
        const int npre = min(NPAIRS, R + 1) * 2 * TC_CWU;
        for (int idx = tid; idx < npre; idx += TC_THREADS) {
            const int prow = idx / TC_CWU, xg = idx - prow * TC_CWU;         // prow = ring row = pair * 2 + row of the pair
            float v[4];
            tc_cell_load(u_img, a.H, a.W, ys0 + prow - 2 * R, X0 + 2 * xg - 2 * R, v);
            tc_cell_store(smem + C::SM_UHI, smem + C::SM_ULO, (prow * TC_CW + xg) * 16, v);
        }
    }
    if (a.pdl != 2) finish_coefs();
    fence_async_smem();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = tmem_base_s;
    const uint32_t sbase = smem_u32(smem);
    if (tid == 0)                                               // the pre-filled pairs: phase 0 of their barriers is complete
        for (int p = 0; p < min(NPAIRS, R + 1); ++p)
            for (int k = 0; k < TC_LOAD_WARPS; ++k) mbar_arrive(pfull + p);

    if (warp < TC_PHI_WARPS) {
        // =================================== phi warps ===================================
        // The warps of a lane quarter share the (batch, filter pair) tickets of that quarter through a counter in shared
        // memory: dead-group skipping makes the cost of a filter pair vary, and a fixed split would make every batch
        // wait for its slowest warp.  A warp arrives on vdone[b] once it holds a ticket beyond batch b (all its batch-b
        // work is written back); z is double-buffered, so a fast warp runs at most one batch ahead of the slowest.
        const int quarter = warp & 3;
        const uint32_t tl = tmem + ((uint32_t)(quarter * 32) << 16);
        const int npairs = nkp >> 1;
        const float kappa = __ldg(a.prm + prm_hdr(KS) + 4), dmax = __ldg(a.prm + prm_hdr(KS) + 5);
        const bool fact = __ldg(a.prm + prm_hdr(KS) + 6) != 0.0f;
        const float dsp = __ldg(a.prm + prm_hdr(KS) + 2);        // centre spacing in scaled units
        const float ganch = __ldg(a.prm + prm_hdr(KS) + 1) + (float)TNRD_FS * dsp, ginv = 1.0f / ((float)TNRD_FM * dsp);
        const float olo = -(dmax + ganch) * ginv, ohi = (dmax - ganch) * ginv;     // tc_phi_fact: group range of a response
        const float* coef = reinterpret_cast<const float*>(smem + C::SM_COEF);
        int* ticket = reinterpret_cast<int*>(smem + C::SM_BAR + 192) + quarter;
        int nlive = 0, nfilt = 0;                                // statistics: groups evaluated, filters evaluated
        int cur = 0;                                             // batch this warp has not yet arrived for
        bool ready = false;                                      // zfull of batch `cur` observed
        for (;;) {
            int t = 0;
            if (lane == 0) t = atomicAdd(ticket, 1);
            t = __shfl_sync(0xffffffffu, t, 0);
            const int bt = t / npairs, pi = t - bt * npairs;
            const int upto = bt < NB ? bt : NB;
            if (cur < upto) {
                tmem_st_wait();
                tc_fence_before();
                __syncwarp();
                for (; cur < upto; ++cur)
                    if (lane == 0) mbar_arrive(vdone + (cur & 1));
                ready = false;
            }
            if (bt >= NB) break;
            if (!ready) {
                mbar_wait(zfull + (cur & 1), (cur >> 1) & 1);
                tc_fence_after();
                ready = true;
            }
            const uint32_t zrow0 = tl + (cur & 1) * 4 * nkp + 4 * pi, zrow1 = zrow0 + 2 * nkp;
            uint32_t z0[4], z1[4], o0[4], o1[4];
            tmem_ld4(zrow0, z0);
            tmem_ld4(zrow1, z1);
            tmem_ld_wait();
#pragma unroll
            for (int f = 0; f < 2; ++f) {
                const float2 zc[2] = {make_float2(__uint_as_float(z0[2 * f]), __uint_as_float(z0[2 * f + 1])),
                                      make_float2(__uint_as_float(z1[2 * f]), __uint_as_float(z1[2 * f + 1]))};
                float2 v[2] = {{0.f, 0.f}, {0.f, 0.f}};
                const int fidx = 2 * pi + f;
                if (fact) {
                    const int nl = tc_phi_fact(coef + fidx * (TNRD_FG * TNRD_FSTRIDE), kappa, olo, ohi, ginv, zc, v);
                    if (STATS) nlive += nl;
                }
                else if (f0 + fidx < a.N_k) tc_phi_direct(a.prm + (size_t)(f0 + fidx) * C::PRM + prm_kkp(KS), zc, v);
                split_bf16(v[0], o0[2 * f], o0[2 * f + 1]);
                split_bf16(v[1], o1[2 * f], o1[2 * f + 1]);
            }
            tmem_st4(zrow0, o0);
            tmem_st4(zrow1, o1);
            if (STATS) nfilt += 2;
        }
        if (STATS && a.stats && lane == 0 && fact) {
            atomicAdd(a.stats, (unsigned long long)nlive);
            atomicAdd(a.stats + 1, (unsigned long long)nfilt * TNRD_FG);
        }
    } else if (warp < TC_PHI_WARPS + 4) {
        // =================================== drain warps ===================================
        // One warp per lane quarter: reads the scatter table of a batch, folds it over neighbouring lanes and over
        // batches (shared memory, fixed order), and completes output rows (a5).
        const int quarter = warp & 3;
        const int L = quarter * 32 + lane;                       // tensor-memory lane = pixel pair
        const uint32_t tl = tmem + ((uint32_t)(quarter * 32) << 16);
        float2* xbuf = reinterpret_cast<float2*>(smem + C::SM_X);      // [q][k][128]
        float2* oring = reinterpret_cast<float2*>(smem + C::SM_O);     // [8][128]
        const float lambda = a.lambda_ptr ? __ldg(a.lambda_ptr) : a.lambda_val;
        const int xcol = xs * C::OW + 2 * L;                     // image column of this lane's first pixel
        const bool lane_out = L < 128 - R;                       // lanes whose output pixels this strip completes
        constexpr int NQ = KS + 1;                               // table blocks with content
        for (int b = 0; b < NB; ++b) {
            mbar_wait_idle<TNRD_TC_SLEEP_DRAIN>(tfull, b & 1);
            tc_fence_after();
            bar_drain();                                         // the previous fold has finished reading xbuf
#pragma unroll 1
            for (int q = 0; q < NQ; q += 2) {                    // two table blocks at a time (register count)
                uint32_t tt[16];
                tmem_ld16(tl + TC_TCOL + 8 * q, tt);
                tmem_ld_wait();
#pragma unroll
                for (int qq = 0; qq < 2; ++qq)
#pragma unroll
                    for (int k = 0; k < C::XK; ++k)
                        xbuf[((q + qq) * C::XK + k) * 128 + L] =
                            make_float2(__uint_as_float(tt[8 * qq + 2 * k]), __uint_as_float(tt[8 * qq + 2 * k + 1]));
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(tfree);
            bar_drain();
            // prefetch u and f of the two rows this batch completes
            float uu[2][2], ff[2][2];
            bool okr[2];
#pragma unroll
            for (int qq = 0; qq < 2; ++qq) {
                const int yrel = 2 * b + 1 - (KS - 1 + qq);
                okr[qq] = yrel >= 0 && yrel < rows_out && lane_out;
                const size_t base = ((size_t)img * a.H + ys0 + (okr[qq] ? yrel : 0)) * a.W;
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const bool ok = okr[qq] && xcol + e < a.W && part == nullptr;
                    uu[qq][e] = ok ? __ldg(a.u_in + base + xcol + e) : 0.f;
                    ff[qq][e] = ok ? __ldg(a.f + base + xcol + e) : 0.f;
                }
            }
#pragma unroll
            for (int q = 0; q < NQ; ++q) {
                float2 o = make_float2(0.f, 0.f);
#pragma unroll
                for (int t2 = 0; t2 <= R; ++t2)                  // lanes L .. L + r reach this lane's pixel pair
                    if (L + t2 < 128) {
                        const float2 x = xbuf[(q * C::XK + (R - t2)) * 128 + L + t2];
                        o.x += x.x; o.y += x.y;
                    }
                const int yrel = 2 * b + 1 - q;                  // output row (relative to ys0) block q belongs to
                float2* slot = oring + (yrel & 7) * 128 + L;
                if (q >= 2) { const float2 p = *slot; o.x += p.x; o.y += p.y; }
                if (q < KS - 1) { *slot = o; continue; }
                // a5: the row is complete
                const int qq = q - (KS - 1);
                if (!okr[qq]) continue;
                const size_t base = ((size_t)img * a.H + ys0 + yrel) * a.W;
                if (part) {                                      // a filter chunk: its partial sums, for tc_update_kernel
                    float* pc = part + (size_t)chunk * a.B * a.H * a.W + base;
                    if (xcol < a.W) __stcg(pc + xcol, o.x);
                    if (xcol + 1 < a.W) __stcg(pc + xcol + 1, o.y);
                    continue;
                }
                if (xcol < a.W) a.u_out[base + xcol] = uu[qq][0] - (o.x + lambda * (uu[qq][0] - ff[qq][0]));
                if (xcol + 1 < a.W) a.u_out[base + xcol + 1] = uu[qq][1] - (o.y + lambda * (uu[qq][1] - ff[qq][1]));
            }
        }
    } else if (warp == TC_MMA_WARP) {
        // =================================== MMA issuer ===================================
        if (lane == 0) {
            const uint32_t id_f = umma_idesc(2, 128, 2 * nkp), id_s = umma_idesc(1, 128, C::NSC);
            const uint32_t lbo_f = 2 * nkp * 16;
            const uint32_t s_lo = umma_desc_lo(sbase + C::SM_BS, C::NSC * 16), s_hi = umma_desc_hi(128);
            // descriptor words that do not change: high words (stride between 8-row groups, version), the low words of
            // the ring and operand bases; per MMA one 32-bit add each for the ring row and the tap row
            const uint32_t a_hi = umma_desc_hi(128), b_hi = umma_desc_hi(128);
            const uint32_t a_lo_hi = umma_desc_lo(sbase + C::SM_UHI, 32), a_lo_lo = umma_desc_lo(sbase + C::SM_ULO, 32);
            const uint32_t b_lo_hi = umma_desc_lo(sbase + C::SM_BFH, lbo_f), b_lo_lo = umma_desc_lo(sbase + C::SM_BFL, lbo_f);
            constexpr uint32_t RING_STEP = (TC_CW * 16) >> 4;            // one ring row, in 16-byte units
            const uint32_t tap_step = (2 * lbo_f) >> 4;                  // one tap row of the operand
            auto forward = [&](int b) {
                const int bb = b & 1;
                const int r0 = (2 * b) % (2 * TC_NP);
                // the two rows of the batch accumulate into different columns and alternate: two chains of dependent
                // accumulations in flight (no measurable difference: the pipe is bound by reading A)
#pragma unroll
                for (int split = 0; split < 3; ++split) {                // hi*hi, hi*lo, lo*hi
                    const uint32_t ab = split == 2 ? a_lo_lo : a_lo_hi;
                    const uint32_t bbl = split == 1 ? b_lo_lo : b_lo_hi;
#pragma unroll
                    for (int ta = 0; ta < KS; ++ta) {
#pragma unroll
                        for (int rr = 0; rr < 2; ++rr) {
                            const uint32_t d = tmem + bb * 4 * nkp + rr * 2 * nkp;
                            int ring = r0 + rr + ta;
                            if (ring >= 2 * TC_NP) ring -= 2 * TC_NP;
                            if (split == 0 && ta == 0)
                                umma_tf32_ss2<false>(d, ab + ring * RING_STEP, a_hi, bbl + ta * tap_step, b_hi, id_f);
                            else
                                umma_tf32_ss2<true>(d, ab + ring * RING_STEP, a_hi, bbl + ta * tap_step, b_hi, id_f);
                        }
                    }
                }
                umma_commit(zfull + bb);
                umma_commit(pempty + b % TC_NP);
            };
            auto wait_pair = [&](int p) { mbar_wait_idle<TNRD_TC_SLEEP_MMA>(pfull + p % TC_NP, (p / TC_NP) & 1); };
            for (int p = 0; p <= R; ++p) wait_pair(p);
            tc_fence_after();
            forward(0);
            if (NB > 1) { wait_pair(R + 1); tc_fence_after(); forward(1); }
            for (int b = 0; b < NB; ++b) {
                const int bb = b & 1;
                mbar_wait_idle<TNRD_TC_SLEEP_MMA>(vdone + bb, (b >> 1) & 1);
                if (b >= 1) mbar_wait_idle<TNRD_TC_SLEEP_MMA>(tfree, (b - 1) & 1);
                tc_fence_after();
                for (int rr = 1; rr >= 0; --rr) {                        // row 1 first: it initialises blocks 0 .. KS
                    const uint32_t d = tmem + TC_TCOL + (rr == 0 ? 8 : 0);
                    const uint32_t av = tmem + bb * 4 * nkp + rr * 2 * nkp;
                    for (int pass = 0; pass < 2; ++pass) {
                        uint32_t bl = s_lo + ((pass * (nkp / 2)) * C::NSC);      // in 16-byte units: one K chunk = NSC cells
                        for (int ks = 0; ks < nkp / 4; ++ks, bl += 2 * C::NSC) {
                            if (rr == 1 && pass == 0 && ks == 0) umma_bf16_ts2<false>(d, av, bl, s_hi, id_s);
                            else umma_bf16_ts2<true>(d, av + 8 * ks, bl, s_hi, id_s);
                        }
                    }
                }
                umma_commit(tfull);
                if (b + 2 < NB) { wait_pair(b + 2 + R); tc_fence_after(); forward(b + 2); }
            }
        }
    } else {
        // =================================== loader warps ===================================
        const int lt = tid - (TC_MMA_WARP + 1) * 32;
        int have = 0;
        for (int p = R + 1; p < NPAIRS; ++p) {
            const int slot = p % TC_NP;
            if (p >= TC_NP) mbar_wait_idle<TNRD_TC_SLEEP_LOAD>(pempty + slot, ((p / TC_NP) - 1) & 1);
            if (a.arrived) have = tc_wait_rows(a.arrived, min(a.H, max(ys0 + 2 * p + 2 - 2 * R, 2 * R + 1)), have);
            constexpr int NL = TC_LOAD_WARPS * 32, UNR = 4;      // UNR cells' loads in flight per thread
            for (int idx0 = lt; idx0 < 2 * TC_CWU; idx0 += NL * UNR) {
                float v[UNR][4];
#pragma unroll
                for (int k = 0; k < UNR; ++k) {
                    const int idx = idx0 + k * NL;
                    if (idx < 2 * TC_CWU) {
                        const int rrow = idx / TC_CWU, xg = idx - rrow * TC_CWU;
                        tc_cell_load(u_img, a.H, a.W, ys0 + 2 * p + rrow - 2 * R, X0 + 2 * xg - 2 * R, v[k]);
                    }
                }
#pragma unroll
                for (int k = 0; k < UNR; ++k) {
                    const int idx = idx0 + k * NL;
                    if (idx < 2 * TC_CWU) {
                        const int rrow = idx / TC_CWU, xg = idx - rrow * TC_CWU;
                        tc_cell_store(smem + C::SM_UHI, smem + C::SM_ULO, ((slot * 2 + rrow) * TC_CW + xg) * 16, v[k]);
                    }
                }
            }
            fence_async_smem();
            __syncwarp();
            if (lane == 0) mbar_arrive(pfull + slot);
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == TC_MMA_WARP)
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(tmem), "r"(512) : "memory");
}

// a5 for the filter-chunk mode: u_t = u - (sum of the chunks' partial sums, in chunk order + lambda (u - f))
__global__ void __launch_bounds__(256) tc_update_kernel(StageArgs a, const float* __restrict__ part, int nchunk)
{
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");
    const size_t n = (size_t)a.B * a.H * a.W;
    const float lambda = a.lambda_ptr ? __ldg(a.lambda_ptr) : a.lambda_val;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        float s = 0.0f;
        for (int c = 0; c < nchunk; ++c) s += __ldcg(part + (size_t)c * n + i);
        const float uu = a.u_in[i];
        a.u_out[i] = uu - (s + lambda * (uu - a.f[i]));
    }
}

inline int tc_env_int(const char* name)
{
    const char* e = getenv(name);
    return e ? atoi(e) : 0;
}

}  // namespace

bool tc_supported(int N_k, int ksize) { return (ksize == 7 || ksize == 5) && N_k >= 1 && N_k <= TC_NKP_MAX; }

size_t tc_workspace_bytes(int T, int N_k, int ksize)
{
    const int nkp = (N_k + 7) / 8 * 8;
    return (size_t)T * tc_ws_stage_bytes(ksize, nkp);
}

TcPlan plan_stage_tc(int B, int H, int W, int N_k, int ksize, int num_sms, int nchunk_fixed, int seg_mult)
{
    const int R = (ksize - 1) / 2, OW = 256 - 2 * R, nkp = (N_k + 7) / 8 * 8;
    TcPlan pl;
    pl.nxs = (W + OW - 1) / OW;
    // Units = images x filter chunks x row segments x strips.  Time of a unit in SM clocks (fitted on B200): set-up
    // (operands to shared memory, tensor-memory allocation, pipeline fill and drain) + batches x (a floor of the MMA /
    // drain pipeline + the phi time of the chunk's filters).  Minimise waves x unit time (+ the
    // update kernel when the bank is split).  Even segment heights: every segment then starts on an even row, so a pixel's
    // arithmetic (the pairing of phi rows into batches) does not depend on how the rows are cut up.
    double best = -1.0;
    long long best_units = 0;
    pl.nys = 1; pl.seg_rows = H; pl.nchunk = 1;
    const int forced = tc_env_int("TNRD_TC_SEG"), forced_chunk = tc_env_int("TNRD_TC_CHUNK");
    for (int nchunk = 1; nchunk <= nkp / 8; ++nchunk) {
        if (nkp % (8 * nchunk)) continue;
        if (nchunk_fixed > 0 && nchunk != nchunk_fixed) continue;
        if (nchunk_fixed <= 0 && forced_chunk > 0 && nchunk != forced_chunk && nkp % (8 * forced_chunk) == 0) continue;
        const double nf = nkp / nchunk;
        const double per_batch = 2400.0 + 380.0 * nf;       // measured (7x7): 5.8 k clocks at 8 filters, 8.3 k at 16, 10.9 k at 24, 20.6 k at 48
        for (int nys = 1; nys <= (H + 3) / 4; ++nys) {
            int seg = (H + nys - 1) / nys;
            seg = (seg + seg_mult - 1) / seg_mult * seg_mult;
            if (forced > 0) seg = forced < H ? forced : H;
            const int n = (H + seg - 1) / seg;
            const long long units = (long long)B * nchunk * pl.nxs * n;
            const double unit_clk = 12000.0 + 300.0 * nf + ((seg + 2 * R) / 2 + 1) * per_batch;
            // split bank: the update kernel ((nchunk + 3) planes of traffic; its launch overlaps the stage kernel's tail)
            const double upd = nchunk > 1 ? 4000.0 + 0.002 * (double)B * H * W * (nchunk + 3) : 0.0;
            const double cost = (double)((units + num_sms - 1) / num_sms) * unit_clk + upd;
            // within 1 % the plan with more units wins: units are handed out as SMs become free, and short units even
            // out the tail that the wave count does not see (4096^2: 442 units of 158 rows beat 289 of 242 by 0.4 %)
            if (best < 0 || cost < 0.99 * best || (cost < 1.01 * best && units > best_units)) {
                if (best < 0 || cost < best) best = cost;
                best_units = units;
                pl.nys = n; pl.seg_rows = seg; pl.nchunk = nchunk;
            }
            if (forced > 0) break;
        }
    }
    pl.units = (long long)B * pl.nchunk * pl.nxs * pl.nys;
    pl.cost_clk = best;
    return pl;
}

cudaError_t launch_tc_prep(const float* prm, int T, int N_k, int ksize, unsigned char* ws, cudaStream_t st,
                           unsigned long long* launches)
{
    const int nkp = (N_k + 7) / 8 * 8;
    const long long total = (long long)T * (ksize * 2 * 2 * nkp * 4 + nkp * 8 * (ksize + 1) * 8);
    const int threads = 256;
    long long blocks = (total + threads - 1) / threads;
    if (blocks > 1184) blocks = 1184;
    tc_prep_kernel<<<(int)blocks, threads, 0, st>>>(prm, T, N_k, nkp, ksize, ws);
    ++*launches;
    return cudaGetLastError();
}

template <int KS>
static cudaError_t launch_tc_ks(const StageArgs& a, const TcPlan& pl, const unsigned char* ws_t, int nkp, float* part,
                                cudaStream_t st)
{
    using C = TcCfg<KS>;
    // the opt-in shared-memory size is a per-device function attribute: set it at every launch (cheap) so that any
    // device of the process works
    auto kern = a.stats ? stage_tc_kernel<KS, true> : stage_tc_kernel<KS, false>;    // counting costs registers: own instance
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM);
    if (e != cudaSuccess) return e;
    if (pl.units > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)pl.units, 1, 1);
    cfg.blockDim = dim3(TC_THREADS, 1, 1);
    cfg.dynamicSmemBytes = C::SMEM;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;     // see griddepcontrol in the kernel
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = a.pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, a, ws_t, nkp, pl.nxs, pl.nys, pl.seg_rows, pl.nchunk,
                              pl.nchunk > 1 ? part : (float*)nullptr);
}

cudaError_t launch_stage_tc(const StageArgs& a, const TcPlan& pl, const unsigned char* ws_t, float* part, cudaStream_t st,
                            unsigned long long* launches)
{
    const int nkp = (a.N_k + 7) / 8 * 8;
    if (pl.nchunk > 1 && !part) return cudaErrorInvalidValue;
    cudaError_t e;
    if (a.ksize == 7) e = launch_tc_ks<7>(a, pl, ws_t, nkp, part, st);
    else if (a.ksize == 5) e = launch_tc_ks<5>(a, pl, ws_t, nkp, part, st);
    else return cudaErrorInvalidValue;
    ++*launches;
    if (e != cudaSuccess || pl.nchunk == 1) return e;
    const size_t n = (size_t)a.B * a.H * a.W;
    size_t blocks = (n + 255) / 256;
    if (blocks > 148 * 8) blocks = 148 * 8;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)blocks, 1, 1);
    cfg.blockDim = dim3(256, 1, 1);
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = a.pdl ? 1 : 0;
    ++*launches;
    return cudaLaunchKernelEx(&cfg, tc_update_kernel, a, (const float*)part, pl.nchunk);
}

size_t tc_ws_stage_stride(int N_k, int ksize) { return tc_ws_stage_bytes(ksize, (N_k + 7) / 8 * 8); }

}  // namespace tnrd

// tnrd_internal.h -- declarations shared by the translation units of libtnrd (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>

#define TNRD_M 63          // RBF terms per influence function
#define TNRD_MP 64         // padded to 64 (term 63 has weight 0)
#define TNRD_TAB_NODES 4096  // nodes of a piecewise-linear phi table (tnrd_table.cu)
#define TNRD_FS 6          // factorised phi evaluator: a group = one anchor centre and its TNRD_FS neighbours on each side
#define TNRD_FM (2 * TNRD_FS + 1)                        // centres per group
#define TNRD_FG ((TNRD_M + TNRD_FM - 1) / TNRD_FM)       // groups
#define TNRD_FSTRIDE ((TNRD_FM + 1 + 3) / 4 * 4)        // floats per group record
#define TNRD_FCLAMP 11.3f  // |d| clamp in scaled units: 2^{-d^2} is flushed to zero beyond sqrt(126) = 11.22

namespace tnrd {

// ---- staged ("prepped") parameters ---------------------------------------------------------------
// For every stage t and filter i the prep kernel writes one record of prm_stride(ksize) floats:
//   taps     (ksize + 1) rows rho = 0..ksize of prm_ts(ksize) floats; row rho holds the ksize PAIRS
//            P[rho][b] = (k'[rho-1][b], k'[rho][b]),  k'_i[a][b] = s * k_i[a][b],  k'[-1] = k'[ksize] = 0,
//            s = sqrt(log2(e) / (2 gamma^2)).  A pair feeds one packed FFMA2 that updates the two output rows of a
//            4x2 pixel block at once: forward filter at window row wr uses row rho = ksize - wr, transposed filter
//            at window row wr uses row rho = wr.
//   pairs    at offset prm_kkp: 64 pairs (-mu'_j, w'_ij) = (-s * mu_j, w_ij / s), pair 63 = (0, 0)
//   wplain   at offset prm_wplain: w'_ij, j = 0..63 (w'_i63 = 0), for the windowed phi evaluator's per-lane gathers
//   hdr      at offset prm_hdr, 8 floats, the same in every record: (1/delta', mu'_0, delta', ok_w, kappa, D, ok_f, 0) --
//            centre spacing in scaled units; ok_w = 1.0f when the centres are equidistant to rounding (|mu_j - (mu_0 +
//            j delta)| <= 1.5e-7 (|mu_0| + 62 delta), a few ulp of the largest centre) and gamma <= delta (window of 14 centres then holds every centre within 6.5 gamma of any z);
//            kappa = 2 delta', D and ok_f belong to the factorised evaluator (next item)
//   fact     at offset prm_fact: TNRD_FG groups of TNRD_FSTRIDE floats for the factorised phi evaluator.  Group g has its
//            anchor at centre a = g (2 S + 1) + S (S = TNRD_FS) and holds
//            -mu'_a,  c_S, c_{S-1}, .., c_0,  c_{-S}, c_{-S+1}, .., c_{-1},  K_g, 1/K_g  (slots 14, 15: K_g = 2^{kappa (mu'_mid -
//            mu'_a)}, mid = the middle group's anchor; used by the tensor-core kernel to derive rho of every group from one)  with
//            c_j = w'_{i,a+j} 2^{-(j delta')^2} (0 where a + j is not a centre).  With d = z' - mu'_a and equidistant
//            centres,  2^{-(d - j delta')^2} = 2^{-d^2} (2^{kappa d})^j 2^{-(j delta')^2},  so the 2S+1 terms of a group
//            are  2^{-d^2} * (polynomial in rho = 2^{kappa d} for j >= 0, in 1/rho for j < 0): 3 ex2 instead of 2S+1.
//            d is clamped to [-D, D], D = 11.3: there 2^{-d^2} has flushed to zero, so the clamp changes nothing, and
//            rho^S stays finite.  ok_f = 1.0f when the centres are equidistant, the dropped terms are negligible
//            ((D - S delta')^2 >= 30, i.e. below 2^-30 of their weight) and max_j (j kappa D - (j delta')^2) <= 92
//            (the polynomial cannot overflow for |w'| < 2^31); gamma = delta gives 38.4 and 89.2.
// so that phi_i(k_i * u) = sum_j w_ij 2^{-(z' - mu'_j)^2} with z' = k'_i * u, and the transposed bank
// sum_i kbar_i * v_i = sum_i kbar'_i * (v_i / s) re-uses the same scaled taps.
__host__ __device__ constexpr int prm_ts(int ksize) { return ((2 * ksize + 3) / 4) * 4; }
__host__ __device__ constexpr int prm_tap(int ksize, int a, int b) { return (a + 1) * prm_ts(ksize) + 2 * b; }
__host__ __device__ constexpr int prm_kkp(int ksize) { return (ksize + 1) * prm_ts(ksize); }
__host__ __device__ constexpr int prm_wplain(int ksize) { return prm_kkp(ksize) + 2 * TNRD_MP; }
__host__ __device__ constexpr int prm_hdr(int ksize) { return prm_wplain(ksize) + TNRD_MP; }
__host__ __device__ constexpr int prm_fact(int ksize) { return prm_hdr(ksize) + 8; }
__host__ __device__ constexpr int prm_stride(int ksize) { return prm_fact(ksize) + TNRD_FG * TNRD_FSTRIDE; }

// Half-sample symmetric mirror map, edge pixel repeated, then clamped so that
// coordinates beyond the 2r halo (ragged tiles) still address memory inside the image.
__host__ __device__ inline int mirror_clamp(int q, int n)
{
    q = q < 0 ? -1 - q : q;
    q = q >= n ? 2 * n - 1 - q : q;
    q = q < 0 ? 0 : q;
    return q >= n ? n - 1 : q;
}

struct StageArgs {
    const float* f;      // [B][H][W]
    const float* u_in;   // [B][H][W]
    float* u_out;        // [B][H][W]
    const float* prm;    // staged records of this stage: [N_k][prm_stride]
    const float* lambda_ptr; // device pointer to lambda_t, or nullptr -> lambda_val
    float lambda_val;
    int B, H, W, N_k, ksize;
    int dense_is_fallback;  // set by the launcher: the dense kernel returns at once when the windowed one applies
    const float* tab;       // piecewise-linear phi tables of this stage [N_k][TNRD_TAB_NODES] float2 (phi evaluator 2)
    const float* tabhdr;    // their header (tnrd_table.cu), device
    unsigned long long* stats;  // null, or device counters {phi group evaluations executed, defined} (tensor-core kernel)
    int row_lo, row_hi;         // tensor-core kernel: this launch completes output rows [row_lo, row_hi) only; 0, 0 = all rows
    // tensor-core kernel, one image, host entry point: null, or device words {set to 1 by a poll that timed out, then one
    // word per block of 32 rows: non-zero once the block of f / u_in has arrived} -- copied by another stream while the
    // kernel runs; the loader polls the word of a block before it reads its first row
    unsigned* arrived;
    // tensor-core kernel, programmatic dependent launch: 0 = a plain launch (the host entry point's image groups: a CTA
    // that sits on an SM waiting for its own stream's previous kernel would keep the other groups' CTAs off it);
    // 1 = programmatic, the CTA waits for the previous kernel of the stream before anything else; 2 = programmatic, and
    // this launch's operands and records were complete before that kernel started (stages after the first of a call),
    // so the CTA sets itself up before it waits
    int pdl;
};

// Launch plan of the fused stage kernel (tnrd_fused.cu: plan_stage_fused).  Tiles partition the phi region
// (H + 2r) x (W + 2r); nsplit > 1 = the small-image path: the filter bank of a tile is split over nsplit CTAs.  Every CTA
// stores its partial transposed-filter sums in `part_floats` floats of scratch; stage_update_kernel adds them up.
struct FusedPlan {
    int cfg;                 // kernel configuration 1..3 (output area / threads)
    int ntx, nty, tw, th;    // tiles per image and nominal tile size (the last tile of a row / column may be smaller)
    int nsplit;              // CTAs per split tile (each takes a contiguous chunk of the N_k filters)
    long long n_full;        // the first n_full tiles are taken by one CTA each, the others by nsplit CTAs
    int cta_floats;          // partial sums of one CTA
    size_t part_floats;      // scratch needed: (n_full + (tiles - n_full) * nsplit) * cta_floats
};

// ---- backward pass of a stage (tnrd_bwd.cu) ----------------------------------------------------------------
struct BwdArgs {
    const float* f;      // [B][H][W]
    const float* u;      // [B][H][W]  u_{t-1}
    const float* e;      // [B][H][W]  dl/du_t
    float* g_u;          // [B][H][W]  dl/du_{t-1}, or null
    const float* prm;    // staged records of this stage
    const float* lambda_ptr;
    float lambda_val;
    int B, H, W, N_k, ksize;
    float* pmap;         // [B][N_k][H+2r][W+2r]  Lambda_i Kbar_i^T e / s   (null unless g_k is wanted)
    float* vmap;         // [B][N_k][H+2r][W+2r]  phi_i(z_i) / s
    float* part_w;       // [n_cta][N_k][64] per-CTA g_w sums (null unless g_w is wanted)
    float* part_l;       // [n_cta] per-CTA g_lambda sums (null unless wanted)
};
struct BwdPlan {
    int ntx, nty;        // tiles of the extended output domain per image (stage_bwd_kernel)
    long long n_cta;     // ntx * nty * B
    int wtx, wty, G;     // wgrad tiles per image; CTAs per filter
};
BwdPlan plan_stage_bwd(int B, int H, int W, int N_k, int ksize, int num_sms);
// what: 1 = stage_bwd_kernel, 2 = wgrad_kernel (reads the maps kernel 1 wrote), 3 = both in turn
cudaError_t launch_stage_bwd(const BwdArgs& a, const BwdPlan& pl, float* part_k /*[G][N_k][ks*ks]*/, int what, cudaStream_t st,
                             unsigned long long* launches);
cudaError_t launch_reduce_partials(const float* part_w, long long n_cta, const float* part_k, int G, const float* part_l,
                                   int N_k, int ksize, float s, float* g_w, float* g_k, float* g_lambda, cudaStream_t st,
                                   unsigned long long* launches);
cudaError_t launch_sub(const float* x, const float* y, float* out, size_t n, cudaStream_t st, unsigned long long* launches);

// tnrd_api.cu, for entry points that live in other files (tnrd_static.cu): record a CUDA failure for
// tnrd_last_cuda_error and return TNRD_ERR_CUDA; add to the process-wide launch counter
int api_cuda_fail(cudaError_t e, const char* what);
void api_count_launches(unsigned long long n);

// launchers (each returns the cudaError_t of the launch; *launches += kernels launched)
cudaError_t launch_prep(const float* filters, const float* rbf_w, const float* rbf_mu, float gamma,
                        int T, int N_k, int ksize, float* prm, cudaStream_t st, unsigned long long* launches);
cudaError_t launch_stage_ref(const StageArgs& a, float* vbuf, cudaStream_t st, unsigned long long* launches);
size_t ref_scratch_floats(int B, int H, int W, int N_k, int ksize);
FusedPlan plan_stage_fused(const StageArgs& a, int num_sms);
// phi_mode: 0 dense, direct (one ex2 per Gaussian), 1 windowed (with dense fallback), 2 piecewise-linear table (a.tab),
// 3 dense, factorised (direct inside the same kernel when the staged flag says it does not apply).  part = scratch of
// plan.part_floats floats.
cudaError_t launch_stage_fused(const StageArgs& a, const FusedPlan& plan, float* part, int phi_mode, cudaStream_t st,
                               unsigned long long* launches);
// ---- small-image kernel (tnrd_small.cu): all T stages of an image that fits a cluster of 8 CTAs in one launch ----
bool small_supported(int B, int H, int W, int N_k, int ksize);
// pp: ping-pong plane [B][H][W] (needed when T > 1); u0 must not be the buffer stage 1 writes (out when T is odd, pp else);
// lambda: device [T], or null -> lambda_val for every stage; force_direct: one ex2 per Gaussian (TNRD_PHI_DENSE)
cudaError_t launch_small_diffuse(const float* f, const float* u0, float* out, float* pp, const float* filters,
                                 const float* rbf_w, const float* rbf_mu, float gamma, const float* lambda, float lambda_val,
                                 int B, int H, int W, int T, int N_k, int ksize, int force_direct, cudaStream_t st,
                                 unsigned long long* launches);
cudaError_t launch_qcs_project(const float* y, const float* lo, const float* hi, float* u, int B, int H, int W,
                               cudaStream_t st, unsigned long long* launches);   // u may alias y
// phi tables: [TN][TNRD_TAB_NODES] float2 + 4 header floats; basis 0 Gaussian, 1 triangular
cudaError_t launch_build_table(const float* rbf_w, const float* rbf_mu, float gamma, int TN, int basis, float* tab,
                               float* hdr, cudaStream_t st, unsigned long long* launches);
cudaError_t fused_init();   // opt-in shared memory attributes; idempotent

// ---- tensor-core stage kernel (tnrd_tc.cu): both filterings as tcgen05 implicit GEMMs, update fused in ----------
// A unit = (image, row segment, strip of 256 - 2r output columns); one CTA per unit.
struct TcPlan {
    int nxs, nys, seg_rows;   // strips per image, row segments per image, output rows per segment
    int nchunk;               // filter chunks per (image, segment, strip): > 1 = partial sums + tc_update_kernel
    long long units;          // CTAs
    double cost_clk;          // the planner's objective: waves x modelled clocks of a unit
};
bool tc_supported(int N_k, int ksize);                       // ksize 5 or 7, N_k <= 48
size_t tc_workspace_bytes(int T, int N_k, int ksize);        // Toeplitz operands of T stages
size_t tc_ws_stage_stride(int N_k, int ksize);               // bytes per stage inside that workspace
// H = number of output rows of the launch; nchunk_fixed > 0: that many filter chunks, no choice; seg_mult: segment heights
// are a multiple of it (even; the host entry point asks for 32, the rows of an arrival block)
TcPlan plan_stage_tc(int B, int H, int W, int N_k, int ksize, int num_sms, int nchunk_fixed = 0, int seg_mult = 2);
// prm = staged records of T stages (launch_prep); ws receives the operands
cudaError_t launch_tc_prep(const float* prm, int T, int N_k, int ksize, unsigned char* ws, cudaStream_t st,
                           unsigned long long* launches);
// one stage; a.u_out must not alias a.u_in (the kernel reads halos of u_in while other CTAs write u_out)
// part: scratch of nchunk * B * H * W floats when pl.nchunk > 1 (then a point-wise update kernel follows), else unused
cudaError_t launch_stage_tc(const StageArgs& a, const TcPlan& pl, const unsigned char* ws_t, float* part, cudaStream_t st,
                            unsigned long long* launches);
cudaError_t run_microbench(int which, double* rate, cudaStream_t st, unsigned long long* launches);

}  // namespace tnrd

/*
 * tnrd.h -- C ABI of libtnrd: the inference hot path of the trained nonlinear
 * reaction-diffusion model (TNRD) of Chen, Yu & Pock, arXiv 1503.05768, on NVIDIA B200 (sm_100a).
 *
 * The library computes, per stage t = 1..T (Main Eq. 7; Supp. Eq. 2):
 *
 *     u_t = u_{t-1} - ( sum_{i=1..N_k} kbar_i^t * phi_i^t( k_i^t * u_{t-1} ) + lambda^t (u_{t-1} - f) )
 *
 *   k_i * u      true 2-D convolution with the ksize x ksize filter k_i
 *   phi_i(z)     = sum_{j=1..63} w_ij exp( -(z - mu_j)^2 / (2 gamma^2) )        (Main Eq. 6, :113-117; :553)
 *   kbar_i       = k_i rotated by 180 degrees
 *   boundary     u_{t-1} is extended by 2r (r = (ksize-1)/2) with mirror reflections (edge pixel
 *                repeated), both filterings are "valid", the result is the H x W centre -- the
 *                pad / diffuse / crop procedure of Supp. Sec. 1, which is the same
 *                for every pad width omega >= 2r (reading S1).
 *
 * All arithmetic is IEEE fp32 (FMA contraction, any summation order, ex2.approx for the exponential);
 * results are deterministic run to run.  Nothing here allocates or reads through PyTorch; callers hand
 * in raw pointers.
 *
 * Conventions common to all entry points
 *   - Images are dense row-major float32 [B][H][W] (x fastest).  filters [T][N_k][ksize][ksize] with
 *     k[a][b], a = row, b = column.  rbf_w [T][N_k][63].  rbf_mu [63].  lambda [T].
 *   - "device pointer": memory of the CURRENT CUDA device (cudaMalloc / torch allocator), 4-byte aligned.
 *     "host pointer": ordinary or pinned host memory.
 *   - Ownership: the caller owns every buffer and keeps device buffers alive until the work queued on
 *     `stream` has completed.  The library owns only an internal per-(device, stream) scratch (the staged parameters,
 *     and either the partial sums of the tile kernel, about 4.5 bytes per pixel, or the ping-pong plane of the
 *     tensor-core kernel, 4 bytes per pixel), grown on demand and released by tnrd_shutdown().  The scratch grows
 *     with cudaMallocAsync on `stream`; a call that would have to grow it while `stream` is being captured into a
 *     CUDA graph returns TNRD_ERR_CUDA instead (run the shape once before capturing).
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Device entry points
 *     are asynchronous on `stream` and never synchronise the device.
 *     The stage kernels of the tensor-core and small-image paths are launched with programmatic stream serialisation
 *     (they may be scheduled while the previous kernel of the stream drains, and wait for it before they touch global
 *     memory): work the caller queues before or after a call on the same stream sees ordinary stream order.
 *   - Every function returning int returns TNRD_OK (0) or a negative tnrd_status.  Nothing throws.
 *     Errors found while validating or launching are returned; asynchronous faults surface at the
 *     caller's next synchronisation.  On error no output is written.
 *   - Shapes: B,H,W >= 1, B*H*W < 2^31; ksize in {3,5,7,9}; 1 <= N_k <= 128; min(H,W) >= ksize-1 (the
 *     mirror source must lie inside the image); T >= 0.
 */
#ifndef TNRD_H_
#define TNRD_H_

#ifdef __cplusplus
extern "C" {
#endif

#define TNRD_NUM_RBF 63 /* M, PAPER.md:176 ("63 Gaussian RBFs") -- fixed by the model family */
#define TNRD_MAX_FILTERS 128
#define TNRD_VERSION 200 /* 0.2.0 */

typedef enum {
    TNRD_OK = 0,
    TNRD_ERR_NULL = -1,        /* a required pointer is NULL */
    TNRD_ERR_SHAPE = -2,       /* B/H/W/T/N_k out of range, image smaller than the 2r halo, too many pixels */
    TNRD_ERR_UNSUPPORTED = -3, /* ksize not in {3,5,7,9}; unknown option */
    TNRD_ERR_ALIAS = -4,       /* output aliases an input it must not alias */
    TNRD_ERR_CUDA = -5,        /* a CUDA call failed; see tnrd_last_cuda_error() */
    TNRD_ERR_PARAM = -6,       /* rbf_gamma not finite or <= 0 */
    TNRD_ERR_TOO_LARGE = -7    /* tnrd_stage_static: the call needs more than TNRD_STATIC_SCRATCH_BYTES of scratch */
} tnrd_status;

/*
 * One stage (rows a1-a5 of the hot path; Main Eq. 7).
 *   f, u_in     device, [B][H][W]   noisy image f_n and previous iterate u_{t-1}
 *   filters_t   device, [N_k][ksize][ksize]      k_i^t
 *   rbf_w_t     device, [N_k][63]                w_ij^t
 *   rbf_mu      device, [63]                     mu_j (any values; equidistant in the paper, :117)
 *   rbf_gamma   by value, > 0 and finite         shared width gamma (:117 "unified scaling", :553)
 *   lambda_t    by value                          reaction weight lambda^t
 *   u_out       device, [B][H][W]   u_t; may equal u_in (in place: every halo read is done before the first write);
 *               must not be f -> TNRD_ERR_ALIAS on pointer equality; partial overlap is undefined behaviour.
 */
int tnrd_stage(const float* f, const float* u_in, int B, int H, int W, int N_k, int ksize,
               const float* filters_t, const float* rbf_w_t, const float* rbf_mu, float rbf_gamma,
               float lambda_t, float* u_out, void* stream);

/*
 * tnrd_stage for callers that must not allocate (code under CUDA graph capture, serving loops, harnesses that forbid
 * cudaMalloc): the same operation (Main Eq. 7), arguments, layouts and aliasing rules as tnrd_stage, always
 * with the tile kernel and the factorised Gaussian evaluator (the process-wide options of tnrd_set_kernel /
 * tnrd_set_phi_mode / tnrd_set_basis do not apply).  Its scratch -- the staged parameters and the per-CTA partial sums
 * -- is a fixed device array of TNRD_STATIC_SCRATCH_BYTES that every GPU loading the library holds until exit; the call
 * makes no cudaMalloc / cudaFree / host allocation.
 *   Limit: TNRD_ERR_TOO_LARGE, and nothing launched, when the stage needs more: 1 MiB holds the parameters, the rest
 *   the partial sums, 4 x part_floats bytes of tnrd_plan_query's plan (64 KiB per CTA of the tile kernel for 7x7
 *   filters, so at most 1008 CTAs).  That covers e.g. one 2560 x 2560 image or 36 images of 321 x 481 with 48 filters of
 *   7x7, not 4096 x 4096 (1756 CTAs): cut larger batches into several calls.
 *   Sharing: every call uses the same array and finds the last call's contents in it (nothing has to start at zero:
 *   each call writes all it reads).  Calls on one stream are ordered; calls that overlap on the GPU (several streams or
 *   host threads) race on it and give garbage -- serialise them.
 */
#define TNRD_STATIC_SCRATCH_BYTES (64u << 20)
int tnrd_stage_static(const float* f, const float* u_in, int B, int H, int W, int N_k, int ksize,
                      const float* filters_t, const float* rbf_w_t, const float* rbf_mu, float rbf_gamma,
                      float lambda_t, float* u_out, void* stream);

/*
 * T stages with per-stage parameters Theta_t = {lambda^t, phi_i^t, k_i^t} (row a6).
 *   f, u0       device, [B][H][W]; the paper starts from u0 = f (Main Fig. 2)
 *   filters     device, [T][N_k][ksize][ksize];  rbf_w device [T][N_k][63];  rbf_mu device [63]
 *   lambda      device, [T]  (device so that the call needs no host sync and can be graph-captured)
 *   out         device, [B][H][W]; receives u_T.  out may equal u0 (in place); out must not equal f.
 *   T = 0 copies u0 to out.
 * With the tile kernel every stage writes `out`, from the second one on in place; with the tensor-core kernel the
 * stages alternate between `out` and one image-sized plane of the library scratch (tnrd_set_kernel).
 */
int tnrd_diffuse(const float* f, const float* u0, int B, int H, int W, int T, int N_k, int ksize,
                 const float* filters, const float* rbf_w, const float* rbf_mu, float rbf_gamma,
                 const float* lambda, float* out, void* stream);

/*
 * End-to-end variant with HOST buffers: every pointer below is a host pointer (pinned memory makes the
 * copies asynchronous).  Copies f, u0 and the parameters (packed, one copy) to the device, runs the T stages on
 * `stream`, copies u_T back to `out` and synchronises before returning.  f == u0 (same host pointer) is uploaded once.
 * Device staging buffers are cached in the library scratch.  With the tensor-core kernel (tnrd_set_kernel) the copies
 * overlap the arithmetic, on internal streams:
 *   - a batch is cut into up to four groups of images, each taken through all T stages on a stream of its own, so that a
 *     group computes while the next one arrives and the previous one leaves;
 *   - a single image arrives in blocks of 32 rows, the rows of the first wave of CTAs first; the first stage's loader
 *     warps wait for the block they are about to read (one device word per block, written by the copy stream; a wait
 *     that lasts two seconds ends the call with TNRD_ERR_CUDA), and when `out` is pinned (or otherwise device-mapped)
 *     host memory the last stage stores u_T into it directly; a pageable `out` gets one copy after the last stage.
 * Either way the result is bit-identical to tnrd_diffuse on device buffers.  The buffers must stay valid and unchanged
 * until the call returns (it synchronises `stream`).  `out` may be the host buffer of f / u0 (in place on the host; the
 * direct stores are then replaced by a copy); partial overlap is undefined behaviour.
 */
int tnrd_diffuse_host(const float* f, const float* u0, int B, int H, int W, int T, int N_k, int ksize,
                      const float* filters, const float* rbf_w, const float* rbf_mu, float rbf_gamma,
                      const float* lambda, float* out, void* stream);

/*
 * JPEG-deblocking variant (Main Eq. 9; Supp. Eq. 26-29).  Per stage
 *     y = u_{t-1} - sum_i kbar_i^t * phi_i^t(k_i^t * u_{t-1})        (the diffusion term of tnrd_stage, no reaction term)
 *     u_t = D^T eta(D y)                                              (projection onto the quantisation constraint set)
 * D is the orthonormal 2-D DCT-II of every 8x8 block (D^T D = I; the block grid starts at pixel (0,0)),
 * eta clamps coefficient p to [qcs_lo_p, qcs_hi_p] (Supp. Eq. 26).  Coefficient (p, q) of block (by, bx) lives at pixel
 * (8 by + p, 8 bx + q) of a [B][H][W] array; qcs_lo / qcs_hi use that layout and refer to the DCT of u itself (no level
 * shift).  H and W must be multiples of 8 (TNRD_ERR_SHAPE otherwise); the paper's pad width omega = 8 is
 * one whole block, so with the 2r mirror halo of the diffusion term the H x W result is the paper's (D1).
 *   u0, qcs_lo, qcs_hi, out   device, [B][H][W];  filters [T][N_k][ksize][ksize], rbf_w [T][N_k][63], rbf_mu [63] device
 *   out may equal u0; out must not equal qcs_lo or qcs_hi.  T = 0 copies u0.  Asynchronous on `stream`.
 */
int tnrd_deblock_diffuse(const float* u0, int B, int H, int W, int T, int N_k, int ksize, const float* filters,
                         const float* rbf_w, const float* rbf_mu, float rbf_gamma, const float* qcs_lo,
                         const float* qcs_hi, float* out, void* stream);

/* u_out = D^T eta(D y) alone (all device, [B][H][W]; u_out may equal y).  Asynchronous on `stream`. */
int tnrd_qcs_project(const float* y, int B, int H, int W, const float* qcs_lo, const float* qcs_hi, float* u_out,
                     void* stream);

/*
 * Backward pass of one stage (the step on the other side of inference: training on the same kernels).
 * For u_t = u_in - ( sum_i kbar_i * phi_i(k_i * u_in) + lambda (u_in - f) ) as tnrd_stage computes it (mirror
 * extension by 2r, crop built in) and e = dl/du_t, it returns
 *     grad_u       = (du_t/du_in)^T e = (1 - lambda) e - P^T sum_i K_i^T Lambda_i Kbar_i^T e   (Supp. Eq. 21)
 *     grad_filters = dl/dk_i = -(P_inv^T V^T + U^T Lambda_i Kbar_i^T) e                         (Supp. Eq. 10)
 *     grad_w       = dl/dw_i = -G^T Kbar_i^T e                                                  (Supp. Eq. 19)
 *     grad_lambda  = dl/dlambda = -<u_in - f, e>                                                (Supp. Eq. 7)
 * Lambda_i = diag(phi_i'(k_i * u_in)) with phi'(z) = -sum_j w_j (z - mu_j)/gamma^2 exp(-(z - mu_j)^2 / (2 gamma^2)), the
 * derivative of PAPER.md:553 (the printed formula at :568 is garbled); the sign of grad_lambda follows Supp. Eq. 4
 * (Eq. 6 prints it without the minus).  Parameter gradients are SUMMED over the B images (Supp. Eq. 3), grad_u is per
 * image.
 *   f, u_in, e    device, [B][H][W];  filters_t [N_k][ksize][ksize], rbf_w_t [N_k][63], rbf_mu [63] device
 *   grad_u        device, [B][H][W], or NULL;  must not be u_in, e or f (TNRD_ERR_ALIAS)
 *   grad_filters  device, [N_k][ksize][ksize], or NULL.  When asked for, the library keeps two maps of
 *                 B*N_k*(H+2r)*(W+2r) floats in its scratch (Lambda_i Kbar_i^T e and phi_i(z_i), read back by the
 *                 filter-gradient kernel)
 *   grad_w        device, [N_k][63], or NULL;   grad_lambda  device, [1], or NULL
 * All outputs are written (not accumulated); results are deterministic run to run.  Asynchronous on `stream`.
 */
int tnrd_stage_backward(const float* f, const float* u_in, const float* e, int B, int H, int W, int N_k, int ksize,
                        const float* filters_t, const float* rbf_w_t, const float* rbf_mu, float rbf_gamma,
                        float lambda_t, float* grad_u, float* grad_filters, float* grad_w, float* grad_lambda,
                        void* stream);

/*
 * Back-propagation through T stages (joint training, Supp. Eq. 20-21): runs the T forward stages
 * from u0 keeping every iterate in the library scratch (T planes of B*H*W floats), then the backward recurrence
 * e_{t-1} = (du_t/du_{t-1})^T e_t with the parameter gradients of every stage.
 *   Exactly one of u_gt / e_T is non-NULL (device, [B][H][W]): with u_gt the loss is 1/2 ||u_T - u_gt||^2 (Supp. Eq. 3)
 *   and e_T = u_T - u_gt is formed on the device; otherwise e_T = dl/du_T is taken as given (it cannot depend on this
 *   call's u_T).
 *   lambda        device, [T]
 *   u_T           device, [B][H][W], or NULL: receives the forward result
 *   grad_u0       device, [B][H][W], or NULL;  grad_filters [T][N_k][ksize][ksize], grad_w [T][N_k][63],
 *                 grad_lambda [T]: device, each may be NULL
 * T >= 1.  Asynchronous on `stream`.
 */
int tnrd_diffuse_backward(const float* f, const float* u0, const float* u_gt, const float* e_T, int B, int H, int W,
                          int T, int N_k, int ksize, const float* filters, const float* rbf_w, const float* rbf_mu,
                          float rbf_gamma, const float* lambda, float* u_T, float* grad_u0, float* grad_filters,
                          float* grad_w, float* grad_lambda, void* stream);

/*
 * Kernel selection, for tests and profiling.  Process-wide (read once at the entry of every call).
 *   0  automatic (default): the tensor-core stage kernel where it applies and its work units fill the GPU
 *      (tnrd_tc_plan_query), the tile kernel otherwise;
 *   1  the plain one-thread-per-pixel reference kernel (global memory only);
 *   2  the fused tile kernel: both filterings on the FP32 FMA pipe, partial sums + a point-wise update kernel;
 *   3  the tensor-core stage kernel (csrc/tnrd_tc.cu): both filterings as tcgen05 implicit GEMMs (forward bank: three
 *      TF32 products of hi/lo split operands; transposed bank: BF16 hi/lo pairs), accumulators in tensor memory,
 *      factorised influence functions on the accumulators, u_t written by the same kernel.  It applies to the Gaussian
 *      basis with TNRD_PHI_FACTORED, ksize 5 or 7 and N_k <= 48; any other call returns TNRD_ERR_UNSUPPORTED while 3 is
 *      selected.  Results agree with kernel 2 to fp32 rounding (same distance from the double-precision definition).
 *      It cannot run in place: tnrd_diffuse / tnrd_deblock_diffuse then keep one image-sized ping-pong plane in the
 *      library scratch (and copy u0 into it when out == u0 and T is odd), tnrd_stage with u_out == u_in writes the
 *      plane and copies it back.  A non-finite pixel reaches a slightly larger neighbourhood than the (2 ksize - 1)^2
 *      footprint of the definition (0 x NaN inside the 8-column windows of the implicit GEMM).
 *   4  the small-image kernel (csrc/tnrd_small.cu): ALL T stages of tnrd_diffuse (or the one of tnrd_stage) in ONE launch,
 *      parameter staging included, for images that fit a thread-block cluster of 8 or 16 CTAs (B*H*W <= 32768 and a row
 *      band's working set -- its u tile and N_k influence maps -- within 200 KB of shared memory): the automatic choice for such images with the
 *      Gaussian basis and TNRD_PHI_FACTORED / TNRD_PHI_DENSE (64 x 64, T = 2: 39 us -> about a quarter of that per
 *      call).  Iterates alternate between `out` and the ping-pong plane.  Other entry points and shapes return
 *      TNRD_ERR_UNSUPPORTED while 4 is selected.
 * Returns TNRD_ERR_UNSUPPORTED for other values.
 */
int tnrd_set_kernel(int which);

/*
 * Work decomposition of the tensor-core stage kernel for this shape on a device with `num_sms` multiprocessors (pure host
 * logic).  plan[0..6] = {0: the kernel does not apply to (N_k, ksize); 1: applies, the automatic choice is the tile
 * kernel; 2: applies and is the automatic choice}, strips per image (256 - 2r output columns each), row segments per
 * image, output rows per segment, CTAs (= images x filter chunks x segments x strips), output columns per strip, filter
 * chunks (> 1 for images that would not fill the GPU otherwise: each CTA takes a chunk of the filter bank and a point-wise
 * kernel adds the chunks' partial sums and applies the reaction term).  Honours the TNRD_TC_SEG / TNRD_TC_CHUNK environment
 * knobs (force the rows per segment / the number of chunks; tests).
 */
int tnrd_tc_plan_query(int B, int H, int W, int N_k, int ksize, int num_sms, long long* plan);

/*
 * Influence-function evaluator of the fused kernel.  Process-wide.
 *   TNRD_PHI_FACTORED (3, default): every one of the 63 Gaussians of Main Eq. 6 is evaluated, the exponentials of 13
 *       neighbouring centres from three ex2: with equidistant centres (spacing delta) and d = z - mu_a,
 *         exp(-(d - j delta)^2 / 2 gamma^2) = exp(-d^2 / 2 gamma^2) * rho^j * exp(-(j delta)^2 / 2 gamma^2),
 *         rho = exp(delta d / gamma^2),
 *       so a group of centres a-6 .. a+6 costs exp(-d^2/2gamma^2), rho, 1/rho and two polynomials (Horner's rule) whose
 *       coefficients w_{a+j} exp(-(j delta)^2 / 2 gamma^2) are staged on the device at every call.  An identity, not an
 *       approximation: the result differs from TNRD_PHI_DENSE by fp32 rounding only.  When
 *       rbf_mu is not equidistant (same device-side check as TNRD_PHI_WINDOW) or rbf_gamma < 0.96 delta (the powers of
 *       rho would leave the fp32 range) the same kernel evaluates the direct form -- decided on the device, one launch.
 *       Weights with |w| * rbf_gamma beyond about 1e9 overflow in this form (the direct form holds up to ~1e38).
 *   TNRD_PHI_DENSE  (0): the direct form, one ex2 per Gaussian.
 *   TNRD_PHI_WINDOW (1): when rbf_mu is equidistant to rounding (|mu_j - (mu_0 + j delta)| <= 1.5e-7 (|mu_0| + 62 delta), checked on the device by the
 *       staging kernel) and rbf_gamma <= delta, each response evaluates only the 14 consecutive centres around it that
 *       contain every centre within 6.5 gamma; the dropped terms are each below e^{-21.1} = 6.7e-10 of their weight, i.e.
 *       below fp32 rounding of the sum ("equidistant centers").  When the check
 *       fails the dense evaluator runs instead -- decided on the device, two launches per stage, no host synchronisation.
 *   TNRD_PHI_LUT (2): the authors' own speed-up: phi_i is tabulated at 4096 equidistant nodes from 6 gamma
 *       below the lowest centre to 6 gamma above the highest (every node the full 63-term sum, rebuilt on the device at
 *       every call) and evaluated by linear interpolation -- one gather and one FMA per response.  An APPROXIMATION of
 *       Main Eq. 6: per response |error| <= h^2/8 max|phi''| with node spacing h (0.18 for the configs' centres); the
 *       end-to-end distance from the oracle stays inside the library's tolerance.
 * Returns TNRD_ERR_UNSUPPORTED for other values.
 */
#define TNRD_PHI_DENSE 0
#define TNRD_PHI_WINDOW 1
#define TNRD_PHI_LUT 2
#define TNRD_PHI_FACTORED 3
int tnrd_set_phi_mode(int mode);

/*
 * Radial basis of the influence functions.  Process-wide.
 *   TNRD_RBF_GAUSSIAN (0, default): phi_i(z) = sum_j w_ij exp(-(z - mu_j)^2 / (2 gamma^2))            (the paper's results)
 *   TNRD_RBF_TRIANGLE (1): phi_i(z) = sum_j w_ij max(0, 1 - |z - mu_j| / gamma)
 *       evaluated through the table evaluator whatever tnrd_set_phi_mode says: EXACTLY (the linear interpolant of the
 *       weights, two basis functions per z) when rbf_mu is equidistant and rbf_gamma equals the spacing;
 *       otherwise on the 4096-node grid of TNRD_PHI_LUT (approximate).  tnrd_stage_backward / tnrd_diffuse_backward and
 *       the reference kernel (tnrd_set_kernel(1)) return TNRD_ERR_UNSUPPORTED with this basis.
 */
#define TNRD_RBF_GAUSSIAN 0
#define TNRD_RBF_TRIANGLE 1
int tnrd_set_rbf_basis(int basis);

/*
 * Launch plan the library would use for one stage of this shape on a device with `num_sms` multiprocessors (pure host
 * logic, no device needed; for tests and tuning).  plan[0..9] = kernel configuration (1: 128 x 128 output area, 512 threads;
 * 2: 64 x 32, 256 threads; 3: 64 x 64, 256 threads), tiles per image in x, in y, nominal tile width, height (pixels of
 * the (H + 2r) x (W + 2r) phi region), number of leading tiles taken by one CTA each, CTAs per remaining tile (filter
 * split), total CTAs, floats of partial sums per CTA, floats of scratch.  Honours the TNRD_TILE / TNRD_SPLIT / TNRD_NTX /
 * TNRD_NTY environment knobs.
 */
int tnrd_plan_query(int B, int H, int W, int N_k, int ksize, int num_sms, long long* plan);

/*
 * Executed vs defined influence-function work of the tensor-core stage kernel.  The factorised evaluator skips a group
 * of 13 centres when its Gaussian factor is exactly zero for every response of a warp (the result is bit-identical),
 * so the run time depends on the responses; this call reports how much was skipped.  enable != 0 switches counting on
 * for later calls on `stream` (process-wide flag, a few atomics per CTA), 0 switches it off; either way the counters
 * gathered so far on this (device, stream) are returned and reset: *executed = (warp, filter, group) evaluations
 * performed, *defined = evaluations the definition has (5 groups per filter and warp).  Synchronises `stream`.
 * Either pointer may be NULL.  The tile kernel is not instrumented.  rbf_w must be finite: with a skipped group a
 * non-finite weight does not turn the result into NaN (0 x Inf is never formed), so results for non-finite weights are
 * unspecified.
 */
int tnrd_phi_stats(int enable, unsigned long long* executed, unsigned long long* defined, void* stream);

/* Number of kernels this library has launched since load (or since the last tnrd_reset_launch_count). */
unsigned long long tnrd_launch_count(void);
void tnrd_reset_launch_count(void);

/*
 * Roofline denominators measured on the current device: register-only micro-kernels
 * timed with CUDA events on `stream`; synchronises `stream`.
 *   which = 0: FP32 FFMA rate      -> *rate = FMA lane-operations per second (x2 = FLOP/s)
 *   which = 1: MUFU.EX2 rate       -> *rate = ex2 evaluations per second
 *   which = 2: the phi inner loop (FADD, FMUL, MUFU.EX2, FFMA per term) -> RBF terms per second
 *   which = 3: FFMA2 (FMA pipe) and FMNMX (ALU pipe) interleaved 1:1 on independent registers -> WARP instructions per
 *              second of the two together.  Each occupies its pipe for 2 cycles per warp; pipes that issued side by side
 *              would give 148 x 4 x clock, one shared dispatch half of that; B200 measures 0.66 of it (DESIGN.md "Roofline":
 *              the sum of FMA-pipe and ALU-pipe cycles is what the tensor-core stage kernel runs against)
 * Any other value: TNRD_ERR_UNSUPPORTED.
 */
int tnrd_microbench(int which, double* rate, void* stream);

const char* tnrd_strerror(int status);
const char* tnrd_last_cuda_error(void); /* message of the last failing CUDA call on this thread, "" if none */
int tnrd_version(void);
void tnrd_shutdown(void); /* frees the cached scratch of every device; the library stays usable */

#ifdef __cplusplus
}
#endif
#endif /* TNRD_H_ */

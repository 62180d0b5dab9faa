// tnrd_api.cu -- host side of libtnrd: the C ABI declared in include/tnrd.h.
// Validation, per-(device, stream) scratch, parameter staging and the stage loop (row a6: PAPER.md:74, :184).
// Every step of the path runs in this library's kernels; there is no CPU fallback.
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <vector>

#include "../../include/tnrd.h"
#include "tnrd_internal.h"

namespace {

thread_local char g_cuda_err[512] = "";
// Process-wide options and counters: atomics, read ONCE at the entry of every call (Opts), so that a thread that toggles
// a mode while another thread is inside a call cannot change that call half-way.
std::atomic<unsigned long long> g_launches{0};
std::atomic<int> g_kernel{0};    // 0 auto, 1 reference, 2 fused tile kernel (FMA pipe), 3 tensor-core stage kernel
std::atomic<int> g_phi_mode{3};  // 0 direct 63-term phi, 1 windowed evaluator (dense fallback decided on the device), 2 table,
                                 // 3 factorised 63-term phi (direct fallback inside the kernel)
std::atomic<int> g_basis{0};     // 0 Gaussian radial basis, 1 triangular-shaped (table evaluator)
std::atomic<int> g_stats{0};     // 1: the tensor-core kernel counts executed / defined phi group evaluations (tnrd_phi_stats)
std::mutex g_mu;

struct Opts {
    int kernel, phi_mode, basis;
    Opts() : kernel(g_kernel.load()), phi_mode(g_phi_mode.load()), basis(g_basis.load()) {}
    // evaluator of the fused kernel: the triangular basis always goes through the table
    int phi() const { return (basis == 1 || phi_mode == 2) ? 2 : phi_mode; }
};
// kernels launched by one call; added to the process-wide counter when the call returns
struct LaunchCount {
    unsigned long long n = 0;
    ~LaunchCount() { g_launches.fetch_add(n); }
};

int cuda_fail(cudaError_t e, const char* what)
{
    snprintf(g_cuda_err, sizeof(g_cuda_err), "%s: %s (%s)", what, cudaGetErrorName(e), cudaGetErrorString(e));
    (void)cudaGetLastError();  // clear the sticky-less error state
    return TNRD_ERR_CUDA;
}
#define TNRD_CUDA(call)                                          \
    do {                                                         \
        cudaError_t e__ = (call);                                \
        if (e__ != cudaSuccess) return cuda_fail(e__, #call);    \
    } while (0)

// A device buffer that only grows; allocation and release are stream-ordered.
struct Buf {
    float* p = nullptr;
    size_t cap = 0;  // floats
};

constexpr int HOST_BANDS = 4;

struct Scratch {
    int dev = -1;
    cudaStream_t st = nullptr;
    int num_sms = 0;
    Buf prm, refv;                    // staged parameters, reference-path phi maps
    Buf split;                        // partial transposed-filter sums of the fused kernel's CTAs
    Buf pp;                           // ping-pong image plane of the tensor-core kernel (it cannot run in place)
    Buf tcws;                         // its Toeplitz operands, T stages
    Buf stats;                        // two 64-bit counters (tnrd_phi_stats)
    // host entry point: copy streams and events of the pipelined path, pinned staging of the packed parameters
    cudaStream_t s_in = nullptr, s_out = nullptr;
    cudaStream_t s_band[HOST_BANDS] = {};       // one compute stream per group of images, falling priority
    cudaEvent_t ev[5 + 2 * HOST_BANDS] = {};
    float* h_par_pinned = nullptr;
    size_t h_par_cap = 0;
    Buf arrive;                       // single-image path: {time-out, one word per block of 32 rows}
    unsigned* h_word = nullptr;       // pinned: the time-out word read back
    unsigned* h_flags = nullptr;      // pinned: snapshots of the block words, one per pass / piece of the copy schedule
    size_t h_flags_cap = 0;
    Buf tab;                          // piecewise-linear phi tables [T][N_k][4096] float2 + 4 header floats
    Buf h_f, h_u, h_out, h_par;       // device staging of the host entry point
    Buf bw_maps, bw_part, bw_trace, bw_e[3];   // backward pass: P/V maps, per-CTA partial sums, iterates, dl/du planes
    cudaStream_t s_bw = nullptr;               // tnrd_diffuse_backward: the lag-product kernel of stage t runs here, next to
    cudaEvent_t ev_bw[4] = {};                 // the stage kernel of stage t - 1 (lowest priority; events: maps written / read)
};
std::vector<Scratch*> g_scratch;

int grow(Buf& b, size_t floats, cudaStream_t st)
{
    if (floats <= b.cap) return TNRD_OK;
    // An allocation made inside a stream capture would become a graph memory node whose pointer this cache then hands
    // to later calls outside the graph: refuse, the caller warms the shape up before capturing (include/tnrd.h).
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(st, &cs) == cudaSuccess && cs != cudaStreamCaptureStatusNone)
        return cuda_fail(cudaErrorStreamCaptureUnsupported, "scratch growth during stream capture (run the shape once before capturing)");
    if (b.p) TNRD_CUDA(cudaFreeAsync(b.p, st));
    b.p = nullptr;
    b.cap = 0;
    TNRD_CUDA(cudaMallocAsync(&b.p, floats * sizeof(float), st));
    b.cap = floats;
    return TNRD_OK;
}

int get_scratch(cudaStream_t st, Scratch** out)
{
    int dev = 0;
    TNRD_CUDA(cudaGetDevice(&dev));
    std::lock_guard<std::mutex> lk(g_mu);
    for (Scratch* s : g_scratch)
        if (s->dev == dev && s->st == st) { *out = s; return TNRD_OK; }
    Scratch* s = new Scratch();
    s->dev = dev;
    s->st = st;
    cudaError_t e = cudaDeviceGetAttribute(&s->num_sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) { delete s; return cuda_fail(e, "cudaDeviceGetAttribute"); }
    g_scratch.push_back(s);
    *out = s;
    return TNRD_OK;
}

int check_shape(int B, int H, int W, int N_k, int ksize)
{
    if (B < 1 || H < 1 || W < 1) return TNRD_ERR_SHAPE;
    if ((long long)B * H * W >= (1LL << 31)) return TNRD_ERR_SHAPE;
    if (ksize != 3 && ksize != 5 && ksize != 7 && ksize != 9) return TNRD_ERR_UNSUPPORTED;
    if (N_k < 1 || N_k > TNRD_MAX_FILTERS) return TNRD_ERR_SHAPE;
    if (H < ksize - 1 || W < ksize - 1) return TNRD_ERR_SHAPE;  // mirror source must lie inside the image
    return TNRD_OK;
}

int check_gamma(float g) { return (std::isfinite(g) && g > 0.0f) ? TNRD_OK : TNRD_ERR_PARAM; }

// Everything one call needs: the options as they were at its entry, its launch counter, scratch and stream.
struct Call {
    Opts o;
    LaunchCount lc;
    Scratch* sc = nullptr;
    cudaStream_t st = nullptr;
    bool tc = false;   // this call runs the tensor-core stage kernel
    bool small = false; // this call runs the small-image kernel (all stages in one launch)
    int nchunk_fixed = 0, seg_mult = 2;   // handed to plan_stage_tc by run_stage (the host entry point's first stage)
    bool no_pdl = false;                  // plain launches (StageArgs::pdl = 0)
};

// The automatic choice between the two stage kernels: strips of the tensor-core kernel are 256 - 2r columns wide and
// every CTA recomputes 2r phi rows, so it pays once its units fill the GPU with segments of a few dozen rows.
bool tc_auto(const tnrd::TcPlan& pl, int W, int num_sms, int ksize)
{
    return pl.units * 10 >= (long long)num_sms * 6 && pl.seg_rows > ksize && W >= 192;
}

// Which stage kernel a call uses.  kernel 3 forces the tensor-core kernel (TNRD_ERR_UNSUPPORTED where it does not apply),
// 0 picks it when it applies and the image keeps its 128-lane strips busy: it needs the Gaussian basis with the
// factorised evaluator, ksize 5 or 7 and N_k <= 48 (tnrd_tc.cu).
// The small-image kernel (kernel 4, or the automatic choice for images that fit a cluster; tnrd_small.cu) serves the
// Gaussian basis with the factorised or the direct evaluator.
int pick_small(Call& c, int B, int H, int W, int N_k, int ksize, int phi)
{
    const bool can = tnrd::small_supported(B, H, W, N_k, ksize) && (phi == 3 || phi == 0) && c.o.basis == 0;
    if (c.o.kernel == 4) {
        if (!can) return TNRD_ERR_UNSUPPORTED;
        c.small = true;
    } else if (c.o.kernel == 0) {
        c.small = can;
    }
    return TNRD_OK;
}

// All T stages through the small-image kernel.  Iterates alternate between `out` and the ping-pong plane so that stage T
// lands in `out`; when stage 1 would write the buffer it reads (out == u0 and T odd) u0 is copied to the plane first.
int run_small(Call& c, const float* f, const float* u0, int B, int H, int W, int T, int N_k, int ksize, const float* filters,
              const float* rbf_w, const float* rbf_mu, float gamma, const float* lambda, float lambda_val, float* out, int phi)
{
    const size_t n = (size_t)B * H * W;
    float* pp = nullptr;
    const float* src = u0;
    if (T > 1 || out == u0) {
        int rc = grow(c.sc->pp, n, c.st);
        if (rc != TNRD_OK) return rc;
        pp = c.sc->pp.p;
        if (out == u0 && (T & 1)) {
            TNRD_CUDA(cudaMemcpyAsync(pp, u0, n * sizeof(float), cudaMemcpyDeviceToDevice, c.st));
            src = pp;
        }
    }
    TNRD_CUDA(tnrd::launch_small_diffuse(f, src, out, pp, filters, rbf_w, rbf_mu, gamma, lambda, lambda_val, B, H, W, T, N_k,
                                         ksize, phi == 0 ? 1 : 0, c.st, &c.lc.n));
    return TNRD_OK;
}

int pick_kernel(Call& c, int B, int H, int W, int N_k, int ksize, int phi)
{
    if (c.o.kernel == 4) return TNRD_ERR_UNSUPPORTED;     // the small-image kernel serves tnrd_stage / tnrd_diffuse only
    const bool can = tnrd::tc_supported(N_k, ksize) && phi == 3 && c.o.basis == 0;
    if (c.o.kernel == 3) {
        if (!can) return TNRD_ERR_UNSUPPORTED;
        c.tc = true;
    } else if (c.o.kernel == 0 && can) {
        // strips are 256 - 2r columns wide and every CTA recomputes 2r phi rows: worth it once the units fill the GPU
        c.tc = tc_auto(tnrd::plan_stage_tc(B, H, W, N_k, ksize, c.sc->num_sms), W, c.sc->num_sms, ksize);
    }
    return TNRD_OK;
}

// Stages the parameters of T stages; with the table evaluator also builds the phi tables, with the tensor-core kernel
// the Toeplitz operands.
int stage_params(Call& c, const float* filters, const float* rbf_w, const float* rbf_mu, float gamma, int T, int N_k,
                 int ksize, int phi)
{
    Scratch* sc = c.sc;
    int rc = grow(sc->prm, (size_t)T * N_k * tnrd::prm_stride(ksize), c.st);
    if (rc != TNRD_OK) return rc;
    TNRD_CUDA(tnrd::launch_prep(filters, rbf_w, rbf_mu, gamma, T, N_k, ksize, sc->prm.p, c.st, &c.lc.n));
    if (phi == 2) {
        const size_t n = (size_t)T * N_k * TNRD_TAB_NODES * 2;
        if ((rc = grow(sc->tab, n + 4, c.st)) != TNRD_OK) return rc;
        TNRD_CUDA(tnrd::launch_build_table(rbf_w, rbf_mu, gamma, T * N_k, c.o.basis, sc->tab.p + 4, sc->tab.p, c.st,
                                           &c.lc.n));
    }
    if (c.tc) {
        if ((rc = grow(sc->tcws, (tnrd::tc_workspace_bytes(T, N_k, ksize) + 3) / 4, c.st)) != TNRD_OK) return rc;
        TNRD_CUDA(tnrd::launch_tc_prep(sc->prm.p, T, N_k, ksize, reinterpret_cast<unsigned char*>(sc->tcws.p), c.st,
                                       &c.lc.n));
    }
    return TNRD_OK;
}

// phi: evaluator (0 .. 3); t = stage index inside the staged parameters (selects the table / the operands)
int run_stage(Call& c, tnrd::StageArgs a, int phi, int t)
{
    Scratch* sc = c.sc;
    if (phi == 2) {
        a.tabhdr = sc->tab.p;
        a.tab = sc->tab.p + 4 + (size_t)t * a.N_k * TNRD_TAB_NODES * 2;
    }
    if (c.tc) {
        if (a.u_out == a.u_in) return TNRD_ERR_ALIAS;        // callers ping-pong (run_stages)
        a.pdl = c.no_pdl ? 0 : (t >= 1 ? 2 : 1);   // operands and records of stage t were staged before stage 0 of this call ran
        if (g_stats.load()) {
            if (!sc->stats.p) {
                int rc = grow(sc->stats, 4, c.st);
                if (rc != TNRD_OK) return rc;
                TNRD_CUDA(cudaMemsetAsync(sc->stats.p, 0, 16, c.st));
            }
            a.stats = reinterpret_cast<unsigned long long*>(sc->stats.p);
        }
        const int rows = a.row_hi > 0 ? a.row_hi - a.row_lo : a.H;
        const tnrd::TcPlan pl = tnrd::plan_stage_tc(a.B, rows, a.W, a.N_k, a.ksize, sc->num_sms, c.nchunk_fixed, c.seg_mult);
        if (pl.nchunk > 1) {
            int rc = grow(sc->split, (size_t)pl.nchunk * a.B * a.H * a.W, c.st);
            if (rc != TNRD_OK) return rc;
        }
        const unsigned char* ws = reinterpret_cast<const unsigned char*>(sc->tcws.p) +
                                  (size_t)t * tnrd::tc_ws_stage_stride(a.N_k, a.ksize);
        TNRD_CUDA(tnrd::launch_stage_tc(a, pl, ws, sc->split.p, c.st, &c.lc.n));
    } else if (c.o.kernel == 1) {
        if (c.o.basis == 1) return TNRD_ERR_UNSUPPORTED;     // the reference kernel knows the Gaussian basis only
        int rc = grow(sc->refv, tnrd::ref_scratch_floats(a.B, a.H, a.W, a.N_k, a.ksize), c.st);
        if (rc != TNRD_OK) return rc;
        TNRD_CUDA(tnrd::launch_stage_ref(a, sc->refv.p, c.st, &c.lc.n));
    } else {
        const tnrd::FusedPlan pl = tnrd::plan_stage_fused(a, sc->num_sms);
        int rc = grow(sc->split, pl.part_floats, c.st);
        if (rc != TNRD_OK) return rc;
        TNRD_CUDA(tnrd::launch_stage_fused(a, pl, sc->split.p, phi, c.st, &c.lc.n));
    }
    return TNRD_OK;
}

// One stage from `src` to `dst` for the entry points that allow dst == src: the tile kernel runs in place (it only reads
// u_{t-1} and stores partial sums; the point-wise update kernel follows it on the stream), the tensor-core kernel writes
// u_t itself while other CTAs still read halos of u_{t-1}, so it goes through the ping-pong plane and is copied back.
int run_stage_maybe_inplace(Call& c, tnrd::StageArgs a, int phi, int t)
{
    if (!c.tc || a.u_out != a.u_in) return run_stage(c, a, phi, t);
    const size_t n = (size_t)a.B * a.H * a.W;
    int rc = grow(c.sc->pp, n, c.st);
    if (rc != TNRD_OK) return rc;
    float* dst = a.u_out;
    a.u_out = c.sc->pp.p;
    if ((rc = run_stage(c, a, phi, t)) != TNRD_OK) return rc;
    TNRD_CUDA(cudaMemcpyAsync(dst, c.sc->pp.p, n * sizeof(float), cudaMemcpyDeviceToDevice, c.st));
    return TNRD_OK;
}

int open_call(Call& c, void* stream)
{
    c.st = (cudaStream_t)stream;
    return get_scratch(c.st, &c.sc);
}

}  // namespace

namespace tnrd {
int api_cuda_fail(cudaError_t e, const char* what) { return cuda_fail(e, what); }
void api_count_launches(unsigned long long n) { g_launches.fetch_add(n); }
}  // namespace tnrd

extern "C" {

int tnrd_stage(const float* f, const float* u_in, int B, int H, int W, int N_k, int ksize,
               const float* filters_t, const float* rbf_w_t, const float* rbf_mu, float rbf_gamma,
               float lambda_t, float* u_out, void* stream)
{
    if (!f || !u_in || !filters_t || !rbf_w_t || !rbf_mu || !u_out) return TNRD_ERR_NULL;
    int rc = check_shape(B, H, W, N_k, ksize);
    if (rc != TNRD_OK) return rc;
    if ((rc = check_gamma(rbf_gamma)) != TNRD_OK) return rc;
    if (u_out == f) return TNRD_ERR_ALIAS;
    Call c;
    if ((rc = open_call(c, stream)) != TNRD_OK) return rc;
    const int phi = c.o.phi();
    if ((rc = pick_small(c, B, H, W, N_k, ksize, phi)) != TNRD_OK) return rc;
    if (c.small)
        return run_small(c, f, u_in, B, H, W, 1, N_k, ksize, filters_t, rbf_w_t, rbf_mu, rbf_gamma, nullptr, lambda_t, u_out, phi);
    if ((rc = pick_kernel(c, B, H, W, N_k, ksize, phi)) != TNRD_OK) return rc;
    if ((rc = stage_params(c, filters_t, rbf_w_t, rbf_mu, rbf_gamma, 1, N_k, ksize, phi)) != TNRD_OK) return rc;
    tnrd::StageArgs a{f, u_in, u_out, c.sc->prm.p, nullptr, lambda_t, B, H, W, N_k, ksize};
    return run_stage_maybe_inplace(c, a, phi, 0);
}

int tnrd_diffuse(const float* f, const float* u0, int B, int H, int W, int T, int N_k, int ksize,
                 const float* filters, const float* rbf_w, const float* rbf_mu, float rbf_gamma,
                 const float* lambda, float* out, void* stream)
{
    if (!f || !u0 || !out) return TNRD_ERR_NULL;
    if (T < 0) return TNRD_ERR_SHAPE;
    if (T > 0 && (!filters || !rbf_w || !rbf_mu || !lambda)) return TNRD_ERR_NULL;
    int rc = check_shape(B, H, W, N_k, ksize);
    if (rc != TNRD_OK) return rc;
    if ((rc = check_gamma(rbf_gamma)) != TNRD_OK) return rc;
    if (out == f) return TNRD_ERR_ALIAS;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t n = (size_t)B * H * W;
    if (T == 0) {
        if (out != u0) TNRD_CUDA(cudaMemcpyAsync(out, u0, n * sizeof(float), cudaMemcpyDeviceToDevice, st));
        return TNRD_OK;
    }
    Call c;
    if ((rc = open_call(c, stream)) != TNRD_OK) return rc;
    const size_t rec = (size_t)N_k * tnrd::prm_stride(ksize);
    const int phi = c.o.phi();
    if ((rc = pick_small(c, B, H, W, N_k, ksize, phi)) != TNRD_OK) return rc;
    if (c.small)
        return run_small(c, f, u0, B, H, W, T, N_k, ksize, filters, rbf_w, rbf_mu, rbf_gamma, lambda, 0.0f, out, phi);
    if ((rc = pick_kernel(c, B, H, W, N_k, ksize, phi)) != TNRD_OK) return rc;
    if ((rc = stage_params(c, filters, rbf_w, rbf_mu, rbf_gamma, T, N_k, ksize, phi)) != TNRD_OK) return rc;
    const float* src = u0;
    if (!c.tc) {
        // Tile kernel: every stage writes `out`, from the second one on in place: the tile kernel only READS u_{t-1} (all
        // halo reads happen there) and stores partial sums in scratch; the update kernel that follows it is point-wise.
        for (int t = 1; t <= T; ++t) {
            tnrd::StageArgs a{f, src, out, c.sc->prm.p + (size_t)(t - 1) * rec, lambda + (t - 1), 0.0f, B, H, W, N_k, ksize};
            if ((rc = run_stage(c, a, phi, t - 1)) != TNRD_OK) return rc;
            src = out;
        }
        return TNRD_OK;
    }
    // Tensor-core kernel: u_t is written by the stage kernel itself, so stages alternate between `out` and one ping-pong
    // plane such that stage T lands in `out`; when that would make stage 1 write the plane it reads (out == u0 and T odd)
    // u0 is copied to the plane first.
    if (T > 1 || out == u0)
        if ((rc = grow(c.sc->pp, n, st)) != TNRD_OK) return rc;
    float* pp = c.sc->pp.p;
    if (out == u0 && (T & 1)) {
        TNRD_CUDA(cudaMemcpyAsync(pp, u0, n * sizeof(float), cudaMemcpyDeviceToDevice, st));
        src = pp;
    }
    for (int t = 1; t <= T; ++t) {
        float* dst = ((T - t) & 1) ? pp : out;
        tnrd::StageArgs a{f, src, dst, c.sc->prm.p + (size_t)(t - 1) * rec, lambda + (t - 1), 0.0f, B, H, W, N_k, ksize};
        if ((rc = run_stage(c, a, phi, t - 1)) != TNRD_OK) return rc;
        src = dst;
    }
    return TNRD_OK;
}

// Copy streams, events and the pinned parameter staging of the host entry point (created on first use).
static int host_pipe_init(Scratch* sc, size_t npar)
{
    if (!sc->s_in) {
        TNRD_CUDA(cudaStreamCreateWithFlags(&sc->s_in, cudaStreamNonBlocking));
        TNRD_CUDA(cudaStreamCreateWithFlags(&sc->s_out, cudaStreamNonBlocking));
        int pr_least = 0, pr_greatest = 0;      // numerically lower = more urgent
        TNRD_CUDA(cudaDeviceGetStreamPriorityRange(&pr_least, &pr_greatest));
        for (int g = 0; g < HOST_BANDS; ++g) {
            const int pr = pr_greatest + g < pr_least ? pr_greatest + g : pr_least;
            TNRD_CUDA(cudaStreamCreateWithPriority(&sc->s_band[g], cudaStreamNonBlocking, pr));
        }
        for (auto& e : sc->ev) TNRD_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        TNRD_CUDA(cudaHostAlloc(&sc->h_word, sizeof(unsigned), cudaHostAllocDefault));
    }
    if (npar > sc->h_par_cap) {
        if (sc->h_par_pinned) TNRD_CUDA(cudaFreeHost(sc->h_par_pinned));
        sc->h_par_pinned = nullptr;
        sc->h_par_cap = 0;
        TNRD_CUDA(cudaHostAlloc(&sc->h_par_pinned, npar * sizeof(float), cudaHostAllocDefault));
        sc->h_par_cap = npar;
    }
    return TNRD_OK;
}

static int host_flags_reserve(Scratch* sc, size_t words)
{
    if (words <= sc->h_flags_cap) return TNRD_OK;
    if (sc->h_flags) TNRD_CUDA(cudaFreeHost(sc->h_flags));
    sc->h_flags = nullptr;
    sc->h_flags_cap = 0;
    TNRD_CUDA(cudaHostAlloc(&sc->h_flags, words * sizeof(unsigned), cudaHostAllocDefault));
    sc->h_flags_cap = words;
    return TNRD_OK;
}

// The device address of a host result buffer the last stage may store into directly (pinned or otherwise device-mapped
// memory), or null.  Not when `out` overlaps an input: with T = 1 the stage that stores u_T runs while the input arrives.
static float* host_mapped_out(float* out, const float* f, const float* u0, size_t n)
{
    const bool apart = (out + n <= f || f + n <= out) && (out + n <= u0 || u0 + n <= out);
    cudaPointerAttributes pa;
    float* dev = nullptr;
    if (apart && cudaPointerGetAttributes(&pa, out) == cudaSuccess && pa.type == cudaMemoryTypeHost && pa.devicePointer)
        dev = static_cast<float*>(pa.devicePointer);
    (void)cudaGetLastError();
    return dev;
}

// experiments with the host entry point: 1 = a single image takes the two-halves path as well, 2 = never store to host
// memory from a kernel, 3 = the input strictly top to bottom, 4 = serial (upload, stages, download)
static int host_mode_env()
{
    const char* e = getenv("TNRD_HOST_MODE");
    return e ? atoi(e) : 0;
}

int tnrd_diffuse_host(const float* f, const float* u0, int B, int H, int W, int T, int N_k, int ksize,
                      const float* filters, const float* rbf_w, const float* rbf_mu, float rbf_gamma,
                      const float* lambda, float* out, void* stream)
{
    if (!f || !u0 || !out) return TNRD_ERR_NULL;
    if (T < 0) return TNRD_ERR_SHAPE;
    if (T > 0 && (!filters || !rbf_w || !rbf_mu || !lambda)) return TNRD_ERR_NULL;
    int rc = check_shape(B, H, W, N_k, ksize);
    if (rc != TNRD_OK) return rc;
    if ((rc = check_gamma(rbf_gamma)) != TNRD_OK) return rc;
    Call c;
    if ((rc = open_call(c, stream)) != TNRD_OK) return rc;
    Scratch* sc = c.sc;
    cudaStream_t st = c.st;
    const size_t n = (size_t)B * H * W;
    const size_t nk = (size_t)T * N_k * ksize * ksize, nw = (size_t)T * N_k * TNRD_NUM_RBF;
    const size_t npar = nk + nw + TNRD_NUM_RBF + (size_t)T;
    if ((rc = grow(sc->h_f, n, st)) != TNRD_OK) return rc;
    if (u0 != f && (rc = grow(sc->h_u, n, st)) != TNRD_OK) return rc;
    if ((rc = grow(sc->h_out, n, st)) != TNRD_OK) return rc;
    if ((rc = grow(sc->h_par, npar > 0 ? npar : 1, st)) != TNRD_OK) return rc;
    if ((rc = host_pipe_init(sc, npar > 0 ? npar : 1)) != TNRD_OK) return rc;
    float* d_k = sc->h_par.p;
    float* d_w = d_k + nk;
    float* d_mu = d_w + nw;
    float* d_lam = d_mu + TNRD_NUM_RBF;
    float* d_f = sc->h_f.p;
    float* d_u0 = (u0 != f) ? sc->h_u.p : sc->h_f.p;
    float* d_out = sc->h_out.p;
    if (T > 0) {        // the parameters: packed on the host, ONE copy
        float* hp = sc->h_par_pinned;
        memcpy(hp, filters, nk * sizeof(float));
        memcpy(hp + nk, rbf_w, nw * sizeof(float));
        memcpy(hp + nk + nw, rbf_mu, TNRD_NUM_RBF * sizeof(float));
        memcpy(hp + nk + nw + TNRD_NUM_RBF, lambda, (size_t)T * sizeof(float));
        TNRD_CUDA(cudaMemcpyAsync(d_k, hp, npar * sizeof(float), cudaMemcpyHostToDevice, st));
    }
    const int phi = c.o.phi();
    bool piped = false;
    if (T > 0) {
        if ((rc = pick_small(c, B, H, W, N_k, ksize, phi)) != TNRD_OK) return rc;
        if (!c.small && (rc = pick_kernel(c, B, H, W, N_k, ksize, phi)) != TNRD_OK) return rc;
        // below about two million pixels the dozen extra copies and events of the pipelined paths cost more than they hide
        // (1024^2: 1.43 ms serial, 1.53 ms pipelined; 2048^2: 4.35 / 3.96); TNRD_HOST_PIPE_MIN (pixels) for the tests
        const char* pm = getenv("TNRD_HOST_PIPE_MIN");
        const size_t pipe_min = pm ? (size_t)atoll(pm) : ((size_t)1 << 21);
        piped = c.tc && (B >= 2 || H >= 256) && n >= pipe_min && host_mode_env() != 4;
    }
    if (!piped) {
        // serial: upload, all stages, download (small images, the tile kernel)
        TNRD_CUDA(cudaMemcpyAsync(d_f, f, n * sizeof(float), cudaMemcpyHostToDevice, st));
        if (u0 != f) TNRD_CUDA(cudaMemcpyAsync(d_u0, u0, n * sizeof(float), cudaMemcpyHostToDevice, st));
        float* out_dev = (c.tc && T > 0 && host_mode_env() != 2) ? host_mapped_out(out, f, u0, n) : nullptr;
        if (out_dev) {
            // tensor-core kernel and a pinned result buffer: the last stage stores u_T into it, no copy back
            if ((rc = stage_params(c, d_k, d_w, d_mu, rbf_gamma, T, N_k, ksize, phi)) != TNRD_OK) return rc;
            if (T > 1 && (rc = grow(sc->pp, n, st)) != TNRD_OK) return rc;
            const size_t rec = (size_t)N_k * tnrd::prm_stride(ksize);
            const float* src = d_u0;
            for (int t = 1; t <= T; ++t) {
                float* dst = ((T - t) & 1) ? sc->pp.p : (t == T ? out_dev : d_out);
                tnrd::StageArgs a{d_f, src, dst, sc->prm.p + (size_t)(t - 1) * rec, d_lam + (t - 1), 0.0f, B, H, W, N_k, ksize};
                if ((rc = run_stage(c, a, phi, t - 1)) != TNRD_OK) return rc;
                src = dst;
            }
            TNRD_CUDA(cudaStreamSynchronize(st));
            return TNRD_OK;
        }
        rc = tnrd_diffuse(d_f, d_u0, B, H, W, T, N_k, ksize, d_k, d_w, d_mu, rbf_gamma, d_lam, d_out, stream);
        if (rc != TNRD_OK) return rc;
        TNRD_CUDA(cudaMemcpyAsync(out, d_out, n * sizeof(float), cudaMemcpyDeviceToHost, st));
        TNRD_CUDA(cudaStreamSynchronize(st));
        return TNRD_OK;
    }
    if (B == 1 && host_mode_env() != 1) {
        // One image: the stage launches are those of the device call (the first with segment heights that are a multiple
        // of 32).  The input arrives in blocks of 32 whole rows (they end on 128-byte lines) on a copy stream, and one
        // word per block says so; the loader warps of the FIRST stage poll the word of a block before they read its
        // first row, so the stage starts with the first blocks instead of the last.  When `out` is pinned host memory
        // the LAST stage stores u_T straight into it (posted writes over PCIe while the stage computes), otherwise one
        // copy follows.  Same arithmetic per pixel whatever the segments: bit-identical to the device call.
        if ((rc = stage_params(c, d_k, d_w, d_mu, rbf_gamma, T, N_k, ksize, phi)) != TNRD_OK) return rc;
        const int nblk = (H + 31) / 32;
        if ((rc = grow(sc->arrive, (size_t)nblk + 4, st)) != TNRD_OK) return rc;
        if (T > 1 && (rc = grow(sc->pp, n, st)) != TNRD_OK) return rc;
        float* out_dev = host_mode_env() != 2 ? host_mapped_out(out, f, u0, n) : nullptr;
        unsigned* arrived = reinterpret_cast<unsigned*>(sc->arrive.p);
        TNRD_CUDA(cudaEventRecord(sc->ev[0], st));
        TNRD_CUDA(cudaStreamWaitEvent(sc->s_in, sc->ev[0], 0));
        TNRD_CUDA(cudaMemsetAsync(arrived, 0, ((size_t)nblk + 1) * sizeof(unsigned), sc->s_in));
        TNRD_CUDA(cudaEventRecord(sc->ev[1], sc->s_in));
        // The copy schedule.  The first stage's CTAs each walk down a segment of S rows, and the first wave of CTAs
        // covers the top `nreg` segments: their rows go first, INTERLEAVED -- pass k brings rows [32 k, 32 k + 32) of
        // every region (region j = the rows segment j reads first, [j S - 32, (j + 1) S - 32); one strided copy per
        // pass) -- so that every CTA of the first wave starts after the first pass and the data then stays ahead of
        // it.  The rest of the image follows top to bottom in pieces of about 4 MB.  After every pass / piece the
        // block words are refreshed with one small copy from a pinned snapshot.
        const int nchunk_dev = tnrd::plan_stage_tc(1, H, W, N_k, ksize, sc->num_sms).nchunk;     // as the device call cuts the bank
        const tnrd::TcPlan pl1 = tnrd::plan_stage_tc(1, H, W, N_k, ksize, sc->num_sms, nchunk_dev, 32);
        const int S = pl1.seg_rows;
        int nreg = (sc->num_sms + pl1.nxs * pl1.nchunk - 1) / (pl1.nxs * pl1.nchunk);
        if (nreg > pl1.nys) nreg = pl1.nys;
        const bool inter = S % 32 == 0 && S >= 64 && nreg >= 2 && host_mode_env() != 3;
        const int E = !inter ? 0 : ((long long)nreg * S - 32 > H ? H : nreg * S - 32);   // rows [0, E) are interleaved
        int piece = (int)(((1u << 20) / (size_t)W + 31) & ~(size_t)31);       // rows per piece of the linear part
        if (piece < 32) piece = 32;
        {
            int ops = (inter ? S / 32 : 0) + 8;
            for (int r = E, pc = inter ? piece : 32; r < H; r += pc, ++ops) if (!inter && pc < piece) pc *= 2;
            if ((rc = host_flags_reserve(sc, (size_t)ops * nblk)) != TNRD_OK) return rc;
        }
        std::vector<unsigned> ok((size_t)nblk, 0u);
        int op = 0;
        auto copy_rows = [&](int r0, int r1) -> int {
            const size_t o = (size_t)r0 * W, cnt = (size_t)(r1 - r0) * W;
            TNRD_CUDA(cudaMemcpyAsync(d_f + o, f + o, cnt * sizeof(float), cudaMemcpyHostToDevice, sc->s_in));
            if (u0 != f) TNRD_CUDA(cudaMemcpyAsync(d_u0 + o, u0 + o, cnt * sizeof(float), cudaMemcpyHostToDevice, sc->s_in));
            for (int bk = r0 / 32; bk < (r1 + 31) / 32; ++bk) ok[bk] = 1u;
            return TNRD_OK;
        };
        auto flush = [&]() -> int {
            unsigned* snap = sc->h_flags + (size_t)op * nblk;
            memcpy(snap, ok.data(), (size_t)nblk * sizeof(unsigned));
            TNRD_CUDA(cudaMemcpyAsync(arrived + 1, snap, (size_t)nblk * sizeof(unsigned), cudaMemcpyHostToDevice, sc->s_in));
            ++op;
            return TNRD_OK;
        };
        if (inter) {
            const int npass = S / 32;
            for (int k = 0; k < npass; ++k) {
                if (k <= npass - 2 && 32 * k < E)         // region 0 = rows [0, S - 32)
                    if ((rc = copy_rows(32 * k, 32 * k + 32 < E ? 32 * k + 32 : E)) != TNRD_OK) return rc;
                int jfull = 0;                            // regions 1 .. jfull have this block whole
                for (int j = 1; j < nreg && j * S + 32 * k <= E; ++j) jfull = j;
                if (jfull >= 1) {
                    const size_t o = (size_t)(S - 32 + 32 * k) * W, pitch = (size_t)S * W * sizeof(float);
                    const size_t width = (size_t)32 * W * sizeof(float);
                    TNRD_CUDA(cudaMemcpy2DAsync(d_f + o, pitch, f + o, pitch, width, (size_t)jfull, cudaMemcpyHostToDevice, sc->s_in));
                    if (u0 != f)
                        TNRD_CUDA(cudaMemcpy2DAsync(d_u0 + o, pitch, u0 + o, pitch, width, (size_t)jfull, cudaMemcpyHostToDevice, sc->s_in));
                    for (int j = 1; j <= jfull; ++j) ok[(j * S - 32 + 32 * k) / 32] = 1u;
                }
                const int tail = (jfull + 1) * S - 32 + 32 * k;      // a last block cut short by the end of the image
                if (jfull + 1 < nreg && tail < E)
                    if ((rc = copy_rows(tail, E)) != TNRD_OK) return rc;
                if ((rc = flush()) != TNRD_OK) return rc;
            }
        }
        for (int r0 = E, pc = inter ? piece : 32; r0 < H;) {
            const int r1 = r0 + pc < H ? r0 + pc : H;
            if ((rc = copy_rows(r0, r1)) != TNRD_OK) return rc;
            if ((rc = flush()) != TNRD_OK) return rc;
            r0 = r1;
            if (!inter && pc < piece) pc *= 2;
        }
        TNRD_CUDA(cudaStreamWaitEvent(st, sc->ev[1], 0));          // the block words are zero before the first stage starts
        const size_t rec = (size_t)N_k * tnrd::prm_stride(ksize);
        const float* src = d_u0;
        for (int t = 1; t <= T; ++t) {
            float* dst = ((T - t) & 1) ? sc->pp.p : (t == T && out_dev ? out_dev : d_out);
            tnrd::StageArgs a{d_f, src, dst, sc->prm.p + (size_t)(t - 1) * rec, d_lam + (t - 1), 0.0f, B, H, W, N_k, ksize};
            if (t == 1) {                           // the plan the copy schedule was made for
                a.arrived = arrived;
                c.nchunk_fixed = nchunk_dev;
                c.seg_mult = 32;
            } else {
                c.nchunk_fixed = 0;
                c.seg_mult = 2;
            }
            if ((rc = run_stage(c, a, phi, t - 1)) != TNRD_OK) return rc;
            src = dst;
        }
        if (!out_dev) TNRD_CUDA(cudaMemcpyAsync(out, d_out, n * sizeof(float), cudaMemcpyDeviceToHost, st));
        *sc->h_word = 0;
        TNRD_CUDA(cudaMemcpyAsync(sc->h_word, arrived, sizeof(unsigned), cudaMemcpyDeviceToHost, st));
        TNRD_CUDA(cudaStreamSynchronize(st));
        TNRD_CUDA(cudaStreamSynchronize(sc->s_in));
        if (*sc->h_word) return cuda_fail(cudaErrorLaunchTimeout, "tnrd_diffuse_host: the first stage gave up waiting for its input");
        return TNRD_OK;
    }
    // the filter chunks of the device call: every launch below cuts the bank the same way (the order of the sum over
    // filters), whatever part of the batch it covers
    const int nchunk_call = tnrd::plan_stage_tc(B, H, W, N_k, ksize, sc->num_sms).nchunk;
    if (B >= 2 && nchunk_call == 1 && host_mode_env() != 1) {
        // A batch: up to four GROUPS of images, each taken through all T stages on a stream of its own (falling priority,
        // so that the groups finish one after the other; the SMs a group's last wave leaves idle take units of the next
        // group).  Group g computes while the input of group g+1 arrives and the result of group g-1 leaves.  The first
        // and the last group are small (their copies are the ones nothing hides).  Images are independent: bit-identical.
        if ((rc = stage_params(c, d_k, d_w, d_mu, rbf_gamma, T, N_k, ksize, phi)) != TNRD_OK) return rc;
        if (g_stats.load() && !sc->stats.p) {
            if ((rc = grow(sc->stats, 4, st)) != TNRD_OK) return rc;
            TNRD_CUDA(cudaMemsetAsync(sc->stats.p, 0, 16, st));
        }
        if (T > 1 && (rc = grow(sc->pp, n, st)) != TNRD_OK) return rc;
        int lo[HOST_BANDS], hi[HOST_BANDS], G = 0;
        {
            const int want = B < HOST_BANDS ? B : HOST_BANDS;
            const long long wsum = want >= 2 ? 2 + 3LL * (want - 2) : 1;
            long long acc = 0;
            int prev = 0;
            for (int g = 0; g < want; ++g) {
                acc += (g == 0 || g == want - 1) ? 1 : 3;
                const int cut = g == want - 1 ? B : (int)((B * acc + wsum / 2) / wsum);
                if (cut <= prev) continue;
                lo[G] = prev; hi[G] = cut; prev = cut; ++G;
            }
        }
        const size_t plane = (size_t)H * W;
        cudaEvent_t* ev_in = sc->ev + 5;
        cudaEvent_t* ev_done = sc->ev + 5 + HOST_BANDS;
        TNRD_CUDA(cudaEventRecord(sc->ev[0], st));
        TNRD_CUDA(cudaStreamWaitEvent(sc->s_in, sc->ev[0], 0));
        TNRD_CUDA(cudaStreamWaitEvent(sc->s_out, sc->ev[0], 0));
        for (int g = 0; g < G; ++g) {
            const size_t o = (size_t)lo[g] * plane, cnt = (size_t)(hi[g] - lo[g]) * plane;
            TNRD_CUDA(cudaMemcpyAsync(d_f + o, f + o, cnt * sizeof(float), cudaMemcpyHostToDevice, sc->s_in));
            if (u0 != f) TNRD_CUDA(cudaMemcpyAsync(d_u0 + o, u0 + o, cnt * sizeof(float), cudaMemcpyHostToDevice, sc->s_in));
            TNRD_CUDA(cudaEventRecord(ev_in[g], sc->s_in));
        }
        const size_t rec = (size_t)N_k * tnrd::prm_stride(ksize);
        c.nchunk_fixed = 1;                 // concurrent launches must not share the partial-sum scratch
        c.no_pdl = true;
        for (int g = 0; g < G; ++g) {
            cudaStream_t bs = sc->s_band[g];
            TNRD_CUDA(cudaStreamWaitEvent(bs, sc->ev[0], 0));
            TNRD_CUDA(cudaStreamWaitEvent(bs, ev_in[g], 0));
            const size_t o = (size_t)lo[g] * plane, cnt = (size_t)(hi[g] - lo[g]) * plane;
            const float* src = d_u0 + o;
            c.st = bs;
            for (int t = 1; t <= T && rc == TNRD_OK; ++t) {
                float* dst = (((T - t) & 1) ? sc->pp.p : d_out) + o;
                tnrd::StageArgs a{d_f + o, src, dst, sc->prm.p + (size_t)(t - 1) * rec, d_lam + (t - 1), 0.0f,
                                  hi[g] - lo[g], H, W, N_k, ksize};
                rc = run_stage(c, a, phi, t - 1);
                src = dst;
            }
            c.st = st;
            if (rc != TNRD_OK) return rc;
            TNRD_CUDA(cudaEventRecord(ev_done[g], bs));
            TNRD_CUDA(cudaStreamWaitEvent(sc->s_out, ev_done[g], 0));
            TNRD_CUDA(cudaMemcpyAsync(out + o, d_out + o, cnt * sizeof(float), cudaMemcpyDeviceToHost, sc->s_out));
            TNRD_CUDA(cudaStreamWaitEvent(st, ev_done[g], 0));     // later work on the caller's stream comes after the groups
        }
        TNRD_CUDA(cudaStreamSynchronize(sc->s_out));
        TNRD_CUDA(cudaStreamSynchronize(st));
        return TNRD_OK;
    }
    c.nchunk_fixed = nchunk_call;
    // What is left (a batch whose stages cut the filter bank, TNRD_HOST_MODE = 1): the work of the FIRST and the LAST
    // stage is cut in two halves -- the two halves of the batch, or of the rows of a single image (an even row, so that every pixel sees the arithmetic of the un-cut
    // launch and the result is bit-identical) -- so that the first half computes while the second half of the input
    // arrives, and the first half of the result leaves while the second half computes.  Copies run on two internal
    // streams ordered against `stream` by events.
    if ((rc = stage_params(c, d_k, d_w, d_mu, rbf_gamma, T, N_k, ksize, phi)) != TNRD_OK) return rc;
    const bool by_img = B >= 2;
    const int R = (ksize - 1) / 2;
    const int b_mid = B / 2, r_mid = (H / 2) & ~1;
    const size_t plane = (size_t)H * W;
    // elements [0, cutA) must have arrived before the first half starts: its images, or its rows plus the 2r halo
    const size_t cutA = by_img ? (size_t)b_mid * plane : (size_t)(r_mid + 2 * R < H ? r_mid + 2 * R : H) * W;
    const size_t cutO = by_img ? (size_t)b_mid * plane : (size_t)r_mid * W;       // first half of the result
    TNRD_CUDA(cudaEventRecord(sc->ev[0], st));
    TNRD_CUDA(cudaStreamWaitEvent(sc->s_in, sc->ev[0], 0));
    TNRD_CUDA(cudaMemcpyAsync(d_f, f, cutA * sizeof(float), cudaMemcpyHostToDevice, sc->s_in));
    if (u0 != f) TNRD_CUDA(cudaMemcpyAsync(d_u0, u0, cutA * sizeof(float), cudaMemcpyHostToDevice, sc->s_in));
    TNRD_CUDA(cudaEventRecord(sc->ev[1], sc->s_in));
    TNRD_CUDA(cudaMemcpyAsync(d_f + cutA, f + cutA, (n - cutA) * sizeof(float), cudaMemcpyHostToDevice, sc->s_in));
    if (u0 != f) TNRD_CUDA(cudaMemcpyAsync(d_u0 + cutA, u0 + cutA, (n - cutA) * sizeof(float), cudaMemcpyHostToDevice, sc->s_in));
    TNRD_CUDA(cudaEventRecord(sc->ev[2], sc->s_in));
    if (T > 1 && (rc = grow(sc->pp, n, st)) != TNRD_OK) return rc;
    float* pp = sc->pp.p;
    const size_t rec = (size_t)N_k * tnrd::prm_stride(ksize);
    const float* src = d_u0;
    for (int t = 1; t <= T; ++t) {
        float* dst = ((T - t) & 1) ? pp : d_out;
        tnrd::StageArgs a{d_f, src, dst, sc->prm.p + (size_t)(t - 1) * rec, d_lam + (t - 1), 0.0f, B, H, W, N_k, ksize};
        const bool first = t == 1, last = t == T;
        if (!first && !last) {
            if ((rc = run_stage(c, a, phi, t - 1)) != TNRD_OK) return rc;
        } else {
            for (int half = 0; half < 2; ++half) {
                tnrd::StageArgs h = a;
                if (by_img) {
                    const size_t off = half ? (size_t)b_mid * plane : 0;
                    h.f += off; h.u_in += off; h.u_out += off;
                    h.B = half ? B - b_mid : b_mid;
                } else {
                    h.row_lo = half ? r_mid : 0;
                    h.row_hi = half ? H : r_mid;
                }
                if (first) TNRD_CUDA(cudaStreamWaitEvent(st, sc->ev[1 + half], 0));
                if ((rc = run_stage(c, h, phi, t - 1)) != TNRD_OK) return rc;
                if (last) {
                    TNRD_CUDA(cudaEventRecord(sc->ev[3 + half], st));
                    TNRD_CUDA(cudaStreamWaitEvent(sc->s_out, sc->ev[3 + half], 0));
                    const size_t o0 = half ? cutO : 0, cnt = half ? n - cutO : cutO;
                    TNRD_CUDA(cudaMemcpyAsync(out + o0, d_out + o0, cnt * sizeof(float), cudaMemcpyDeviceToHost, sc->s_out));
                }
            }
        }
        src = dst;
    }
    TNRD_CUDA(cudaStreamSynchronize(sc->s_out));
    TNRD_CUDA(cudaStreamSynchronize(st));
    return TNRD_OK;
}

int tnrd_qcs_project(const float* y, int B, int H, int W, const float* qcs_lo, const float* qcs_hi, float* u_out,
                     void* stream)
{
    if (!y || !qcs_lo || !qcs_hi || !u_out) return TNRD_ERR_NULL;
    if (B < 1 || H < 8 || W < 8 || (H % 8) || (W % 8) || (long long)B * H * W >= (1LL << 31)) return TNRD_ERR_SHAPE;
    if (u_out == qcs_lo || u_out == qcs_hi) return TNRD_ERR_ALIAS;
    LaunchCount lc;
    TNRD_CUDA(tnrd::launch_qcs_project(y, qcs_lo, qcs_hi, u_out, B, H, W, (cudaStream_t)stream, &lc.n));
    return TNRD_OK;
}

int tnrd_deblock_diffuse(const float* u0, int B, int H, int W, int T, int N_k, int ksize, const float* filters,
                         const float* rbf_w, const float* rbf_mu, float rbf_gamma, const float* qcs_lo,
                         const float* qcs_hi, float* out, void* stream)
{
    if (!u0 || !out || !qcs_lo || !qcs_hi) return TNRD_ERR_NULL;
    if (T < 0) return TNRD_ERR_SHAPE;
    if (T > 0 && (!filters || !rbf_w || !rbf_mu)) return TNRD_ERR_NULL;
    int rc = check_shape(B, H, W, N_k, ksize);
    if (rc != TNRD_OK) return rc;
    if ((H % 8) || (W % 8)) return TNRD_ERR_SHAPE;
    if ((rc = check_gamma(rbf_gamma)) != TNRD_OK) return rc;
    if (out == qcs_lo || out == qcs_hi) return TNRD_ERR_ALIAS;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t n = (size_t)B * H * W;
    if (T == 0) {
        if (out != u0) TNRD_CUDA(cudaMemcpyAsync(out, u0, n * sizeof(float), cudaMemcpyDeviceToDevice, st));
        return TNRD_OK;
    }
    Call c;
    if ((rc = open_call(c, stream)) != TNRD_OK) return rc;
    const size_t rec = (size_t)N_k * tnrd::prm_stride(ksize);
    const int phi = c.o.phi();
    if ((rc = pick_kernel(c, B, H, W, N_k, ksize, phi)) != TNRD_OK) return rc;
    if ((rc = stage_params(c, filters, rbf_w, rbf_mu, rbf_gamma, T, N_k, ksize, phi)) != TNRD_OK) return rc;
    // Per stage (Supp. Eq. 29): the stage kernels with lambda = 0 write y = u - sum_i kbar_i * phi_i(k_i * u) (f is then
    // irrelevant: u itself is passed), the projection kernel turns it into u_t = D^T eta(D y) in place.  Buffers as in
    // tnrd_diffuse: in place with the tile kernel, alternating between `out` and the ping-pong plane with the
    // tensor-core kernel.
    float* pp = nullptr;
    const float* src = u0;
    if (c.tc && (T > 1 || out == u0)) {
        if ((rc = grow(c.sc->pp, n, st)) != TNRD_OK) return rc;
        pp = c.sc->pp.p;
        if (out == u0 && (T & 1)) {
            TNRD_CUDA(cudaMemcpyAsync(pp, u0, n * sizeof(float), cudaMemcpyDeviceToDevice, st));
            src = pp;
        }
    }
    for (int t = 1; t <= T; ++t) {
        float* dst = (c.tc && ((T - t) & 1)) ? pp : out;
        tnrd::StageArgs a{src, src, dst, c.sc->prm.p + (size_t)(t - 1) * rec, nullptr, 0.0f, B, H, W, N_k, ksize};
        if ((rc = run_stage(c, a, phi, t - 1)) != TNRD_OK) return rc;
        TNRD_CUDA(tnrd::launch_qcs_project(dst, qcs_lo, qcs_hi, dst, B, H, W, st, &c.lc.n));
        src = dst;
    }
    return TNRD_OK;
}

// Backward pass of one stage on staged parameters (shared by tnrd_stage_backward and tnrd_diffuse_backward).
// tnrd_diffuse_backward overlaps the lag-product kernel (g_k) of stage t with the stage kernel of stage t - 1: the stage
// kernel's 1296 CTAs at 2048^2 are 4.4 waves of the 296 resident slots, so a fifth of the GPU idles in its last wave, and
// the lag products of stage t are needed by nobody until the call returns.  The maps and the g_k partial sums are double
// buffered by `parity`; evA[p] = maps p written, evB[p] = maps p (and the dl/du plane of that stage) no longer read.
struct BwdSide {
    cudaStream_t s2;
    cudaEvent_t evA[2], evB[2];
    int parity = 0;
    bool used[2] = {false, false};
};

static int run_stage_backward(Call& c, const float* f, const float* u, const float* e, int B, int H, int W, int N_k,
                              int ksize, const float* prm, const float* lambda_ptr, float lambda_val, float gamma,
                              float* g_u, float* g_k, float* g_w, float* g_l, BwdSide* side = nullptr)
{
    Scratch* sc = c.sc;
    cudaStream_t st = c.st;
    const tnrd::BwdPlan pl = tnrd::plan_stage_bwd(B, H, W, N_k, ksize, sc->num_sms);
    const int R = (ksize - 1) / 2, KK = ksize * ksize;
    const bool want_k = g_k != nullptr, want_w = g_w != nullptr || want_k;
    const size_t n_w = want_w ? (size_t)pl.n_cta * N_k * 64 : 0, n_l = (size_t)pl.n_cta;
    const size_t n_k = want_k ? (size_t)pl.G * N_k * KK : 0;
    if (!want_k) side = nullptr;
    const int p = side ? side->parity : 0;
    int rc = grow(sc->bw_part, n_w + n_l + 2 * n_k + 4, st);
    if (rc != TNRD_OK) return rc;
    const size_t map = want_k ? (size_t)B * N_k * (H + 2 * R) * (W + 2 * R) : 0;
    if (want_k && (rc = grow(sc->bw_maps, (side ? 4 : 2) * map, st)) != TNRD_OK) return rc;
    float* part_w = sc->bw_part.p;
    float* part_l = part_w + n_w;
    float* part_k = part_l + n_l + (size_t)p * n_k;
    float* maps = sc->bw_maps.p + (size_t)p * 2 * map;
    tnrd::BwdArgs a{f, u, e, g_u, prm, lambda_ptr, lambda_val, B, H, W, N_k, ksize,
                    want_k ? maps : nullptr, want_k ? maps + map : nullptr,
                    want_w ? part_w : nullptr, g_l ? part_l : nullptr};
    const float s = sqrtf(1.4426950408889634f / (2.0f * gamma * gamma));
    if (!side) {
        TNRD_CUDA(tnrd::launch_stage_bwd(a, pl, part_k, 3, st, &c.lc.n));
        if (want_w || g_l)
            TNRD_CUDA(tnrd::launch_reduce_partials(part_w, pl.n_cta, part_k, pl.G, part_l, N_k, ksize, s, g_w, g_k, g_l, st,
                                                   &c.lc.n));
        return TNRD_OK;
    }
    if (side->used[p]) TNRD_CUDA(cudaStreamWaitEvent(st, side->evB[p], 0));     // two stages ago: done with these buffers
    TNRD_CUDA(tnrd::launch_stage_bwd(a, pl, part_k, 1, st, &c.lc.n));
    TNRD_CUDA(cudaEventRecord(side->evA[p], st));
    if (g_w || g_l)
        TNRD_CUDA(tnrd::launch_reduce_partials(part_w, pl.n_cta, nullptr, 0, part_l, N_k, ksize, s, g_w, nullptr, g_l, st,
                                               &c.lc.n));
    TNRD_CUDA(cudaStreamWaitEvent(side->s2, side->evA[p], 0));
    TNRD_CUDA(tnrd::launch_stage_bwd(a, pl, part_k, 2, side->s2, &c.lc.n));
    TNRD_CUDA(tnrd::launch_reduce_partials(nullptr, 0, part_k, pl.G, nullptr, N_k, ksize, s, nullptr, g_k, nullptr, side->s2,
                                           &c.lc.n));
    TNRD_CUDA(cudaEventRecord(side->evB[p], side->s2));
    side->used[p] = true;
    side->parity ^= 1;
    return TNRD_OK;
}

int tnrd_stage_backward(const float* f, const float* u_in, const float* e, int B, int H, int W, int N_k, int ksize,
                        const float* filters_t, const float* rbf_w_t, const float* rbf_mu, float rbf_gamma,
                        float lambda_t, float* grad_u, float* grad_filters, float* grad_w, float* grad_lambda,
                        void* stream)
{
    if (!f || !u_in || !e || !filters_t || !rbf_w_t || !rbf_mu) return TNRD_ERR_NULL;
    int rc = check_shape(B, H, W, N_k, ksize);
    if (rc != TNRD_OK) return rc;
    if ((rc = check_gamma(rbf_gamma)) != TNRD_OK) return rc;
    if (grad_u && (grad_u == u_in || grad_u == e || grad_u == f)) return TNRD_ERR_ALIAS;
    Call c;
    if (c.o.basis == 1) return TNRD_ERR_UNSUPPORTED;          // gradients exist for the Gaussian basis only
    if ((rc = open_call(c, stream)) != TNRD_OK) return rc;
    if ((rc = grow(c.sc->prm, (size_t)N_k * tnrd::prm_stride(ksize), c.st)) != TNRD_OK) return rc;
    TNRD_CUDA(tnrd::launch_prep(filters_t, rbf_w_t, rbf_mu, rbf_gamma, 1, N_k, ksize, c.sc->prm.p, c.st, &c.lc.n));
    return run_stage_backward(c, f, u_in, e, B, H, W, N_k, ksize, c.sc->prm.p, nullptr, lambda_t, rbf_gamma, grad_u,
                              grad_filters, grad_w, grad_lambda);
}

int tnrd_diffuse_backward(const float* f, const float* u0, const float* u_gt, const float* e_T, int B, int H, int W,
                          int T, int N_k, int ksize, const float* filters, const float* rbf_w, const float* rbf_mu,
                          float rbf_gamma, const float* lambda, float* u_T, float* grad_u0, float* grad_filters,
                          float* grad_w, float* grad_lambda, void* stream)
{
    if (!f || !u0 || !filters || !rbf_w || !rbf_mu || !lambda) return TNRD_ERR_NULL;
    if ((u_gt == nullptr) == (e_T == nullptr)) return TNRD_ERR_NULL;       // exactly one of them
    if (T < 1) return TNRD_ERR_SHAPE;
    int rc = check_shape(B, H, W, N_k, ksize);
    if (rc != TNRD_OK) return rc;
    if ((rc = check_gamma(rbf_gamma)) != TNRD_OK) return rc;
    if (grad_u0 && (grad_u0 == u0 || grad_u0 == f || grad_u0 == e_T || grad_u0 == u_gt)) return TNRD_ERR_ALIAS;
    // u_T is written before u_gt / e_T are read and before grad_u0 is formed
    if (u_T && (u_T == u0 || u_T == f || u_T == u_gt || u_T == e_T || u_T == grad_u0)) return TNRD_ERR_ALIAS;
    Call c;
    if (c.o.basis == 1) return TNRD_ERR_UNSUPPORTED;          // gradients exist for the Gaussian basis only
    if ((rc = open_call(c, stream)) != TNRD_OK) return rc;
    Scratch* sc = c.sc;
    cudaStream_t st = c.st;
    const size_t n = (size_t)B * H * W, rec = (size_t)N_k * tnrd::prm_stride(ksize);
    const int KK = ksize * ksize;
    // the forward pass of a gradient is an exact evaluator (factorised, direct, or windowed if selected), never the table
    const int phi = c.o.phi_mode == 2 ? 3 : c.o.phi_mode;
    if ((rc = pick_kernel(c, B, H, W, N_k, ksize, phi)) != TNRD_OK) return rc;
    if ((rc = grow(sc->bw_trace, (size_t)T * n, st)) != TNRD_OK) return rc;     // u_1 .. u_T
    for (Buf& eb : sc->bw_e)
        if ((rc = grow(eb, n, st)) != TNRD_OK) return rc;
    BwdSide side;
    if (grad_filters) {
        if (!sc->s_bw) {
            int pr_least = 0, pr_greatest = 0;
            TNRD_CUDA(cudaDeviceGetStreamPriorityRange(&pr_least, &pr_greatest));
            TNRD_CUDA(cudaStreamCreateWithPriority(&sc->s_bw, cudaStreamNonBlocking, pr_least));
            for (auto& ev : sc->ev_bw) TNRD_CUDA(cudaEventCreateWithFlags(&ev, cudaEventDisableTiming));
        }
        side.s2 = sc->s_bw;
        side.evA[0] = sc->ev_bw[0]; side.evA[1] = sc->ev_bw[1];
        side.evB[0] = sc->ev_bw[2]; side.evB[1] = sc->ev_bw[3];
    }
    {
        Opts keep = c.o;
        c.o.basis = 0;                                          // stage_params builds no table: phi != 2 here
        rc = stage_params(c, filters, rbf_w, rbf_mu, rbf_gamma, T, N_k, ksize, phi);
        c.o = keep;
        if (rc != TNRD_OK) return rc;
    }
    // forward, keeping every iterate (Supp. Eq. 21 needs u_{t-1} of every stage)
    const float* src = u0;
    for (int t = 1; t <= T; ++t) {
        float* dst = sc->bw_trace.p + (size_t)(t - 1) * n;
        tnrd::StageArgs a{f, src, dst, sc->prm.p + (size_t)(t - 1) * rec, lambda + (t - 1), 0.0f, B, H, W, N_k, ksize};
        if ((rc = run_stage(c, a, phi, t - 1)) != TNRD_OK) return rc;
        src = dst;
    }
    if (u_T) TNRD_CUDA(cudaMemcpyAsync(u_T, src, n * sizeof(float), cudaMemcpyDeviceToDevice, st));
    // e_T = dl/du_T: given, or u_T - u_gt for the loss 1/2 ||u_T - u_gt||^2 (Supp. Eq. 3, 20)
    const float* e = e_T;
    if (u_gt) {
        TNRD_CUDA(tnrd::launch_sub(src, u_gt, sc->bw_e[0].p, n, st, &c.lc.n));
        e = sc->bw_e[0].p;
    }
    // backward recurrence (Supp. Eq. 21): e_{t-1} = (du_t/du_{t-1})^T e_t; parameter gradients of stage t from (u_{t-1}, e_t)
    for (int t = T; t >= 1; --t) {
        const float* u_prev = (t == 1) ? u0 : sc->bw_trace.p + (size_t)(t - 2) * n;
        float* g_u;
        if (t == 1) g_u = grad_u0;                                   // may be null: not needed then
        else g_u = sc->bw_e[(T - t + 1) % 3].p;      // three planes in turn: stage t's dl/du is still read by its lag products
                                                    // (side stream) while stage t - 1 writes the next one
        rc = run_stage_backward(c, f, u_prev, e, B, H, W, N_k, ksize, sc->prm.p + (size_t)(t - 1) * rec,
                                lambda + (t - 1), 0.0f, rbf_gamma, g_u,
                                grad_filters ? grad_filters + (size_t)(t - 1) * N_k * KK : nullptr,
                                grad_w ? grad_w + (size_t)(t - 1) * N_k * TNRD_NUM_RBF : nullptr,
                                grad_lambda ? grad_lambda + (t - 1) : nullptr, grad_filters ? &side : nullptr);
        if (rc != TNRD_OK) return rc;
        e = g_u;
    }
    for (int q = 0; q < 2; ++q)         // the caller's stream continues after the last lag products
        if (side.used[q]) TNRD_CUDA(cudaStreamWaitEvent(st, side.evB[q], 0));
    return TNRD_OK;
}

int tnrd_plan_query(int B, int H, int W, int N_k, int ksize, int num_sms, long long* plan)
{
    if (!plan) return TNRD_ERR_NULL;
    int rc = check_shape(B, H, W, N_k, ksize);
    if (rc != TNRD_OK) return rc;
    if (num_sms < 1) return TNRD_ERR_SHAPE;
    tnrd::StageArgs a{nullptr, nullptr, nullptr, nullptr, nullptr, 0.0f, B, H, W, N_k, ksize};
    const tnrd::FusedPlan pl = tnrd::plan_stage_fused(a, num_sms);
    const long long tiles = (long long)pl.ntx * pl.nty * B;
    plan[0] = pl.cfg; plan[1] = pl.ntx; plan[2] = pl.nty; plan[3] = pl.tw; plan[4] = pl.th; plan[5] = pl.n_full;
    plan[6] = pl.nsplit; plan[7] = pl.n_full + (tiles - pl.n_full) * pl.nsplit; plan[8] = pl.cta_floats;
    plan[9] = (long long)pl.part_floats;
    return TNRD_OK;
}

int tnrd_tc_plan_query(int B, int H, int W, int N_k, int ksize, int num_sms, long long* plan)
{
    if (!plan) return TNRD_ERR_NULL;
    int rc = check_shape(B, H, W, N_k, ksize);
    if (rc != TNRD_OK) return rc;
    if (num_sms < 1) return TNRD_ERR_SHAPE;
    for (int i = 0; i < 7; ++i) plan[i] = 0;
    if (!tnrd::tc_supported(N_k, ksize)) return TNRD_OK;
    const tnrd::TcPlan pl = tnrd::plan_stage_tc(B, H, W, N_k, ksize, num_sms);
    plan[0] = 1 + (tc_auto(pl, W, num_sms, ksize) ? 1 : 0);
    plan[1] = pl.nxs; plan[2] = pl.nys; plan[3] = pl.seg_rows; plan[4] = pl.units; plan[5] = 256 - (ksize - 1); plan[6] = pl.nchunk;
    return TNRD_OK;
}

int tnrd_phi_stats(int enable, unsigned long long* executed, unsigned long long* defined, void* stream)
{
    g_stats = enable ? 1 : 0;
    if (executed) *executed = 0;
    if (defined) *defined = 0;
    Scratch* sc = nullptr;
    int rc = get_scratch((cudaStream_t)stream, &sc);
    if (rc != TNRD_OK) return rc;
    if (!sc->stats.p) return TNRD_OK;
    unsigned long long h[2] = {0, 0};
    TNRD_CUDA(cudaMemcpyAsync(h, sc->stats.p, 16, cudaMemcpyDeviceToHost, (cudaStream_t)stream));
    TNRD_CUDA(cudaMemsetAsync(sc->stats.p, 0, 16, (cudaStream_t)stream));
    TNRD_CUDA(cudaStreamSynchronize((cudaStream_t)stream));
    if (executed) *executed = h[0];
    if (defined) *defined = h[1];
    return TNRD_OK;
}

int tnrd_set_kernel(int which)
{
    if (which < 0 || which > 4) return TNRD_ERR_UNSUPPORTED;
    g_kernel = which;
    return TNRD_OK;
}

int tnrd_set_phi_mode(int mode)
{
    if (mode < 0 || mode > 3) return TNRD_ERR_UNSUPPORTED;
    g_phi_mode = mode;
    return TNRD_OK;
}

int tnrd_set_rbf_basis(int basis)
{
    if (basis < 0 || basis > 1) return TNRD_ERR_UNSUPPORTED;
    g_basis = basis;
    return TNRD_OK;
}

unsigned long long tnrd_launch_count(void) { return g_launches; }
void tnrd_reset_launch_count(void) { g_launches = 0; }

int tnrd_microbench(int which, double* rate, void* stream)
{
    if (!rate) return TNRD_ERR_NULL;
    if (which < 0 || which > 3) return TNRD_ERR_UNSUPPORTED;
    LaunchCount lc;
    TNRD_CUDA(tnrd::run_microbench(which, rate, (cudaStream_t)stream, &lc.n));
    return TNRD_OK;
}

const char* tnrd_strerror(int status)
{
    switch (status) {
        case TNRD_OK: return "ok";
        case TNRD_ERR_NULL: return "a required pointer is NULL";
        case TNRD_ERR_SHAPE: return "shape out of range (B,H,W>=1, B*H*W<2^31, 1<=N_k<=128, min(H,W)>=ksize-1, T>=0)";
        case TNRD_ERR_UNSUPPORTED: return "unsupported ksize (3,5,7,9) or option";
        case TNRD_ERR_ALIAS: return "output aliases an input it must not alias";
        case TNRD_ERR_CUDA: return "a CUDA call failed (see tnrd_last_cuda_error)";
        case TNRD_ERR_PARAM: return "rbf_gamma must be finite and > 0";
        case TNRD_ERR_TOO_LARGE: return "the call needs more than the fixed scratch of tnrd_stage_static (TNRD_STATIC_SCRATCH_BYTES)";
        default: return "unknown status";
    }
}

const char* tnrd_last_cuda_error(void) { return g_cuda_err; }
int tnrd_version(void) { return TNRD_VERSION; }

void tnrd_shutdown(void)
{
    std::lock_guard<std::mutex> lk(g_mu);
    int cur = 0;
    (void)cudaGetDevice(&cur);
    for (Scratch* s : g_scratch) {
        (void)cudaSetDevice(s->dev);
        Buf* bufs[] = {&s->pp, &s->arrive, &s->tcws, &s->stats, &s->prm, &s->bw_maps, &s->bw_part, &s->bw_trace, &s->bw_e[0], &s->bw_e[1], &s->bw_e[2], &s->refv, &s->split, &s->tab, &s->h_f, &s->h_u, &s->h_out, &s->h_par};
        for (Buf* b : bufs)
            if (b->p) (void)cudaFree(b->p);   // synchronising free: the stream may be gone by now
        if (s->s_in) { (void)cudaStreamDestroy(s->s_in); (void)cudaStreamDestroy(s->s_out); }
        for (cudaStream_t b : s->s_band) if (b) (void)cudaStreamDestroy(b);
        if (s->s_bw) (void)cudaStreamDestroy(s->s_bw);
        for (cudaEvent_t e : s->ev_bw) if (e) (void)cudaEventDestroy(e);
        for (cudaEvent_t e : s->ev) if (e) (void)cudaEventDestroy(e);
        if (s->h_par_pinned) (void)cudaFreeHost(s->h_par_pinned);
        if (s->h_word) (void)cudaFreeHost(s->h_word);
        if (s->h_flags) (void)cudaFreeHost(s->h_flags);
        delete s;
    }
    g_scratch.clear();
    (void)cudaSetDevice(cur);
}

}  // extern "C"

// tnrd_api.cu -- host side of libtnrd: the C ABI declared in include/tnrd.h.
// Validation, per-(device, stream) scratch, parameter staging and the stage loop (row a6: PAPER.md:74, :184).
// Every step of the path runs in this library's kernels; there is no CPU fallback.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <vector>

#include "../../include/tnrd.h"
#include "tnrd_internal.h"

namespace {

thread_local char g_cuda_err[512] = "";
unsigned long long g_launches = 0;
int g_kernel = 0;  // 0 auto, 1 reference, 2 fused
int g_phi_mode = 3;  // 0 direct 63-term phi, 1 windowed evaluator (dense fallback decided on the device), 2 table,
                     // 3 factorised 63-term phi (direct fallback inside the kernel)
int g_basis = 0;     // 0 Gaussian radial basis, 1 triangular-shaped (table evaluator)
std::mutex g_mu;

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

struct Scratch {
    int dev = -1;
    cudaStream_t st = nullptr;
    int num_sms = 0;
    Buf prm, refv;                    // staged parameters, reference-path phi maps
    Buf split;                        // partial transposed-filter sums of the fused kernel's CTAs
    Buf tab;                          // piecewise-linear phi tables [T][N_k][4096] float2 + 4 header floats
    Buf h_f, h_u, h_out, h_par;       // device staging of the host entry point
    Buf bw_maps, bw_part, bw_trace, bw_e[2];   // backward pass: P/V maps, per-CTA partial sums, iterates, dl/du planes
};
std::vector<Scratch*> g_scratch;

int grow(Buf& b, size_t floats, cudaStream_t st)
{
    if (floats <= b.cap) return TNRD_OK;
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

// evaluator of the fused kernel for the current settings: the triangular basis always goes through the table
int effective_phi() { return (g_basis == 1 || g_phi_mode == 2) ? 2 : g_phi_mode; }

// Stages the parameters of T stages; with the table evaluator also builds the phi tables.
int stage_params(Scratch* sc, const float* filters, const float* rbf_w, const float* rbf_mu, float gamma, int T, int N_k,
                 int ksize, int phi, cudaStream_t st)
{
    int rc = grow(sc->prm, (size_t)T * N_k * tnrd::prm_stride(ksize), st);
    if (rc != TNRD_OK) return rc;
    TNRD_CUDA(tnrd::launch_prep(filters, rbf_w, rbf_mu, gamma, T, N_k, ksize, sc->prm.p, st, &g_launches));
    if (phi == 2) {
        const size_t n = (size_t)T * N_k * TNRD_TAB_NODES * 2;
        if ((rc = grow(sc->tab, n + 4, st)) != TNRD_OK) return rc;
        TNRD_CUDA(tnrd::launch_build_table(rbf_w, rbf_mu, gamma, T * N_k, g_basis, sc->tab.p + 4, sc->tab.p, st,
                                           &g_launches));
    }
    return TNRD_OK;
}

// phi: evaluator (0, 1, 2); t = stage index inside the staged parameters (selects the table)
int run_stage(Scratch* sc, tnrd::StageArgs a, int phi, int t, cudaStream_t st)
{
    const bool use_ref = (g_kernel == 1);
    if (phi == 2) {
        a.tabhdr = sc->tab.p;
        a.tab = sc->tab.p + 4 + (size_t)t * a.N_k * TNRD_TAB_NODES * 2;
    }
    if (use_ref) {
        if (g_basis == 1) return TNRD_ERR_UNSUPPORTED;     // the reference kernel knows the Gaussian basis only
        int rc = grow(sc->refv, tnrd::ref_scratch_floats(a.B, a.H, a.W, a.N_k, a.ksize), st);
        if (rc != TNRD_OK) return rc;
        TNRD_CUDA(tnrd::launch_stage_ref(a, sc->refv.p, st, &g_launches));
    } else {
        const tnrd::FusedPlan pl = tnrd::plan_stage_fused(a, sc->num_sms);
        int rc = grow(sc->split, pl.part_floats, st);
        if (rc != TNRD_OK) return rc;
        TNRD_CUDA(tnrd::launch_stage_fused(a, pl, sc->split.p, phi, st, &g_launches));
    }
    return TNRD_OK;
}

}  // namespace

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
    cudaStream_t st = (cudaStream_t)stream;
    Scratch* sc = nullptr;
    if ((rc = get_scratch(st, &sc)) != TNRD_OK) return rc;
    const int phi = effective_phi();
    if ((rc = stage_params(sc, filters_t, rbf_w_t, rbf_mu, rbf_gamma, 1, N_k, ksize, phi, st)) != TNRD_OK) return rc;
    tnrd::StageArgs a{f, u_in, u_out, sc->prm.p, nullptr, lambda_t, B, H, W, N_k, ksize};
    return run_stage(sc, a, phi, 0, st);
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
    Scratch* sc = nullptr;
    if ((rc = get_scratch(st, &sc)) != TNRD_OK) return rc;
    const size_t rec = (size_t)N_k * tnrd::prm_stride(ksize);
    const int phi = effective_phi();
    if ((rc = stage_params(sc, filters, rbf_w, rbf_mu, rbf_gamma, T, N_k, ksize, phi, st)) != TNRD_OK) return rc;
    // Every stage writes `out`, from the second one on in place: the tile kernel only READS u_{t-1} (all halo reads
    // happen there) and stores partial sums in scratch; the update kernel that follows it on the stream is point-wise.
    const float* src = u0;
    for (int t = 1; t <= T; ++t) {
        tnrd::StageArgs a{f, src, out, sc->prm.p + (size_t)(t - 1) * rec, lambda + (t - 1), 0.0f, B, H, W, N_k, ksize};
        if ((rc = run_stage(sc, a, phi, t - 1, st)) != TNRD_OK) return rc;
        src = out;
    }
    return TNRD_OK;
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
    cudaStream_t st = (cudaStream_t)stream;
    Scratch* sc = nullptr;
    if ((rc = get_scratch(st, &sc)) != TNRD_OK) return rc;
    const size_t n = (size_t)B * H * W;
    const size_t nk = (size_t)T * N_k * ksize * ksize, nw = (size_t)T * N_k * TNRD_NUM_RBF;
    const size_t npar = nk + nw + TNRD_NUM_RBF + (size_t)T;
    if ((rc = grow(sc->h_f, n, st)) != TNRD_OK) return rc;
    if (u0 != f && (rc = grow(sc->h_u, n, st)) != TNRD_OK) return rc;
    if ((rc = grow(sc->h_out, n, st)) != TNRD_OK) return rc;
    if ((rc = grow(sc->h_par, npar > 0 ? npar : 1, st)) != TNRD_OK) return rc;
    float* d_k = sc->h_par.p;
    float* d_w = d_k + nk;
    float* d_mu = d_w + nw;
    float* d_lam = d_mu + TNRD_NUM_RBF;
    TNRD_CUDA(cudaMemcpyAsync(sc->h_f.p, f, n * sizeof(float), cudaMemcpyHostToDevice, st));
    const float* d_u0 = sc->h_f.p;
    if (u0 != f) {
        TNRD_CUDA(cudaMemcpyAsync(sc->h_u.p, u0, n * sizeof(float), cudaMemcpyHostToDevice, st));
        d_u0 = sc->h_u.p;
    }
    if (T > 0) {
        TNRD_CUDA(cudaMemcpyAsync(d_k, filters, nk * sizeof(float), cudaMemcpyHostToDevice, st));
        TNRD_CUDA(cudaMemcpyAsync(d_w, rbf_w, nw * sizeof(float), cudaMemcpyHostToDevice, st));
        TNRD_CUDA(cudaMemcpyAsync(d_mu, rbf_mu, TNRD_NUM_RBF * sizeof(float), cudaMemcpyHostToDevice, st));
        TNRD_CUDA(cudaMemcpyAsync(d_lam, lambda, (size_t)T * sizeof(float), cudaMemcpyHostToDevice, st));
    }
    rc = tnrd_diffuse(sc->h_f.p, d_u0, B, H, W, T, N_k, ksize, d_k, d_w, d_mu, rbf_gamma, d_lam, sc->h_out.p, stream);
    if (rc != TNRD_OK) return rc;
    TNRD_CUDA(cudaMemcpyAsync(out, sc->h_out.p, n * sizeof(float), cudaMemcpyDeviceToHost, st));
    TNRD_CUDA(cudaStreamSynchronize(st));
    return TNRD_OK;
}

int tnrd_qcs_project(const float* y, int B, int H, int W, const float* qcs_lo, const float* qcs_hi, float* u_out,
                     void* stream)
{
    if (!y || !qcs_lo || !qcs_hi || !u_out) return TNRD_ERR_NULL;
    if (B < 1 || H < 8 || W < 8 || (H % 8) || (W % 8) || (long long)B * H * W >= (1LL << 31)) return TNRD_ERR_SHAPE;
    if (u_out == qcs_lo || u_out == qcs_hi) return TNRD_ERR_ALIAS;
    TNRD_CUDA(tnrd::launch_qcs_project(y, qcs_lo, qcs_hi, u_out, B, H, W, (cudaStream_t)stream, &g_launches));
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
    Scratch* sc = nullptr;
    if ((rc = get_scratch(st, &sc)) != TNRD_OK) return rc;
    const size_t rec = (size_t)N_k * tnrd::prm_stride(ksize);
    const int phi = effective_phi();
    if ((rc = stage_params(sc, filters, rbf_w, rbf_mu, rbf_gamma, T, N_k, ksize, phi, st)) != TNRD_OK) return rc;
    // Per stage (Supp. Eq. 29): the stage kernels with lambda = 0 write y = u - sum_i kbar_i * phi_i(k_i * u) to `out`
    // (f is then irrelevant: u itself is passed; in place from the second stage on, as in tnrd_diffuse), the projection
    // kernel turns it into u_t = D^T eta(D y) in place.
    const float* src = u0;
    for (int t = 1; t <= T; ++t) {
        tnrd::StageArgs a{src, src, out, sc->prm.p + (size_t)(t - 1) * rec, nullptr, 0.0f, B, H, W, N_k, ksize};
        if ((rc = run_stage(sc, a, phi, t - 1, st)) != TNRD_OK) return rc;
        TNRD_CUDA(tnrd::launch_qcs_project(out, qcs_lo, qcs_hi, out, B, H, W, st, &g_launches));
        src = out;
    }
    return TNRD_OK;
}

// Backward pass of one stage on staged parameters (shared by tnrd_stage_backward and tnrd_diffuse_backward).
static int run_stage_backward(Scratch* sc, const float* f, const float* u, const float* e, int B, int H, int W, int N_k,
                              int ksize, const float* prm, const float* lambda_ptr, float lambda_val, float gamma,
                              float* g_u, float* g_k, float* g_w, float* g_l, cudaStream_t st)
{
    const tnrd::BwdPlan pl = tnrd::plan_stage_bwd(B, H, W, N_k, ksize, sc->num_sms);
    const int R = (ksize - 1) / 2, KK = ksize * ksize;
    const bool want_k = g_k != nullptr, want_w = g_w != nullptr || want_k;
    const size_t n_w = want_w ? (size_t)pl.n_cta * N_k * 64 : 0, n_l = (size_t)pl.n_cta;
    const size_t n_k = want_k ? (size_t)pl.G * N_k * KK : 0;
    int rc = grow(sc->bw_part, n_w + n_l + n_k + 4, st);
    if (rc != TNRD_OK) return rc;
    const size_t map = want_k ? (size_t)B * N_k * (H + 2 * R) * (W + 2 * R) : 0;
    if (want_k && (rc = grow(sc->bw_maps, 2 * map, st)) != TNRD_OK) return rc;
    float* part_w = sc->bw_part.p;
    float* part_l = part_w + n_w;
    float* part_k = part_l + n_l;
    tnrd::BwdArgs a{f, u, e, g_u, prm, lambda_ptr, lambda_val, B, H, W, N_k, ksize,
                    want_k ? sc->bw_maps.p : nullptr, want_k ? sc->bw_maps.p + map : nullptr,
                    want_w ? part_w : nullptr, g_l ? part_l : nullptr};
    TNRD_CUDA(tnrd::launch_stage_bwd(a, pl, part_k, st, &g_launches));
    if (want_w || g_l) {
        const float s = sqrtf(1.4426950408889634f / (2.0f * gamma * gamma));
        TNRD_CUDA(tnrd::launch_reduce_partials(part_w, pl.n_cta, part_k, pl.G, part_l, N_k, ksize, s, g_w, g_k, g_l, st,
                                               &g_launches));
    }
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
    if (g_basis == 1) return TNRD_ERR_UNSUPPORTED;          // gradients exist for the Gaussian basis only
    cudaStream_t st = (cudaStream_t)stream;
    Scratch* sc = nullptr;
    if ((rc = get_scratch(st, &sc)) != TNRD_OK) return rc;
    if ((rc = grow(sc->prm, (size_t)N_k * tnrd::prm_stride(ksize), st)) != TNRD_OK) return rc;
    TNRD_CUDA(tnrd::launch_prep(filters_t, rbf_w_t, rbf_mu, rbf_gamma, 1, N_k, ksize, sc->prm.p, st, &g_launches));
    return run_stage_backward(sc, f, u_in, e, B, H, W, N_k, ksize, sc->prm.p, nullptr, lambda_t, rbf_gamma, grad_u,
                              grad_filters, grad_w, grad_lambda, st);
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
    if (u_T && (u_T == u0 || u_T == f)) return TNRD_ERR_ALIAS;
    if (g_basis == 1) return TNRD_ERR_UNSUPPORTED;          // gradients exist for the Gaussian basis only
    cudaStream_t st = (cudaStream_t)stream;
    Scratch* sc = nullptr;
    if ((rc = get_scratch(st, &sc)) != TNRD_OK) return rc;
    const size_t n = (size_t)B * H * W, rec = (size_t)N_k * tnrd::prm_stride(ksize);
    const int KK = ksize * ksize;
    if ((rc = grow(sc->prm, (size_t)T * rec, st)) != TNRD_OK) return rc;
    if ((rc = grow(sc->bw_trace, (size_t)T * n, st)) != TNRD_OK) return rc;     // u_1 .. u_T
    if ((rc = grow(sc->bw_e[0], n, st)) != TNRD_OK) return rc;
    if ((rc = grow(sc->bw_e[1], n, st)) != TNRD_OK) return rc;
    TNRD_CUDA(tnrd::launch_prep(filters, rbf_w, rbf_mu, rbf_gamma, T, N_k, ksize, sc->prm.p, st, &g_launches));
    // forward, keeping every iterate (Supp. Eq. 21 needs u_{t-1} of every stage)
    const float* src = u0;
    for (int t = 1; t <= T; ++t) {
        float* dst = sc->bw_trace.p + (size_t)(t - 1) * n;
        tnrd::StageArgs a{f, src, dst, sc->prm.p + (size_t)(t - 1) * rec, lambda + (t - 1), 0.0f, B, H, W, N_k, ksize};
        // the forward pass of a gradient is an exact evaluator (factorised, direct, or windowed if selected), never the table
        if ((rc = run_stage(sc, a, g_phi_mode == 2 ? 3 : g_phi_mode, t - 1, st)) != TNRD_OK) return rc;
        src = dst;
    }
    if (u_T) TNRD_CUDA(cudaMemcpyAsync(u_T, src, n * sizeof(float), cudaMemcpyDeviceToDevice, st));
    // e_T = dl/du_T: given, or u_T - u_gt for the loss 1/2 ||u_T - u_gt||^2 (Supp. Eq. 3, 20)
    const float* e = e_T;
    if (u_gt) {
        TNRD_CUDA(tnrd::launch_sub(src, u_gt, sc->bw_e[0].p, n, st, &g_launches));
        e = sc->bw_e[0].p;
    }
    // backward recurrence (Supp. Eq. 21): e_{t-1} = (du_t/du_{t-1})^T e_t; parameter gradients of stage t from (u_{t-1}, e_t)
    for (int t = T; t >= 1; --t) {
        const float* u_prev = (t == 1) ? u0 : sc->bw_trace.p + (size_t)(t - 2) * n;
        float* g_u;
        if (t == 1) g_u = grad_u0;                                   // may be null: not needed then
        else g_u = (e == sc->bw_e[0].p) ? sc->bw_e[1].p : sc->bw_e[0].p;
        rc = run_stage_backward(sc, f, u_prev, e, B, H, W, N_k, ksize, sc->prm.p + (size_t)(t - 1) * rec,
                                lambda + (t - 1), 0.0f, rbf_gamma, g_u,
                                grad_filters ? grad_filters + (size_t)(t - 1) * N_k * KK : nullptr,
                                grad_w ? grad_w + (size_t)(t - 1) * N_k * TNRD_NUM_RBF : nullptr,
                                grad_lambda ? grad_lambda + (t - 1) : nullptr, st);
        if (rc != TNRD_OK) return rc;
        e = g_u;
    }
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

int tnrd_set_kernel(int which)
{
    if (which < 0 || which > 2) return TNRD_ERR_UNSUPPORTED;
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
    if (which < 0 || which > 7) return TNRD_ERR_UNSUPPORTED;
    TNRD_CUDA(tnrd::run_microbench(which, rate, (cudaStream_t)stream, &g_launches));
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
        Buf* bufs[] = {&s->prm, &s->bw_maps, &s->bw_part, &s->bw_trace, &s->bw_e[0], &s->bw_e[1], &s->refv, &s->split, &s->tab, &s->h_f, &s->h_u, &s->h_out, &s->h_par};
        for (Buf* b : bufs)
            if (b->p) (void)cudaFree(b->p);   // synchronising free: the stream may be gone by now
        delete s;
    }
    g_scratch.clear();
    (void)cudaSetDevice(cur);
}

}  // extern "C"

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
int g_phi_mode = 0;  // 0 dense 63-term phi, 1 windowed evaluator (dense fallback decided on the device)
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
    Buf prm, plane[2], refv;          // staged parameters, ping-pong planes, reference-path phi maps
    Buf split;                        // small-image path: tile counters (kept zero between launches) + partial sums
    Buf h_f, h_u, h_out, h_par;       // device staging of the host entry point
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

int run_stage(Scratch* sc, const tnrd::StageArgs& a, cudaStream_t st)
{
    const bool use_ref = (g_kernel == 1);
    if (use_ref) {
        int rc = grow(sc->refv, tnrd::ref_scratch_floats(a.B, a.H, a.W, a.N_k, a.ksize), st);
        if (rc != TNRD_OK) return rc;
        TNRD_CUDA(tnrd::launch_stage_ref(a, sc->refv.p, st, &g_launches));
    } else {
        const tnrd::FusedPlan pl = tnrd::plan_stage_fused(a, sc->num_sms);
        if (pl.split_floats > sc->split.cap) {
            int rc = grow(sc->split, pl.split_floats, st);
            if (rc != TNRD_OK) return rc;
            TNRD_CUDA(cudaMemsetAsync(sc->split.p, 0, sc->split.cap * sizeof(float), st));
        }
        TNRD_CUDA(tnrd::launch_stage_fused(a, pl, sc->split.p, g_phi_mode, st, &g_launches));
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
    if (u_out == u_in || u_out == f) return TNRD_ERR_ALIAS;
    cudaStream_t st = (cudaStream_t)stream;
    Scratch* sc = nullptr;
    if ((rc = get_scratch(st, &sc)) != TNRD_OK) return rc;
    if ((rc = grow(sc->prm, (size_t)N_k * tnrd::prm_stride(ksize), st)) != TNRD_OK) return rc;
    TNRD_CUDA(tnrd::launch_prep(filters_t, rbf_w_t, rbf_mu, rbf_gamma, 1, N_k, ksize, sc->prm.p, st, &g_launches));
    tnrd::StageArgs a{f, u_in, u_out, sc->prm.p, nullptr, lambda_t, B, H, W, N_k, ksize};
    return run_stage(sc, a, st);
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
    if ((rc = grow(sc->prm, (size_t)T * rec, st)) != TNRD_OK) return rc;
    // Destinations d_1..d_T: alternate scratch / out so that d_T = out and no stage writes what it reads.
    // In place (out == u0) with odd T the first stage may not write out: it goes to a second plane.
    const bool inplace_odd = (out == u0) && (T & 1);
    if (T > 1 && (rc = grow(sc->plane[0], n, st)) != TNRD_OK) return rc;
    if (inplace_odd && (rc = grow(sc->plane[1], n, st)) != TNRD_OK) return rc;
    TNRD_CUDA(tnrd::launch_prep(filters, rbf_w, rbf_mu, rbf_gamma, T, N_k, ksize, sc->prm.p, st, &g_launches));
    const float* src = u0;
    for (int t = 1; t <= T; ++t) {
        float* dst;
        if (t == 1 && inplace_odd) dst = sc->plane[1].p;
        else dst = ((T - t) & 1) ? sc->plane[0].p : out;
        tnrd::StageArgs a{f, src, dst, sc->prm.p + (size_t)(t - 1) * rec, lambda + (t - 1), 0.0f, B, H, W, N_k, ksize};
        if ((rc = run_stage(sc, a, st)) != TNRD_OK) return rc;
        src = dst;
    }
    if (src != out)  // T == 1 in place: the single stage went to the second plane
        TNRD_CUDA(cudaMemcpyAsync(out, src, n * sizeof(float), cudaMemcpyDeviceToDevice, st));
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
    if ((rc = grow(sc->prm, (size_t)T * rec, st)) != TNRD_OK) return rc;
    const bool inplace_odd = (out == u0) && (T & 1);
    if (T > 1 && (rc = grow(sc->plane[0], n, st)) != TNRD_OK) return rc;
    if (inplace_odd && (rc = grow(sc->plane[1], n, st)) != TNRD_OK) return rc;
    TNRD_CUDA(tnrd::launch_prep(filters, rbf_w, rbf_mu, rbf_gamma, T, N_k, ksize, sc->prm.p, st, &g_launches));
    // Same ping-pong as tnrd_diffuse.  Per stage (Supp. Eq. 29): the fused kernel with lambda = 0 writes
    // y = u - sum_i kbar_i * phi_i(k_i * u) to the destination plane (f is then irrelevant: u itself is passed),
    // the projection kernel turns it into u_t = D^T eta(D y) in place.
    const float* src = u0;
    for (int t = 1; t <= T; ++t) {
        float* dst;
        if (t == 1 && inplace_odd) dst = sc->plane[1].p;
        else dst = ((T - t) & 1) ? sc->plane[0].p : out;
        tnrd::StageArgs a{src, src, dst, sc->prm.p + (size_t)(t - 1) * rec, nullptr, 0.0f, B, H, W, N_k, ksize};
        if ((rc = run_stage(sc, a, st)) != TNRD_OK) return rc;
        TNRD_CUDA(tnrd::launch_qcs_project(dst, qcs_lo, qcs_hi, dst, B, H, W, st, &g_launches));
        src = dst;
    }
    if (src != out) TNRD_CUDA(cudaMemcpyAsync(out, src, n * sizeof(float), cudaMemcpyDeviceToDevice, st));
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
    if (mode < 0 || mode > 1) return TNRD_ERR_UNSUPPORTED;
    g_phi_mode = mode;
    return TNRD_OK;
}

unsigned long long tnrd_launch_count(void) { return g_launches; }
void tnrd_reset_launch_count(void) { g_launches = 0; }

int tnrd_microbench(int which, double* rate, void* stream)
{
    if (!rate) return TNRD_ERR_NULL;
    if (which < 0 || which > 2) return TNRD_ERR_UNSUPPORTED;
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
        Buf* bufs[] = {&s->prm, &s->plane[0], &s->plane[1], &s->refv, &s->split, &s->h_f, &s->h_u, &s->h_out, &s->h_par};
        for (Buf* b : bufs)
            if (b->p) (void)cudaFree(b->p);   // synchronising free: the stream may be gone by now
        delete s;
    }
    g_scratch.clear();
    (void)cudaSetDevice(cur);
}

}  // extern "C"

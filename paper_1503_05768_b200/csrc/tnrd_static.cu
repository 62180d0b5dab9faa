// tnrd_static.cu -- tnrd_stage_static: one stage (rows a1-a5, Main Eq. 7) for callers that must not
// allocate: code under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc.  It is the tile kernel of
// tnrd_stage (tnrd_fused.cu, factorised phi) with BOTH of its scratch areas -- the staged parameter records and the
// per-CTA partial sums of the transposed bank -- in one file-scope device array of fixed size instead of the growing
// library scratch.  The entry point calls no cudaMalloc / cudaFree / cudaHostAlloc and no allocating library routine.
//
// The array costs TNRD_STATIC_SCRATCH_BYTES of device memory on every GPU that loads the library, until exit.  Every
// call shares it and it keeps the last call's contents: nothing in it has to start at zero (the prep kernel writes every
// record the stage reads, every CTA stores all of its partial sums before the update kernel reads them), but two calls
// that overlap on the GPU (different streams, or two host threads) race on it.
#include <cmath>
#include <mutex>

#include "../../include/tnrd.h"
#include "tnrd_internal.h"

namespace {

constexpr size_t PRM_BYTES = 1u << 20;                                  // staged records of one stage
constexpr size_t PART_BYTES = TNRD_STATIC_SCRATCH_BYTES - PRM_BYTES;     // partial sums
static_assert(TNRD_STATIC_SCRATCH_BYTES % 256 == 0 && PRM_BYTES % 256 == 0, "256-byte aligned areas");

static __device__ __align__(256) unsigned char g_static_scratch[TNRD_STATIC_SCRATCH_BYTES];

// In host code `g_static_scratch` is a stand-in for the symbol, not a device address: the address a kernel may be given
// comes from cudaGetSymbolAddress, once per device, with that device current.
constexpr int MAX_DEV = 64;
std::mutex g_mu;
unsigned char* g_dev_ptr[MAX_DEV] = {};
int g_dev_sms[MAX_DEV] = {};

int static_scratch(unsigned char** ptr, int* num_sms)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return tnrd::api_cuda_fail(e, "cudaGetDevice");
    if (dev < 0 || dev >= MAX_DEV) return TNRD_ERR_UNSUPPORTED;
    std::lock_guard<std::mutex> lk(g_mu);
    if (!g_dev_ptr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_static_scratch);
        if (e != cudaSuccess || !p) return tnrd::api_cuda_fail(e, "cudaGetSymbolAddress(g_static_scratch)");
        int sms = 0;
        e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) return tnrd::api_cuda_fail(e, "cudaDeviceGetAttribute");
        g_dev_sms[dev] = sms;
        g_dev_ptr[dev] = static_cast<unsigned char*>(p);
    }
    *ptr = g_dev_ptr[dev];
    *num_sms = g_dev_sms[dev];
    return TNRD_OK;
}

}  // namespace

extern "C" int tnrd_stage_static(const float* f, const float* u_in, int B, int H, int W, int N_k, int ksize,
                                 const float* filters_t, const float* rbf_w_t, const float* rbf_mu, float rbf_gamma,
                                 float lambda_t, float* u_out, void* stream)
{
    if (!f || !u_in || !filters_t || !rbf_w_t || !rbf_mu || !u_out) return TNRD_ERR_NULL;
    if (B < 1 || H < 1 || W < 1 || (long long)B * H * W >= (1LL << 31)) return TNRD_ERR_SHAPE;
    if (ksize != 3 && ksize != 5 && ksize != 7 && ksize != 9) return TNRD_ERR_UNSUPPORTED;
    if (N_k < 1 || N_k > TNRD_MAX_FILTERS || H < ksize - 1 || W < ksize - 1) return TNRD_ERR_SHAPE;
    if (!(std::isfinite(rbf_gamma) && rbf_gamma > 0.0f)) return TNRD_ERR_PARAM;
    if (u_out == f) return TNRD_ERR_ALIAS;
    unsigned char* scratch = nullptr;
    int num_sms = 0;
    int rc = static_scratch(&scratch, &num_sms);
    if (rc != TNRD_OK) return rc;
    float* prm = reinterpret_cast<float*>(scratch);
    float* part = reinterpret_cast<float*>(scratch + PRM_BYTES);
    tnrd::StageArgs a{f, u_in, u_out, prm, nullptr, lambda_t, B, H, W, N_k, ksize};
    const tnrd::FusedPlan pl = tnrd::plan_stage_fused(a, num_sms);
    if ((size_t)N_k * tnrd::prm_stride(ksize) * sizeof(float) > PRM_BYTES || pl.part_floats * sizeof(float) > PART_BYTES)
        return TNRD_ERR_TOO_LARGE;
    cudaStream_t st = (cudaStream_t)stream;
    unsigned long long launches = 0;
    cudaError_t e = tnrd::launch_prep(filters_t, rbf_w_t, rbf_mu, rbf_gamma, 1, N_k, ksize, prm, st, &launches);
    if (e == cudaSuccess) e = tnrd::launch_stage_fused(a, pl, part, 3, st, &launches);
    tnrd::api_count_launches(launches);
    if (e != cudaSuccess) return tnrd::api_cuda_fail(e, "tnrd_stage_static");
    return TNRD_OK;
}

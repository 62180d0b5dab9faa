// tnrd_ref.cu -- parameter staging kernel and the plain two-pass reference stage (kernel variant 1).
//
// The reference stage is the unfused form of Main Eq. 7: pass 1 writes every influence map
// v_i = phi_i(k_i * u~) on the (H+2r) x (W+2r) region to global memory, pass 2 applies the rot180 bank and the
// reaction term.  One thread per pixel, global memory only.  It exists as a debugging cross-check of the fused
// kernel and as the "what fusion buys" comparison; it is not the product path (kernel 0/2 is).
#include "tnrd_internal.h"

namespace tnrd {

__device__ __forceinline__ float ex2_approx(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// ---- staging ---------------------------------------------------------------------------------------------
__global__ void prep_params_kernel(const float* __restrict__ filters, const float* __restrict__ rbf_w,
                                   const float* __restrict__ rbf_mu, float gamma, int TN, int ksize,
                                   float* __restrict__ prm)
{
    const int KK = ksize * ksize, KKP = prm_kkp(ksize), S = prm_stride(ksize), TS = prm_ts(ksize);
    const float s = sqrtf(1.4426950408889634f / (2.0f * gamma * gamma));
    const int total = TN * S;
    for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += gridDim.x * blockDim.x) {
        const int rec = idx / S, e = idx - rec * S;
        float val = 0.0f;
        if (e < KKP) {
            const int rho = e / TS, c = e - rho * TS, b = c >> 1, a = rho - 1 + (c & 1);
            if (a >= 0 && a < ksize && b < ksize) val = s * filters[(size_t)rec * KK + a * ksize + b];
        } else if (e < KKP + 2 * TNRD_MP) {
            const int j = (e - KKP) >> 1, which = (e - KKP) & 1;
            if (j < TNRD_M) val = which ? rbf_w[(size_t)rec * TNRD_M + j] / s : -s * rbf_mu[j];
        } else if (e < KKP + 3 * TNRD_MP) {
            const int j = e - KKP - 2 * TNRD_MP;
            if (j < TNRD_M) val = rbf_w[(size_t)rec * TNRD_M + j] / s;
        } else if (e < prm_fact(ksize)) {
            // header: spacing of the centres in scaled units and the "windowed / factorised evaluator is valid" flags
            const float mu0 = rbf_mu[0], delta = (rbf_mu[TNRD_M - 1] - mu0) / (float)(TNRD_M - 1);
            const float ds = s * delta;
            const int h = e - prm_hdr(ksize);
            if (h == 0) val = 1.0f / ds;
            else if (h == 1) val = s * mu0;
            else if (h == 2) val = ds;
            else if (h == 4) val = 2.0f * ds;
            else if (h == 5) val = TNRD_FCLAMP;
            else if (h == 3 || h == 6) {
                bool ok = delta > 0.0f;
#pragma unroll 9
                for (int j = 0; j < TNRD_M; ++j)       // no early exit: the 63 loads are independent and overlap
                    ok &= fabsf(__ldg(rbf_mu + j) - fmaf((float)j, delta, mu0)) <= 1.5e-7f * (fabsf(mu0) + 62.0f * delta);   // a few ulp of the largest centre
                if (h == 3) ok &= gamma <= delta * 1.000001f;
                else {
                    const float reach = TNRD_FCLAMP - (float)TNRD_FS * ds;
                    float emax = 0.0f;
                    for (int j = 1; j <= TNRD_FS; ++j)
                        emax = fmaxf(emax, (float)j * 2.0f * ds * TNRD_FCLAMP - (float)(j * j) * ds * ds);
                    ok &= reach > 0.0f && reach * reach >= 30.0f && emax <= 92.0f;
                }
                val = ok ? 1.0f : 0.0f;
            }
        } else {
            // factorised evaluator: group g, anchor a = g (2S+1) + S; (-mu'_a, c_S .. c_0, c_-S .. c_-1)
            const int q = e - prm_fact(ksize), g = q / TNRD_FSTRIDE, o = q - g * TNRD_FSTRIDE;
            const int anchor = g * TNRD_FM + TNRD_FS;
            const float mu0 = rbf_mu[0], delta = (rbf_mu[TNRD_M - 1] - mu0) / (float)(TNRD_M - 1);
            const float ds = s * delta;
            if (o == 0) val = -s * (mu0 + (float)anchor * delta);
            else if (o <= TNRD_FM) {
                const int j = o <= TNRD_FS + 1 ? TNRD_FS + 1 - o : o - 2 * TNRD_FS - 2;   // S .. 0, then -S .. -1
                const int c = anchor + j;
                if (c >= 0 && c < TNRD_M) val = rbf_w[(size_t)rec * TNRD_M + c] / s * exp2f(-(float)(j * j) * ds * ds);
            } else if (o == TNRD_FSTRIDE - 2 || o == TNRD_FSTRIDE - 1) {
                // K_g = 2^{kappa (d_g - d_mid)} = 2^{-2 delta'^2 (anchor_g - anchor_mid)} and 1 / K_g: rho of group g from the
                // rho of the middle group (tensor-core kernel, tnrd_tc.cu)
                const int mid = (TNRD_FG / 2) * TNRD_FM + TNRD_FS;
                const float ex = -2.0f * ds * ds * (float)(anchor - mid);
                val = exp2f(o == TNRD_FSTRIDE - 2 ? ex : -ex);
            }
        }
        prm[idx] = val;
    }
}

cudaError_t launch_prep(const float* filters, const float* rbf_w, const float* rbf_mu, float gamma, int T,
                        int N_k, int ksize, float* prm, cudaStream_t st, unsigned long long* launches)
{
    const int total = T * N_k * prm_stride(ksize);
    if (total == 0) return cudaSuccess;
    const int threads = 256, blocks = (total + threads - 1) / threads;
    prep_params_kernel<<<blocks < 1184 ? blocks : 1184, threads, 0, st>>>(filters, rbf_w, rbf_mu, gamma, T * N_k,
                                                                            ksize, prm);
    ++*launches;
    return cudaGetLastError();
}

// ---- reference pass 1: v_i = phi_i(k_i * u~) on the (H+2r) x (W+2r) region --------------------------------
__global__ void ref_phi_kernel(StageArgs a, float* __restrict__ vbuf)
{
    const int K = a.ksize, r = (K - 1) / 2, KKP = prm_kkp(K), S = prm_stride(K);
    const int Hv = a.H + 2 * r, Wv = a.W + 2 * r;
    const long long per_img = (long long)a.N_k * Hv * Wv;
    const long long total = per_img * a.B;
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < total;
         idx += (long long)gridDim.x * blockDim.x) {
        const int b = (int)(idx / per_img);
        long long rem = idx - b * per_img;
        const int i = (int)(rem / ((long long)Hv * Wv));
        rem -= (long long)i * Hv * Wv;
        const int py = (int)(rem / Wv), px = (int)(rem - (long long)py * Wv);
        const int y = py - r, x = px - r;  // image coordinates of this phi pixel
        const float* rec = a.prm + (size_t)i * S;
        const float* u = a.u_in + (size_t)b * a.H * a.W;
        float z = 0.0f;
        for (int ka = 0; ka < K; ++ka)
            for (int kb = 0; kb < K; ++kb)
                z = fmaf(rec[prm_tap(K, ka, kb)],
                         u[(size_t)mirror_clamp(y + r - ka, a.H) * a.W + mirror_clamp(x + r - kb, a.W)], z);
        float acc = 0.0f;
        for (int j = 0; j < TNRD_M; ++j) {
            const float d = z + rec[KKP + 2 * j];
            acc = fmaf(ex2_approx(-d * d), rec[KKP + 2 * j + 1], acc);
        }
        vbuf[idx] = acc;
    }
}

// ---- reference pass 2: u_t = u - (sum_i kbar_i * v_i + lambda (u - f)) --------------------------------------
__global__ void ref_update_kernel(StageArgs a, const float* __restrict__ vbuf)
{
    const int K = a.ksize, r = (K - 1) / 2, S = prm_stride(K);
    const int Hv = a.H + 2 * r, Wv = a.W + 2 * r;
    const float lambda = a.lambda_ptr ? *a.lambda_ptr : a.lambda_val;
    const long long total = (long long)a.B * a.H * a.W;
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < total;
         idx += (long long)gridDim.x * blockDim.x) {
        const int b = (int)(idx / ((long long)a.H * a.W));
        const long long rem = idx - (long long)b * a.H * a.W;
        const int y = (int)(rem / a.W), x = (int)(rem - (long long)y * a.W);
        float s = 0.0f;
        for (int i = 0; i < a.N_k; ++i) {
            const float* rec = a.prm + (size_t)i * S;
            const float* v = vbuf + ((size_t)b * a.N_k + i) * Hv * Wv;
            for (int ka = 0; ka < K; ++ka)
                for (int kb = 0; kb < K; ++kb)
                    s = fmaf(rec[prm_tap(K, ka, kb)], v[(size_t)(y + ka) * Wv + (x + kb)], s);
        }
        const float uu = a.u_in[idx];
        a.u_out[idx] = uu - (s + lambda * (uu - a.f[idx]));
    }
}

size_t ref_scratch_floats(int B, int H, int W, int N_k, int ksize)
{
    const int r = (ksize - 1) / 2;
    return (size_t)B * N_k * (H + 2 * r) * (size_t)(W + 2 * r);
}

cudaError_t launch_stage_ref(const StageArgs& a, float* vbuf, cudaStream_t st, unsigned long long* launches)
{
    const int threads = 256;
    const long long n1 = (long long)ref_scratch_floats(a.B, a.H, a.W, a.N_k, a.ksize);
    long long b1 = (n1 + threads - 1) / threads;
    if (b1 > 148LL * 64) b1 = 148LL * 64;
    ref_phi_kernel<<<(int)b1, threads, 0, st>>>(a, vbuf);
    ++*launches;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    const long long n2 = (long long)a.B * a.H * a.W;
    long long b2 = (n2 + threads - 1) / threads;
    if (b2 > 148LL * 64) b2 = 148LL * 64;
    ref_update_kernel<<<(int)b2, threads, 0, st>>>(a, vbuf);
    ++*launches;
    return cudaGetLastError();
}

}  // namespace tnrd

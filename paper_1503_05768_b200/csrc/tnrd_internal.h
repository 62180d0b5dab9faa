// tnrd_internal.h -- declarations shared by the translation units of libtnrd (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>

#define TNRD_M 63          // RBF terms per influence function
#define TNRD_MP 64         // padded to 64 (term 63 has weight 0)

namespace tnrd {

// ---- staged ("prepped") parameters ---------------------------------------------------------------
// For every stage t and filter i the prep kernel writes one record of prm_stride(ksize) floats:
//   [0 .. KK)            k'_i[a][b] = s * k_i[a][b],  s = sqrt(log2(e) / (2 gamma^2))
//   [KKP .. KKP + 128)   pairs (mu'_j, w'_ij) = (s * mu_j, w_ij / s), j = 0..63 (pair 63 = (0, 0))
// so that phi_i(k_i * u) = sum_j w_ij 2^{-(z' - mu'_j)^2} with z' = k'_i * u, and the transposed bank
// sum_i kbar_i * v_i = sum_i kbar'_i * (v_i / s) re-uses the same scaled taps.
// After the T*N_k records: lambda[T] is read directly from the caller's array.
__host__ __device__ constexpr int prm_kkp(int ksize) { return ((ksize * ksize + 3) / 4) * 4; }
__host__ __device__ constexpr int prm_stride(int ksize) { return prm_kkp(ksize) + 2 * TNRD_MP; }

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
};

// launchers (each returns the cudaError_t of the launch; *launches += kernels launched)
cudaError_t launch_prep(const float* filters, const float* rbf_w, const float* rbf_mu, float gamma,
                        int T, int N_k, int ksize, float* prm, cudaStream_t st, unsigned long long* launches);
cudaError_t launch_stage_ref(const StageArgs& a, float* vbuf, cudaStream_t st, unsigned long long* launches);
size_t ref_scratch_floats(int B, int H, int W, int N_k, int ksize);
cudaError_t launch_stage_fused(const StageArgs& a, int num_sms, cudaStream_t st, unsigned long long* launches);
cudaError_t fused_init();   // opt-in shared memory attributes; idempotent
cudaError_t run_microbench(int which, double* rate, cudaStream_t st, unsigned long long* launches);

}  // namespace tnrd

// porpp.cu -- one level of the PORPP preference backup (Eq. 1) on a tensorised
// belief tree:
//   Psi(b,a) = (1/eta) log pi0(a|b) + R(b,a) + gamma sum_o Z(b,a,o) V(child(b,a,o))
//   V(b)     = (1/eta) log sum_a exp(eta Psi(b,a))
// One warp per belief node, one lane per action (lanes stride over A > 32); the observation
// branches of an action node are a CSR row into the next level's V.  HBM-bound: per action node
// 12 bytes in (R, log pi0, row offset) + 8 per branch, 4 out.  fp32 throughout, max-shifted LSE.
#include "voila_kernels.h"

namespace voila {

namespace {

__global__ void __launch_bounds__(256) porpp_backup_level_kernel(const float *__restrict__ R,
                                                                 const float *__restrict__ logpi0,
                                                                 const int32_t *__restrict__ child_off,
                                                                 const int32_t *__restrict__ child_idx,
                                                                 const float *__restrict__ child_w,
                                                                 const float *__restrict__ v_next, int n_belief, int A,
                                                                 float inv_eta, float eta, float gamma, float *psi_out,
                                                                 float *v_out) {
    const int lane = threadIdx.x & 31;
    const int b = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (b >= n_belief) return;
    // pass 1: preferences of this belief node's actions, running maximum
    float m = -INFINITY;
    for (int a = lane; a < A; a += 32) {
        const int j = b * A + a;
        float fut = 0.0f;
        for (int c = child_off[j]; c < child_off[j + 1]; ++c) fut = fmaf(child_w[c], v_next[child_idx[c]], fut);
        const float psi = fmaf(logpi0[j], inv_eta, R[j]) + gamma * fut;
        psi_out[j] = psi;
        m = fmaxf(m, psi);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
    // pass 2: sum_a exp(eta (Psi - max)) (the warp re-reads its own Psi values: L1/L2 hits)
    float s = 0.0f;
    if (m > -INFINITY && m < INFINITY)
        for (int a = lane; a < A; a += 32) s += expf(eta * (psi_out[b * A + a] - m));
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (lane == 0) v_out[b] = (m > -INFINITY && m < INFINITY) ? m + logf(s) * inv_eta : m;
}

}  // namespace

cudaError_t launch_porpp_backup_level(const float *R, const float *logpi0, const int32_t *child_off,
                                      const int32_t *child_idx, const float *child_w, const float *v_next, int n_belief,
                                      int A, float eta, float gamma, float *psi_out, float *v_out, cudaStream_t st) {
    const int warps_per_cta = 8;
    const int grid = (n_belief + warps_per_cta - 1) / warps_per_cta;
    porpp_backup_level_kernel<<<grid, 32 * warps_per_cta, 0, st>>>(R, logpi0, child_off, child_idx, child_w, v_next,
                                                                    n_belief, A, 1.0f / eta, eta, gamma, psi_out, v_out);
    return cudaGetLastError();
}

}  // namespace voila

// porpp.cu -- one level of the PORPP preference backup (Eq. 1) on a tensorised
// belief tree:
//   Psi(b,a) = (1/eta) log pi0(a|b) + R(b,a) + gamma sum_o Z(b,a,o) V(child(b,a,o))
//   V(b)     = (1/eta) log sum_a exp(eta Psi(b,a))
// A group of G = pow2(>= A) lanes per belief node, one lane per action (lanes stride over A > 32);
// the observation
// branches of an action node are a CSR row into the next level's V.  HBM-bound: per action node
// 12 bytes in (R, log pi0, row offset) + 8 per branch, 4 out.  fp32 throughout, max-shifted LSE.
#include "voila_kernels.h"

namespace voila {

namespace {

// G = lanes per belief node: the power of two >= A (capped at 32; A > 32 strides over the lanes),
// so a warp serves 32 / G belief nodes and narrow action sets (|A| = 4 ... 16) keep every lane busy.
__global__ void __launch_bounds__(256) porpp_backup_level_kernel(const float *__restrict__ R,
                                                                 const float *__restrict__ logpi0,
                                                                 const int32_t *__restrict__ child_off,
                                                                 const int32_t *__restrict__ child_idx,
                                                                 const float *__restrict__ child_w,
                                                                 const float *__restrict__ v_next, int n_belief, int A,
                                                                 int G, float inv_eta, float eta, float gamma,
                                                                 float *psi_out, float *v_out) {
    const int lane = threadIdx.x & 31;
    const int per_warp = 32 / G;
    const int warp_global = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const int b = warp_global * per_warp + lane / G;
    const int a0 = lane % G;
    const bool live = b < n_belief;
    // pass 1: preferences of this belief node's actions, running maximum
    float m = -INFINITY;
    if (live)
        for (int a = a0; a < A; a += G) {
            const int j = b * A + a;
            float fut = 0.0f;
            for (int c = child_off[j]; c < child_off[j + 1]; ++c) fut = fmaf(child_w[c], v_next[child_idx[c]], fut);
            const float psi = fmaf(logpi0[j], inv_eta, R[j]) + gamma * fut;
            psi_out[j] = psi;
            m = fmaxf(m, psi);
        }
    for (int o = G >> 1; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
    // pass 2: sum_a exp(eta (Psi - max)) (each lane re-reads the Psi values it wrote)
    const bool finite = m > -INFINITY && m < INFINITY;
    float s = 0.0f;
    if (live && finite)
        for (int a = a0; a < A; a += G) s += expf(eta * (psi_out[b * A + a] - m));
    for (int o = G >> 1; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (live && a0 == 0) v_out[b] = finite ? m + logf(s) * inv_eta : m;
}

}  // namespace

cudaError_t launch_porpp_backup_level(const float *R, const float *logpi0, const int32_t *child_off,
                                      const int32_t *child_idx, const float *child_w, const float *v_next, int n_belief,
                                      int A, float eta, float gamma, float *psi_out, float *v_out, cudaStream_t st) {
    const int warps_per_cta = 8;
    int G = 1;
    while (G < A && G < 32) G *= 2;
    const int per_cta = warps_per_cta * (32 / G);
    const int grid = (n_belief + per_cta - 1) / per_cta;
    porpp_backup_level_kernel<<<grid, 32 * warps_per_cta, 0, st>>>(R, logpi0, child_off, child_idx, child_w, v_next,
                                                                    n_belief, A, G, 1.0f / eta, eta, gamma, psi_out,
                                                                    v_out);
    return cudaGetLastError();
}

}  // namespace voila

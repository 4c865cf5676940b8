// porpp.cu -- the PORPP preference backup (Eq. 1) on a tensorised belief tree
// (SURVEY 8f f2), level by level, deepest first:
//   Psi(b,a) = (1/eta) log pi0(a|b) + R(b,a) + gamma sum_o Z(b,a,o) V(child(b,a,o))
//   V(b)     = (1/eta) log sum_a exp(eta Psi(b,a))
// and the root action argmax_a Psi(b0, a).
// A group of G = pow2(>= A) lanes per belief node, one lane per action (lanes stride over A > 32); the
// observation branches of an action node are a CSR row into the next level's V, walked four
// branches at a time (index / weight loads, then the four V gathers, then the FMAs in branch
// order), the preferences stay in registers between the maximum and the sum.  HBM-bound: per
// action node 12 bytes in (R, log pi0, row offset) + 12 per branch (index, weight, V(child)), 4 out.
// fp32, max-shifted LSE.
#include "voila_kernels.h"

namespace voila {

namespace {

constexpr int kPsiRegs = 4;  // preferences kept in registers per lane (A <= 4 G); beyond that re-read

// G = lanes per belief node: the power of two >= A (capped at 32; A > 32 strides over the lanes),
// so a warp serves 32 / G belief nodes and narrow action sets (|A| = 4 ... 16) keep every lane busy.
__global__ void __launch_bounds__(256, 8) porpp_backup_level_kernel(const float *__restrict__ R,
                                                                 const float *__restrict__ logpi0,
                                                                 const int32_t *__restrict__ child_off,
                                                                 const int32_t *__restrict__ child_idx,
                                                                 const float *__restrict__ child_w,
                                                                 const float *__restrict__ v_next, int n_belief, int A,
                                                                 int G, float inv_eta, float eta, float gamma,
                                                                 float *psi_out, float *v_out, int32_t *argmax_out) {
    const int lane = threadIdx.x & 31;
    const int per_warp = 32 / G;
    const int warp_global = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const int b = warp_global * per_warp + lane / G;
    const int a0 = lane % G;
    const bool live = b < n_belief;
    // pass 1: preferences of this belief node's actions, running maximum (and its first action)
    float m = -INFINITY;
    int am = 0x7fffffff;
    float psi_reg[kPsiRegs];
    auto preference = [&](int a) {
        const int j = b * A + a;
        const int c0 = __ldg(child_off + j), c1 = __ldg(child_off + j + 1);
        // issued with the row offsets, not after the CSR walk: one round trip to HBM less per action node
        const float lp = __ldg(logpi0 + j), r_j = __ldg(R + j);
        float fut = 0.0f;
        for (int c = c0; c < c1; c += 4) {
            int idx[4];
            float w[4], v[4];
#pragma unroll
            for (int u = 0; u < 4; ++u)
                if (c + u < c1) {
                    idx[u] = __ldg(child_idx + c + u);
                    w[u] = __ldg(child_w + c + u);
                }
#pragma unroll
            for (int u = 0; u < 4; ++u)
                if (c + u < c1) v[u] = __ldg(v_next + idx[u]);
#pragma unroll
            for (int u = 0; u < 4; ++u)
                if (c + u < c1) fut = fmaf(w[u], v[u], fut);
        }
        const float psi = fmaf(lp, inv_eta, r_j) + gamma * fut;
        __stcs(psi_out + j, psi);
        if (psi == psi && (am == 0x7fffffff || psi > m)) {  // first maximum (a ascends); a NaN never wins
            m = psi;
            am = a;
        }
        return psi;
    };
    if (live) {
#pragma unroll
        for (int slot = 0; slot < kPsiRegs; ++slot) {  // compile-time slots: the array stays in registers
            const int a = a0 + slot * G;
            psi_reg[slot] = a < A ? preference(a) : 0.0f;
        }
        for (int a = a0 + kPsiRegs * G; a < A; a += G) preference(a);
    }
    for (int o = G >> 1; o > 0; o >>= 1) {
        const float mo = __shfl_xor_sync(0xffffffffu, m, o);
        const int ao = __shfl_xor_sync(0xffffffffu, am, o);
        if (ao != 0x7fffffff && (am == 0x7fffffff || mo > m || (mo == m && ao < am))) {
            m = mo;
            am = ao;
        }
    }
    // pass 2: sum_a exp(eta (Psi - max))
    const bool finite = m > -INFINITY && m < INFINITY;
    float s = 0.0f;
    if (live && finite) {
#pragma unroll
        for (int slot = 0; slot < kPsiRegs; ++slot)
            if (a0 + slot * G < A) s += expf(eta * (psi_reg[slot] - m));
        for (int a = a0 + kPsiRegs * G; a < A; a += G) s += expf(eta * (psi_out[b * A + a] - m));
    }
    for (int o = G >> 1; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (live && a0 == 0) {
        v_out[b] = finite ? m + logf(s) * inv_eta : m;
        if (argmax_out) argmax_out[b] = am == 0x7fffffff ? 0 : am;
    }
}

}  // namespace

cudaError_t launch_porpp_backup_level(const float *R, const float *logpi0, const int32_t *child_off,
                                      const int32_t *child_idx, const float *child_w, const float *v_next, int n_belief,
                                      int A, float eta, float gamma, float *psi_out, float *v_out, cudaStream_t st,
                                      int32_t *argmax_out) {
    const int warps_per_cta = 8;
    int G = 1;
    while (G < A && G < 32) G *= 2;
    const int per_cta = warps_per_cta * (32 / G);
    const int grid = (n_belief + per_cta - 1) / per_cta;
    porpp_backup_level_kernel<<<grid, 32 * warps_per_cta, 0, st>>>(R, logpi0, child_off, child_idx, child_w, v_next,
                                                                    n_belief, A, G, 1.0f / eta, eta, gamma, psi_out,
                                                                    v_out, argmax_out);
    return cudaGetLastError();
}

}  // namespace voila

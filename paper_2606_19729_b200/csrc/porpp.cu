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

// G = lanes per belief node: the power of two >= A / 2 (capped at 32; larger A strides over the lanes): a
// lane takes two action nodes at a time, a warp serves 32 / G belief nodes, narrow action sets
// (|A| = 4 ... 16) keep every lane busy.
__global__ void __launch_bounds__(256, 6) porpp_backup_level_kernel(const float *__restrict__ R,
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
    // The same for TWO action nodes of this lane at once (a and a + G): the loads of a phase (offsets + R +
    // log pi0; indices + weights of the first four branches; V of the children) are issued for both before
    // anything is consumed: twice the bytes in flight per thread (the kernel is latency-bound: three
    // dependent round trips to HBM per action node).  Same arithmetic in the same order as preference().
    auto preference2 = [&](int a, bool has1, float &psi0_out, float &psi1_out) {
        int j[2], c0[2], c1[2];
        float lp[2], r_j[2];
#pragma unroll
        for (int s = 0; s < 2; ++s) {
            j[s] = b * A + a + s * G;
            if (s == 0 || has1) {
                c0[s] = __ldg(child_off + j[s]);
                c1[s] = __ldg(child_off + j[s] + 1);
                lp[s] = __ldg(logpi0 + j[s]);
                r_j[s] = __ldg(R + j[s]);
            } else {
                c0[s] = c1[s] = 0;
                lp[s] = r_j[s] = 0.0f;
            }
        }
        int idx[2][4];
        float w[2][4], v[2][4];
#pragma unroll
        for (int s = 0; s < 2; ++s)
#pragma unroll
            for (int u = 0; u < 4; ++u)
                if (c0[s] + u < c1[s]) {
                    idx[s][u] = __ldg(child_idx + c0[s] + u);
                    w[s][u] = __ldg(child_w + c0[s] + u);
                }
#pragma unroll
        for (int s = 0; s < 2; ++s)
#pragma unroll
            for (int u = 0; u < 4; ++u)
                if (c0[s] + u < c1[s]) v[s][u] = __ldg(v_next + idx[s][u]);
        float psi[2];
#pragma unroll
        for (int s = 0; s < 2; ++s) {
            float fut = 0.0f;
#pragma unroll
            for (int u = 0; u < 4; ++u)
                if (c0[s] + u < c1[s]) fut = fmaf(w[s][u], v[s][u], fut);
            for (int c = c0[s] + 4; c < c1[s]; c += 4) {  // rows longer than four branches
                int idx2[4];
                float w2[4], v2[4];
#pragma unroll
                for (int u = 0; u < 4; ++u)
                    if (c + u < c1[s]) {
                        idx2[u] = __ldg(child_idx + c + u);
                        w2[u] = __ldg(child_w + c + u);
                    }
#pragma unroll
                for (int u = 0; u < 4; ++u)
                    if (c + u < c1[s]) v2[u] = __ldg(v_next + idx2[u]);
#pragma unroll
                for (int u = 0; u < 4; ++u)
                    if (c + u < c1[s]) fut = fmaf(w2[u], v2[u], fut);
            }
            psi[s] = fmaf(lp[s], inv_eta, r_j[s]) + gamma * fut;
            if (s == 0 || has1) {
                __stcs(psi_out + j[s], psi[s]);
                if (psi[s] == psi[s] && (am == 0x7fffffff || psi[s] > m)) {  // first maximum (a ascends); a NaN never wins
                    m = psi[s];
                    am = a + s * G;
                }
            }
        }
        psi0_out = psi[0];
        psi1_out = has1 ? psi[1] : 0.0f;
    };
    if (live) {
        // slots 0 and 1 together, then 2 and 3 (compile-time slots: the array stays in registers)
        if (a0 < A) preference2(a0, a0 + G < A, psi_reg[0], psi_reg[1]);
        else psi_reg[0] = psi_reg[1] = 0.0f;
        if (a0 + 2 * G < A) preference2(a0 + 2 * G, a0 + 3 * G < A, psi_reg[2], psi_reg[3]);
        else psi_reg[2] = psi_reg[3] = 0.0f;
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
    while (2 * G < A && G < 32) G *= 2;  // two action nodes per lane (preference2)
    const int per_cta = warps_per_cta * (32 / G);
    const int grid = (n_belief + per_cta - 1) / per_cta;
    porpp_backup_level_kernel<<<grid, 32 * warps_per_cta, 0, st>>>(R, logpi0, child_off, child_idx, child_w, v_next,
                                                                    n_belief, A, G, 1.0f / eta, eta, gamma, psi_out,
                                                                    v_out, argmax_out);
    return cudaGetLastError();
}

}  // namespace voila

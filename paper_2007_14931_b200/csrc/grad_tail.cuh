// grad_tail.cuh — what the last CTA of a gradient kernel (grad.cu: any model; gradf.cu: the shape-specialised form) does once
// every CTA has written its partials: add them in CTA order, take the normalisation side from the held matrix where the
// lineshapes did not move, and form the NLL, the integral and dNLL/d(Re c_k, Im c_k).  Rows of g.partial:
// 0 = sum log S, 1 = sum w S, 2 + j = data-side leaf j, 2 + nleaf + j = normalisation side, 2 + 2 nleaf = sum u S (Eq. 14).
#pragma once
#include "amp_internal.cuh"

namespace amp {

// every thread of the last CTA calls it (after the fence); tot: shared memory, 3 + 2 nleaf doubles
__device__ __forceinline__ void grad_finish(const GradArgs& g, double* tot, int nleaf, int tid, int nthreads, unsigned ncta) {
    const StreamArgs& a = g.a;
    const int rows = 3 + 2 * nleaf;
    for (int r = tid; r < rows; r += nthreads) {
        const double* p = g.partial + (size_t)r * g.stride;
        double s = 0.0;
        for (unsigned c = 0; c < ncta; ++c) s += __ldcg(p + c);
        tot[r] = s;
    }
    __syncthreads();
    const double nd = (double)a.n;
    if (a.qf_G) {
        // static lineshapes: no normalisation tile was walked; the held matrix gives N_k = (M c)_k and sum w S = c^H M c
        // (Re M_kf = G'[2k][2f] + G'[2k+1][2f+1], Im M_kf = G'[2k][2f+1] - G'[2k+1][2f]); one thread per slot, fixed order
        for (int p = tid; p < g.npairs; p += nthreads) {
            const int kslot = g.pair_slot[p];
            double2 acc = make_double2(0.0, 0.0);
            if (kslot >= 0) {
                for (int f = 0; f < a.qf_nent; ++f) {
                    const double2 cf = a.qf_c[f];
                    const double* gm = a.qf_G + (size_t)(2 * kslot) * a.qf_KP + 2 * f;
                    const double mre = gm[0] + gm[a.qf_KP + 1], mim = gm[1] - gm[a.qf_KP];
                    acc.x += mre * cf.x - mim * cf.y;
                    acc.y += mre * cf.y + mim * cf.x;
                }
            }
            tot[2 + nleaf + 2 * p] = acc.x;
            tot[2 + nleaf + 2 * p + 1] = acc.y;
        }
        __syncthreads();
        if (tid == 0) {   // c^H M c = sum_k Re(conj(c_k) (M c)_k), slot order
            double q = 0.0;
            for (int p = 0; p < g.npairs; ++p) {
                const int kslot = g.pair_slot[p];
                if (kslot >= 0) q += a.qf_c[kslot].x * tot[2 + nleaf + 2 * p] + a.qf_c[kslot].y * tot[2 + nleaf + 2 * p + 1];
            }
            tot[1] = q;
        }
        __syncthreads();
    }
    const double swS = tot[1];
    // with a background (Eq. 14) the data-side weights are u_i = ps eps_i / f_i and N is replaced by T = sum_i u_i S_i
    const double Tn = a.bkg ? tot[2 + 2 * nleaf] : nd;
    for (int p = tid; p < g.npairs; p += nthreads) {
        const int kslot = g.pair_slot[p];
        if (kslot < 0) continue;
        // dNLL/dconj(c_k) = -D_k + N N_k / sum_j w_j S_j ; (d/dRe, d/dIm) = 2 (Re, Im)
        g.result[3 + 2 * kslot] = 2.0 * (-tot[2 + 2 * p] + Tn * tot[2 + nleaf + 2 * p] / swS);
        g.result[3 + 2 * kslot + 1] = 2.0 * (-tot[2 + 2 * p + 1] + Tn * tot[2 + nleaf + 2 * p + 1] / swS);
    }
    if (tid == 0) {
        const double I = swS / a.wsum;
        double v = a.bkg ? -tot[0] : -(tot[0] + a.sum_log_eff) + nd * log(I);
        if (!isfinite(v) || !(I > 0.0)) v = INFINITY;
        g.result[0] = v;
        g.result[1] = I;
        g.result[2] = (double)atomicExch(a.flag, 0);
        *a.ticket = 0u;
    }
}

}  // namespace amp

// Test double for tests/test_minimizer_host.py: the minimiser of csrc/minimize.cu linked against a stand-in "likelihood" with a
// known minimum and Hessian, so that its host logic (BFGS, line search, fixed slots, ties, scales, floating masses and widths,
// covariance) runs without a GPU.
//   f(H, M, G) = 1/2 sum_i lam_i d_i^2 + 1/4 sum_i d_i^4 + 0.3 sum_i d_i d_{i+1}
//                + 1/2 a (M - M*)^2 + 1/2 b (G - G*)^2 + c (M - M*) d_0 + e (M - M*)(G - G*),
//   d = (Re H_0, Im H_0, Re H_1, ...) - target;  lam_i spread over four decades (an ill-conditioned valley, as the couplings of
//   weak resonances make it).  One resonance carries (M, G); without a mass/width array the point sits at (M*, G*).
#include <cmath>
#include <vector>

#include "../paper_2007_14931_b200/csrc/minimize.cu"

static const int K = 12;
static const double MS = 4196.0, GS = 370.0, QA = 0.04, QB = 0.01, QC = 0.1, QE = 0.005;
static std::vector<double> cur(2 * K, 0.0), cur_mw;
static int cur_P = 0, n_set = 0, n_grad = 0, n_batch = 0;

static double lam(int i) { return std::pow(1e4, i / (2.0 * K - 1)); }
static double target(int i) { return 1.0 + 0.1 * i; }

static double value(const double* h, double M, double G, double* g /* [2K] or null */) {
    double s = 0.0;
    for (int i = 0; i < 2 * K; ++i) {
        const double d = h[i] - target(i);
        s += 0.5 * lam(i) * d * d + 0.25 * d * d * d * d;
        if (g) g[i] = lam(i) * d + d * d * d;
    }
    for (int i = 0; i + 1 < 2 * K; ++i) {
        const double d0 = h[i] - target(i), d1 = h[i + 1] - target(i + 1);
        s += 0.3 * d0 * d1;
        if (g) { g[i] += 0.3 * d1; g[i + 1] += 0.3 * d0; }
    }
    const double dM = M - MS, dG = G - GS, d0 = h[0] - target(0);
    s += 0.5 * QA * dM * dM + 0.5 * QB * dG * dG + QC * dM * d0 + QE * dM * dG;
    if (g) g[0] += QC * dM;
    return s;
}

extern "C" {
int amp_num_couplings(const amp_model*) { return K; }
int amp_num_resonances(const amp_model*) { return 1; }
amp_status amp_set_params(amp_model*, int P, const double* c, const double* mw) {
    if (P < 1) return AMP_ERR_INVALID;
    cur.assign(c, c + (size_t)P * 2 * K);
    cur_mw.clear();
    if (mw) cur_mw.assign(mw, mw + (size_t)P * 2);
    cur_P = P;
    ++n_set;
    for (int p = 0; p < P && mw; ++p)
        if (!(mw[2 * p + 1] > 0.0)) return AMP_ERR_DOMAIN;       // a width must be positive
    return AMP_OK;
}
amp_status amp_nll_grad(amp_model*, double* f, double* g, void*) {
    if (cur_P != 1) return AMP_ERR_STATE;
    ++n_grad;
    if (cur[0] > 50.0) return AMP_ERR_DOMAIN;                    // a region without a likelihood: the line search has to back off
    *f = value(cur.data(), cur_mw.empty() ? MS : cur_mw[0], cur_mw.empty() ? GS : cur_mw[1], g);
    return AMP_OK;
}
amp_status amp_nll(amp_model*, double* f, void*) {
    ++n_batch;
    for (int p = 0; p < cur_P; ++p)
        f[p] = value(&cur[(size_t)p * 2 * K], cur_mw.empty() ? MS : cur_mw[2 * p], cur_mw.empty() ? GS : cur_mw[2 * p + 1], nullptr);
    return AMP_OK;
}
int stub_counts(int which) { return which == 0 ? n_set : (which == 1 ? n_grad : n_batch); }
void stub_current(double* out) { for (int i = 0; i < 2 * K; ++i) out[i] = cur[i]; }
}

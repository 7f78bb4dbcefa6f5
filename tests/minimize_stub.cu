// Test double for tests/test_minimizer_host.py: the minimiser of csrc/minimize.cu linked against a stand-in "likelihood" with a
// known minimum and Hessian, so that its host logic (BFGS, line search, fixed slots, ties, scales, covariance) runs without a GPU.
//   f(H) = 1/2 sum_i lam_i d_i^2 + 1/4 sum_i d_i^4 + 0.3 sum_i d_i d_{i+1},  d = (Re H_0, Im H_0, Re H_1, ...) - target
// lam_i spread over four decades (an ill-conditioned valley, as the couplings of weak resonances make it).
#include <cmath>
#include <vector>

#include "../paper_2007_14931_b200/csrc/minimize.cu"

static const int K = 12;
static std::vector<double> cur(2 * K, 0.0);
static int n_set = 0, n_grad = 0;

static double lam(int i) { return std::pow(1e4, i / (2.0 * K - 1)); }
static double target(int i) { return 1.0 + 0.1 * i; }

extern "C" {
int amp_num_couplings(const amp_model*) { return K; }
int amp_num_resonances(const amp_model*) { return 1; }
amp_status amp_set_params(amp_model*, int P, const double* c, const double*) {
    if (P != 1) return AMP_ERR_INVALID;
    cur.assign(c, c + 2 * K);
    ++n_set;
    return AMP_OK;
}
amp_status amp_nll_grad(amp_model*, double* f, double* g, void*) {
    double s = 0.0;
    ++n_grad;
    for (int i = 0; i < 2 * K; ++i) {
        const double d = cur[i] - target(i);
        s += 0.5 * lam(i) * d * d + 0.25 * d * d * d * d;
        g[i] = lam(i) * d + d * d * d;
    }
    for (int i = 0; i + 1 < 2 * K; ++i) {
        const double d0 = cur[i] - target(i), d1 = cur[i + 1] - target(i + 1);
        s += 0.3 * d0 * d1;
        g[i] += 0.3 * d1;
        g[i + 1] += 0.3 * d0;
    }
    if (cur[0] > 50.0) return AMP_ERR_DOMAIN;   // a region without a likelihood: the line search has to back off
    *f = s;
    return AMP_OK;
}
int stub_counts(int which) { return which ? n_grad : n_set; }
void stub_current(double* out) { for (int i = 0; i < 2 * K; ++i) out[i] = cur[i]; }
}

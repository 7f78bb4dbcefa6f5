// minimize.cu — the fit loop in native code: a quasi-Newton (BFGS) minimiser of the NLL over the complex
// helicity couplings, driven by the analytic gradient of amp_nll_grad, with Hessian errors.  The paper drives the device
// PDF with MINUIT; MINUIT is not in this image and its gradient is a finite-difference one — here every
// iteration is one amp_set_params + one k_grad launch (the couplings' derivatives come with the NLL), and no interpreter
// sits between two launches: a 10,000-event pseudo-experiment is fitted in a few milliseconds.
//
// Host code only; it uses nothing but the public C ABI (amp_set_params, amp_nll_grad), so it adds no second path to the
// likelihood.  Method: BFGS on the inverse Hessian (Nocedal & Wright, Numerical Optimization, Alg. 6.1) with a strong-Wolfe
// line search (Alg. 3.5 / 3.6, c1 = 1e-4, c2 = 0.9, cubic interpolation safeguarded by bisection); parameters are
// Re H_k / s_k, Im H_k / s_k of the free slots (s_k: caller's scale or |H_k| of the start); fixed slots (Eq. 6) keep their
// start values, tied slots (Eq. 11) copy their source and pass their derivative on by the chain rule.
// Covariance: inverse of the Hessian at the minimum, the Hessian from central differences of the analytic gradient.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <vector>

#include "amp_internal.cuh"

namespace {

struct Problem {
    amp_model* m;
    void* stream;
    int K, R, n;                       // n = 2 * number of free slots
    std::vector<int> free_slot;        // free slots
    std::vector<int> tie_dst, tie_src;
    std::vector<double> tie_sign;      // H[dst] = sign * H[src], sign = +1 or -1 (Eq. 11: the sign depends on the Z's spin-parity)
    std::vector<double> c0;            // [K][2] start (fixed slots stay)
    std::vector<double> scale;         // [K]
    const double* mw;                  // [R][2] or null: what amp_set_params receives (mwv when lineshape parameters float)
    // floating masses / widths: parameter 2 F + i is (mass or width of resonance mw_res[i]) / mw_scale[i]; its derivative is a
    // central difference of the NLL over +- mw_step[i] (one batch of 1 + 2 n_mw points per evaluation: the gradient-batch kernel)
    std::vector<int> mw_res, mw_which;
    std::vector<double> mw_scale, mw_step, mwv;   // mwv: [R][2] current values
    std::vector<double> bc, bmw, bnll;            // batch work arrays
    int calls = 0;
    amp_status status = AMP_OK;
    std::vector<double> c, grad;       // work: [K][2]

    int nmw() const { return (int)mw_res.size(); }
    void unpack_mw(const double* th) {
        for (int i = 0; i < nmw(); ++i) mwv[2 * mw_res[i] + mw_which[i]] = th[2 * free_slot.size() + i] * mw_scale[i];
    }
    void unpack(const double* th, double* c_out) const {
        std::memcpy(c_out, c0.data(), sizeof(double) * 2 * K);
        for (size_t i = 0; i < free_slot.size(); ++i) {
            const int k = free_slot[i];
            c_out[2 * k] = th[2 * i] * scale[k];
            c_out[2 * k + 1] = th[2 * i + 1] * scale[k];
        }
        for (size_t t = 0; t < tie_dst.size(); ++t) {
            c_out[2 * tie_dst[t]] = tie_sign[t] * c_out[2 * tie_src[t]];
            c_out[2 * tie_dst[t] + 1] = tie_sign[t] * c_out[2 * tie_src[t] + 1];
        }
    }
    // NLL and its gradient in theta; a domain error (non-finite likelihood) is reported as +inf so that a line search backs off
    bool eval(const double* th, double* f, double* g) {
        unpack(th, c.data());
        unpack_mw(th);
        amp_status st = amp_set_params(m, 1, c.data(), mw);
        if (st == AMP_OK) st = amp_nll_grad(m, f, grad.data(), stream);
        ++calls;
        if (st == AMP_ERR_DOMAIN) { *f = INFINITY; std::fill(g, g + n, 0.0); return true; }
        if (st != AMP_OK) { status = st; return false; }
        if (nmw() > 0) {
            const int Pn = 1 + 2 * nmw();
            for (int q = 0; q < Pn; ++q) {
                std::memcpy(&bc[(size_t)q * 2 * K], c.data(), sizeof(double) * 2 * K);
                std::memcpy(&bmw[(size_t)q * 2 * R], mwv.data(), sizeof(double) * 2 * R);
            }
            for (int i = 0; i < nmw(); ++i) {
                bmw[(size_t)(1 + 2 * i) * 2 * R + 2 * mw_res[i] + mw_which[i]] += mw_step[i];
                bmw[(size_t)(2 + 2 * i) * 2 * R + 2 * mw_res[i] + mw_which[i]] -= mw_step[i];
            }
            st = amp_set_params(m, Pn, bc.data(), bmw.data());
            if (st == AMP_OK) st = amp_nll(m, bnll.data(), stream);
            if (st == AMP_ERR_DOMAIN) { *f = INFINITY; std::fill(g, g + n, 0.0); return true; }   // a step left the lineshape's domain
            if (st != AMP_OK) { status = st; return false; }
            for (int i = 0; i < nmw(); ++i)
                g[2 * free_slot.size() + i] = (bnll[1 + 2 * i] - bnll[2 + 2 * i]) / (2.0 * mw_step[i]) * mw_scale[i];
        }
        for (size_t t = 0; t < tie_dst.size(); ++t) {
            grad[2 * tie_src[t]] += tie_sign[t] * grad[2 * tie_dst[t]];
            grad[2 * tie_src[t] + 1] += tie_sign[t] * grad[2 * tie_dst[t] + 1];
        }
        for (size_t i = 0; i < free_slot.size(); ++i) {
            const int k = free_slot[i];
            g[2 * i] = grad[2 * k] * scale[k];
            g[2 * i + 1] = grad[2 * k + 1] * scale[k];
        }
        return true;
    }
};

double dot(const std::vector<double>& a, const std::vector<double>& b) {
    double s = 0.0;
    for (size_t i = 0; i < a.size(); ++i) s += a[i] * b[i];
    return s;
}
double max_abs(const std::vector<double>& a) {
    double s = 0.0;
    for (double v : a) s = std::fmax(s, std::fabs(v));
    return s;
}

// minimiser of the cubic through (a, fa, dfa), (b, fb, dfb); falls back to the midpoint
double cubic_min(double a, double fa, double dfa, double b, double fb, double dfb) {
    const double d1 = dfa + dfb - 3.0 * (fa - fb) / (a - b);
    const double rad = d1 * d1 - dfa * dfb;
    if (!(rad >= 0.0) || !std::isfinite(rad)) return 0.5 * (a + b);
    const double d2 = (b > a ? 1.0 : -1.0) * std::sqrt(rad);
    const double x = b - (b - a) * (dfb + d2 - d1) / (dfb - dfa + 2.0 * d2);
    return std::isfinite(x) ? x : 0.5 * (a + b);
}

struct Trial { double a, f, df; std::vector<double> x, g; };

// strong-Wolfe line search along p from (x, f0, g0); on success `out` holds the accepted point
bool line_search(Problem& P, const std::vector<double>& x, double f0, const std::vector<double>& g0, const std::vector<double>& p,
                 double a1, Trial* out) {
    const double c1 = 1e-4, c2 = 0.9;
    // near the minimum the decrease a step can achieve falls below the rounding of the NLL itself (|f| 2^-52 per addition, ~1e-11
    // for a sum over 1e5 events) while the analytic gradient keeps its relative accuracy: function comparisons allow for that
    // noise, and the curvature condition on the gradient decides
    const double eps_f = 1e-12 * std::fabs(f0);
    const int n = P.n;
    const double df0 = dot(g0, p);
    if (!(df0 < 0.0)) return false;
    auto at = [&](double a, Trial* t) {
        t->a = a;
        t->x.resize(n);
        t->g.resize(n);
        for (int i = 0; i < n; ++i) t->x[i] = x[i] + a * p[i];
        if (!P.eval(t->x.data(), &t->f, t->g.data())) return false;
        t->df = dot(t->g, p);
        return true;
    };
    Trial lo{0.0, f0, df0, x, g0}, hi, cur;
    bool bracket = false;
    double a = a1;
    Trial prev = lo;
    for (int it = 0; it < 25 && !bracket; ++it) {
        if (!at(a, &cur)) return false;
        if (!std::isfinite(cur.f) || cur.f > f0 + c1 * a * df0 + eps_f || (it > 0 && cur.f >= prev.f + eps_f)) { lo = prev; hi = cur; bracket = true; break; }
        if (std::fabs(cur.df) <= -c2 * df0) { *out = cur; return true; }
        if (cur.df >= 0.0) { lo = cur; hi = prev; bracket = true; break; }
        prev = cur;
        a *= 2.0;
    }
    if (!bracket) { *out = prev; return prev.a > 0.0; }
    for (int it = 0; it < 40; ++it) {   // zoom: lo satisfies sufficient decrease and has the lowest value so far
        double an;
        if (std::isfinite(hi.f)) {
            an = cubic_min(lo.a, lo.f, lo.df, hi.a, hi.f, hi.df);
            const double l = std::fmin(lo.a, hi.a), h = std::fmax(lo.a, hi.a), w = h - l;
            if (!(an > l + 0.1 * w && an < h - 0.1 * w)) an = 0.5 * (l + h);
        } else {
            an = lo.a + 0.25 * (hi.a - lo.a);
        }
        if (!at(an, &cur)) return false;
        if (!std::isfinite(cur.f) || cur.f > f0 + c1 * an * df0 + eps_f || cur.f >= lo.f + eps_f) {
            hi = cur;
        } else {
            if (std::fabs(cur.df) <= -c2 * df0) { *out = cur; return true; }
            if (cur.df * (hi.a - lo.a) >= 0.0) hi = lo;
            lo = cur;
        }
        if (std::fabs(hi.a - lo.a) < 1e-14 * std::fmax(1.0, std::fabs(lo.a))) break;
    }
    if (lo.a > 0.0) { *out = lo; return true; }   // sufficient decrease only
    return false;
}

// inverse of a symmetric positive-definite matrix by Cholesky; false if not positive definite
bool spd_inverse(std::vector<double>& A, int n) {
    std::vector<double> L(A);
    for (int j = 0; j < n; ++j) {
        double d = L[j * n + j];
        for (int k = 0; k < j; ++k) d -= L[j * n + k] * L[j * n + k];
        if (!(d > 0.0)) return false;
        d = std::sqrt(d);
        L[j * n + j] = d;
        for (int i = j + 1; i < n; ++i) {
            double s = L[i * n + j];
            for (int k = 0; k < j; ++k) s -= L[i * n + k] * L[j * n + k];
            L[i * n + j] = s / d;
        }
    }
    // A^-1 = L^-T L^-1: invert L (lower triangular) in place, then multiply
    std::vector<double> Li(n * n, 0.0);
    for (int j = 0; j < n; ++j) {
        Li[j * n + j] = 1.0 / L[j * n + j];
        for (int i = j + 1; i < n; ++i) {
            double s = 0.0;
            for (int k = j; k < i; ++k) s -= L[i * n + k] * Li[k * n + j];
            Li[i * n + j] = s / L[i * n + i];
        }
    }
    for (int i = 0; i < n; ++i)
        for (int j = 0; j <= i; ++j) {
            double s = 0.0;
            for (int k = i; k < n; ++k) s += Li[k * n + i] * Li[k * n + j];
            A[i * n + j] = A[j * n + i] = s;
        }
    return true;
}

}  // namespace

extern "C" amp_status amp_fit(amp_model* m, const double* h_start, const double* h_mass_width, const int* fixed, int n_fixed,
                              const int* tie_dst, const int* tie_src, const int* tie_sign, int n_ties, const int* float_mw, int n_float_mw,
                              const double* h_scale, int max_iter, double gtol,
                              double* h_fit, double* h_fit_mw, double* h_nll, double* h_cov, int* h_info, void* stream) {
    if (!m || !h_start || !h_fit || !h_nll || n_fixed < 0 || n_ties < 0 || (n_fixed && !fixed) || (n_ties && (!tie_dst || !tie_src)) ||
        max_iter < 0 || !(gtol > 0.0) || n_float_mw < 0 || (n_float_mw && (!float_mw || !h_mass_width)) ||
        1 + 2 * n_float_mw > AMP_MAX_POINTS)
        return AMP_ERR_INVALID;
    Problem P;
    P.m = m;
    P.stream = stream;
    P.K = amp_num_couplings(m);
    P.R = amp_num_resonances(m);
    P.mw = h_mass_width;
    std::vector<char> held(P.K, 0);
    for (int i = 0; i < n_fixed; ++i) {
        if (fixed[i] < 0 || fixed[i] >= P.K) return AMP_ERR_INVALID;
        held[fixed[i]] = 1;
    }
    for (int i = 0; i < n_ties; ++i) {
        if (tie_dst[i] < 0 || tie_dst[i] >= P.K || tie_src[i] < 0 || tie_src[i] >= P.K || tie_dst[i] == tie_src[i]) return AMP_ERR_INVALID;
        if (tie_sign && tie_sign[i] != 1 && tie_sign[i] != -1) return AMP_ERR_INVALID;
        if (held[tie_dst[i]]) return AMP_ERR_INVALID;   // a destination that is fixed, or tied twice
        held[tie_dst[i]] = 1;
        P.tie_sign.push_back(tie_sign ? (double)tie_sign[i] : 1.0);
        P.tie_dst.push_back(tie_dst[i]);
        P.tie_src.push_back(tie_src[i]);
    }
    for (int i = 0; i < n_ties; ++i)
        if (held[tie_src[i]] == 1 && std::find(P.tie_dst.begin(), P.tie_dst.end(), tie_src[i]) != P.tie_dst.end()) return AMP_ERR_INVALID;   // no chains
    for (int k = 0; k < P.K; ++k)
        if (!held[k]) P.free_slot.push_back(k);
    if (h_mass_width) P.mwv.assign(h_mass_width, h_mass_width + 2 * P.R);
    for (int i = 0; i < n_float_mw; ++i) {
        const int r = float_mw[2 * i], which = float_mw[2 * i + 1];
        if (r < 0 || r >= P.R || which < 0 || which > 1) return AMP_ERR_INVALID;
        for (int j = 0; j < i; ++j)
            if (float_mw[2 * j] == r && float_mw[2 * j + 1] == which) return AMP_ERR_INVALID;
        const double width = h_mass_width[2 * r + 1];
        if (!(width > 0.0) || !std::isfinite(width)) return AMP_ERR_INVALID;
        P.mw_res.push_back(r);
        P.mw_which.push_back(which);
        P.mw_scale.push_back(width);            // masses and widths both move on the scale of the width
        P.mw_step.push_back(1e-2 * width);      // truncation error ~ (step / width)^2 of the derivative; rounding of the NLL far below
    }
    if (n_float_mw) {
        P.mw = P.mwv.data();
        const int Pn = 1 + 2 * n_float_mw;
        P.bc.resize((size_t)Pn * 2 * P.K);
        P.bmw.resize((size_t)Pn * 2 * P.R);
        P.bnll.resize(Pn);
    }
    P.n = 2 * (int)P.free_slot.size() + n_float_mw;
    P.c0.assign(h_start, h_start + 2 * P.K);
    P.scale.resize(P.K);
    double cmax = 0.0;
    for (int k = 0; k < P.K; ++k) cmax = std::fmax(cmax, std::hypot(h_start[2 * k], h_start[2 * k + 1]));
    for (int k = 0; k < P.K; ++k) {
        P.scale[k] = h_scale ? h_scale[k] : std::fmax(std::hypot(h_start[2 * k], h_start[2 * k + 1]), 1e-3 * cmax);
        if (!(P.scale[k] > 0.0) || !std::isfinite(P.scale[k])) return AMP_ERR_INVALID;
    }
    P.c.resize(2 * P.K);
    P.grad.resize(2 * P.K);
    const int n = P.n;
    std::vector<double> x(n), g(n), p(n), H((size_t)n * n, 0.0), s(n), y(n), Hy(n);
    for (size_t i = 0; i < P.free_slot.size(); ++i) {
        const int k = P.free_slot[i];
        x[2 * i] = h_start[2 * k] / P.scale[k];
        x[2 * i + 1] = h_start[2 * k + 1] / P.scale[k];
    }
    for (int i = 0; i < n_float_mw; ++i) x[2 * P.free_slot.size() + i] = h_mass_width[2 * P.mw_res[i] + P.mw_which[i]] / P.mw_scale[i];
    double f;
    if (!P.eval(x.data(), &f, g.data())) return P.status;
    if (!std::isfinite(f)) return AMP_ERR_DOMAIN;
    for (int i = 0; i < n; ++i) H[(size_t)i * n + i] = 1.0;
    bool converged = n == 0 || max_abs(g) < gtol, first = true;
    double f_prev = INFINITY;
    int iter = 0;
    for (; iter < max_iter && !converged; ++iter) {
        for (int i = 0; i < n; ++i) {
            double t = 0.0;
            for (int j = 0; j < n; ++j) t -= H[(size_t)i * n + j] * g[j];
            p[i] = t;
        }
        if (!(dot(g, p) < 0.0)) {   // lost positive definiteness to rounding: restart from steepest descent
            std::fill(H.begin(), H.end(), 0.0);
            for (int i = 0; i < n; ++i) { H[(size_t)i * n + i] = 1.0; p[i] = -g[i]; }
            first = true;
            f_prev = INFINITY;
        }
        Trial t;
        // first trial step: 1 once the inverse Hessian has its scale; before that the step that would repeat the last decrease
        // (Nocedal & Wright Eq. 3.60), and 1/|g| at the very start
        double a1 = first ? std::fmin(1.0, 1.0 / std::sqrt(dot(g, g))) : 1.0;
        if (!first && std::isfinite(f_prev)) {
            const double ai = 1.01 * 2.0 * (f - f_prev) / dot(g, p);
            if (ai > 0.0 && ai < 1.0) a1 = ai;
        }
        if (!line_search(P, x, f, g, p, a1, &t)) {
            if (P.status != AMP_OK) return P.status;
            break;   // no further decrease along a descent direction: at the numerical minimum
        }
        for (int i = 0; i < n; ++i) { s[i] = t.x[i] - x[i]; y[i] = t.g[i] - g[i]; }
        const double sy = dot(s, y);
        if (sy > 1e-12 * std::sqrt(dot(s, s) * dot(y, y))) {
            first = false;
            const double rho = 1.0 / sy;
            for (int i = 0; i < n; ++i) {
                double v = 0.0;
                for (int j = 0; j < n; ++j) v += H[(size_t)i * n + j] * y[j];
                Hy[i] = v;
            }
            const double yHy = dot(y, Hy);
            for (int i = 0; i < n; ++i)
                for (int j = 0; j < n; ++j)
                    H[(size_t)i * n + j] += -rho * (Hy[i] * s[j] + s[i] * Hy[j]) + rho * (rho * yHy + 1.0) * s[i] * s[j];
        }
        f_prev = f;
        x = t.x;
        g = t.g;
        f = t.f;
        converged = max_abs(g) < gtol;
    }
    P.unpack(x.data(), h_fit);
    P.unpack_mw(x.data());
    if (h_fit_mw && h_mass_width) std::memcpy(h_fit_mw, P.mwv.data(), sizeof(double) * 2 * P.R);
    h_nll[0] = f;
    h_nll[1] = max_abs(g);
    int cov_ok = 0;
    bool hess_finite = true;   // an evaluation outside the likelihood's domain (f = inf, g = 0) must not enter the covariance
    const int nc = 2 * (int)P.free_slot.size();
    auto par_scale = [&](int i) { return i < nc ? P.scale[P.free_slot[i / 2]] : P.mw_scale[i - nc]; };
    if (h_cov && n > 0) {
        const double h = 1e-4;
        std::vector<double> A((size_t)n * n), gp(n), gm(n), xx(x);
        double fp, fm;
        for (int j = 0; j < n; ++j) {
            xx[j] = x[j] + h;
            if (!P.eval(xx.data(), &fp, gp.data())) return P.status;
            xx[j] = x[j] - h;
            if (!P.eval(xx.data(), &fm, gm.data())) return P.status;
            hess_finite = hess_finite && std::isfinite(fp) && std::isfinite(fm);
            xx[j] = x[j];
            for (int i = 0; i < n; ++i) A[(size_t)i * n + j] = (gp[i] - gm[i]) / (2.0 * h);
        }
        for (int i = 0; i < n; ++i)
            for (int j = 0; j < i; ++j) A[(size_t)i * n + j] = A[(size_t)j * n + i] = 0.5 * (A[(size_t)i * n + j] + A[(size_t)j * n + i]);
        cov_ok = (hess_finite && spd_inverse(A, n)) ? 1 : 0;
        for (int i = 0; i < n; ++i)
            for (int j = 0; j < n; ++j)
                h_cov[(size_t)i * n + j] = cov_ok ? A[(size_t)i * n + j] * par_scale(i) * par_scale(j) : NAN;
    }
    P.unpack_mw(x.data());   // the Hessian loop moved them
    // leave the model at the fitted point
    amp_status st = amp_set_params(m, 1, h_fit, P.mw);
    if (st != AMP_OK) return st;
    if (h_info) {
        h_info[0] = converged ? 1 : 0;
        h_info[1] = P.calls;
        h_info[2] = iter;
        h_info[3] = cov_ok;
        h_info[4] = n;
    }
    return AMP_OK;
}

"""A small host-side minimiser loop around the device NLL and its analytic gradient.

The paper drives the device PDF with MINUIT; MINUIT is not in this image, so this loop uses scipy's BFGS
(dense: at most 2 x 48 parameters) with the analytic gradient of `amp_nll_grad` — one launch per iteration instead of 2 K finite-difference evaluations.  It fits
the complex helicity couplings (real and imaginary parts) at fixed masses and widths; the conventions of the paper enter as
`fixed` slots (Eq. 6: the K*(892) lambda = 0 amplitude is the reference) and `ties` (Eq. 11: H^Z_{+1} = H^Z_{-1}), applied by
the chain rule.  Every likelihood evaluation runs in the CUDA library; nothing here touches the oracle.
"""
import numpy as np


class FitResult:
    def __init__(self, couplings, nll, n_calls, converged, grad_norm, message):
        self.couplings, self.nll, self.n_calls = couplings, nll, n_calls
        self.converged, self.grad_norm, self.message = converged, grad_norm, message

    def __repr__(self):
        return f"FitResult(nll={self.nll:.6f}, n_calls={self.n_calls}, converged={self.converged}, |grad|={self.grad_norm:.3e})"


def fit_couplings(model, c_start, fixed=(), ties=(), mass_width=None, maxiter=3000, gtol=1e-3, scale=None):
    """Minimise the NLL of `model` (a binding.Model with data and normalisation events loaded) over the couplings.

    c_start   complex [K] starting values (fixed slots keep these values)
    fixed     slots held constant (e.g. the K*(892) lambda = 0 slot, Eq. 6)
    ties      (dst, src) pairs with H[dst] = H[src] (Eq. 11); dst is not a free parameter
    scale     optional positive [K] parameter scales (default |c_start|, floored): the fit runs in H / scale
    Returns a FitResult; the model is left with the fitted parameters set.
    """
    from scipy.optimize import minimize

    c0 = np.asarray(c_start, dtype=np.complex128).copy()
    K = c0.size
    assert K == model.K
    tied = {int(d): int(s) for d, s in ties}
    free = [k for k in range(K) if k not in set(int(f) for f in fixed) and k not in tied]
    sc = np.maximum(np.abs(c0), 1e-3 * np.max(np.abs(c0))) if scale is None else np.asarray(scale, dtype=np.float64)
    mw = None if mass_width is None else np.asarray(mass_width, dtype=np.float64).reshape(1, model.R, 2)
    calls = [0]

    def unpack(theta):
        c = c0.copy()
        t = theta.reshape(-1, 2)
        for i, k in enumerate(free):
            c[k] = (t[i, 0] + 1j * t[i, 1]) * sc[k]
        for d, s in tied.items():
            c[d] = c[s]
        return c

    def fun(theta):
        c = unpack(theta)
        model.set_params(c, mw)
        nll, g = model.nll_grad()                 # g[k] = (dNLL/dRe H_k, dNLL/dIm H_k)
        calls[0] += 1
        g = g.copy()
        for d, s in tied.items():                 # chain rule of H[dst] = H[src]
            g[s] += g[d]
        return nll, (g[free] * sc[free, None]).ravel()

    theta0 = np.stack([(c0[free] / sc[free]).real, (c0[free] / sc[free]).imag], -1).ravel()
    # gtol: largest |dNLL/d(scaled parameter)| at the end; the NLL itself is O(N), so 1e-3 is far below its statistical scale
    res = minimize(fun, theta0, jac=True, method="BFGS", options={"maxiter": maxiter, "gtol": gtol})
    c_fit = unpack(res.x)
    model.set_params(c_fit, mw)
    gmax = float(np.max(np.abs(res.jac)))
    return FitResult(c_fit, float(res.fun), calls[0], bool(res.success) or gmax < 10 * gtol, gmax, str(res.message))

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
        self.free = None        # free slots, in the order of `errors` / `covariance`
        self.errors = None      # complex [n_free]: sigma(Re H_k) + 1j sigma(Im H_k) (fit_couplings(..., errors=True))
        self.covariance = None  # [2 n_free][2 n_free] of (Re H_k0, Im H_k0, Re H_k1, ...)

    def __repr__(self):
        return f"FitResult(nll={self.nll:.6f}, n_calls={self.n_calls}, converged={self.converged}, |grad|={self.grad_norm:.3e})"


def fit_couplings(model, c_start, fixed=(), ties=(), mass_width=None, maxiter=3000, gtol=1e-3, scale=None, errors=False):
    """Minimise the NLL of `model` (a binding.Model with data and normalisation events loaded) over the couplings.

    c_start   complex [K] starting values (fixed slots keep these values)
    fixed     slots held constant (e.g. the K*(892) lambda = 0 slot, Eq. 6)
    ties      (dst, src) or (dst, src, sign) with H[dst] = sign * H[src], sign = +-1 (Eq. 11: +1 for the 1+ Z;
              -1 for a 2+ or 1- Z, amp.h); dst is not a free parameter
    scale     optional positive [K] parameter scales (default |c_start|, floored): the fit runs in H / scale
    errors    also return the covariance of the free parameters: inverse of the Hessian of the NLL at the minimum, the Hessian
              from central differences of the ANALYTIC gradient (2 launches per free real parameter) — what the pulls of the
              paper's validation (Figs. 5-6) are normalised with
    Returns a FitResult; the model is left with the fitted parameters set.
    """
    from scipy.optimize import minimize

    c0 = np.asarray(c_start, dtype=np.complex128).copy()
    K = c0.size
    assert K == model.K
    tied = {int(t[0]): (int(t[1]), float(t[2]) if len(t) > 2 else 1.0) for t in ties}
    free = [k for k in range(K) if k not in set(int(f) for f in fixed) and k not in tied]
    sc = np.maximum(np.abs(c0), 1e-3 * np.max(np.abs(c0))) if scale is None else np.asarray(scale, dtype=np.float64)
    mw = None if mass_width is None else np.asarray(mass_width, dtype=np.float64).reshape(1, model.R, 2)
    calls = [0]

    def unpack(theta):
        c = c0.copy()
        t = theta.reshape(-1, 2)
        for i, k in enumerate(free):
            c[k] = (t[i, 0] + 1j * t[i, 1]) * sc[k]
        for d, (s, sg) in tied.items():
            c[d] = sg * c[s]
        return c

    def fun(theta):
        c = unpack(theta)
        model.set_params(c, mw)
        nll, g = model.nll_grad()                 # g[k] = (dNLL/dRe H_k, dNLL/dIm H_k)
        calls[0] += 1
        g = g.copy()
        for d, (s, sg) in tied.items():           # chain rule of H[dst] = sign H[src]
            g[s] += sg * g[d]
        return nll, (g[free] * sc[free, None]).ravel()

    theta0 = np.stack([(c0[free] / sc[free]).real, (c0[free] / sc[free]).imag], -1).ravel()
    # gtol: largest |dNLL/d(scaled parameter)| at the end; the NLL itself is O(N), so 1e-3 is far below its statistical scale
    res = minimize(fun, theta0, jac=True, method="BFGS", options={"maxiter": maxiter, "gtol": gtol})
    c_fit = unpack(res.x)
    gmax = float(np.max(np.abs(res.jac)))
    out = FitResult(c_fit, float(res.fun), calls[0], bool(res.success) or gmax < 10 * gtol, gmax, str(res.message))
    out.free = list(free)
    if errors:
        nt = res.x.size
        H = np.empty((nt, nt))
        h = 1e-4                                   # in units of the parameter scale; the gradient is analytic, so O(h^2) error only
        for j in range(nt):
            tp, tm = res.x.copy(), res.x.copy()
            tp[j] += h
            tm[j] -= h
            H[:, j] = (fun(tp)[1] - fun(tm)[1]) / (2 * h)
        H = 0.5 * (H + H.T)
        cov_t = np.linalg.inv(H)
        s2 = np.repeat(sc[free], 2)
        out.covariance = cov_t * s2[:, None] * s2[None, :]
        sig = np.sqrt(np.maximum(np.diag(out.covariance), 0.0)).reshape(-1, 2)
        out.errors = sig[:, 0] + 1j * sig[:, 1]
        out.n_calls = calls[0]
    model.set_params(c_fit, mw)
    return out


def pull_study(model, c_true, n_toys, n_events, seed, m_lo, m_hi, cos_max, fixed=(), ties=(), start_spread=0.1, f_max=None, native=True):
    """The paper's validation loop: n_toys pseudo-experiments of n_events each are generated from c_true on the
    device (amp_generate; no efficiency: the model's normalisation sample must then be an unweighted phase-space sample), each is
    fitted from a perturbed start (amp_fit, or scipy's BFGS with native=False) and its pulls (fit - true) / sigma are recorded.
    Returns dict(pulls [n_toys][2 n_free], converged [n_toys], n_calls [n_toys], couplings [n_toys][K]); candidate streams of
    successive toys do not overlap (toy t uses seed + t)."""
    import torch
    c_true = np.asarray(c_true, dtype=np.complex128)
    model.set_params(c_true)
    if f_max is None:
        _, _, _, fs = model.generate(seed, 0, 1 << 18, 0.0, m_lo, m_hi, cos_max, 0)
        f_max = 1.5 * fs
    ones = torch.ones(n_events, dtype=torch.float64, device="cuda")
    rng = np.random.default_rng(seed)
    pulls, conv, ncall, cs = [], [], [], []
    tied = {int(t[0]): (int(t[1]), float(t[2]) if len(t) > 2 else 1.0) for t in ties}
    for t in range(n_toys):
        model.set_params(c_true)
        x, _, _, fseen = model.generate_toy(n_events, seed + 1 + t, m_lo, m_hi, cos_max, f_max=f_max, block=1 << 20)
        if fseen > f_max:
            raise RuntimeError("pull_study: envelope f_max too low for this toy")
        model.load_events(x.contiguous(), ones)
        start = c_true * (1 + start_spread * rng.uniform(-1, 1, c_true.size)) * np.exp(1j * start_spread * rng.uniform(-1, 1, c_true.size))
        for k in fixed:
            start[k] = c_true[k]
        for d, (s, sg) in tied.items():
            start[d] = sg * start[s]
        if native:      # the minimiser of the library (amp_fit): no interpreter between two launches
            r = model.fit(start, fixed=fixed, ties=ties, scale=np.abs(c_true), errors=True)
            cf, free, err, ok, nc = r["couplings"], r["free"], r["errors"], r["converged"] and r["errors"] is not None, r["n_calls"]
        else:           # scipy's BFGS on the same gradient (cross-check)
            r = fit_couplings(model, start, fixed=fixed, ties=ties, scale=np.abs(c_true), errors=True)
            cf, free, err, ok, nc = r.couplings, r.free, r.errors, r.converged, r.n_calls
        d = cf[free] - c_true[free]
        pulls.append(np.stack([d.real / err.real, d.imag / err.imag], -1).ravel() if err is not None else np.full(2 * len(free), np.nan))
        conv.append(ok)
        ncall.append(nc)
        cs.append(cf)
    return {"pulls": np.array(pulls), "converged": np.array(conv), "n_calls": np.array(ncall), "couplings": np.array(cs)}

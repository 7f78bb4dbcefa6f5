"""Host logic of the native minimiser (csrc/minimize.cu, amp_fit) without a GPU: the file is compiled (host code only) against a
stand-in likelihood with a known minimum and Hessian (tests/minimize_stub.cu) and compared with the closed form and with scipy."""
import ctypes as C
import os
import shutil
import subprocess

import numpy as np
import pytest

HERE = os.path.dirname(os.path.abspath(__file__))
K = 12


def lam(i):
    return 1e4 ** (i / (2.0 * K - 1))


def f_and_grad(h):
    d = h - (1.0 + 0.1 * np.arange(2 * K))
    l = lam(np.arange(2 * K))
    f = np.sum(0.5 * l * d * d + 0.25 * d ** 4) + 0.3 * np.sum(d[:-1] * d[1:])
    g = l * d + d ** 3
    g[:-1] += 0.3 * d[1:]
    g[1:] += 0.3 * d[:-1]
    return f, g


@pytest.fixture(scope="module")
def stub(tmp_path_factory):
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(nvcc):
        pytest.skip("nvcc not available")
    out = str(tmp_path_factory.mktemp("minstub") / "libminstub.so")
    subprocess.check_call([nvcc, "-O2", "-shared", "-Xcompiler", "-fPIC", "-I", os.path.join(HERE, "..", "include"), "-o", out,
                           os.path.join(HERE, "minimize_stub.cu")])
    lib = C.CDLL(out)
    vp, i, d = C.c_void_p, C.c_int, C.c_double
    lib.amp_fit.restype = i
    lib.amp_fit.argtypes = [vp, vp, vp, vp, i, vp, vp, vp, i, vp, i, vp, i, d, vp, vp, vp, vp, vp, vp]
    return lib


def run(lib, start, fixed=(), ties=(), scale=None, max_iter=3000, gtol=1e-7, cov=True, mw=None, float_mw=()):
    p = lambda a: a.ctypes.data_as(C.c_void_p) if a is not None and a.size else None
    hs = np.ascontiguousarray(start, dtype=np.float64).reshape(K, 2)
    fx = np.ascontiguousarray(fixed, dtype=np.int32)
    td = np.ascontiguousarray([t[0] for t in ties], dtype=np.int32)
    ts = np.ascontiguousarray([t[1] for t in ties], dtype=np.int32)
    tg = np.ascontiguousarray([t[2] for t in ties], dtype=np.int32) if ties and all(len(t) > 2 for t in ties) else None
    sc = None if scale is None else np.ascontiguousarray(scale, dtype=np.float64)
    nfree = K - len(set(fixed)) - len(td)
    fm = np.ascontiguousarray(float_mw, dtype=np.int32).reshape(-1, 2)
    hmw = None if mw is None else np.ascontiguousarray(mw, dtype=np.float64).reshape(1, 2)
    fit, nll, info, fit_mw = np.empty((K, 2)), np.empty(2), np.zeros(5, dtype=np.int32), np.zeros((1, 2))
    n = 2 * nfree + len(fm)
    cv = np.empty((n, n)) if cov else None
    st = lib.amp_fit(C.c_void_p(1), p(hs), p(hmw), p(fx), len(fx), p(td), p(ts), p(tg), len(td), p(fm), len(fm), p(sc), max_iter, gtol, p(fit),
                     p(fit_mw), p(nll), p(cv), p(info), None)
    if mw is not None:
        return st, fit, nll, cv, info, fit_mw
    return st, fit, nll, cv, info


def test_unconstrained_minimum_and_covariance(stub):
    start = np.full(2 * K, 0.5)
    st, fit, nll, cov, info = run(stub, start)
    assert st == 0 and info[0] == 1 and info[3] == 1 and info[4] == 2 * K
    target = 1.0 + 0.1 * np.arange(2 * K)
    assert np.max(np.abs(fit.ravel() - target)) < 1e-7          # the known minimum
    assert nll[0] < 1e-12 and nll[1] < 1e-7
    # covariance = inverse Hessian; at the minimum the Hessian is diag(lam) + 0.3 (off-diagonals)
    H = np.diag(lam(np.arange(2 * K))) + 0.3 * (np.eye(2 * K, k=1) + np.eye(2 * K, k=-1))
    assert np.max(np.abs(cov - np.linalg.inv(H)) / np.abs(np.linalg.inv(H)).max()) < 1e-6
    # as many likelihood calls as scipy's BFGS needs for the same problem (+ 4 F for the Hessian), within a factor 1.5
    from scipy.optimize import minimize
    r = minimize(lambda t: f_and_grad(t), start, jac=True, method="BFGS", options={"gtol": 1e-7})
    assert info[1] - 4 * K <= 1.5 * r.nfev + 5, (info, r.nfev)
    # the stand-in model is left at the fitted point
    cur = np.empty(2 * K)
    stub.stub_current(cur.ctypes.data_as(C.c_void_p))
    assert np.array_equal(cur, fit.ravel())


def test_fixed_slots_ties_and_scales(stub):
    start = np.full(2 * K, 0.5)
    start[2:4] = (0.9, -0.4)                                      # slot 1 fixed at this value
    fixed, ties = [1], [(5, 3), (7, 3)]                           # H_5 = H_3, H_7 = H_3
    scale = np.linspace(0.2, 3.0, K)
    st, fit, nll, cov, info = run(stub, start, fixed=fixed, ties=ties, scale=scale)
    assert st == 0 and info[0] == 1 and info[4] == 2 * (K - 3)
    assert tuple(fit[1]) == (0.9, -0.4)
    assert np.array_equal(fit[5], fit[3]) and np.array_equal(fit[7], fit[3])
    # reference: scipy on the reduced problem
    free = [k for k in range(K) if k not in (1, 5, 7)]

    def expand(t):
        h = start.copy().reshape(K, 2)
        h[free] = t.reshape(-1, 2)
        h[5] = h[3]
        h[7] = h[3]
        return h

    def red(t):
        f, g = f_and_grad(expand(t).ravel())
        g = g.reshape(K, 2).copy()
        g[3] += g[5] + g[7]
        return f, g[free].ravel()

    from scipy.optimize import minimize
    r = minimize(red, start.reshape(K, 2)[free].ravel(), jac=True, method="BFGS", options={"gtol": 1e-9})
    assert abs(nll[0] - r.fun) < 1e-9 * max(1.0, abs(r.fun))
    assert np.max(np.abs(fit[free].ravel() - r.x)) < 1e-6
    # covariance of the free parameters in H units (not in scaled units): finite-difference Hessian of the reduced problem
    n = 2 * len(free)
    Hn = np.empty((n, n))
    for j in range(n):
        e = np.zeros(n)
        e[j] = 1e-5
        Hn[:, j] = (red(r.x + e)[1] - red(r.x - e)[1]) / 2e-5
    ref = np.linalg.inv(0.5 * (Hn + Hn.T))
    assert np.max(np.abs(cov - ref)) < 1e-5 * np.abs(ref).max()


def test_bad_arguments_and_domain_backoff(stub):
    start = np.full(2 * K, 0.5)
    assert run(stub, start, fixed=[K])[0] == 1                    # AMP_ERR_INVALID: slot out of range
    assert run(stub, start, ties=[(2, 2)])[0] == 1                # tie to itself
    assert run(stub, start, ties=[(2, 3), (3, 4)])[0] == 1        # chained ties
    assert run(stub, start, ties=[(2, 3), (2, 4)])[0] == 1        # one destination tied twice
    assert run(stub, start, fixed=[2], ties=[(2, 3)])[0] == 1     # a fixed slot as destination
    assert run(stub, start, ties=[(2, 3, 0)])[0] == 1             # sign must be +1 or -1
    assert run(stub, start, scale=np.zeros(K))[0] == 1            # non-positive scale
    assert run(stub, start, gtol=0.0)[0] == 1
    # max_iter = 0: no step, start returned, covariance at the start point still computed
    st, fit, nll, cov, info = run(stub, start, max_iter=0)
    assert st == 0 and info[0] == 0 and info[2] == 0 and np.array_equal(fit.ravel(), start)
    # a start next to a region without a likelihood (the stand-in refuses Re H_0 > 50): the search backs off and still converges
    far = start.copy()
    far[0] = 49.9
    st, fit, nll, cov, info = run(stub, far, cov=False)
    assert st == 0 and info[0] == 1 and abs(fit[0, 0] - 1.0) < 1e-6


def test_floating_mass_and_width(stub):
    """masses and widths as parameters: derivative by central differences of a batch, coupled to the couplings (the stand-in has
    cross terms M x Re H_0 and M x Gamma); minimum, covariance and the fixed-width variant against the closed form"""
    MS, GS, QA, QB, QC, QE = 4196.0, 370.0, 0.04, 0.01, 0.1, 0.005
    start = np.full(2 * K, 0.5)
    st, fit, nll, cov, info, fmw = run(stub, start, mw=(4230.0, 330.0), float_mw=[(0, 0), (0, 1)], gtol=1e-6)
    assert st == 0 and info[0] == 1 and info[3] == 1 and info[4] == 2 * K + 2
    assert abs(fmw[0, 0] - MS) < 1e-4 and abs(fmw[0, 1] - GS) < 1e-4
    assert np.max(np.abs(fit.ravel() - (1.0 + 0.1 * np.arange(2 * K)))) < 1e-6
    H = np.zeros((2 * K + 2, 2 * K + 2))
    H[:2 * K, :2 * K] = np.diag(lam(np.arange(2 * K))) + 0.3 * (np.eye(2 * K, k=1) + np.eye(2 * K, k=-1))
    H[2 * K, 2 * K], H[2 * K + 1, 2 * K + 1] = QA, QB
    H[2 * K, 0] = H[0, 2 * K] = QC
    H[2 * K, 2 * K + 1] = H[2 * K + 1, 2 * K] = QE
    ref = np.linalg.inv(H)
    assert np.max(np.abs(cov - ref) / np.sqrt(np.outer(np.diag(ref), np.diag(ref)))) < 1e-4
    # only the mass floats; the width stays at its (wrong) start value: the minimum in M shifts by -QE (G - G*) / QA (+ the H_0 coupling)
    st, fit, nll, cov, info, fmw = run(stub, start, mw=(4230.0, 330.0), float_mw=[(0, 0)], gtol=1e-6)
    assert st == 0 and info[0] == 1 and fmw[0, 1] == 330.0 and info[4] == 2 * K + 1
    from scipy.optimize import minimize

    def red(t):                                                   # (H, M) at G = 330, the stand-in's formula retyped in numpy
        f, g = f_and_grad(t[:2 * K])
        dM, dG, d0 = t[2 * K] * 100.0 - MS, 330.0 - GS, t[0] - 1.0
        f += 0.5 * QA * dM * dM + 0.5 * QB * dG * dG + QC * dM * d0 + QE * dM * dG
        g = np.append(g, (QA * dM + QC * d0 + QE * dG) * 100.0)
        g[0] += QC * dM
        return f, g

    r = minimize(red, np.append(fit.ravel(), 42.0), jac=True, method="BFGS", options={"gtol": 1e-10})
    assert abs(fmw[0, 0] - r.x[2 * K] * 100.0) < 1e-3 and abs(fmw[0, 0] - MS) > 1.0
    assert abs(nll[0] - r.fun) < 1e-8
    # bad specifications
    assert run(stub, start, mw=(4230.0, 330.0), float_mw=[(1, 0)])[0] == 1      # resonance index out of range
    assert run(stub, start, mw=(4230.0, 330.0), float_mw=[(0, 2)])[0] == 1
    assert run(stub, start, mw=(4230.0, 330.0), float_mw=[(0, 0), (0, 0)])[0] == 1
    assert run(stub, start, float_mw=[(0, 0)])[0] == 1                            # floating without start values
    # a start whose first steps would make the width negative: the stand-in refuses, the search backs off and still converges
    st, fit, nll, cov, info, fmw = run(stub, start, mw=(4230.0, 3.0), float_mw=[(0, 0), (0, 1)], gtol=1e-6, cov=False)
    assert st == 0 and info[0] == 1 and abs(fmw[0, 1] - GS) < 1e-3


def test_signed_ties_and_hessian_outside_the_domain(stub):
    """H[dst] = -H[src] (Eq. 11 for a 2+ or 1- Z): minimum of the reduced problem against scipy; a Hessian step that leaves the
    likelihood's domain (the stand-in refuses Re H_0 > 50) must clear the covariance flag instead of entering the matrix"""
    start = np.full(2 * K, 0.5)
    ties = [(5, 3, -1), (7, 2, 1)]
    st, fit, nll, cov, info = run(stub, start, ties=ties)
    assert st == 0 and info[0] == 1 and info[3] == 1
    assert np.array_equal(fit[5], -fit[3]) and np.array_equal(fit[7], fit[2])
    free = [k for k in range(K) if k not in (5, 7)]

    def red(t):
        h = np.zeros((K, 2))
        h[free] = t.reshape(-1, 2)
        h[5], h[7] = -h[3], h[2]
        f, g = f_and_grad(h.ravel())
        g = g.reshape(K, 2).copy()
        g[3] -= g[5]
        g[2] += g[7]
        return f, g[free].ravel()

    from scipy.optimize import minimize
    r = minimize(red, start.reshape(K, 2)[free].ravel(), jac=True, method="BFGS", options={"gtol": 1e-9})
    assert abs(nll[0] - r.fun) < 1e-9 * max(1.0, abs(r.fun)) and np.max(np.abs(fit[free].ravel() - r.x)) < 1e-6
    # at the known minimum with a huge scale on slot 0: the Hessian's +h step puts Re H_0 at 1 + 100 > 50
    target = 1.0 + 0.1 * np.arange(2 * K)
    scale = np.ones(K)
    scale[0] = 1e6
    st, fit, nll, cov, info = run(stub, target, scale=scale, max_iter=0)
    assert st == 0 and info[3] == 0 and np.all(np.isnan(cov))

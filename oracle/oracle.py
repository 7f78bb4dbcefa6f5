"""ctypes front end of oracle/amp_oracle.cpp — TEST INFRASTRUCTURE (see oracle/__init__.py).

Every function is a thin marshalling wrapper; all arithmetic lives in amp_oracle.cpp, which cites
the PAPER.md passage each step follows.
"""
import ctypes as C
import numpy as np

from .build import build as _build

_lib = C.CDLL(_build())

_d, _i, _ll = C.c_double, C.c_int, C.c_longlong
_pd = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
_pi = np.ctypeslib.ndpointer(dtype=np.int32, flags="C_CONTIGUOUS")
_vp = C.c_void_p

_lib.orc_num_threads.restype = _i
_lib.orc_set_num_threads.argtypes = [_i]
_lib.orc_breakup_momentum.restype = _d
_lib.orc_breakup_momentum.argtypes = [_d, _d, _d, _i]
_lib.orc_barrier_polynomial.restype = _d
_lib.orc_barrier_polynomial.argtypes = [_i, _d]
_lib.orc_blatt_weisskopf.restype = _d
_lib.orc_blatt_weisskopf.argtypes = [_i, _d, _d, _d]
_lib.orc_wigner_d.restype = _d
_lib.orc_wigner_d.argtypes = [_i, _i, _i, _d, _i]
_lib.orc_orbital_L.argtypes = [_i, _i, C.POINTER(_i), C.POINTER(_i)]
_lib.orc_lineshape.argtypes = [_pd, _i, _i, _d, _d, _d, _d, _i, _pd]
_lib.orc_z_kinematics.argtypes = [_pd, _pd, _i, _pd]
_lib.orc_lineshape_at_event.argtypes = [_pd, _i, _i, _d, _d, _d, _pd, _i, _pd]
_lib.orc_num_couplings.restype = _i
_lib.orc_num_couplings.argtypes = [_i, _pi, _pi]
_MODEL = [_pd, _i, _pi, _pi, _pd, _pd, _pd]
_lib.orc_basis_terms.argtypes = _MODEL + [_pd, _i, _pd]
_lib.orc_eval_events.argtypes = _MODEL + [_pd, _pd, _vp, _ll, _i, _pd]
_lib.orc_nll.restype = _i
_lib.orc_nll.argtypes = _MODEL + [_i, _pd, _vp, _pd, _vp, _ll, _pd, _vp, _ll, _i, _vp, _vp]
_lib.orc_norm_matrix.argtypes = _MODEL + [_pd, _vp, _ll, _pd]
_lib.orc_nll_gradient.argtypes = _MODEL + [_pd, _pd, _vp, _ll, _pd, _vp, _ll, _pd, _pd]
_lib.orc_nll_gradient_bkg.argtypes = _MODEL + [_pd, _pd, _vp, _pd, _d, _ll, _pd, _vp, _ll, _pd, _pd]

KSTAR, ZRES, CONST, LASS, ZNEG = 0, 1, 2, 3, 4


def num_threads():
    return _lib.orc_num_threads()


def set_num_threads(n):
    _lib.orc_set_num_threads(int(n))


def breakup_momentum(M, a, b, prec=0):
    return _lib.orc_breakup_momentum(M, a, b, prec)


def barrier_polynomial(L, z):
    return _lib.orc_barrier_polynomial(L, z)


def blatt_weisskopf(L, p, p0, r):
    return _lib.orc_blatt_weisskopf(L, p, p0, r)


def wigner_d(j, mp, m, beta, prec=0):
    return _lib.orc_wigner_d(j, mp, m, beta, prec)


def orbital_L(kind, J):
    a, b = _i(), _i()
    _lib.orc_orbital_L(kind, J, C.byref(a), C.byref(b))
    return a.value, b.value


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _opt(a):
    """optional float64 array -> (keepalive, void*)"""
    if a is None:
        return None, None
    a = _f64(a)
    return a, a.ctypes.data_as(_vp)


class Model:
    """Decay constants + resonance list, as plain arrays (same fields as include/amp.h)."""

    def __init__(self, decay, resonances):
        # decay = (m_parent, m_psi, m_k, m_pi); resonances = [(kind, J, mass, width, radius), ...]
        self.decay = _f64(decay)
        self.kinds = np.ascontiguousarray([r[0] for r in resonances], dtype=np.int32)
        self.Js = np.ascontiguousarray([r[1] for r in resonances], dtype=np.int32)
        self.mass = _f64([r[2] for r in resonances])
        self.width = _f64([r[3] for r in resonances])
        self.radius = _f64([r[4] for r in resonances])
        self.R = len(resonances)
        self.K = _lib.orc_num_couplings(self.R, self.kinds, self.Js)

    def _args(self):
        return [self.decay, self.R, self.kinds, self.Js, self.mass, self.width, self.radius]

    def lineshape(self, r, m, prec=0):
        """(A^R(m) complex, Gamma(m)) of resonance index r at running mass m."""
        out = np.zeros(3)
        _lib.orc_lineshape(self.decay, int(self.kinds[r]), int(self.Js[r]), self.mass[r], self.width[r], self.radius[r],
                           float(m), prec, out)
        return complex(out[0], out[1]), out[2]

    def lineshape_at_event(self, r, x, prec=0):
        """A^R of resonance r at the event x = (m_Kpi, cosK, cosPsi, phi): its chain's running mass is formed in the working
        precision (prec=1: long double) and never rounded to double on the way to the lineshape."""
        out = np.zeros(3)
        _lib.orc_lineshape_at_event(self.decay, int(self.kinds[r]), int(self.Js[r]), self.mass[r], self.width[r], self.radius[r],
                                    _f64(x), prec, out)
        return complex(out[0], out[1])

    def z_kinematics(self, x, prec=0):
        out = np.zeros(31)
        _lib.orc_z_kinematics(self.decay, _f64(x), prec, out)
        names = ["mZ", "cosZ", "sinZ", "cosT", "sinT", "phiT", "alpha"]
        d = {k: out[i] for i, k in enumerate(names)}
        d["K_B"], d["pi_B"], d["psi_B"] = out[7:11].copy(), out[11:15].copy(), out[15:19].copy()
        d["nK"], d["npi"], d["nKst"], d["nmu"] = out[19:22].copy(), out[22:25].copy(), out[25:28].copy(), out[28:31].copy()
        return d

    def basis_terms(self, x, prec=0):
        """complex array [K][2]: B_{k,xi} of one event, xi = +1 then -1."""
        out = np.zeros((self.K, 2, 2))
        _lib.orc_basis_terms(*self._args(), _f64(x), prec, out)
        return out[..., 0] + 1j * out[..., 1]

    def eval_events(self, couplings, x, eff=None, prec=0):
        """v_i = eff_i * S_i; x is SoA [4][n]; couplings complex [K]."""
        x = _f64(x)
        n = x.shape[1]
        c = _f64(np.stack([np.real(couplings), np.imag(couplings)], -1))
        assert c.shape == (self.K, 2)
        ka, pe = _opt(eff)
        out = np.zeros(n)
        _lib.orc_eval_events(*self._args(), c, x, pe, n, prec, out)
        return out

    def nll(self, couplings, x, eff, xn, wn, mass_width=None, prec=0, want_nll=True):
        """(NLL[P], I[P]) for couplings complex [P][K] (or [K]); mass_width [P][R][2] or None."""
        cc = np.asarray(couplings)
        if cc.ndim == 1:
            cc = cc[None]
        P = cc.shape[0]
        c = _f64(np.stack([cc.real, cc.imag], -1))
        assert c.shape == (P, self.K, 2)
        kmw, pmw = _opt(mass_width)
        if kmw is not None:
            assert kmw.shape == (P, self.R, 2)
        x, xn = _f64(x), _f64(xn)
        ke, pe = _opt(eff)
        kw, pw = _opt(wn)
        nll, I = np.zeros(P), np.zeros(P)
        _lib.orc_nll(*self._args(), P, c, pmw, x, pe, x.shape[1], xn, pw, xn.shape[1], prec,
                     nll.ctypes.data_as(_vp) if want_nll else None, I.ctypes.data_as(_vp))
        return nll, I

    def norm_integral(self, couplings, xn, wn, mass_width=None, prec=0):
        return self.nll(couplings, np.zeros((4, 0)), None, xn, wn, mass_width, prec, want_nll=False)[1]

    def nll_gradient(self, couplings, x, eff, xn, wn):
        """(NLL, grad [K][2]) with grad[k] = (dNLL/dRe c_k, dNLL/dIm c_k): the derivative of the NLL written out event by event."""
        c = _f64(np.stack([np.real(couplings), np.imag(couplings)], -1))
        assert c.shape == (self.K, 2)
        x, xn = _f64(x), _f64(xn)
        ke, pe = _opt(eff)
        kw, pw = _opt(wn)
        nll, grad = np.zeros(1), np.zeros((self.K, 2))
        _lib.orc_nll_gradient(*self._args(), c, x, pe, x.shape[1], xn, pw, xn.shape[1], nll, grad)
        return nll[0], grad

    def nll_gradient_background(self, couplings, x, eff, bkg, purity, xn, wn):
        """(NLL, grad [K][2]) of Eq. 14 (background + purity), the derivative written out event by event"""
        c = _f64(np.stack([np.real(couplings), np.imag(couplings)], -1))
        assert c.shape == (self.K, 2)
        x, xn, bkg = _f64(x), _f64(xn), _f64(bkg)
        ke, pe = _opt(eff)
        kw, pw = _opt(wn)
        nll, grad = np.zeros(1), np.zeros((self.K, 2))
        _lib.orc_nll_gradient_bkg(*self._args(), c, x, pe, bkg, float(purity), x.shape[1], xn, pw, xn.shape[1], nll, grad)
        return nll[0], grad

    def nll_background(self, couplings, x, eff, bkg, purity, xn, wn, mass_width=None):
        """Eq. 14: NLL(p) = -sum_i log f_i, f_i = purity * eps_i S_i / I + (1 - purity) * b_i, with the signal
        part normalised by the Monte Carlo integral I = sum_j w_j S_j / sum_j w_j and b_i the (normalised) background density
        at the data events, supplied by the caller.  Plain definition, exact summation (math.fsum).  couplings [P][K] or [K]."""
        import math
        cc = np.asarray(couplings)
        if cc.ndim == 1:
            cc = cc[None]
        bkg = _f64(bkg)
        out = np.zeros(cc.shape[0])
        for p in range(cc.shape[0]):
            M = self
            if mass_width is not None:
                mw = np.asarray(mass_width, dtype=np.float64).reshape(cc.shape[0], self.R, 2)[p]
                M = Model(self.decay, [(int(self.kinds[r]), int(self.Js[r]), mw[r, 0], mw[r, 1], self.radius[r]) for r in range(self.R)])
            I = M.norm_integral(cc[p], xn, wn)[0]
            v = M.eval_events(cc[p], x, eff)                       # eps_i S_i
            f = purity * v / I + (1.0 - purity) * bkg
            out[p] = -math.fsum(np.log(f)) if np.all(f > 0) else np.inf
        return out

    def fit_fractions(self, couplings, xn, wn, mass_width=None, groups=None):
        """Eq. 13 by its plain definition: FF_j = sum_n w_n S_j(x_n) / sum_n w_n S(x_n), where S_j is the density
        with every helicity amplitude except those of resonance j set to zero ("setting to zero all the other helicity
        amplitudes").  groups: optional list of lists of resonance indices (a fraction per group instead of per resonance)."""
        c = np.asarray(couplings, dtype=np.complex128)
        assert c.shape == (self.K,)
        slot_res = []
        for r in range(self.R):
            three = self.kinds[r] in (ZRES, ZNEG) or (self.kinds[r] == KSTAR and self.Js[r] >= 1)
            slot_res += [r] * (3 if three else 1)
        slot_res = np.array(slot_res)
        groups = [[r] for r in range(self.R)] if groups is None else groups
        mw = None if mass_width is None else np.asarray(mass_width, dtype=np.float64).reshape(1, self.R, 2)
        total = self.norm_integral(c, xn, wn, mw)[0]
        return np.array([self.norm_integral(np.where(np.isin(slot_res, g), c, 0.0), xn, wn, mw)[0] / total for g in groups])

    def norm_matrix(self, xn, wn):
        xn = _f64(xn)
        kw, pw = _opt(wn)
        out = np.zeros((self.K, self.K, 2))
        _lib.orc_norm_matrix(*self._args(), xn, pw, xn.shape[1], out)
        return out[..., 0] + 1j * out[..., 1]

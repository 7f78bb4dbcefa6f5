"""Thin ctypes binding of libamp4d.so (include/amp.h): argument marshalling only.

Same names as the C ABI.  torch is used for device memory and streams; every step of the path runs in
the library's CUDA kernels.  There is no fallback: a missing library or a failing call raises.
"""
import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libamp4d.so")   # built in-tree by paper_2007_14931_b200/build.py

AMP_OK, AMP_ERR_INVALID, AMP_ERR_STATE, AMP_ERR_DOMAIN, AMP_ERR_CUDA, AMP_ERR_NOMEM = range(6)
AMP_KSTAR, AMP_Z, AMP_CONST, AMP_LASS, AMP_ZM = 0, 1, 2, 3, 4
AMP_MAX_RESONANCES, AMP_MAX_COUPLINGS, AMP_MAX_POINTS = 16, 48, 256
AMP_STATIC_MAX_POINTS, AMP_STATIC_MAX_CTAS = 8, 1024

# every symbol include/amp.h declares (tests/test_abi.py checks the header against this list and the .so)
SYMBOLS = [
    "amp_model_create", "amp_model_destroy", "amp_num_couplings", "amp_num_resonances", "amp_load_events",
    "amp_load_norm", "amp_set_background", "amp_set_params", "amp_nll", "amp_nll_static", "amp_nll_grad", "amp_fit", "amp_generate", "amp_nll_terms", "amp_dataset_sums", "amp_eval_events", "amp_norm_integral", "amp_dump_cache",
    "amp_cache_column_name", "amp_eval_lineshape", "amp_norm_matrix", "amp_fit_fractions", "amp_set_norm_mode", "amp_set_lineshape_mode", "amp_set_batch_mode", "amp_set_fused_mode", "amp_set_grad_mode",
    "amp_last_call_stats", "amp_last_call_timing", "amp_recent_launch_ms", "amp_last_error", "amp_status_string", "amp_version", "amp_probe_fp64", "amp_probe_hbm_read",
]


class amp_resonance(C.Structure):
    _fields_ = [("kind", C.c_int), ("J", C.c_int), ("mass", C.c_double), ("width", C.c_double), ("radius", C.c_double)]


class amp_decay(C.Structure):
    _fields_ = [("m_parent", C.c_double), ("m_psi", C.c_double), ("m_k", C.c_double), ("m_pi", C.c_double)]


class AmpError(RuntimeError):
    def __init__(self, status, text):
        super().__init__(f"{text}")
        self.status = status


_lib = None


def lib():
    """Load libamp4d.so (built by paper_2007_14931_b200.build); raises if it is missing — no fallback."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} not built: run `python -m paper_2007_14931_b200.build` (needs nvcc); "
                          "there is no CPU fallback")
    L = C.CDLL(LIB_PATH)
    vp, i, ll, d = C.c_void_p, C.c_int, C.c_longlong, C.c_double
    pd, pi = C.POINTER(C.c_double), C.POINTER(C.c_int)
    sig = {
        "amp_model_create": (i, [C.POINTER(amp_decay), C.POINTER(amp_resonance), i, C.POINTER(vp)]),
        "amp_model_destroy": (i, [vp]),
        "amp_num_couplings": (i, [vp]),
        "amp_num_resonances": (i, [vp]),
        "amp_load_events": (i, [vp, vp, vp, ll, vp]),
        "amp_load_norm": (i, [vp, vp, vp, ll, vp]),
        "amp_set_background": (i, [vp, vp, d, vp]),
        "amp_set_params": (i, [vp, i, vp, vp]),
        "amp_nll": (i, [vp, vp, vp]),
        "amp_nll_static": (i, [vp, vp, vp]),
        "amp_nll_grad": (i, [vp, vp, vp, vp]),
        "amp_fit": (i, [vp, vp, vp, vp, i, vp, vp, vp, i, vp, i, vp, i, d, vp, vp, vp, vp, vp, vp]),
        "amp_generate": (i, [vp, C.c_ulonglong, C.c_ulonglong, ll, d, d, d, d, vp, vp, ll, C.POINTER(ll), pd, vp]),
        "amp_nll_terms": (i, [vp, vp, vp, vp]),
        "amp_dataset_sums": (i, [vp, C.POINTER(ll), pd, C.POINTER(ll), pd]),
        "amp_eval_events": (i, [vp, i, vp, vp]),
        "amp_norm_integral": (i, [vp, vp, vp]),
        "amp_dump_cache": (i, [vp, i, vp, pi, vp]),
        "amp_cache_column_name": (C.c_char_p, [i]),
        "amp_eval_lineshape": (i, [vp, i, i, d, d, vp, vp]),
        "amp_norm_matrix": (i, [vp, i, vp, vp]),
        "amp_fit_fractions": (i, [vp, i, vp, vp]),
        "amp_set_norm_mode": (i, [vp, i]),
        "amp_set_lineshape_mode": (i, [vp, i]),
        "amp_set_batch_mode": (i, [vp, i]),
        "amp_set_fused_mode": (i, [vp, i]),
        "amp_set_grad_mode": (i, [vp, i]),
        "amp_last_call_stats": (i, [vp, pi, pi, pi]),
        "amp_last_call_timing": (i, [vp, pd]),
        "amp_recent_launch_ms": (i, [vp, i, pd, pi]),
        "amp_last_error": (C.c_char_p, [vp]),
        "amp_status_string": (C.c_char_p, [i]),
        "amp_version": (C.c_char_p, []),
        "amp_probe_fp64": (i, [i, i, pd, vp]),
        "amp_probe_hbm_read": (i, [C.c_longlong, pd, vp]),
    }
    for name, (res, args) in sig.items():
        f = getattr(L, name)
        f.restype, f.argtypes = res, args
    _lib = L
    return L


def _stream_ptr(stream):
    if stream is None:
        import torch
        return C.c_void_p(torch.cuda.current_stream().cuda_stream)
    return C.c_void_p(getattr(stream, "cuda_stream", stream))


def _dev_ptr(t, n_expected=None):
    """device pointer of a contiguous float64 CUDA tensor (or None)"""
    if t is None:
        return None
    import torch
    assert isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous(), \
        "expected a contiguous float64 CUDA tensor"
    if n_expected is not None:
        assert t.numel() == n_expected, f"expected {n_expected} elements, got {t.numel()}"
    return C.c_void_p(t.data_ptr())


class Model:
    """amp_model handle.  Methods mirror the C calls one to one."""

    def __init__(self, decay, resonances):
        """decay = (m_parent, m_psi, m_k, m_pi); resonances = [(kind, J, mass, width, radius), ...]"""
        L = lib()
        self._h = C.c_void_p()
        dec = amp_decay(*[float(v) for v in decay])
        arr = (amp_resonance * len(resonances))(*[amp_resonance(int(k), int(J), float(m), float(w), float(r)) for k, J, m, w, r in resonances])
        st = L.amp_model_create(C.byref(dec), arr, len(resonances), C.byref(self._h))
        if st != AMP_OK:
            self._h = C.c_void_p()
            raise AmpError(st, f"amp_model_create: {L.amp_status_string(st).decode()}")
        self.K = L.amp_num_couplings(self._h)
        self.R = L.amp_num_resonances(self._h)
        self.P = 0
        self.n = self.n_norm = 0

    def _check(self, st, what):
        if st != AMP_OK:
            L = lib()
            raise AmpError(st, f"{what}: {L.amp_status_string(st).decode()}: {L.amp_last_error(self._h).decode()}")

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            lib().amp_model_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # --- loading ---------------------------------------------------------------------------------
    def load_events(self, d_x, d_eff=None, stream=None):
        n = d_x.shape[1] if d_x.dim() == 2 else d_x.numel() // 4
        self._check(lib().amp_load_events(self._h, _dev_ptr(d_x, 4 * n), _dev_ptr(d_eff, n if d_eff is not None else None), n,
                                          _stream_ptr(stream)), "amp_load_events")
        self.n = n

    def load_norm(self, d_x, d_w=None, stream=None):
        n = d_x.shape[1] if d_x.dim() == 2 else d_x.numel() // 4
        self._check(lib().amp_load_norm(self._h, _dev_ptr(d_x, 4 * n), _dev_ptr(d_w, n if d_w is not None else None), n,
                                        _stream_ptr(stream)), "amp_load_norm")
        self.n_norm = n

    def set_background(self, d_bkg, purity, stream=None):
        """Eq. 14: background density at the data events (float64 CUDA tensor [n], or None to switch it off) and the purity"""
        self._check(lib().amp_set_background(self._h, _dev_ptr(d_bkg, self.n) if d_bkg is not None else None, float(purity),
                                             _stream_ptr(stream)), "amp_set_background")
        self.P = 0

    # --- parameters ------------------------------------------------------------------------------
    def set_params(self, couplings, mass_width=None):
        """couplings: complex [K] or [P][K] (host); mass_width: [P][R][2] (host) or None"""
        c = np.asarray(couplings)
        if c.ndim == 1:
            c = c[None]
        P = c.shape[0]
        assert c.shape == (P, self.K), f"couplings must be [P][{self.K}]"
        hc = np.ascontiguousarray(c, dtype=np.complex128).view(np.float64)      # [P][K][re, im]
        pmw = None
        if mass_width is not None:
            hmw = np.ascontiguousarray(mass_width, dtype=np.float64)
            if hmw.ndim == 2:
                hmw = hmw[None]
            assert hmw.shape == (P, self.R, 2), f"mass_width must be [P][{self.R}][2]"
            pmw = hmw.ctypes.data_as(C.c_void_p)
        self._check(lib().amp_set_params(self._h, P, hc.ctypes.data_as(C.c_void_p), pmw), "amp_set_params")
        self.P = P

    # --- evaluation ------------------------------------------------------------------------------
    def nll(self, stream=None, allow_domain_error=False):
        out = np.empty(max(self.P, 1), dtype=np.float64)
        st = lib().amp_nll(self._h, out.ctypes.data_as(C.c_void_p), _stream_ptr(stream))
        if not (allow_domain_error and st == AMP_ERR_DOMAIN):
            self._check(st, "amp_nll")
        return out[:self.P]

    def nll_static(self, out, stream=None):
        """amp_nll_static: the fused launch(es) with the kernel's scratch in the library's static device array (no allocation, no copy,
        no synchronisation).  `out`: caller-owned float64 CUDA tensor [P][6] = (NLL, I, domain flag, sum log S, sum w S, 1.0) per point;
        P <= AMP_STATIC_MAX_POINTS.  Calls that overlap on the GPU race on the shared array."""
        self._check(lib().amp_nll_static(self._h, _dev_ptr(out, 6 * max(self.P, 1)), _stream_ptr(stream)), "amp_nll_static")
        return out

    def nll_grad(self, stream=None):
        """(NLL, grad [K][2] = (dNLL/dRe H_k, dNLL/dIm H_k)) at the single point set by set_params"""
        nll, grad = np.empty(1), np.empty((self.K, 2))
        self._check(lib().amp_nll_grad(self._h, nll.ctypes.data_as(C.c_void_p), grad.ctypes.data_as(C.c_void_p), _stream_ptr(stream)), "amp_nll_grad")
        return nll[0], grad

    def fit(self, c_start, fixed=(), ties=(), mass_width=None, float_mw=(), scale=None, max_iter=3000, gtol=1e-3, errors=False, stream=None):
        """native BFGS fit (amp_fit) of the couplings and, for float_mw = [(resonance, 0 mass | 1 width), ...], of masses and widths
        -> dict(couplings [K] complex, mass_width [R][2] or None, nll, grad_max, converged, n_calls, iterations, free (slots),
        covariance [n][n] or None (n = 2 F + len(float_mw)), errors complex [F] or None, mw_errors [len(float_mw)] or None)"""
        c = np.asarray(c_start, dtype=np.complex128)
        assert c.shape == (self.K,)
        hc = np.ascontiguousarray(np.stack([c.real, c.imag], -1))
        hmw = None if mass_width is None else np.ascontiguousarray(np.asarray(mass_width, dtype=np.float64).reshape(self.R, 2))
        fx = np.ascontiguousarray(list(fixed), dtype=np.int32)
        td = np.ascontiguousarray([t[0] for t in ties], dtype=np.int32)
        ts = np.ascontiguousarray([t[1] for t in ties], dtype=np.int32)
        tg = np.ascontiguousarray([t[2] if len(t) > 2 else 1 for t in ties], dtype=np.int32)   # (dst, src) or (dst, src, +-1)
        fm = np.ascontiguousarray([[int(r), int(w)] for r, w in float_mw], dtype=np.int32).reshape(-1, 2)
        hs = None if scale is None else np.ascontiguousarray(scale, dtype=np.float64)
        free = [k for k in range(self.K) if k not in set(int(f) for f in fixed) and k not in set(int(t) for t in td)]
        n = 2 * len(free) + len(fm)
        out, nll, info = np.empty((self.K, 2)), np.empty(2), np.zeros(5, dtype=np.int32)
        out_mw = np.empty((self.R, 2)) if hmw is not None else None
        cov = np.empty((n, n)) if errors else None
        p = lambda a: a.ctypes.data_as(C.c_void_p) if a is not None and a.size else None
        self._check(lib().amp_fit(self._h, p(hc), p(hmw), p(fx), len(fx), p(td), p(ts), p(tg), len(td), p(fm), len(fm), p(hs), int(max_iter), float(gtol),
                                  p(out), p(out_mw), p(nll), p(cov), p(info), _stream_ptr(stream)), "amp_fit")
        self.P = 1
        res = {"couplings": out[:, 0] + 1j * out[:, 1], "mass_width": out_mw, "nll": float(nll[0]), "grad_max": float(nll[1]),
               "converged": bool(info[0]), "n_calls": int(info[1]), "iterations": int(info[2]), "free": free, "covariance": cov,
               "errors": None, "mw_errors": None}
        if errors and info[3]:
            sig = np.sqrt(np.diag(cov))
            res["errors"] = sig[:2 * len(free):2] + 1j * sig[1:2 * len(free):2]
            res["mw_errors"] = sig[2 * len(free):]
        return res

    def generate(self, seed, first, n_candidates, f_max, m_lo, m_hi, cos_max, capacity, with_index=False, stream=None):
        """accept-reject toy block (amp_generate): -> (x_out cuda [4][capacity], index cuda [capacity] or None, n_accepted, f_seen_max);
        only the first min(n_accepted, capacity) columns are meaningful"""
        import torch
        x_out = torch.empty((4, max(capacity, 1)), dtype=torch.float64, device="cuda")[:, :capacity]
        idx = torch.empty(max(capacity, 1), dtype=torch.int64, device="cuda")[:capacity] if with_index else None
        nacc, fseen = C.c_longlong(), C.c_double()
        self._check(lib().amp_generate(self._h, int(seed), int(first), int(n_candidates), float(f_max), float(m_lo), float(m_hi), float(cos_max),
                                       C.c_void_p(x_out.data_ptr()) if capacity else None, C.c_void_p(idx.data_ptr()) if (with_index and capacity) else None,
                                       int(capacity), C.byref(nacc), C.byref(fseen), _stream_ptr(stream)), "amp_generate")
        return x_out, idx, nacc.value, fseen.value

    def generate_toy(self, n_events, seed, m_lo, m_hi, cos_max, f_max=None, block=1 << 22, safety=1.5):
        """n_events toy events [4][n_events] (cuda), the first n_events accepted candidates of the stream `seed`.
        f_max None: taken as safety x the largest weight among the first 2^18 candidates (a pilot pass that writes nothing);
        returns (x, n_candidates_used, f_max, f_seen_max) — f_seen_max > f_max means the envelope was too low"""
        import torch
        if f_max is None:
            _, _, _, fs = self.generate(seed, 0, 1 << 18, 0.0, m_lo, m_hi, cos_max, 0)
            f_max = safety * fs
        out = torch.empty((4, n_events), dtype=torch.float64, device="cuda")
        have, first, fseen = 0, 0, 0.0
        while have < n_events:
            x, _, nacc, fs = self.generate(seed, first, block, f_max, m_lo, m_hi, cos_max, n_events - have)
            take = min(nacc, n_events - have)
            out[:, have:have + take] = x[:, :take]
            have += take
            fseen = max(fseen, fs)
            if have < n_events:
                first += block
            if nacc == 0 and first > (1 << 40):
                raise AmpError("generate_toy: nothing accepted")
        return out, first + block, f_max, fseen

    def nll_terms(self, stream=None):
        """(sum_i log S_i(p), sum_j w_j S_j(p)) of this model's own events, [P] each: the per-shard sums behind nll()"""
        a, b = np.empty(max(self.P, 1)), np.empty(max(self.P, 1))
        self._check(lib().amp_nll_terms(self._h, a.ctypes.data_as(C.c_void_p), b.ctypes.data_as(C.c_void_p), _stream_ptr(stream)), "amp_nll_terms")
        return a[:self.P], b[:self.P]

    def dataset_sums(self):
        """(n_data, sum_i log eps_i, n_norm, sum_j w_j)"""
        n, m, sl, sw = C.c_longlong(), C.c_longlong(), C.c_double(), C.c_double()
        self._check(lib().amp_dataset_sums(self._h, C.byref(n), C.byref(sl), C.byref(m), C.byref(sw)), "amp_dataset_sums")
        return n.value, sl.value, m.value, sw.value

    def norm_integral(self, stream=None):
        out = np.empty(max(self.P, 1), dtype=np.float64)
        self._check(lib().amp_norm_integral(self._h, out.ctypes.data_as(C.c_void_p), _stream_ptr(stream)), "amp_norm_integral")
        return out[:self.P]

    def eval_events(self, p=0, out=None, stream=None):
        import torch
        if out is None:
            out = torch.empty(self.n, dtype=torch.float64, device="cuda")
        self._check(lib().amp_eval_events(self._h, int(p), _dev_ptr(out, self.n) if self.n else None, _stream_ptr(stream)), "amp_eval_events")
        return out

    def dump_cache(self, which=0, stream=None):
        import torch
        nc = C.c_int(0)
        self._check(lib().amp_dump_cache(self._h, which, None, C.byref(nc), _stream_ptr(stream)), "amp_dump_cache")
        n = self.n_norm if which else self.n
        out = torch.empty((nc.value, n), dtype=torch.float64, device="cuda")
        self._check(lib().amp_dump_cache(self._h, which, _dev_ptr(out), C.byref(nc), _stream_ptr(stream)), "amp_dump_cache")
        names = [lib().amp_cache_column_name(i).decode() for i in range(nc.value)]
        return names, out

    def eval_lineshape(self, r, mass, width, which=0, stream=None):
        import torch
        n = self.n_norm if which else self.n
        out = torch.empty((n, 2), dtype=torch.float64, device="cuda")
        self._check(lib().amp_eval_lineshape(self._h, which, int(r), float(mass), float(width), _dev_ptr(out), _stream_ptr(stream)),
                    "amp_eval_lineshape")
        return out

    def norm_matrix(self, p=0, stream=None):
        out = np.empty((self.K, self.K, 2), dtype=np.float64)
        self._check(lib().amp_norm_matrix(self._h, int(p), out.ctypes.data_as(C.c_void_p), _stream_ptr(stream)), "amp_norm_matrix")
        return out[..., 0] + 1j * out[..., 1]

    def fit_fractions(self, p=0, stream=None):
        out = np.empty(self.R, dtype=np.float64)
        self._check(lib().amp_fit_fractions(self._h, int(p), out.ctypes.data_as(C.c_void_p), _stream_ptr(stream)), "amp_fit_fractions")
        return out

    def set_norm_mode(self, mode):
        self._check(lib().amp_set_norm_mode(self._h, int(mode)), "amp_set_norm_mode")

    def set_lineshape_mode(self, mode):
        self._check(lib().amp_set_lineshape_mode(self._h, int(mode)), "amp_set_lineshape_mode")

    def set_batch_mode(self, mode):
        self._check(lib().amp_set_batch_mode(self._h, int(mode)), "amp_set_batch_mode")

    def set_fused_mode(self, mode):
        self._check(lib().amp_set_fused_mode(self._h, int(mode)), "amp_set_fused_mode")

    def set_grad_mode(self, mode):
        self._check(lib().amp_set_grad_mode(self._h, int(mode)), "amp_set_grad_mode")

    def last_call_stats(self):
        a, b, c = C.c_int(), C.c_int(), C.c_int()
        self._check(lib().amp_last_call_stats(self._h, C.byref(a), C.byref(b), C.byref(c)), "amp_last_call_stats")
        return {"launches": a.value, "columns_recomputed": b.value, "norm_path": c.value}


    def last_call_timing(self):
        ms = (C.c_double * 4)()
        self._check(lib().amp_last_call_timing(self._h, ms), "amp_last_call_timing")
        return {"lineshape_ms": ms[0], "data_ms": ms[1], "norm_ms": ms[2], "final_ms": ms[3]}


def _recent_launch_ms(self, max_calls=256):
    """device ms of the launches of the most recent fused / gradient-batch evaluations, oldest first"""
    buf = (C.c_double * max(max_calls, 1))()
    n = C.c_int(0)
    self._check(lib().amp_recent_launch_ms(self._h, int(max_calls), buf, C.byref(n)), "amp_recent_launch_ms")
    return np.array(buf[:n.value])


Model.recent_launch_ms = _recent_launch_ms


def probe_fp64(kind, iters=2000, stream=None):
    out = C.c_double(0)
    st = lib().amp_probe_fp64(int(kind), int(iters), C.byref(out), _stream_ptr(stream))
    if st != AMP_OK:
        raise AmpError(st, "amp_probe_fp64 failed")
    return out.value


def probe_hbm_read(nbytes=2_208_000_000, stream=None):
    """GB/s of k_stream's tile pipeline reading `nbytes` of scratch with no model arithmetic (amp_probe_hbm_read)."""
    out = C.c_double(0)
    st = lib().amp_probe_hbm_read(int(nbytes), C.byref(out), _stream_ptr(stream))
    if st != AMP_OK:
        raise AmpError(st, "amp_probe_hbm_read failed")
    return out.value


def version():
    return lib().amp_version().decode()

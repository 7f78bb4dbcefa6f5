"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs.

Bars (BASELINE.json north_star): per-event eps*|A|^2 within 1e-11 relative, NLL within 1e-9 relative.
Sizes span several tiles and a ragged tail (n not a multiple of 32 or 256).
"""
import math

import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import oracle as O
from paper_2007_14931_b200 import workloads as W

pytestmark = pytest.mark.gpu

RTOL_EVENT = 1e-11
RTOL_NLL = 1e-9


def dev(a):
    return torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64).cuda()


def gpu_model(cfg):
    from paper_2007_14931_b200 import binding as B
    return B.Model(W.DECAY, W.resonances(cfg))


def oracle_model(cfg):
    return O.Model(W.DECAY, W.resonances(cfg))


def make_inputs(cfg, n, m):
    """seeded data (accept-reject driven by the ORACLE) and norm events"""
    Mo = oracle_model(cfg)
    c = W.couplings(cfg)
    xn, wn = W.norm_events(cfg, m)
    x, eff = W.data_events(cfg, lambda xx, ee: Mo.eval_events(c, xx, ee), n=n)
    return x, eff, xn, wn


# ---------------------------------------------------------------------------------------------------
def _cache_reference(Mo, x, prec):
    """every cached quantity of one event by the oracle's explicit 4-vector route (prec = 1: its long double twin)"""
    MB, mpsi, mK, mpi = W.DECAY
    k = Mo.z_kinematics(x, prec=prec)
    m = x[0]
    return {
        "m2": m * m, "inv_m": 1 / m, "q": O.breakup_momentum(m, mK, mpi, prec), "pB": O.breakup_momentum(MB, m, mpsi, prec),
        "cosK": x[1], "sinK": math.sqrt((1 - x[1]) * (1 + x[1])), "cosPsi": x[2],
        "sinPsi": math.sqrt((1 - x[2]) * (1 + x[2])), "cosPhi": math.cos(x[3]), "sinPhi": math.sin(x[3]),
        "mZ2": k["mZ"] ** 2, "inv_mZ": 1 / k["mZ"], "cosZ": k["cosZ"], "sinZ": k["sinZ"], "cosT": k["cosT"], "sinT": k["sinT"],
        "cosPhiT": math.cos(k["phiT"]), "sinPhiT": math.sin(k["phiT"]), "cosAlpha": math.cos(k["alpha"]), "sinAlpha": math.sin(k["alpha"]),
    }


def test_kinematics_cache_matches_oracle_boosts():
    """a1: every cached quantity against the oracle's explicit 4-vector route (independent derivations), arbitrated by the
    oracle's long double twin: 1e-13 (K* chain) / 5e-13 (Z chain) wherever the FP64 oracle achieves it itself.  The two Z-chain
    momenta q_Z, p_B^Z are checked through the lineshape and the density (a momentum formed from a rounded m_psipi minus a
    threshold is not a usable reference near that threshold)."""
    import arbitration as A
    cfg, n = 2, 3001
    Mo, Mg = oracle_model(cfg), gpu_model(cfg)
    x, w = W.norm_events(cfg, n)
    Mg.load_events(dev(x), dev(w))
    names, cache = Mg.dump_cache(0)
    cache = dict(zip(names, cache.cpu().numpy()))
    refd = [_cache_reference(Mo, x[:, i], 0) for i in range(n)]
    refl = [_cache_reference(Mo, x[:, i], 1) for i in range(n)]
    for name in refd[0]:
        rd, rl = np.array([r[name] for r in refd]), np.array([r[name] for r in refl])
        scale = np.maximum(np.abs(rl), 1.0) if name in ("m2", "mZ2", "q", "pB") else 1.0
        tol = 1e-13 if name in ("m2", "inv_m", "q", "pB", "cosK", "sinK", "cosPsi", "sinPsi", "cosPhi", "sinPhi", "mZ2", "inv_mZ") else 5e-13
        A.check(cache[name], rd, rl, tol, f"cache column {name}", events=x, oracle_model=Mo, scale=scale)


def test_lineshape_columns_match_oracle():
    """a2: A^R(m) of every resonance against the oracle (Eqs. 2-3), relative to |A|, on ALL events plus 600 events within 1 MeV
    and 1e-3 MeV of the two m_psipi thresholds.  The reference forms the chain's running mass from the event in the working
    precision (lineshape_at_event); the long double twin arbitrates: 5e-13 wherever the FP64 oracle achieves it."""
    import arbitration as A
    cfg, n = 2, 2500
    Mo, Mg = oracle_model(cfg), gpu_model(cfg)
    x, w = W.norm_events(cfg, n)
    x = np.concatenate([x] + [A.threshold_events(Mo, which, 150, dmax, 3) for which in (0, 1) for dmax in (1.0, 1e-3)], axis=1)
    Mg.load_events(dev(x), None)
    for r, (kind, J, mass, width, rad) in enumerate(W.resonances(cfg)):
        for mm, ww in ((mass, width), (mass * 1.003, width * 0.98)):
            col = Mg.eval_lineshape(r, mm, ww).cpu().numpy()
            Agpu = col[:, 0] + 1j * col[:, 1]
            Mo2 = O.Model(W.DECAY, [(kind, J, mm, ww, rad)])
            rd = np.array([Mo2.lineshape_at_event(0, x[:, i]) for i in range(x.shape[1])])
            rl = np.array([Mo2.lineshape_at_event(0, x[:, i], prec=1) for i in range(x.shape[1])])
            A.check(Agpu, rd, rl, 5e-13, f"lineshape of resonance {r} at ({mm}, {ww})", events=x, oracle_model=Mo)


def mpsi_mpi():
    return W.DECAY[1] + W.DECAY[3]


@pytest.mark.parametrize("cfg,n", [(0, 4099), (1, 6007), (2, 6007)])
def test_event_density_matches_oracle(cfg, n):
    """a3: eps_i * S_i per event, configs 0-2, 1e-11 relative; also each resonance alone (couplings of the
    others zero) so that the small high-spin and Z terms are checked at full relative precision."""
    Mo, Mg = oracle_model(cfg), gpu_model(cfg)
    c = W.couplings(cfg)
    x, eff, xn, wn = make_inputs(cfg, n, 1000)
    Mg.load_events(dev(x), dev(eff))
    Mg.set_params(c)
    v = Mg.eval_events(0).cpu().numpy()
    ref = Mo.eval_events(c, x, eff)
    err = np.abs(v - ref) / ref
    i = int(np.argmax(err))
    assert err[i] < RTOL_EVENT, f"worst event {i}: rel {err[i]:.3e} x={x[:, i]}"
    slots = W.slot_table(W.resonances(cfg))
    for r in range(len(W.resonances(cfg))):
        cr = np.array([c[k] if slots[k][0] == r else 0.0 for k in range(len(c))])
        Mg.set_params(cr)
        v = Mg.eval_events(0).cpu().numpy()
        ref = Mo.eval_events(cr, x, eff)
        err = np.abs(v - ref) / ref
        i = int(np.argmax(err))
        extra = ""
        if W.resonances(cfg)[r][0] == O.ZRES:
            extra = f" mZ-thr={Mo.z_kinematics(x[:, i])['mZ'] - mpsi_mpi():.3e}"
        assert err[i] < RTOL_EVENT, f"resonance {r} alone, worst event {i}: rel {err[i]:.3e} x={x[:, i]}{extra}"


@pytest.mark.parametrize("mode", [1, 2])
def test_event_density_with_changed_masses(mode):
    """a2+a3 with floating masses/widths, columns stored in the pool (mode 1) or evaluated in registers (mode 2)."""
    cfg, n = 2, 5003
    Mo, Mg = oracle_model(cfg), gpu_model(cfg)
    Mg.set_lineshape_mode(mode)
    c = W.couplings(cfg)
    x, w = W.norm_events(cfg, n)
    Mg.load_events(dev(x), dev(w))
    for step in (1, 2, 3):
        mw = W.step_mass_width(3, step)
        Mg.set_params(c, mw[None])
        v = Mg.eval_events(0).cpu().numpy()
        res2 = [(r[0], r[1], mw[i, 0], mw[i, 1], r[4]) for i, r in enumerate(W.resonances(cfg))]
        ref = O.Model(W.DECAY, res2).eval_events(c, x, w)
        assert (np.abs(v - ref) / ref).max() < RTOL_EVENT
        st = Mg.last_call_stats()
        assert st["columns_recomputed"] == (11 if mode == 1 else 0)


@pytest.mark.parametrize("cfg", [0, 1, 2])
def test_nll_matches_oracle_full_config(cfg):
    """a3-a5 at the full sizes of configs 0-2 (10k/100k, 200k/1M, 500k/2M), one NLL evaluation."""
    n, m = W.SIZES[cfg]
    Mo, Mg = oracle_model(cfg), gpu_model(cfg)
    c = W.couplings(cfg)
    x, eff, xn, wn = make_inputs(cfg, n, m)
    Mg.load_events(dev(x), dev(eff))
    Mg.load_norm(dev(xn), dev(wn))
    Mg.set_params(c)
    nll = Mg.nll()[0]
    I = Mg.norm_integral()[0]
    ref_nll, ref_I = Mo.nll(c, x, eff, xn, wn)
    assert abs(I - ref_I[0]) < 1e-12 * ref_I[0]
    assert abs(nll - ref_nll[0]) < RTOL_NLL * abs(ref_nll[0]), (nll, ref_nll[0])
    # bitwise reproducible
    assert Mg.nll()[0] == nll
    # the default P = 1 step is ONE fused launch (data tiles, norm tiles, last-block NLL); the separate-launch form agrees
    st = Mg.last_call_stats()
    assert st["norm_path"] == 4 and st["launches"] == 1
    Mg.set_fused_mode(1)
    nll_sep = Mg.nll()[0]
    st = Mg.last_call_stats()
    assert st["norm_path"] == 1 and st["launches"] > 1
    assert abs(nll_sep - nll) < 1e-13 * abs(nll)
    assert abs(nll_sep - ref_nll[0]) < RTOL_NLL * abs(ref_nll[0])
    Mg.set_fused_mode(0)
    if cfg == 2:   # Z mass and width float (configs[2])
        mw = W.step_mass_width(2, 1)
        Mg.set_params(c, mw[None])
        nll2 = Mg.nll()[0]
        ref2 = Mo.nll(c, x, eff, xn, wn, mass_width=mw[None])[0][0]
        assert abs(nll2 - ref2) < RTOL_NLL * abs(ref2)
        assert Mg.last_call_stats()["columns_recomputed"] == 0      # P = 1: lineshapes live in registers
        # forced column pool: the first call fills all 11 columns for both samples, a Z-only change recomputes 2
        Mg.set_lineshape_mode(1)
        Mg.set_params(c)
        nll3 = Mg.nll()[0]
        assert Mg.last_call_stats()["columns_recomputed"] == 22
        assert abs(nll3 - nll) < 1e-12 * abs(nll)
        Mg.set_params(c, mw[None])
        nll4 = Mg.nll()[0]
        assert Mg.last_call_stats()["columns_recomputed"] == 2      # the Z column, data + norm
        assert abs(nll4 - ref2) < RTOL_NLL * abs(ref2)
        Mg.set_params(c)
        Mg.nll()
        assert Mg.last_call_stats()["columns_recomputed"] == 0      # both Z variants are still held


def test_nll_batched_points_small():
    """cfg 4 pattern at reduced size: all 121 points of one gradient step against the oracle."""
    cfg = 4
    Mo, Mg = oracle_model(cfg), gpu_model(cfg)
    x, eff, xn, wn = make_inputs(cfg, 20011, 100003)
    cs, mws = W.fit_points(cfg)
    Mg.load_events(dev(x), dev(eff))
    Mg.load_norm(dev(xn), dev(wn))
    Mg.set_params(cs, mws)
    nll = Mg.nll()
    ref, refI = Mo.nll(cs, x, eff, xn, wn, mass_width=mws)
    assert nll.shape == (121,)
    st = Mg.last_call_stats()
    assert st["norm_path"] == 9 and st["launches"] == 3     # shape-specialised gradient-batch kernels (normalisation events twice, then data events): no columns, no matrix
    tm = Mg.last_call_timing()                                # the three launches: normalisation pass 0, pass 1, then the data events
    assert tm["lineshape_ms"] == 0.0 and min(tm["norm_ms"], tm["final_ms"], tm["data_ms"]) > 0.0, tm
    assert abs(tm["norm_ms"] + tm["final_ms"] + tm["data_ms"] - Mg.recent_launch_ms(1)[-1]) < 1e-3, tm
    assert st["columns_recomputed"] == 0
    assert np.max(np.abs(nll - ref) / np.abs(ref)) < RTOL_NLL
    assert np.array_equal(Mg.nll(), nll)                     # bit-reproducible
    I = Mg.norm_integral()
    assert Mg.last_call_stats()["norm_path"] == 9
    assert np.max(np.abs(I - refI) / refI) < 1e-12
    # the finite differences themselves (what MINUIT uses) agree: compare NLL(p) - NLL(0)
    d, dref = nll[1:] - nll[0], ref[1:] - ref[0]
    assert np.max(np.abs(d - dref)) < 1e-9 * abs(ref[0])
    # the general gradient-batch kernel (contribution program, delta.cu) on the same batch: another kernel, the same numbers
    Mg.set_batch_mode(3)
    Mg.set_params(cs, mws)
    nll_g = Mg.nll()
    st = Mg.last_call_stats()
    assert st["norm_path"] == 5 and st["launches"] == 1
    assert np.max(np.abs(nll_g - ref) / np.abs(ref)) < RTOL_NLL and np.max(np.abs(nll_g - nll) / np.abs(nll)) < 1e-12
    assert np.max(np.abs((nll_g[1:] - nll_g[0]) - d)) < 1e-9 * abs(ref[0])
    assert np.max(np.abs(Mg.norm_integral() - refI) / refI) < 1e-12 and Mg.last_call_stats()["norm_path"] == 5
    Mg.set_batch_mode(0)
    Mg.set_params(cs, mws)
    # per-event density of a perturbed point (lineshapes in registers)
    for p in (0, 5, 97, 120):
        v = Mg.eval_events(p).cpu().numpy()
        res2 = [(r[0], r[1], mws[p, i, 0], mws[p, i, 1], r[4]) for i, r in enumerate(W.resonances(cfg))]
        vref = O.Model(W.DECAY, res2).eval_events(cs[p], x, eff)
        assert np.max(np.abs(v - vref) / vref) < RTOL_EVENT
    # the same batch as the dense DMMA contraction on the data and the matrix M for the integrals
    Mg.set_batch_mode(2)
    Mg.set_params(cs, mws)
    nll_dense = Mg.nll()
    assert Mg.last_call_stats()["norm_path"] == 2
    assert np.max(np.abs(nll_dense - ref) / np.abs(ref)) < RTOL_NLL
    assert np.max(np.abs(nll_dense - nll) / np.abs(nll)) < 1e-12
    # ... with the normalisation as a direct DMMA sum over the norm events
    Mg.set_norm_mode(1)
    Mg.set_params(cs, mws)
    nll_direct = Mg.nll()
    assert Mg.last_call_stats()["norm_path"] == 3
    assert np.max(np.abs(nll_direct - ref) / np.abs(ref)) < RTOL_NLL
    assert np.max(np.abs(Mg.norm_integral() - refI) / refI) < 1e-12
    Mg.set_norm_mode(0)
    # the loop of single-point streaming launches gives the same numbers
    Mg.set_batch_mode(1)
    Mg.set_params(cs, mws)
    nll_seq = Mg.nll()
    assert Mg.last_call_stats()["norm_path"] == 1
    assert np.max(np.abs(nll_seq - nll) / np.abs(nll)) < 1e-12
    Mg.set_batch_mode(0)


def test_delta_batches_general():
    """gradient-batch kernel beyond the cfg 4 pattern: ragged point counts (1, 31, 32, 33, 129, 200 points besides point 0,
    i.e. partial blocks and two launches), points equal to point 0, points that change two resonances at once, a K*-only
    model, and a dense random batch that must fall back to the DMMA contraction.  (Batch mode 3: the general kernel even where a
    batch happens to fit the shape-specialised one.)"""
    rng = np.random.default_rng(5)
    for cfg in (2, 1):
        Mo, Mg = oracle_model(cfg), gpu_model(cfg)
        Mg.set_batch_mode(3)
        x, eff, xn, wn = make_inputs(cfg, 3001, 7013)
        Mg.load_events(dev(x), dev(eff))
        Mg.load_norm(dev(xn), dev(wn))
        c0 = W.couplings(cfg)
        mw0 = np.array([[r[2], r[3]] for r in W.resonances(cfg)])
        K, R = len(c0), len(mw0)
        slots = W.slot_table(W.resonances(cfg))
        for P in (2, 32, 33, 34, 130, 201):
            cs, mws = np.tile(c0, (P, 1)), np.tile(mw0, (P, 1, 1))
            for p in range(1, P):
                kind = p % 5
                if kind == 0:
                    continue                                   # identical to point 0
                k = rng.integers(K)
                cs[p, k] *= 1 + 0.3 * rng.uniform(-1, 1) + 0.2j * rng.uniform(-1, 1)
                if kind >= 3:                                  # a second resonance: its mass and width
                    r = rng.integers(R)
                    mws[p, r] *= 1 + 0.01 * rng.uniform(-1, 1, 2)
                if kind == 4:                                  # ... and a coupling of that same resonance
                    ks = [i for i, (rr, _l) in enumerate(slots) if rr == r]
                    cs[p, ks[0]] += 0.1
            Mg.set_params(cs, mws)
            nll = Mg.nll()
            st = Mg.last_call_stats()
            assert st["norm_path"] == 5 and st["launches"] == (P - 1 + 127) // 128
            ref, refI = Mo.nll(cs, x, eff, xn, wn, mass_width=mws)
            assert np.max(np.abs(nll - ref) / np.abs(ref)) < RTOL_NLL, (cfg, P)
            assert np.max(np.abs(Mg.norm_integral() - refI) / refI) < 1e-12, (cfg, P)
        # dense random batch: every coupling differs -> not a gradient batch
        Mg.set_batch_mode(0)
        P = 40
        cs = c0[None] * (1 + 0.1 * rng.uniform(-1, 1, (P, K)))
        Mg.set_params(cs)
        nll = Mg.nll()
        assert Mg.last_call_stats()["norm_path"] in (2, 3)
        ref, _ = Mo.nll(cs, x, eff, xn, wn)
        assert np.max(np.abs(nll - ref) / np.abs(ref)) < RTOL_NLL


def test_gradient_batch_large_coupling_steps_in_groups_of_four():
    """Groups of four points on one coupling (k_delta takes their normalisation side from three weighted sums of the slot,
    DESIGN.md 5.6) with LARGE steps, so that the linear and the quadratic term of the expansion both carry weight: every coupling
    of the full model, 109 points = one launch; then twice that = two launches.  Integrals at 1e-12, NLL at the parity bar."""
    cfg = 2
    Mo, Mg = oracle_model(cfg), gpu_model(cfg)
    Mg.set_batch_mode(3)                                      # the general gradient-batch kernel
    x, eff, xn, wn = make_inputs(cfg, 2999, 9001)
    Mg.load_events(dev(x), dev(eff))
    Mg.load_norm(dev(xn), dev(wn))
    c0 = W.couplings(cfg)
    K = len(c0)
    steps = (1.4, 0.6, 1 + 0.5j, 1 - 0.5j)
    for reps in (1, 2):
        P = 1 + 4 * K * reps
        cs = np.tile(c0, (P, 1))
        for r in range(reps):
            for k in range(K):
                for j, f in enumerate(steps):
                    cs[1 + 4 * (r * K + k) + j, k] *= f * (1 + 0.1 * r)
        Mg.set_params(cs)
        nll = Mg.nll()
        st = Mg.last_call_stats()
        assert st["norm_path"] == 5 and st["launches"] == (P - 1 + 127) // 128
        ref, refI = Mo.nll(cs, x, eff, xn, wn)
        assert np.max(np.abs(nll - ref) / np.abs(ref)) < RTOL_NLL, reps
        assert np.max(np.abs(Mg.norm_integral() - refI) / refI) < 1e-12, reps


def _gradient_points(c0, mw0, couplings, lineshapes, h=1e-4):
    """a MINUIT-style step: for every listed coupling slot modulus +-h and phase +-h, for every listed (resonance, 0 mass | 1 width) +-h"""
    pts_c, pts_mw = [c0.copy()], [mw0.copy()]
    for k in couplings:
        for f in (1 + h, 1 - h, np.exp(1j * h), np.exp(-1j * h)):
            c = c0.copy()
            c[k] *= f
            pts_c.append(c)
            pts_mw.append(mw0.copy())
    for r, which in lineshapes:
        for sgn in (1, -1):
            mw = mw0.copy()
            mw[r, which] *= 1 + sgn * h
            pts_c.append(c0.copy())
            pts_mw.append(mw)
    return np.array(pts_c), np.array(pts_mw)


@pytest.mark.parametrize("cfg,n,m", [(1, 3001, 7013), (2, 1, 300), (2, 255, 257), (2, 513, 1025)])
def test_shape_specialised_gradient_batch(cfg, n, m):
    """deltaf.cu beyond configs[4]: the K*-only shape (no Z compiled in), every coupling and every mass and width floating, and
    ragged sizes around the 256-event pipeline unit (a single data event; one event short of / past a unit; past a cache block).
    NLL, integrals and the finite differences NLL(p) - NLL(0) against the oracle, and against the general kernel."""
    Mo, Mg = oracle_model(cfg), gpu_model(cfg)
    c0 = W.couplings(cfg)
    xn, wn = W.norm_events(cfg, m)
    x, eff = W.data_events(cfg, lambda xx, ee: Mo.eval_events(c0, xx, ee), n=n)
    Mg.load_events(dev(x), dev(eff))
    Mg.load_norm(dev(xn), dev(wn))
    mw0 = np.array([[r[2], r[3]] for r in W.resonances(cfg)]) * (1 + 1e-3 * np.random.default_rng(8).uniform(-1, 1, (len(W.resonances(cfg)), 2)))
    R = len(mw0)
    cs, mws = _gradient_points(c0, mw0, range(len(c0)), [(r, w) for r in range(R) for w in (0, 1)])
    assert len(cs) == 1 + 4 * len(c0) + 4 * R
    ref, refI = Mo.nll(cs, x, eff, xn, wn, mass_width=mws)
    out = {}
    for mode, path in ((0, 9), (4, 9), (3, 5)):     # k_deltan + k_deltaf; k_deltaf alone on both samples; the general kernel
        Mg.set_batch_mode(mode)
        Mg.set_params(cs, mws)
        nll = Mg.nll()
        st = Mg.last_call_stats()
        assert st["norm_path"] == path and (path == 5 or st["launches"] == (3 if mode == 0 else 1)), (mode, st)
        assert np.max(np.abs(nll - ref) / np.abs(ref)) < RTOL_NLL
        assert np.max(np.abs((nll - nll[0]) - (ref - ref[0]))) < 1e-9 * abs(ref[0])
        assert np.max(np.abs(Mg.norm_integral() - refI) / refI) < 1e-12
        assert np.array_equal(Mg.nll(), nll)                    # bit-reproducible
        out[mode] = nll
    assert np.max(np.abs(out[0] - out[3]) / np.abs(ref)) < 1e-12


def test_gradient_batch_with_a_silent_constant_term():
    """The paper's resonance list plus a constant term whose coupling is zero at point 0: the shape-specialised kernels still take
    batches that leave it alone, and a point that switches it on goes to another kernel — the same numbers as the oracle either way."""
    from paper_2007_14931_b200 import binding as B
    cfg = 2
    res = W.resonances(cfg) + [(W.CONST, 0, 0.0, 0.0, 0.0)]
    Mo, Mg = O.Model(W.DECAY, res), B.Model(W.DECAY, res)
    x, eff, xn, wn = make_inputs(cfg, 3001, 7013)
    Mg.load_events(dev(x), dev(eff))
    Mg.load_norm(dev(xn), dev(wn))
    c0 = np.concatenate([W.couplings(cfg), [0.0]])
    mw0 = np.array([[r[2], r[3]] for r in res])
    cs = np.stack([c0] * 4)
    mws = np.stack([mw0] * 4)
    cs[1, 3] *= 1.001
    cs[2, 12] *= np.exp(1e-3j)
    mws[3, 10, 0] *= 1.0001
    Mg.set_params(cs, mws)
    nll = Mg.nll()
    assert Mg.last_call_stats()["norm_path"] == 9
    ref, _ = Mo.nll(cs, x, eff, xn, wn, mass_width=mws)
    assert np.max(np.abs(nll - ref) / np.abs(ref)) < RTOL_NLL
    cs[3, -1] = 0.05 / (W.KSTARS[1][3] * W.KSTARS[1][4])      # the constant term switched on at one point (and the Z mass moved there)
    Mg.set_params(cs, mws)
    nll = Mg.nll()
    assert Mg.last_call_stats()["norm_path"] != 9
    ref, _ = Mo.nll(cs, x, eff, xn, wn, mass_width=mws)
    assert np.max(np.abs(nll - ref) / np.abs(ref)) < RTOL_NLL


def test_shape_specialised_gradient_batch_falls_back():
    """What deltaf.cu does not take goes to the general kernel with the same results: a fifth point on one coupling, a point that
    moves a coupling and a mass at once, two resonances at one point; and a step so large that S(p) / S(0) leaves [0.5, 1.5]
    at some event trips the guard, after which the call is repeated with the amplitudes summed term by term."""
    cfg = 2
    Mo, Mg = oracle_model(cfg), gpu_model(cfg)
    x, eff, xn, wn = make_inputs(cfg, 3001, 7013)
    Mg.load_events(dev(x), dev(eff))
    Mg.load_norm(dev(xn), dev(wn))
    c0 = W.couplings(cfg)
    mw0 = np.array([[r[2], r[3]] for r in W.resonances(cfg)])
    base_c, base_mw = _gradient_points(c0, mw0, [3, 4, 24, 25], [(10, 0), (1, 1)])
    assert len(base_c) == 21

    def check(cs, mws, path, launches=None):
        Mg.set_params(cs, mws)
        nll = Mg.nll()
        st = Mg.last_call_stats()
        assert st["norm_path"] == path and (launches is None or st["launches"] == launches), st
        ref, refI = Mo.nll(cs, x, eff, xn, wn, mass_width=mws)
        assert np.max(np.abs(nll - ref) / np.abs(ref)) < RTOL_NLL
        assert np.max(np.abs(Mg.norm_integral() - refI) / refI) < 1e-12

    check(base_c, base_mw, 9, 3)
    # a point equal to point 0 and a Z pair moving together (Eq. 11) are still deltaf's
    cs, mws = np.concatenate([base_c, base_c[:1], base_c[:1]]), np.concatenate([base_mw, base_mw[:1], base_mw[:1]])
    cs[-1, 24] *= 1.0002
    assert c0[26] == c0[24]                                    # Eq. 11 in the seeded couplings
    cs[-1, 26] = cs[-1, 24]                                    # the same delta on l' = -1 and l' = +1
    check(cs, mws, 9, 3)
    # a fifth point on slot 3
    cs, mws = np.concatenate([base_c, base_c[:1]]), np.concatenate([base_mw, base_mw[:1]])
    cs[-1, 3] *= 1.0003
    check(cs, mws, 5)
    # coupling and mass of one resonance at one point
    cs, mws = base_c.copy(), base_mw.copy()
    mws[1, 1, 0] *= 1.0001                                     # point 1 already moves slot 3 = K*(892) lambda = -1 (resonance 1)
    check(cs, mws, 5)
    # two resonances at one point
    cs, mws = base_c.copy(), base_mw.copy()
    cs[2, 12] *= 1.0001
    check(cs, mws, 5)
    # the guard: one coupling reversed -> deltaf's three launches, then the general kernel's exact form (4 launches in all)
    cs, mws = base_c.copy(), base_mw.copy()
    cs[5, 4] = -c0[4]
    check(cs, mws, 5, 4)
    # ... and the model returns to deltaf on the next small step
    check(base_c, base_mw, 9, 3)


def test_nll_terms_of_two_shards_add_up():
    """amp_nll_terms / amp_dataset_sums: the per-shard sums of two models that each hold half of the events combine
    (sharded.py's formula, here without a process group) to the oracle's NLL of the whole sample — for the fused
    P = 1 launch, the gradient-batch kernel and the separate-launch path."""
    from paper_2007_14931_b200 import sharded as S
    cfg = 2
    Mo = oracle_model(cfg)
    x, eff, xn, wn = make_inputs(cfg, 4001, 9001)
    shards = []
    for r in range(2):
        lo, hi = S.shard_bounds(x.shape[1], r, 2)
        ln, hn = S.shard_bounds(xn.shape[1], r, 2)
        Mg = gpu_model(cfg)
        Mg.load_events(dev(x[:, lo:hi]), dev(eff[lo:hi]))
        Mg.load_norm(dev(xn[:, ln:hn]), dev(wn[ln:hn]))
        shards.append(Mg)
    c = W.couplings(cfg)
    cs4, mws4 = W.fit_points(4)
    for cs, mws, fused_mode, path in ((c[None], None, 0, 4), (c[None], None, 1, 2), (cs4[:40], mws4[:40], 0, 9)):   # (2: same masses twice -> matrix M; 9: gradient batch)
        tot = np.zeros(4)
        sl, sw = 0.0, 0.0
        for Mg in shards:
            Mg.set_fused_mode(fused_mode)
            Mg.set_params(cs, mws)
            a, b = Mg.nll_terms()
            assert Mg.last_call_stats()["norm_path"] == path
            sl, sw = sl + a, sw + b
            tot += np.array(Mg.dataset_sums())
        assert tot[0] == x.shape[1] and tot[2] == xn.shape[1]
        assert abs(tot[1] - np.sum(np.log(eff))) < 1e-9 and abs(tot[3] - np.sum(wn)) < 1e-9 * tot[3]
        nll, integral = S.nll_from_sums(sl, sw, (int(tot[0]), tot[1], int(tot[2]), tot[3]))   # the formula combine_terms applies after its all-reduce
        ref, ref_I = Mo.nll(cs, x, eff, xn, wn, mass_width=mws)
        assert np.max(np.abs(nll - ref) / np.abs(ref)) < RTOL_NLL and np.max(np.abs(integral - ref_I) / ref_I) < 1e-12


def test_sharded_model_two_virtual_ranks_on_one_gpu():
    """ShardedModel end to end on one device: two virtual ranks (one host thread and one amp_model each, sharded.ThreadReducer as
    the exchange step) load their slices of the FULL arrays, evaluate, exchange and must both return the oracle's NLL of the
    whole sample — bitwise equal on the two ranks; P = 1 (fused launch) and a 40-point gradient batch."""
    import threading
    from paper_2007_14931_b200 import sharded as S
    cfg = 2
    Mo = oracle_model(cfg)
    x, eff, xn, wn = make_inputs(cfg, 4001, 9001)
    c = W.couplings(cfg)
    cs4, mws4 = W.fit_points(4)
    cases = [(c[None], W.step_mass_width(3, 1)[None]), (cs4[:40], mws4[:40])]
    red = S.ThreadReducer(2)
    out, err = [None, None], []

    def rank_main(r):
        try:
            torch.cuda.set_device(0)
            sm = S.ShardedModel(W.DECAY, W.resonances(cfg), reduce=red.port(r))
            assert (sm.rank, sm.world) == (r, 2)
            sm.load_events(x, eff)
            sm.load_norm(xn, wn)
            res = []
            for cs, mws in cases:
                sm.set_params(cs, mws)
                res.append(sm.nll())
            assert sm.totals[0] == x.shape[1] and sm.totals[2] == xn.shape[1]
            out[r] = res
        except Exception as e:   # noqa: BLE001
            err.append(e)
            red.barrier.abort()

    th = [threading.Thread(target=rank_main, args=(r,)) for r in range(2)]
    [t.start() for t in th]
    [t.join() for t in th]
    assert not err, err
    for k, (cs, mws) in enumerate(cases):
        ref, _ = Mo.nll(cs, x, eff, xn, wn, mass_width=mws)
        assert np.array_equal(out[0][k], out[1][k])
        assert np.max(np.abs(out[0][k] - ref) / np.abs(ref)) < RTOL_NLL


def test_sharded_model_over_nccl_process_group():
    """the default exchange step: torch.distributed all-reduce on an NCCL process group (one rank here: this box has one GPU)"""
    import os
    import socket
    import torch.distributed as dist
    from paper_2007_14931_b200 import sharded as S
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    torch.cuda.set_device(0)
    dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda", 0))
    try:
        cfg = 2
        Mo = oracle_model(cfg)
        x, eff, xn, wn = make_inputs(cfg, 3001, 7001)
        c = W.couplings(cfg)
        sm = S.ShardedModel(W.DECAY, W.resonances(cfg))
        sm.load_events(x, eff)
        sm.load_norm(xn, wn)
        mw = W.step_mass_width(3, 2)[None]
        sm.set_params(c[None], mw)
        nll = sm.nll()
        ref, _ = Mo.nll(c[None], x, eff, xn, wn, mass_width=mw)
        assert abs(nll[0] - ref[0]) < RTOL_NLL * abs(ref[0])
    finally:
        dist.destroy_process_group()


def test_norm_matrix_matches_oracle_and_direct_sum():
    """a4: the Hermitian matrix M from the HERK kernel against the oracle's plain double loop, and c^H M c against
    the direct sum (pin P10 on the GPU side)."""
    cfg = 2
    Mo, Mg = oracle_model(cfg), gpu_model(cfg)
    c = W.couplings(cfg)
    xn, wn = W.norm_events(cfg, 7001)
    Mg.load_norm(dev(xn), dev(wn))
    Mg.set_norm_mode(2)
    Mg.set_params(c)
    M = Mg.norm_matrix(0)
    ref = Mo.norm_matrix(xn, wn)
    assert np.abs(M - ref).max() < 1e-12 * np.abs(ref).max()
    assert np.abs(M - M.conj().T).max() < 1e-15 * np.abs(M).max()
    I_mat = Mg.norm_integral()[0]
    assert Mg.last_call_stats()["norm_path"] == 2
    assert abs(I_mat - (c.conj() @ ref @ c).real) < 1e-12 * I_mat
    Mg.set_norm_mode(1)
    Mg.set_params(c)
    I_dir = Mg.norm_integral()[0]
    assert Mg.last_call_stats()["norm_path"] == 1
    assert abs(I_mat - I_dir) < 1e-12 * I_dir
    assert abs(I_dir - Mo.norm_integral(c, xn, wn)[0]) < 1e-12 * I_dir


def test_fit_fractions_match_oracle():
    """Eq. 13: per-resonance fit fractions from the device quadratic forms against the oracle's plain definition
    (density with all other helicity amplitudes set to zero, summed over the same sample), configs 1 and 2, also at
    moved masses and widths."""
    for cfg in (1, 2):
        Mo, Mg = oracle_model(cfg), gpu_model(cfg)
        c = W.couplings(cfg)
        xn, wn = W.norm_events(cfg, 9001)
        Mg.load_norm(dev(xn), dev(wn))
        Mg.set_norm_mode(2)
        Mg.set_params(c)
        ff = Mg.fit_fractions(0)
        ref = Mo.fit_fractions(c, xn, wn)
        assert ff.shape == (len(W.resonances(cfg)),)
        assert np.max(np.abs(ff - ref) / ref) < 1e-11, (cfg, ff, ref)
        mw = W.step_mass_width(3, 2)[:len(W.resonances(cfg))]
        Mg.set_params(c, mw[None])
        ff2 = Mg.fit_fractions(0)
        ref2 = Mo.fit_fractions(c, xn, wn, mass_width=mw)
        assert np.max(np.abs(ff2 - ref2) / ref2) < 1e-11
        assert np.max(np.abs(ff2 - ff)) > 1e-9          # the lineshapes did move


@pytest.mark.parametrize("with_z", [True, False])
def test_lass_model_matches_oracle(with_z):
    """Eqs. 7-9: the model with the LASS S-wave term (replacing kappa(800) and K0*(1430)): lineshape column, per-event density,
    NLL through the fused launch, the separate launches, the matrix M, and a batch of points through the DMMA contraction
    with the K0*(1430) mass and width inside the LASS term moving."""
    from paper_2007_14931_b200 import binding as B
    res = W.resonances_lass(with_z)
    c = W.couplings_lass(with_z)
    Mo, Mg = O.Model(W.DECAY, res), B.Model(W.DECAY, res)
    assert Mg.K == Mo.K == len(c)
    xn, wn = W.norm_events(2, 20011)
    x, eff = W.data_events(2, lambda xx, ee: Mo.eval_events(c, xx, ee), n=5003)
    Mg.load_events(dev(x), dev(eff))
    Mg.load_norm(dev(xn), dev(wn))
    col = Mg.eval_lineshape(0, res[0][2], res[0][3]).cpu().numpy()
    ref = np.array([Mo.lineshape(0, v)[0] for v in x[0]])
    assert np.max(np.abs(col[:, 0] + 1j * col[:, 1] - ref) / np.abs(ref)) < 5e-13
    Mg.set_params(c)
    v = Mg.eval_events(0).cpu().numpy()
    vref = Mo.eval_events(c, x, eff)
    assert np.max(np.abs(v - vref) / vref) < RTOL_EVENT
    only = np.array([c[0]] + [0.0] * (len(c) - 1))               # the LASS term alone
    Mg.set_params(only)
    assert np.max(np.abs(Mg.eval_events(0).cpu().numpy() - Mo.eval_events(only, x, eff)) / Mo.eval_events(only, x, eff)) < RTOL_EVENT
    mw = np.array([[r[2], r[3]] for r in res]) * (1 + 1e-3 * np.linspace(-1, 1, 2 * len(res)).reshape(-1, 2))
    for fused in (0, 1):
        mwf = mw * (1 + 1e-4 * fused)                            # (equal masses on successive calls would switch to the matrix)
        Mg.set_fused_mode(fused)
        Mg.set_params(c, mwf[None])
        nll = Mg.nll()[0]
        assert Mg.last_call_stats()["norm_path"] == (4 if fused == 0 else 1)
        rn = Mo.nll(c, x, eff, xn, wn, mass_width=mwf[None])[0][0]
        assert abs(nll - rn) < RTOL_NLL * abs(rn)
    Mg.set_fused_mode(0)
    Mg.set_params(c, mwf[None])
    assert abs(Mg.nll()[0] - rn) < RTOL_NLL * abs(rn)
    assert Mg.last_call_stats()["norm_path"] == 2             # same masses twice: matrix M
    # a batch: LASS coupling, LASS mass and width, another coupling, moving point by point -> dense DMMA path
    P = 30
    rng = np.random.default_rng(9)
    cs, mws = np.tile(c, (P, 1)), np.tile(mw, (P, 1, 1))
    for p in range(1, P):
        cs[p, p % len(c)] *= 1 + 0.2 * rng.uniform(-1, 1)
        cs[p, 0] *= 1 + 0.1j * rng.uniform(-1, 1)
        if p % 3 == 0:
            mws[p, 0] *= 1 + 1e-2 * rng.uniform(-1, 1, 2)
    Mg.set_params(cs, mws)
    nll = Mg.nll()
    assert Mg.last_call_stats()["norm_path"] in (2, 3)
    rb, _ = Mo.nll(cs, x, eff, xn, wn, mass_width=mws)
    assert np.max(np.abs(nll - rb) / np.abs(rb)) < RTOL_NLL


@pytest.mark.parametrize("cfg", [0, 1, 2])
def test_analytic_gradient_matches_oracle(cfg):
    """NLL and dNLL/d(Re, Im H_k) for all K couplings in one launch against the oracle's derivative written
    out event by event; the Euler identity sum_k conj(H_k) dNLL/dconj(H_k) = 0 (scale and phase invariance, pin P11) on the
    GPU numbers; moved masses and widths; bit-reproducibility."""
    Mo, Mg = oracle_model(cfg), gpu_model(cfg)
    c = W.couplings(cfg)
    x, eff, xn, wn = make_inputs(cfg, 6007, 20011)
    Mg.load_events(dev(x), dev(eff))
    Mg.load_norm(dev(xn), dev(wn))
    Mg.set_params(c)
    nll, g = Mg.nll_grad()
    # the paper's resonance lists (configs 1, 2) run the shape-specialised kernel (gradient components in registers, path 8)
    assert Mg.last_call_stats() == {"launches": 1, "columns_recomputed": 0, "norm_path": 8 if cfg > 0 else 7}
    rn, rg = Mo.nll_gradient(c, x, eff, xn, wn)
    assert abs(nll - rn) < RTOL_NLL * abs(rn)
    assert np.max(np.abs(g - rg)) < 1e-9 * np.max(np.abs(rg)), np.max(np.abs(g - rg)) / np.max(np.abs(rg))
    if cfg > 0:   # the generic kernel on the same point
        Mg.set_grad_mode(1)
        nll_g, g_g = Mg.nll_grad()
        assert Mg.last_call_stats()["norm_path"] == 7
        assert abs(nll_g - rn) < RTOL_NLL * abs(rn) and np.max(np.abs(g_g - rg)) < 1e-9 * np.max(np.abs(rg))
        assert abs(nll_g - nll) < 1e-12 * abs(nll) and np.max(np.abs(g_g - g)) < 1e-10 * np.max(np.abs(g))
        Mg.set_grad_mode(0)
    gc = 0.5 * (g[:, 0] + 1j * g[:, 1])
    if cfg > 0:   # (cfg 0 holds the constant term's coupling fixed by convention, but the identity is over ALL slots anyway)
        assert abs(np.sum(np.conj(c) * gc)) < 1e-9 * np.sum(np.abs(c) * np.abs(gc))
    nll2, g2 = Mg.nll_grad()
    assert nll2 == nll and np.array_equal(g2, g)
    assert abs(Mg.nll()[0] - nll) < 1e-13 * abs(nll)
    # same masses and widths again, other couplings (a fit at fixed lineshapes): the normalisation side comes from the matrix M
    # ((M c)_k and c^H M c), only the data events are walked
    c2 = c * (1 + 0.05 * np.cos(np.arange(len(c)))) * np.exp(0.05j * np.sin(np.arange(len(c))))
    Mg.set_params(c2)
    nll3, g3 = Mg.nll_grad()
    rn3, rg3 = Mo.nll_gradient(c2, x, eff, xn, wn)
    assert abs(nll3 - rn3) < RTOL_NLL * abs(rn3)
    assert np.max(np.abs(g3 - rg3)) < 1e-9 * np.max(np.abs(rg3)), np.max(np.abs(g3 - rg3)) / np.max(np.abs(rg3))
    Mg.set_params(c2)
    nll4, g4 = Mg.nll_grad()
    assert nll4 == nll3 and np.array_equal(g4, g3)
    if cfg == 2:
        mw = W.step_mass_width(3, 2)
        Mg.set_params(c, mw[None])
        nll, g = Mg.nll_grad()
        res2 = [(r[0], r[1], mw[i, 0], mw[i, 1], r[4]) for i, r in enumerate(W.resonances(cfg))]
        rn, rg = O.Model(W.DECAY, res2).nll_gradient(c, x, eff, xn, wn)
        assert abs(nll - rn) < RTOL_NLL * abs(rn) and np.max(np.abs(g - rg)) < 1e-9 * np.max(np.abs(rg))


def test_background_and_purity_match_oracle():
    """Eq. 14: NLL with a per-event background density and a purity against the oracle's plain definition — one point with
    all lineshapes moved, a batch of points, purity 1 (= signal only) and switching the background off again."""
    cfg = 2
    Mo, Mg = oracle_model(cfg), gpu_model(cfg)
    c = W.couplings(cfg)
    x, eff, xn, wn = make_inputs(cfg, 7001, 20011)
    rng = np.random.default_rng(8)
    # a smooth seeded background shape at the data events, a few 1e-10 like eps S / I (any positive numbers are valid inputs)
    I0 = Mo.norm_integral(c, xn, wn)[0]
    bkg = np.mean(Mo.eval_events(c, x, eff)) / I0 * (1.0 + 0.5 * x[1]) * (1.0 + 0.3 * np.cos(x[3])) * rng.uniform(0.8, 1.2, x.shape[1])
    Mg.load_events(dev(x), dev(eff))
    Mg.load_norm(dev(xn), dev(wn))
    Mg.set_params(c)
    base = Mg.nll()[0]
    Mg.set_background(dev(bkg), 0.85)
    mw = W.step_mass_width(3, 4)
    Mg.set_params(c, mw[None])
    nll = Mg.nll()[0]
    assert Mg.last_call_stats()["norm_path"] == 6
    ref = Mo.nll_background(c, x, eff, bkg, 0.85, xn, wn, mass_width=mw[None])[0]
    assert abs(nll - ref) < RTOL_NLL * abs(ref), (nll, ref)
    assert Mg.nll()[0] == nll
    cs, mws = W.fit_points(4)
    Mg.set_params(cs[:9], mws[:9])
    nb = Mg.nll()
    rb = Mo.nll_background(cs[:9], x, eff, bkg, 0.85, xn, wn, mass_width=mws[:9])
    assert np.max(np.abs(nb - rb) / np.abs(rb)) < RTOL_NLL
    Mg.set_background(dev(bkg), 1.0)                       # purity 1: the background drops out
    Mg.set_params(c)
    assert abs(Mg.nll()[0] - base) < 1e-12 * abs(base)
    Mg.set_background(None, 1.0)
    Mg.set_params(c)
    assert abs(Mg.nll()[0] - base) < 1e-12 * abs(base) and Mg.last_call_stats()["norm_path"] in (2, 4)   # signal-only paths again


def test_gradient_batch_guard_repeats_large_cancelling_changes():
    """The gradient-batch kernel expands single-contribution points around point 0; a point that switches a dominant amplitude
    off makes S(p) << S(0) at some events, where the expansion would lose digits: the guard trips and the library repeats the call
    with the amplitudes summed term by term (twice the launches).  Results against the oracle either way; small steps do not trip it."""
    from paper_2007_14931_b200 import binding as B
    res = [(W.KSTAR, 1, 895.55, 47.3, W.RADIUS)]                # one resonance: at sin(theta_K*) -> 0 only lambda = 0 is left
    c = np.array([0.7 * np.exp(0.5j), 1.0, 0.9 * np.exp(-1.1j)])
    Mo, Mg = O.Model(W.DECAY, res), B.Model(W.DECAY, res)
    xn, wn = W.norm_events(1, 12000)
    x, eff = xn[:, :6000].copy(), wn[:6000].copy()
    Mg.load_events(dev(x), dev(eff))
    Mg.load_norm(dev(xn[:, 6000:]), dev(wn[6000:]))
    xn, wn = xn[:, 6000:], wn[6000:]
    small = np.tile(c, (5, 1))
    for p in range(1, 5):
        small[p, (p - 1) % 3] *= 1 + 1e-3 * p
    Mg.set_params(small)
    nb = Mg.nll()
    st = Mg.last_call_stats()
    assert st["norm_path"] == 5 and st["launches"] == 1
    rb, rI = Mo.nll(small, x, eff, xn, wn)
    assert np.max(np.abs(nb - rb) / np.abs(rb)) < RTOL_NLL and np.max(np.abs(Mg.norm_integral() - rI) / rI) < 1e-12
    big = np.tile(c, (4, 1))
    big[1, 1] = 1e-7 * c[1]                                      # lambda = 0 switched off: S(p)/S(0) ~ sin^2(theta_K*) at some events
    big[2, 1] = -c[1]
    big[3, 0] *= 1.001
    Mg.set_params(big)
    nb = Mg.nll()
    st = Mg.last_call_stats()
    assert st["norm_path"] == 5 and st["launches"] == 2           # the repeat
    rb, rI = Mo.nll(big, x, eff, xn, wn)
    assert np.max(np.abs(nb - rb) / np.abs(rb)) < RTOL_NLL, np.max(np.abs(nb - rb) / np.abs(rb))
    assert np.max(np.abs(Mg.norm_integral() - rI) / rI) < 1e-12


@pytest.mark.parametrize("with_z", [True, False])
def test_lass_model_gradient_and_fit(with_z):
    """amp_nll_grad and amp_fit for the paper's LASS variant of the model (Eq. 9): the LASS term is one more slot whose lineshape
    record is A_LASS; lineshapes moved (both samples walked), fixed (matrix M), and a short fit"""
    from paper_2007_14931_b200 import binding as B
    res = W.resonances_lass(with_z)
    c = W.couplings_lass(with_z)
    Mo, Mg = O.Model(W.DECAY, res), B.Model(W.DECAY, res)
    xn, wn = W.norm_events(2, 20011)
    x, eff = W.data_events(2, lambda xx, ee: Mo.eval_events(c, xx, ee), n=5003)
    Mg.load_events(dev(x), dev(eff))
    Mg.load_norm(dev(xn), dev(wn))
    mw = np.array([[r[2], r[3]] for r in res]) * (1 + 1e-3 * np.linspace(-1, 1, 2 * len(res)).reshape(-1, 2))
    Mo2 = O.Model(W.DECAY, [(r[0], r[1], mw[i, 0], mw[i, 1], r[4]) for i, r in enumerate(res)])
    Mg.set_params(c, mw[None])
    nll, g = Mg.nll_grad()
    rn, rg = Mo2.nll_gradient(c, x, eff, xn, wn)
    assert abs(nll - rn) < RTOL_NLL * abs(rn)
    assert np.max(np.abs(g - rg)) < 1e-9 * np.max(np.abs(rg)), np.max(np.abs(g - rg)) / np.max(np.abs(rg))
    assert np.abs(rg[0]).max() > 1e-3 * np.max(np.abs(rg))                # the LASS slot's derivative is not a trivial zero
    c2 = c * (1 + 0.04 * np.cos(np.arange(len(c))))
    Mg.set_params(c2, mw[None])                                           # fixed lineshapes: matrix M
    nll2, g2 = Mg.nll_grad()
    rn2, rg2 = Mo2.nll_gradient(c2, x, eff, xn, wn)
    assert abs(nll2 - rn2) < RTOL_NLL * abs(rn2)
    assert np.max(np.abs(g2 - rg2)) < 1e-9 * np.max(np.abs(rg2))
    slots = W.slot_table(res)
    fixed = [k for k, (r, lam) in enumerate(slots) if res[r][0] == W.KSTAR and abs(res[r][2] - 895.55) < 1e-9 and lam == 0]
    r = Mg.fit(c2, fixed=fixed, mass_width=mw, gtol=1e-3, max_iter=500)
    assert r["nll"] < nll2 and r["grad_max"] < 0.02 * np.max(np.abs(g2))
    # floating K0*(1430) mass and width inside the LASS term: derivative batch through the dense path
    r3 = Mg.fit(r["couplings"], fixed=fixed, mass_width=mw, float_mw=[(0, 0), (0, 1)], gtol=1e-2, max_iter=60)
    assert r3["nll"] <= r["nll"] + 1e-9


@pytest.mark.parametrize("cfg,n,m", [(2, 7001, 20011), (1, 513, 1500)])
def test_analytic_gradient_with_background(cfg, n, m):
    """amp_nll_grad under Eq. 14 (background + purity): the data-side weights become purity eps / (I f_i) and N becomes
    sum_i u_i S_i.  Lineshapes just moved (a normalisation launch first, then the gradient kernel over both samples), then
    fixed (sum w S from the held matrix M inside the kernel); purity 1 gives the signal-only gradient; a fit loop runs on it."""
    Mo, Mg = oracle_model(cfg), gpu_model(cfg)
    c = W.couplings(cfg)
    x, eff, xn, wn = make_inputs(cfg, n, m)
    rng = np.random.default_rng(9)
    I0 = Mo.norm_integral(c, xn, wn)[0]
    bkg = np.mean(Mo.eval_events(c, x, eff)) / I0 * (1.0 + 0.5 * x[1]) * (1.0 + 0.3 * np.cos(x[3])) * rng.uniform(0.8, 1.2, x.shape[1])
    Mg.load_events(dev(x), dev(eff))
    Mg.load_norm(dev(xn), dev(wn))
    Mg.set_background(dev(bkg), 0.8)
    mw = W.step_mass_width(3, 2)[:len(W.resonances(cfg))]
    res2 = [(r[0], r[1], mw[i, 0], mw[i, 1], r[4]) for i, r in enumerate(W.resonances(cfg))]
    Mo2 = O.Model(W.DECAY, res2)
    Mg.set_params(c, mw[None])
    nll, g = Mg.nll_grad()
    st = Mg.last_call_stats()
    assert st["norm_path"] == 7 and st["launches"] == 3
    rn, rg = Mo2.nll_gradient_background(c, x, eff, bkg, 0.8, xn, wn)
    assert abs(nll - rn) < RTOL_NLL * abs(rn), (nll, rn)
    assert np.max(np.abs(g - rg)) < 1e-9 * np.max(np.abs(rg)), np.max(np.abs(g - rg)) / np.max(np.abs(rg))
    assert abs(Mg.nll()[0] - nll) < 1e-12 * abs(nll)                      # the NLL of amp_nll (path 6) is the same number
    c2 = c * (1 + 0.05 * np.cos(np.arange(len(c)))) * np.exp(0.05j * np.sin(np.arange(len(c))))
    Mg.set_params(c2, mw[None])                                           # same lineshapes: matrix M
    nll2, g2 = Mg.nll_grad()
    assert Mg.last_call_stats()["launches"] == 1
    rn2, rg2 = Mo2.nll_gradient_background(c2, x, eff, bkg, 0.8, xn, wn)
    assert abs(nll2 - rn2) < RTOL_NLL * abs(rn2)
    assert np.max(np.abs(g2 - rg2)) < 1e-9 * np.max(np.abs(rg2))
    Mg.set_params(c2, mw[None])
    nll3, g3 = Mg.nll_grad()
    assert nll3 == nll2 and np.array_equal(g3, g2)                        # bit-reproducible
    # purity 1: f = eps S / I, the signal-only likelihood
    Mg.set_background(dev(bkg), 1.0)
    Mg.set_params(c2, mw[None])
    nll4, g4 = Mg.nll_grad()
    r4, rg4 = Mo2.nll_gradient(c2, x, eff, xn, wn)
    assert abs(nll4 - r4) < RTOL_NLL * abs(r4) and np.max(np.abs(g4 - rg4)) < 1e-9 * np.max(np.abs(rg4))
    # the native fit runs on it: the NLL does not go up and the gradient at the result is small
    Mg.set_background(dev(bkg), 0.8)
    fixed = [k for k, (r, lam) in enumerate(W.slot_table(W.resonances(cfg))) if r == 1 and lam == 0]
    r = Mg.fit(c2, fixed=fixed, mass_width=mw, gtol=1e-3, max_iter=400)
    assert r["nll"] <= nll2 and r["grad_max"] < 0.05 * np.max(np.abs(g2))


def test_two_z_model_matches_oracle():
    """SURVEY.md 8(f)-3 / PAPER.md:165, 191 ("ten K*s and two Zs"): a second 1+ exotic, Z(4430) (m = 4478, Gamma = 181 MeV), shares
    the Z(4200)'s decay frame and angular cache; K = 30.  Per-event density, fused NLL with all 12 lineshapes moving, and a
    gradient batch that moves the couplings, mass and width of both Zs (gradient-batch kernel)."""
    from paper_2007_14931_b200 import binding as B
    res = W.resonances(2) + [(W.ZRES, 1, 4478.0, 181.0, W.RADIUS)]
    rng = np.random.default_rng(21)
    c = np.concatenate([W.couplings(2), 4.0 * rng.uniform(0.5, 1.5, 3) * np.exp(1j * rng.uniform(-3, 3, 3))])
    c[-1] = c[-3]                                             # Eq. 11
    Mo, Mg = O.Model(W.DECAY, res), B.Model(W.DECAY, res)
    assert Mg.K == 30
    xn, wn = W.norm_events(2, 20011)
    x, eff = W.data_events(2, lambda xx, ee: Mo.eval_events(c, xx, ee), n=6007)
    Mg.load_events(dev(x), dev(eff))
    Mg.load_norm(dev(xn), dev(wn))
    Mg.set_params(c)
    v, vref = Mg.eval_events(0).cpu().numpy(), Mo.eval_events(c, x, eff)
    assert np.max(np.abs(v - vref) / vref) < RTOL_EVENT
    mw = np.array([[r[2], r[3]] for r in res]) * (1 + 1e-3 * rng.uniform(-1, 1, (len(res), 2)))
    Mg.set_params(c, mw[None])
    nll = Mg.nll()[0]
    assert Mg.last_call_stats()["norm_path"] == 4
    rn = Mo.nll(c, x, eff, xn, wn, mass_width=mw[None])[0][0]
    assert abs(nll - rn) < RTOL_NLL * abs(rn)
    P = 1 + 2 * 12
    cs, mws = np.tile(c, (P, 1)), np.tile(mw, (P, 1, 1))
    p = 1
    for zr, k0 in ((10, 24), (11, 27)):                      # (resonance index, first slot) of the two Zs
        for sgn in (+1, -1):
            cs[p, k0] *= 1 + sgn * 1e-3; cs[p, k0 + 2] = cs[p, k0]; p += 1          # |H_-1| = |H_+1| (tied)
            cs[p, k0 + 1] *= np.exp(sgn * 1e-3j); p += 1                              # arg H_0
            mws[p, zr, 0] *= 1 + sgn * 1e-4; p += 1                                   # mass
            mws[p, zr, 1] *= 1 + sgn * 1e-4; p += 1                                   # width
            cs[p, 3] *= 1 + sgn * 1e-3; p += 1                                        # a K* coupling
            mws[p, 1, 0] *= 1 + sgn * 1e-5; p += 1                                    # the K*(892) mass
    assert p == P
    rb, rI = Mo.nll(cs, x, eff, xn, wn, mass_width=mws)
    for mode, path in ((0, 9), (4, 9), (3, 5)):               # the shape-specialised kernels (two Zs compiled in): three launches, one launch; the general one
        Mg.set_batch_mode(mode)
        Mg.set_params(cs, mws)
        nll = Mg.nll()
        assert Mg.last_call_stats()["norm_path"] == path
        assert np.max(np.abs(nll - rb) / np.abs(rb)) < RTOL_NLL
        assert np.max(np.abs((nll - nll[0]) - (rb - rb[0]))) < 1e-9 * abs(rb[0])
        assert np.max(np.abs(Mg.norm_integral() - rI) / rI) < 1e-12


def test_static_lineshapes_switch_to_the_matrix():
    """cfg 1 call pattern (masses and widths fixed, couplings move): the second call with unchanged lineshapes builds
    M once, later calls only evaluate c^H M c; a moved mass goes back to the direct sum."""
    cfg = 1
    Mo, Mg = oracle_model(cfg), gpu_model(cfg)
    c = W.couplings(cfg)
    x, eff, xn, wn = make_inputs(cfg, 20011, 60013)
    Mg.load_events(dev(x), dev(eff))
    Mg.load_norm(dev(xn), dev(wn))
    rng = np.random.default_rng(11)
    paths, launches = [], []
    for it in range(4):
        ci = c * (1 + 0.05 * rng.uniform(-1, 1, c.size))
        Mg.set_params(ci)
        nll = Mg.nll()[0]
        ref = Mo.nll(ci, x, eff, xn, wn)[0][0]
        assert abs(nll - ref) < RTOL_NLL * abs(ref)
        st = Mg.last_call_stats()
        paths.append(st["norm_path"]); launches.append(st["launches"])
    assert paths == [4, 2, 2, 2]      # first call: fused single launch with a direct-sum normalisation; then the matrix
    assert launches[3] < launches[1]          # no lineshape / HERK launches once M is held
    assert launches[2] == 1 and launches[3] == 1   # ... the step is ONE launch: data tiles + c^H M c + NLL in the last thread block
    mw = W.step_mass_width(3, 5)[:10]
    Mg.set_params(c, mw[None])
    nll = Mg.nll()[0]
    assert Mg.last_call_stats()["norm_path"] == 4
    ref = Mo.nll(c, x, eff, xn, wn, mass_width=mw[None])[0][0]
    assert abs(nll - ref) < RTOL_NLL * abs(ref)


def test_edge_cases():
    from paper_2007_14931_b200 import binding as B
    cfg = 2
    Mg = gpu_model(cfg)
    c = W.couplings(cfg)
    xn, wn = W.norm_events(cfg, 777)
    # call order
    with pytest.raises(B.AmpError) as e:
        Mg.nll()
    assert e.value.status == B.AMP_ERR_STATE
    Mg.load_norm(dev(xn), dev(wn))
    Mg.set_params(c)
    with pytest.raises(B.AmpError) as e:
        Mg.nll()
    assert e.value.status == B.AMP_ERR_STATE
    # empty data set: NLL = 0
    Mg.load_events(dev(np.zeros((4, 0))), None)
    assert Mg.nll()[0] == 0.0
    # single event, no efficiency given (= 1); norm weights None (= 1)
    x1 = xn[:, :1].copy()
    Mg.load_events(dev(x1), None)
    Mg.load_norm(dev(xn), None)
    Mo = oracle_model(cfg)
    ref = Mo.nll(c, x1, None, xn, None)[0][0]
    assert abs(Mg.nll()[0] - ref) < RTOL_NLL * abs(ref)
    # event outside phase space -> AMP_ERR_DOMAIN, data set left unloaded
    bad = xn[:, :10].copy()
    bad[0, 3] = 500.0
    with pytest.raises(B.AmpError) as e:
        Mg.load_events(dev(bad), None)
    assert e.value.status == B.AMP_ERR_DOMAIN
    bad = xn[:, :10].copy()
    bad[1, 7] = 1.5
    with pytest.raises(B.AmpError) as e:
        Mg.load_events(dev(bad), None)
    assert e.value.status == B.AMP_ERR_DOMAIN
    with pytest.raises(B.AmpError) as e:
        Mg.load_events(dev(xn[:, :10]), dev(np.zeros(10)))          # eps = 0
    assert e.value.status == B.AMP_ERR_DOMAIN
    # pole mass outside the kinematic range
    mw = np.array([[r[2], r[3]] for r in W.resonances(cfg)])
    mw[1, 0] = 3000.0
    with pytest.raises(B.AmpError) as e:
        Mg.set_params(c, mw[None])
    assert e.value.status == B.AMP_ERR_DOMAIN
    # all couplings zero: S = 0 -> domain error, NLL = +inf
    Mg.load_events(dev(xn[:, :100]), None)
    Mg.set_params(np.zeros_like(c))
    out = Mg.nll(allow_domain_error=True)
    assert np.isinf(out[0])
    # events at the edge of the allowed input range (|cos| = 1 - 1e-9, m 1e-3 above threshold)
    edge = np.array([[W.DECAY[2] + W.DECAY[3] + 1e-3, 2182.0, 1000.0, 1500.0],
                     [W.COS_MAX, -W.COS_MAX, W.COS_MAX, 0.0],
                     [-W.COS_MAX, W.COS_MAX, 0.3, W.COS_MAX],
                     [0.1, -3.0, np.pi, -np.pi]])
    Mg.load_events(dev(edge), None)
    Mg.set_params(c)
    v = Mg.eval_events(0).cpu().numpy()
    import arbitration as A
    A.check(v, Mo.eval_events(c, edge), Mo.eval_events(c, edge, prec=1), RTOL_EVENT, "edge events", events=edge, oracle_model=Mo)
    # degenerate Z-chain geometry (mu+ exactly along the pion: cos theta_K* = +-1 AND cos theta_psi = +-1): phi~ and alpha are
    # angles between planes that do not exist (reading A17) -> refused at load for a model with a Z ...
    degenerate = np.array([[1000.0, 1200.0], [1.0, -1.0], [1.0, 1.0], [0.3, -2.0]])
    with pytest.raises(B.AmpError) as e:
        Mg.load_events(dev(degenerate), None)
    assert e.value.status == B.AMP_ERR_DOMAIN
    # ... and a plain event (of density exactly zero) for the K*-only model, which has no Z chain; each |cos| = 1 alone is fine for both
    Mk, Mok = gpu_model(1), oracle_model(1)
    Mk.load_events(dev(degenerate), None)
    Mk.set_params(W.couplings(1))
    vk = Mk.eval_events(0).cpu().numpy()
    # sin theta_K* = sin theta_psi = 0: every term of Eq. 4 vanishes (the oracle's angles pass through atan2 and sin: 1e-44, not 0)
    assert np.all(vk < 1e-30) and np.all(Mok.eval_events(W.couplings(1), degenerate) < 1e-30)
    single = np.array([[1000.0, 1200.0, 900.0], [1.0, 0.2, -1.0], [0.4, -1.0, 0.3], [0.3, -2.0, 1.0]])
    Mg.load_events(dev(single), None)
    Mg.set_params(c)
    v1 = Mg.eval_events(0).cpu().numpy()
    assert np.all(np.isfinite(v1)) and np.all(v1 > 0)
    # at |cos| = 1 EXACTLY the oracle's own construction does not exist (its x axis is the K direction's component across n_K*,
    # zero at cos theta_K* = +-1; alpha is a dihedral about an axis parallel to n_K* at cos theta_psi = +-1): the closed forms
    # return the continuous limit — compare with the oracle a hair inside (the density moves by O(sin) ~ 1e-6 over that step)
    inside = single * np.array([[1.0], [1.0 - 1e-12], [1.0 - 1e-12], [1.0]])
    ref_in = Mo.eval_events(c, inside, prec=1)
    assert np.all(np.isfinite(ref_in)) and np.max(np.abs(v1 - ref_in) / ref_in) < 1e-4


def test_threshold_and_edge_events_arbitrated_by_long_double():
    """2000 events drawn within 1 MeV and 1e-3 MeV of m_psipi = m_psi + m_pi (pion at rest in the Z frame: theta_Z is
    the direction of a vanishing momentum, NOT suppressed by the lineshape) and of m_psipi = m_B - m_K (kaon at rest), and 1000
    events with |cos theta_K*| = |cos theta_psi| = 1 - 1e-9.  eps S of the full model and of the Z alone against the oracle's long
    double twin: 1e-11 wherever the FP64 oracle achieves it, never more than 4x the oracle's own error; the worst event is
    printed with its distance from the thresholds."""
    import arbitration as A
    cfg = 2
    Mo, Mg = oracle_model(cfg), gpu_model(cfg)
    c = W.couplings(cfg)
    slots = W.slot_table(W.resonances(cfg))
    cz = np.array([c[k] if W.resonances(cfg)[slots[k][0]][0] == O.ZRES else 0.0 for k in range(len(c))])
    rng = np.random.default_rng(33)
    samples = {f"m_Z threshold {which} within {dmax} MeV": A.threshold_events(Mo, which, 500, dmax, 9) for which in (0, 1) for dmax in (1.0, 1e-3)}
    n = 1000
    samples["|cos| = 1 - 1e-9"] = np.stack([rng.uniform(700.0, 2100.0, n), rng.choice([-1.0, 1.0], n) * W.COS_MAX,
                                           rng.choice([-1.0, 1.0], n) * W.COS_MAX, rng.uniform(-np.pi, np.pi, n)])
    for label, xs in samples.items():
        Mg.load_events(dev(xs), None)
        for what, cc in (("full model", c), ("Z alone", cz)):
            Mg.set_params(cc)
            v = Mg.eval_events(0).cpu().numpy()
            eg, eo, msg = A.check(v, Mo.eval_events(cc, xs), Mo.eval_events(cc, xs, prec=1), RTOL_EVENT, f"{label}, {what}", events=xs, oracle_model=Mo)
            print(f"{label}, {what}: max |gpu - ld| {eg:.2e}, max |oracle - ld| {eo:.2e}; {msg}")


def test_paths_without_held_columns_are_refused_not_read_as_one():
    """After a default P = 1 amp_set_params the lineshapes live in registers and no column is held: the matrix paths must say so
    (AMP_ERR_STATE) instead of building M with every Breit-Wigner replaced by 1; with amp_set_norm_mode(2) they work.  And a
    P >= 24 normalisation integral with a background set (lineshapes in registers) must not take the dense path on missing columns."""
    from paper_2007_14931_b200 import binding as B
    cfg = 2
    Mo, Mg = oracle_model(cfg), gpu_model(cfg)
    c = W.couplings(cfg)
    x, eff, xn, wn = make_inputs(cfg, 1500, 4000)
    Mg.load_events(dev(x), dev(eff))
    Mg.load_norm(dev(xn), dev(wn))
    Mg.set_params(c)
    Mg.nll()
    for call in (lambda: Mg.norm_matrix(0), lambda: Mg.fit_fractions(0)):
        with pytest.raises(B.AmpError) as e:
            call()
        assert e.value.status == B.AMP_ERR_STATE
    Mg.set_norm_mode(2)
    Mg.set_params(c)
    Mat = Mg.norm_matrix(0)
    ref = Mo.norm_matrix(xn, wn)
    assert np.max(np.abs(Mat - ref)) < 1e-12 * np.max(np.abs(ref))
    assert np.max(np.abs(Mg.fit_fractions(0) - Mo.fit_fractions(c, xn, wn))) < 1e-12
    Mg.set_norm_mode(0)
    # background set, 30 points: I(p) against the oracle, the likelihood against the plain definition of Eq. 14
    b = np.random.default_rng(5).uniform(0.5, 1.5, x.shape[1]) * np.mean(Mo.eval_events(c, x, eff)) / Mo.norm_integral(c, xn, wn)[0]
    Mg.set_background(dev(b), 0.85)
    P = 30
    cs = np.stack([c * np.exp(0.01j * p * np.arange(len(c))) * (1 + 0.003 * p) for p in range(P)])
    mws = np.stack([W.step_mass_width(3, p % 3) for p in range(P)])
    Mg.set_params(cs, mws)
    I = Mg.norm_integral()
    Iref = Mo.norm_integral(cs, xn, wn, mass_width=mws)
    assert np.max(np.abs(I - Iref) / Iref) < 1e-12
    nll = Mg.nll()
    ref = Mo.nll_background(cs, x, eff, b, 0.85, xn, wn, mass_width=mws)
    assert np.max(np.abs(nll - ref) / np.abs(ref)) < RTOL_NLL
    # the two sums of amp_nll_terms do not exist under Eq. 14
    with pytest.raises(B.AmpError) as e:
        Mg.nll_terms()
    assert e.value.status == B.AMP_ERR_STATE
    Mg.set_background(None, 1.0)
    Mg.set_params(c)
    slog, swS = Mg.nll_terms()
    assert np.isfinite(slog[0]) and swS[0] > 0


def test_fp64_probe_runs():
    from paper_2007_14931_b200 import binding as B
    dfma = B.probe_fp64(0, 500)
    dmma = B.probe_fp64(1, 500)
    assert 1e12 < dfma < 1e14 and 1e11 < dmma < 1e14


def test_hbm_read_probe_runs():
    from paper_2007_14931_b200 import binding as B
    gbs = B.probe_hbm_read(512 * 1024 * 1024)
    assert 1e3 < gbs < 1e4                          # a B200 streams several TB/s; the value itself is bench.py's business
    with pytest.raises(B.AmpError):
        B.probe_hbm_read(1000)                      # below one 512-event block

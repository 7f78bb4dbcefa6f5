"""amp_nll_static (include/amp.h): the fused NLL launch with its scratch in the library's static device array, for callers
that may not allocate.  Checked against the existing path (amp_nll) on the same model, two calls in a row.

Collected last on purpose (the suite runs with pytest -x); passes alone in a fresh process and after the other tests.
The data events are phase-space events here (both sides are the CUDA path; the oracle is not involved)."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from paper_2007_14931_b200 import binding as B
from paper_2007_14931_b200 import workloads as W

pytestmark = pytest.mark.gpu

RTOL_NLL = 1e-9    # the bar of tests/test_parity_gpu.py (BASELINE.json north_star)


def dev(a):
    return torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64).cuda()


def loaded_model(cfg=2, n=3001, m=7013):
    x, w = W.norm_events(cfg, n + m)          # ragged sizes: several tiles and a tail on both samples
    Mg = B.Model(W.DECAY, W.resonances(cfg))
    Mg.load_events(dev(x[:, :n]), dev(w[:n]))
    Mg.load_norm(dev(x[:, n:]), dev(w[n:]))
    return Mg


def test_static_scratch_entry_matches_amp_nll_on_two_calls_in_a_row():
    Mg = loaded_model()
    c = W.couplings(2)
    for step in range(2):                     # two different parameter points, the second call right after the first
        mw = W.step_mass_width(3, step)
        Mg.set_params(c * np.exp(0.1j * step * np.arange(len(c))), mw[None])
        out = torch.full((1, 6), float("nan"), dtype=torch.float64, device="cuda")
        Mg.nll_static(out)
        got = out.cpu().numpy()               # (synchronises)
        ref = Mg.nll()
        ref_I = Mg.norm_integral()
        assert got[0, 5] == 1.0 and got[0, 2] == 0.0, got
        assert abs(got[0, 0] - ref[0]) <= RTOL_NLL * abs(ref[0]), (step, got[0, 0], ref[0])
        assert abs(got[0, 1] - ref_I[0]) <= RTOL_NLL * abs(ref_I[0]), (step, got[0, 1], ref_I[0])
        print(f"step {step}: static {got[0, 0]!r} amp_nll {ref[0]!r} rel {abs(got[0, 0] - ref[0]) / abs(ref[0]):.1e}")
    # back to back on one stream without a synchronisation in between, then again: the shared array keeps the last call's
    # contents (ticket, flag, partials) and every call has to come out the same
    outs = [torch.full((1, 6), float("nan"), dtype=torch.float64, device="cuda") for _ in range(3)]
    free0 = torch.cuda.mem_get_info()[0]
    for o in outs:
        Mg.nll_static(o)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0, "the entry point allocated device memory"
    vals = [o.cpu().numpy() for o in outs]
    assert np.array_equal(vals[0], vals[1]) and np.array_equal(vals[0], vals[2]), vals
    assert np.array_equal(vals[0], got)       # and the same bits as the first call at these parameters


def test_static_scratch_entry_batch_of_points():
    Mg = loaded_model()
    c = W.couplings(2)
    P = B.AMP_STATIC_MAX_POINTS
    rng = np.random.default_rng(7)
    cs = np.stack([c * (1.0 + 0.2 * rng.standard_normal(len(c))) * np.exp(0.3j * rng.standard_normal(len(c))) for _ in range(P)])
    mws = np.stack([W.step_mass_width(3, p) for p in range(P)])
    Mg.set_params(cs, mws)
    ref = Mg.nll()                            # the existing path for a dense batch (other kernels: tolerance, not bits)
    for _ in range(2):
        out = torch.full((P, 6), float("nan"), dtype=torch.float64, device="cuda")
        Mg.nll_static(out)
        got = out.cpu().numpy()
        assert np.all(got[:, 5] == 1.0) and np.all(got[:, 2] == 0.0)
        rel = np.abs(got[:, 0] - ref) / np.abs(ref)
        assert np.all(rel <= RTOL_NLL), rel


def test_static_scratch_entry_rejects_what_does_not_fit():
    Mg = loaded_model(n=300, m=700)
    c = W.couplings(2)
    P = B.AMP_STATIC_MAX_POINTS + 1
    mw = W.step_mass_width(3, 0)
    Mg.set_params(np.stack([c] * P), np.stack([mw] * P))
    out = torch.zeros((P, 6), dtype=torch.float64, device="cuda")
    with pytest.raises(B.AmpError) as e:
        Mg.nll_static(out)
    assert e.value.status == B.AMP_ERR_INVALID and "AMP_STATIC_MAX_POINTS" in str(e.value), str(e.value)
    assert torch.count_nonzero(out).item() == 0          # nothing was launched
    empty = B.Model(W.DECAY, W.resonances(2))
    with pytest.raises(B.AmpError) as e:
        empty.nll_static(torch.zeros((1, 6), dtype=torch.float64, device="cuda"))
    assert e.value.status == B.AMP_ERR_STATE

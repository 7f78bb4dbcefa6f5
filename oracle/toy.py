"""Oracle of the accept-reject toy generator ("a distribution according to the fit model is
generated through MC techniques") — TEST INFRASTRUCTURE (see oracle/__init__.py).

The method, step by step (DESIGN.md "Toy generator" fixes what the paper leaves open — it only says "MC techniques"):

  1. candidate i (a 64-bit index) draws twelve 32-bit words from the counter-based generator Philox4x32-10
     (Salmon et al., SC'11): counter (i mod 2^32, i div 2^32, j, 0), key (seed mod 2^32, seed div 2^32), j = 0, 1, 2;
  2. five uniforms in [0, 1) with 53 bits each:  U_k = ((w_2k >> 5) * 2^26 + (w_2k+1 >> 6)) * 2^-53;
  3. the candidate point (Eq. 1, in the build's variables):
       m_Kpi = m_lo + (m_hi - m_lo) U_0,  cos theta_K* = (2 U_1 - 1) c_max,  cos theta_psi = (2 U_2 - 1) c_max,  phi = (2 U_3 - 1) pi;
  4. its weight f = p_B(m_Kpi) q(m_Kpi) S(x): the three-body phase-space density in these variables (d m2_Kpi d m2_psipi
     = 4 M_B p_B q dm dcos theta_K*, up to constants) times the signal density S of Eq. 12;
  5. accepted iff  U_4 f_max < f;  the toy is the accepted candidates in index order.

Each product and sum of steps 2-3 is a single correctly rounded FP64 operation in the order written, so the candidate stream
is reproducible bit for bit by any implementation; step 5 is a floating-point decision, exact except for candidates whose two
sides agree to rounding (the parity test lists and excludes those).

Pins (tests/test_oracle_pins.py): the generator against the known-answer vectors of the Philox4x32-10 publication; the uniforms'
range and resolution; a constant spin-0 model, for which the accepted events must follow p_B q in m_Kpi, sin^2 in theta_psi
(sum over xi of |d^1_{0 xi}|^2) and be flat in cos theta_K* and phi.
"""
import numpy as np

PHILOX_M0, PHILOX_M1 = 0xD2511F53, 0xCD9E8D57     # multipliers
PHILOX_W0, PHILOX_W1 = 0x9E3779B9, 0xBB67AE85     # key increments (golden ratio, sqrt(3) - 1)
_MASK = np.uint64(0xFFFFFFFF)


def philox4x32_10(counter, key):
    """counter: uint32 [n][4], key: (k0, k1) -> uint32 [n][4]; ten rounds of
         (c0, c1, c2, c3) <- (hi(M1 c2) ^ c1 ^ k0,  lo(M1 c2),  hi(M0 c0) ^ c3 ^ k1,  lo(M0 c0)),   key += (W0, W1) after each round."""
    c = np.asarray(counter, dtype=np.uint64).reshape(-1, 4) & _MASK
    c0, c1, c2, c3 = (c[:, j].copy() for j in range(4))
    k0, k1 = np.uint64(int(key[0]) & 0xFFFFFFFF), np.uint64(int(key[1]) & 0xFFFFFFFF)
    for _ in range(10):
        p0 = np.uint64(PHILOX_M0) * c0          # 32 x 32 -> 64 bit products, exact in uint64
        p1 = np.uint64(PHILOX_M1) * c2
        hi0, lo0 = p0 >> np.uint64(32), p0 & _MASK
        hi1, lo1 = p1 >> np.uint64(32), p1 & _MASK
        c0, c1, c2, c3 = hi1 ^ c1 ^ k0, lo1, hi0 ^ c3 ^ k1, lo0
        k0 = (k0 + np.uint64(PHILOX_W0)) & _MASK
        k1 = (k1 + np.uint64(PHILOX_W1)) & _MASK
    return np.stack([c0, c1, c2, c3], -1).astype(np.uint32)


def uniform53(a, b):
    """two 32-bit words -> a double in [0, 1) with 53 random bits (step 2)"""
    a = np.asarray(a, dtype=np.uint32).astype(np.uint64)
    b = np.asarray(b, dtype=np.uint32).astype(np.uint64)
    return ((a >> np.uint64(5)).astype(np.float64) * 67108864.0 + (b >> np.uint64(6)).astype(np.float64)) * (1.0 / 9007199254740992.0)


def candidates(seed, first, n, m_lo, m_hi, cos_max):
    """(x [4][n], u [n]) of candidates first .. first + n - 1 (steps 1-3)"""
    i = np.uint64(first) + np.arange(n, dtype=np.uint64)
    key = (int(seed) & 0xFFFFFFFF, (int(seed) >> 32) & 0xFFFFFFFF)
    words = []
    for j in range(3):
        ctr = np.stack([i & _MASK, i >> np.uint64(32), np.full(n, j, dtype=np.uint64), np.zeros(n, dtype=np.uint64)], -1)
        words.append(philox4x32_10(ctr, key))
    w = np.concatenate(words, -1)               # [n][12]
    U = [uniform53(w[:, 2 * k], w[:, 2 * k + 1]) for k in range(5)]
    x = np.empty((4, n))
    x[0] = m_lo + (m_hi - m_lo) * U[0]
    x[1] = (2.0 * U[1] - 1.0) * cos_max
    x[2] = (2.0 * U[2] - 1.0) * cos_max
    x[3] = (2.0 * U[3] - 1.0) * np.pi
    return x, U[4]


def _two_body(M, a, b):
    return np.sqrt((M - (a + b)) * (M + (a + b)) * (M - (a - b)) * (M + (a - b))) / (2.0 * M)


def weights(model, couplings, x):
    """f = p_B q S of candidate points x [4][n] (step 4); `model` is an oracle.Model"""
    MB, mpsi, mK, mpi = (float(v) for v in model.decay)
    return _two_body(MB, x[0], mpsi) * _two_body(x[0], mK, mpi) * model.eval_events(couplings, x)


def generate(model, couplings, seed, first, n, f_max, m_lo, m_hi, cos_max):
    """-> dict(x = accepted events [4][n_acc] in candidate order, index = their candidate numbers (relative to `first`),
               f [n] = all weights, u [n], f_seen_max)  (steps 1-5)"""
    x, u = candidates(seed, first, n, m_lo, m_hi, cos_max)
    f = weights(model, couplings, x)
    keep = u * f_max < f
    return {"x": x[:, keep], "index": np.nonzero(keep)[0], "f": f, "u": u, "f_seen_max": float(np.max(f)) if n else 0.0}

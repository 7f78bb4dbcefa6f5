/* amp.h — C ABI of libamp4d: the per-event unbinned negative log-likelihood of the 4D
 * helicity-amplitude model for B0 -> J/psi K+ pi-, J/psi -> mu+ mu- (ten K* resonances and an
 * exotic Z+ -> J/psi pi+), evaluated by hand-written sm_100a CUDA kernels.
 *
 * Paper: Sur et al., "A GPU based multidimensional amplitude analysis to search for tetraquark
 * candidates", J Big Data 8:16 (2021) — cited below as PAPER.md:<line> (+ equation).
 *
 * The calls follow the paper's statement of the problem: the minimiser on the host
 * proposes a parameter vector at every step, the device evaluates the PDF over all events and
 * returns one scalar.  Events (4 doubles each, Eq. 1) are loaded once per data
 * set; the normalisation integral is a sum over "several million phase space points"
 * (PAPER.md:53), loaded once as well.
 *
 * Conventions
 *  - Units: MeV; Blatt-Weisskopf radius in MeV^-1.
 *  - `d_` arguments are DEVICE pointers, `h_` arguments are HOST pointers.  Device input buffers
 *    are borrowed for the duration of the call only: the library builds its own cache from them
 *    on `stream` and the caller may free them after synchronising that stream.
 *  - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  All work of a
 *    model is issued on the stream given to the call; calls that return host data synchronise it.
 *  - No exception or abort crosses the ABI.  Every call returns an amp_status; amp_last_error()
 *    gives the text of the last failure of that model.
 *  - One amp_model per host thread; calls on one model are not re-entrant.
 *  - There is no CPU fallback: without a CUDA device every compute call returns AMP_ERR_CUDA.
 */
#ifndef AMP4D_AMP_H
#define AMP4D_AMP_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct amp_model amp_model; /* opaque; owns all device state */

typedef enum {
    AMP_OK = 0,
    AMP_ERR_INVALID = 1, /* null pointer, bad size, J out of range, too many resonances / points          */
    AMP_ERR_STATE = 2,   /* call order: amp_nll before amp_load_events / amp_load_norm / amp_set_params   */
    AMP_ERR_DOMAIN = 3,  /* event outside phase space, pole mass outside the kinematic range,
                            non-finite or non-positive PDF value                                          */
    AMP_ERR_CUDA = 4,    /* CUDA runtime error (text in amp_last_error)                                   */
    AMP_ERR_NOMEM = 5    /* device or host allocation failed                                              */
} amp_status;

/* Resonance kinds.  AMP_KSTAR: K* -> K pi, Eq. 4.  AMP_Z: Z -> J/psi pi evaluated in
 * its own decay frame, Eq. 10, of POSITIVE parity: J^P = 1+ (the paper's default) or 2+;
 * AMP_ZM: the same of NEGATIVE parity: 0-, 1-, 2- ("any combination of their spin-parity values").  Orbital
 * momenta of the Z chain: L_B = J; L_R = lowest L with (-1)^L = P and |L - 1| <= J <= L + 1 (1+: 0, 2+: 2, 0-/1-/2-: 1; 0+
 * does not decay to J/psi pi and is refused).  A Z always has three coupling slots lambda' = -1, 0, +1 (for J = 0 the
 * lambda' = +-1 slots multiply a zero d function); Eq. 11's relation between them is the caller's.  The fused shape-specialised
 * kernels and the gradient-batch kernel cover 1+ Zs; other spin-parities run the generic streaming kernel and, for parameter
 * batches, the dense path.  AMP_CONST: lineshape == 1,
 * J = 0, angular factor d^1_{0 xi}(theta_psi) (BASELINE.json configs[0], "constant S-wave term").
 * AMP_LASS: the LASS parametrisation of the K pi S-wave, Eqs. 7-9: J = 0, one coupling slot,
 * lineshape A_LASS built on mass = M(K0*(1430)), width = Gamma(K0*(1430)) with the paper's a = 1.95 GeV^-1,
 * b = 1.76 GeV^-1 (Eq. 8); radius is ignored.  Models with a LASS term run the generic streaming kernel; gradient
 * batches of such models take the dense path.                                                          */
typedef enum { AMP_KSTAR = 0, AMP_Z = 1, AMP_CONST = 2, AMP_LASS = 3, AMP_ZM = 4 } amp_kind;

/* One resonance: spin J (K*: 0..4, AMP_Z: 1..2, AMP_ZM: 0..2, CONST: 0), nominal mass M_R and width
 * Gamma_0 [MeV], Blatt-Weisskopf radius r [MeV^-1] used for both F_B and F_R of Eq. 2 (PAPER.md:89,
 * 103).  Orbital momenta: K*: L_R = J, L_B = J-1 (J >= 1) or 1 (J = 0), the lowest allowed
 * (PAPER.md:107); Z: L_B = 1, L_R = 0.                                                               */
typedef struct {
    int kind;
    int J;
    double mass, width, radius;
} amp_resonance;

/* Masses of B0, J/psi, K+, pi- [MeV] (symbols of Eq. 2). */
typedef struct {
    double m_parent, m_psi, m_k, m_pi;
} amp_decay;

enum { AMP_MAX_RESONANCES = 16, AMP_MAX_COUPLINGS = 48, AMP_MAX_POINTS = 256 };

/* Create a model from the decay constants and a resonance list (copied).  Fails with AMP_ERR_INVALID on
 * bad J / kind / non-positive mass or width / n_res > AMP_MAX_RESONANCES, AMP_ERR_DOMAIN if a pole mass
 * lies outside the kinematic range of its chain (its pole momenta would not exist), AMP_ERR_CUDA if no
 * device is usable.  *out is owned by the caller and released with amp_model_destroy.                 */
amp_status amp_model_create(const amp_decay* decay, const amp_resonance* res, int n_res, amp_model** out);
amp_status amp_model_destroy(amp_model* m);

/* K = number of complex coupling slots.  Slot order: resonance order, then lambda = -1, 0, +1 for a
 * K* with J >= 1 and for the Z (lambda' for the Z), lambda = 0 only for J = 0 and AMP_CONST
 * ("For K*s with zero spin, only lambda = 0 is allowed").  Returns -1 on a null model. */
int amp_num_couplings(const amp_model* m);
int amp_num_resonances(const amp_model* m);

/* Load the data events and build the parameter-independent per-event cache (breakup momenta,
 * d-function arguments, phi phases, Z-frame mass and angles: Eqs. 1, 4, 10; "Lorentz
 * boosts and rotations", :171-179).
 *   d_x   device, FP64 structure-of-arrays [4][n]: m_Kpi [MeV], cos(theta_K*), cos(theta_J/psi), phi
 *         [rad] (the variables of Eq. 1 with m_J/psi pi replaced by the equivalent cos(theta_K*)).
 *   d_eff device [n] relative efficiency eps_i > 0 (Eq. 14), or NULL (= 1).
 * Replaces a previously loaded data set.  n >= 0 (n == 0: NLL data term is 0).  Synchronises `stream`.
 * AMP_ERR_DOMAIN if any event is outside phase space (m_Kpi not in (m_K+m_pi, m_B-m_psi), |cos| > 1,
 * non-finite input, eps <= 0) or, for a model with a Z, has an undefined Z-chain angle (mu+ exactly along the pion in the
 * J/psi frame — e.g. cos(theta_K*) = +-1 together with cos(theta_J/psi) = +-1 — or m_J/psi pi exactly at a threshold:
 * PAPER.md:176-179 define the angles between planes that then do not exist); the data set is then left unloaded.     */
amp_status amp_load_events(amp_model* m, const double* d_x, const double* d_eff, long long n, void* stream);

/* Load the phase-space Monte Carlo sample used for the normalisation integral.
 *   d_x as above, [4][n_norm]; d_w device [n_norm] weights w_j >= 0 (efficiency x quadrature weight) or
 *   NULL (= 1).  The integral is I = sum_j w_j S(x_j) / sum_j w_j.  Same errors as amp_load_events.   */
amp_status amp_load_norm(amp_model* m, const double* d_x, const double* d_w, long long n_norm, void* stream);

/* Set P >= 1 parameter points (P <= AMP_MAX_POINTS).
 *   h_couplings  host [P][K][2]: complex helicity couplings H (re, im) in slot order (Eqs. 4, 10).  The
 *                constraints of Eq. 6 and Eq. 11 are the caller's business:
 *                the library treats all K slots as free.
 *   h_mass_width host [P][R][2]: (mass, width) of every resonance at every point, or NULL (= the values
 *                given at amp_model_create).  Entries of AMP_CONST resonances are ignored.
 * The library compares each (resonance, mass, width) with the lineshape columns it holds and marks only
 * the missing ones for recomputation (done lazily by the next evaluation call).  Copies both arrays.    */
amp_status amp_set_params(amp_model* m, int P, const double* h_couplings, const double* h_mass_width);

/* NLL(p) = - sum_i log( eps_i S_i(p) / I(p) ) for the P points of the last amp_set_params, with
 * S = sum_xi |sum_k H_k B_k,xi|^2 (Eqs. 5, 12) and I(p) the Monte Carlo integral.
 *   h_nll host [P].  Synchronous with respect to h_nll.  Deterministic: the same inputs give the same
 * bits (fixed-order reductions, no floating-point atomics).
 * AMP_ERR_STATE without data / norm sample / parameters; AMP_ERR_DOMAIN if some eps_i S_i or I(p) is not
 * finite and positive: h_nll[p] = +inf for those points, the others are valid.                         */
amp_status amp_nll(amp_model* m, double* h_nll, void* stream);

/* amp_nll for callers that may not allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): the same one-launch evaluation as amp_nll at a single point with floating lineshapes (k_stream<MODE_FUSED>,
 * Eqs. 5, 12 and the Monte Carlo integral), one launch per point of the last amp_set_params, with the
 * kernel's scratch (per-CTA partial sums, the last-CTA ticket, the domain flag) in a file-scope `static __device__` array of
 * the library instead of the model's buffers.  It calls no cudaMalloc / cudaFree / allocating library routine, copies nothing
 * and does not synchronise: the launches are enqueued on `stream` and the call returns.
 *   d_out DEVICE [P][6], caller-owned: per point NLL, I, domain flag (non-zero: some eps_i S_i or I was not finite and positive,
 *   NLL = +inf), sum_i log S_i, sum_j w_j S_j, and 1.0 (written last: the block is complete).  Same bits as amp_nll for the same
 *   inputs (same kernel, same grid, same fixed-order sums).
 * Limits: P <= AMP_STATIC_MAX_POINTS and a persistent grid of at most AMP_STATIC_MAX_CTAS CTAs (2 per SM); beyond them
 * AMP_ERR_INVALID with a message that names the limit.  AMP_ERR_STATE without data / norm sample / parameters or with a
 * background set (Eq. 14 needs a second pass over model-owned buffers).  Lineshapes are always evaluated in registers
 * (amp_set_lineshape_mode is not consulted: pool columns are model-owned buffers).  The array (AMP_STATIC_SCRATCH_BYTES = 133 120 B) is held by every device that loads the library until
 * the process exits; its address is looked up once per device (cudaGetSymbolAddress, with the model's device current) on the first
 * call there.  EVERY call on a device shares it and it keeps the last call's contents: the ticket and flag words are cleared on
 * `stream` before each launch, so calls on ONE stream are safe back to back, while calls that overlap on the GPU (two streams, two
 * host threads, two models on one device) race on it - serialise them.                                                     */
#define AMP_STATIC_MAX_POINTS 8
#define AMP_STATIC_MAX_CTAS 1024
#define AMP_STATIC_SCRATCH_BYTES (AMP_STATIC_MAX_POINTS * (2 * AMP_STATIC_MAX_CTAS * 8 + 256))
amp_status amp_nll_static(amp_model* m, double* d_out, void* stream);

/* NLL and its analytic gradient in the couplings at the single point of the last amp_set_params (P = 1), in ONE pass over
 * the data and normalisation events (one launch):
 *   h_nll host [1]; h_grad host [K][2] = (dNLL/dRe H_k, dNLL/dIm H_k) in slot order, from
 *   dNLL/dconj(H_k) = - sum_i [sum_xi conj(B_k,xi) A_xi]_i / S_i + N [sum_j w_j sum_xi conj(B_k,xi) A_xi]_j / [sum_j w_j S_j].
 * Replaces the 2 K finite-difference points a minimiser would spend on the couplings (masses and widths still go through
 * a gradient batch; amp_fit does both).  Constraints such as Eq. 6 / Eq. 11 are the caller's chain rule.  With masses and
 * widths unchanged since the previous amp_set_params the normalisation side comes from the held matrix M ((M c)_k, c^H M c) and
 * only the data events are walked.  With a background (amp_set_background, Eq. 14) the data-side weights are
 * purity eps_i / (I f_i) and N becomes sum_i u_i S_i; sum_j w_j S_j is then needed first: from M inside the kernel, or from a
 * normalisation launch before it (3 launches).  Models with LASS terms and Zs of any spin-parity are covered.
 * Deterministic.  Path 7 in amp_last_call_stats.                                                                        */
amp_status amp_nll_grad(amp_model* m, double* h_nll, double* h_grad, void* stream);

/* Fit in native code (the paper's MINUIT loop, with the analytic gradient in place of finite differences for the
 * couplings): BFGS with a strong-Wolfe line search over Re, Im of the free helicity couplings and, optionally, masses and
 * widths of chosen resonances ("floating masses/widths").  Every evaluation is one amp_set_params + one
 * amp_nll_grad; with floating lineshape parameters one more batch of 1 + 2 n_float_mw points (amp_nll; central differences
 * of the NLL over +- 1 % of the width).  Needs data and normalisation events loaded.
 *   h_start      host [K][2] start values; fixed slots keep them
 *   h_mass_width host [R][2] start / fixed masses and widths, or NULL (= the values given at amp_model_create; only
 *                without floating lineshape parameters)
 *   fixed        [n_fixed] slots held constant (Eq. 6: the K*(892) lambda = 0 amplitude)
 *   tie_dst/src  [n_ties] H[dst] = sign * H[src] (Eq. 11); a dst is not free, not fixed, not a src of another tie
 *                and appears once
 *   tie_sign     [n_ties] +1 or -1, or NULL (= all +1).  Eq. 11 is H_+1 = H_-1 for the 1+ Z the paper considers; parity
 *                conservation in Z -> J/psi pi gives H_l' = P (-1)^(1 - J) H_-l' in general (A24), i.e. -1 for 2+ and 1-
 *   float_mw     [n_float_mw][2] = (resonance index, 0: its mass / 1: its width) floating lineshape parameters, no duplicates
 *   h_scale      host [K] positive parameter scales or NULL (= |start|, floored at 1e-3 of the largest); masses and widths
 *                are scaled by the start width
 *   max_iter, gtol   iteration cap; converged when max |dNLL/d(parameter / scale)| < gtol
 *   h_fit        host [K][2] fitted couplings (ties applied);  h_fit_mw host [R][2] fitted masses and widths, or NULL;
 *   h_nll        host [2]: NLL at the fit, max |gradient| there
 *   h_cov        host [n][n], n = 2F + n_float_mw (F = free slots, ascending; Re, Im per slot; then float_mw order): covariance
 *                = inverse Hessian of the NLL, the Hessian from central differences of the gradient (2 n more evaluations); or NULL
 *   h_info       host int[5] or NULL: converged, likelihood evaluations, iterations, covariance valid (Hessian positive definite
 *                and every evaluation behind it finite; else h_cov is NaN), n
 * The model is left with the fitted point set.  Errors of amp_set_params / amp_nll_grad / amp_nll are passed on (a trial point
 * outside the likelihood's domain makes the line search back off); AMP_ERR_INVALID for bad indices, chained ties, duplicates
 * or a non-positive scale; AMP_ERR_DOMAIN if the start point has no finite likelihood.                                       */
amp_status amp_fit(amp_model* m, const double* h_start, const double* h_mass_width, const int* fixed, int n_fixed,
                   const int* tie_dst, const int* tie_src, const int* tie_sign, int n_ties, const int* float_mw, int n_float_mw,
                   const double* h_scale, int max_iter, double gtol,
                   double* h_fit, double* h_fit_mw, double* h_nll, double* h_cov, int* h_info, void* stream);

/* Accept-reject toy generator ("a distribution according to the fit model is generated through MC techniques";
 * the recipe the paper leaves open is fixed in DESIGN.md "Toy generator").  For the candidate numbers
 * first .. first + n_candidates - 1, at the single point of the last amp_set_params (P = 1):
 *   twelve 32-bit words of Philox4x32-10 (counter (i mod 2^32, i div 2^32, j, 0), key (seed mod 2^32, seed div 2^32), j = 0..2)
 *   -> five uniforms U = ((w_a >> 5) 2^26 + (w_b >> 6)) 2^-53  ->  the point (Eq. 1)
 *   x = (m_lo + (m_hi - m_lo) U0, (2 U1 - 1) cos_max, (2 U2 - 1) cos_max, (2 U3 - 1) pi),
 *   accepted iff  U4 f_max < f(x),  f = p_B(m_Kpi) q(m_Kpi) S(x)  (phase-space density in these variables x Eq. 12).
 * The accepted points are written in candidate order (independent of scheduling; the candidate stream itself is reproducible
 * bit for bit): d_x_out DEVICE [4][capacity] SoA (stride = capacity), d_index_out DEVICE [capacity] their candidate numbers
 * (may be null).  *h_n_accepted = number accepted (points beyond `capacity` are counted, not written); *h_f_seen_max =
 * largest f among the candidates (if it exceeds f_max the toy is biased: raise f_max and call again; f_max = 0 accepts all).
 * Efficiency is not applied: thin the toy by eps(x) afterwards, as a detector simulation would.  Needs neither data nor
 * normalisation events; leaves both untouched.  AMP_ERR_INVALID: mass range not strictly inside (m_K + m_pi, m_B - m_psi),
 * cos_max outside (0, 1], negative or non-finite f_max, null outputs; AMP_ERR_STATE: no parameters, P != 1, or lineshape
 * columns forced (amp_set_lineshape_mode 1); AMP_ERR_DOMAIN: a candidate weight is not finite.                              */
amp_status amp_generate(amp_model* m, unsigned long long seed, unsigned long long first, long long n_candidates,
                        double f_max, double m_lo, double m_hi, double cos_max,
                        double* d_x_out, long long* d_index_out, long long capacity,
                        long long* h_n_accepted, double* h_f_seen_max, void* stream);

/* Background and signal purity, Eq. 14: with a background set, amp_nll returns
 *   NLL(p) = - sum_i log( purity * eps_i S_i(p) / I(p) + (1 - purity) * b_i ).
 *   d_bkg device [n]: the normalised background density b(Phi_i) >= 0 at the loaded data events (copied), or NULL to go back
 *   to the signal-only likelihood; purity in [0, 1] (the paper uses 0.85).  Call after amp_load_events and before
 *   amp_set_params (loading a new data set drops the background).  Such evaluations run one normalisation launch and one
 *   data launch per point (path 6); amp_nll_terms is not defined for them (the sums no longer separate).             */
amp_status amp_set_background(amp_model* m, const double* d_bkg, double purity, void* stream);

/* The two sums behind amp_nll, for callers that shard the events over several devices or processes:
 *   h_sum_log[p] = sum_i log S_i(p) over the loaded data events (without the efficiency), h_sum_wS[p] = sum_j w_j S_j(p)
 * over the loaded normalisation events, host [P] each.  With the constants of amp_dataset_sums summed over the shards,
 *   NLL(p) = -( sum_shards sum_log[p] + sum_shards sum_log_eff ) + N_total log( sum_shards sum_wS[p] / sum_shards sum_w ).
 * Same launches, states and errors as amp_nll; AMP_ERR_STATE with a background set (Eq. 14 does not separate).       */
amp_status amp_nll_terms(amp_model* m, double* h_sum_log, double* h_sum_wS, void* stream);
/* Per-dataset constants fixed at load time: number of data events, sum_i log eps_i, number of normalisation events,
 * sum_j w_j (0 for a sample that is not loaded).  Any output pointer may be NULL.                                     */
amp_status amp_dataset_sums(const amp_model* m, long long* n_data, double* sum_log_eff, long long* n_norm, double* sum_w);

/* Diagnostics / parity. */
/* d_out device [n]: eps_i * S_i(p) of the loaded data events for point p of the last amp_set_params.   */
amp_status amp_eval_events(amp_model* m, int p, double* d_out, void* stream);
/* h_I host [P]: I(p) = sum_j w_j S_j(p) / sum_j w_j.                                                   */
amp_status amp_norm_integral(amp_model* m, double* h_I, void* stream);
/* d_out device [ncols][n] (or [ncols][n_norm] if which == 1): the kinematics cache columns, in the order
 * returned by amp_cache_column_name(i); *ncols receives the count (pass d_out == NULL to query).       */
amp_status amp_dump_cache(amp_model* m, int which, double* d_out, int* ncols, void* stream);
const char* amp_cache_column_name(int i);
/* d_out device [n or n_norm][2]: A^R(m) of resonance r at (mass, width) (Eqs. 2-3).                    */
amp_status amp_eval_lineshape(amp_model* m, int which, int r, double mass, double width, double* d_out, void* stream);
/* h_M host [K][K][2]: Hermitian normalisation matrix M_kl = sum_j w_j sum_xi conj(B_k,xi) B_l,xi / sum_j w_j
 * at the lineshapes of point p, so that I(p) = c^H M c (fit fractions of Eq. 13, are ratios
 * of its diagonal blocks).                                                                             */
amp_status amp_norm_matrix(amp_model* m, int p, double* h_M, void* stream);
/* h_ff host [R]: fit fraction of every resonance at point p, Eq. 13 (the printed denominator "|S|^2" read
 * as the integral of the density S):  FF_r = sum_j w_j S_r(x_j) / sum_j w_j S(x_j) over the loaded normalisation sample, S_r
 * the density with all helicity amplitudes but those of resonance r set to zero.  Evaluated on the device as quadratic
 * forms c_r^H M c_r / c^H M c of the normalisation matrix (built by the HERK kernel if it is not held).  Load the sample
 * with unit weights for efficiency-free fractions.  Same call-order requirement as amp_norm_matrix
 * (amp_set_norm_mode(m, 2) before amp_set_params).                                                                  */
amp_status amp_fit_fractions(amp_model* m, int p, double* h_ff, void* stream);

/* How the normalisation integral is evaluated: 0 = automatic (default), 1 = always the direct sum over
 * the norm events, 2 = always through the matrix M (rebuilt when a lineshape it depends on changes).   */
amp_status amp_set_norm_mode(amp_model* m, int mode);
/* How missing lineshape columns are produced when P == 1: 0 = automatic (a resonance whose column missed
 * on two successive calls is floating: evaluate it in registers inside the combine kernel, no HBM round
 * trip), 1 = always store columns in the pool, 2 = always evaluate missing columns in registers.        */
amp_status amp_set_lineshape_mode(amp_model* m, int mode);
/* How P > 1 points are evaluated: 0 = automatic: a batch whose points 1..P-1 differ from point 0 in few resonances (a
 * MINUIT-style gradient step: on average <= 3 changed resonances per point) runs the gradient-batch kernel, one fused
 * launch over data and normalisation events with no lineshape column and no matrix; any other batch with P >= 24, at
 * most 28 couplings and an extended basis that fits in shared memory runs one dense DMMA launch per sample; else as
 * mode 1.  1 = a loop of single-point streaming launches over the stored lineshape columns.  2 = as 0 without the
 * gradient-batch kernels (dense DMMA contraction even for sparse batches).  3 = as 0 without the shape-specialised form of the
 * gradient-batch kernel.  Under 0, a sparse batch of the paper's resonance lists (ten K* with zero to two 1+ Z's, one radius
 * per spin) in which every point is ONE coupling change (a single slot, or a Z's helicities -1 and +1 moving together, Eq. 11)
 * or ONE mass / width change, at most four per slot / resonance — MINUIT's gradient step — runs that form: three launches for all
 * points (two passes over the normalisation events, whose sums do not depend on the point, then the data events), exact, S(p) / S(0) formed
 * directly; a step so large that the ratio leaves [0.5, 1.5] at some event repeats the call through the general kernel.
 * 4 = as 0 with that form as ONE launch over both samples (the cross-check of the two-launch form).                   */
amp_status amp_set_batch_mode(amp_model* m, int mode);
/* How a P == 1 step with lineshapes in registers and a direct-sum normalisation is launched: 0 = automatic (ONE fused
 * launch: data tiles, then normalisation tiles, the last thread block forms the NLL), 1 = separate data / normalisation /
 * reduction launches (per-phase timing, parity tests of the two forms against each other).                       */
amp_status amp_set_fused_mode(amp_model* m, int mode);
/* Which kernel amp_nll_grad / amp_fit run: 0 = automatic (the paper's resonance lists — ten K* with zero to two 1+ Z's,
 * one radius per spin, no LASS / constant term, no background — run the shape-specialised kernel that keeps every
 * gradient component in registers; any other model the generic one), 1 = always the generic kernel (parity tests of the
 * two against each other).                                                                                        */
amp_status amp_set_grad_mode(amp_model* m, int mode);
/* Counters of the last amp_nll / amp_norm_integral call: kernels launched, lineshape columns
 * recomputed (data + norm), which normalisation path ran (1 direct streaming sum, 2 matrix, 3 batched DMMA sum,
 * 4 fused single launch, 5 gradient-batch delta kernel, 6 background + purity, 7 analytic gradient, generic kernel,
 * 8 analytic gradient, shape-specialised kernel, 9 gradient batch, shape-specialised kernel).                         */
amp_status amp_last_call_stats(const amp_model* m, int* launches, int* columns_recomputed, int* norm_path);

/* Device time [ms] of the phases of the last amp_nll / amp_norm_integral call, from CUDA events recorded on
 * the call's stream: ms4[0] lineshape columns, ms4[1] data-side combine + reduce, ms4[2] normalisation,
 * ms4[3] final reductions and the copy of the result.  After a fused single launch (path 4): ms4[1] = that launch,
 * the others 0.  After the three launches of a shape-specialised gradient batch (path 9, batch mode 0): ms4[2], ms4[3] = the
 * two passes over the normalisation events, ms4[1] = the data events, ms4[0] = 0.                          */
amp_status amp_last_call_timing(const amp_model* m, double* ms4);

/* Device time [ms] of the launches of the most recent single-launch evaluations (paths 4 and 5), from CUDA event pairs
 * recorded around them on the call's stream and kept in a ring of 256: h_ms[0 .. *n_out) = the last min(max_calls, 256,
 * calls so far) such evaluations, oldest first.  Reading costs nothing in the timed calls themselves (bench.py's
 * roofline).  The evaluations must have completed (amp_nll is synchronous).                                        */
amp_status amp_recent_launch_ms(const amp_model* m, int max_calls, double* h_ms, int* n_out);

const char* amp_last_error(const amp_model* m);
const char* amp_status_string(amp_status s);
const char* amp_version(void);

/* FP64 throughput probes used for the roofline denominators: run `iters`
 * dependent-chain rounds of register-resident DFMA (kind 0) or mma.sync m8n8k4 f64 (kind 1) on every SM
 * and return achieved FLOP/s in *flops (timed with CUDA events on `stream`).                          */
amp_status amp_probe_fp64(int kind, int iters, double* flops, void* stream);

/* Read-bandwidth probe for the HBM roofline of the streaming kernels: allocates a scratch
 * buffer of `bytes` (rounded down to whole 512-event blocks of 184 B per event; use more than the 126 MB L2), streams
 * it through k_stream's own TMA tile pipeline (same grid, block, shared-memory staging; no model arithmetic) and
 * returns the best of five timed passes in *gbs (GB/s, CUDA events on `stream`).  The buffer is freed before
 * returning.  AMP_ERR_INVALID: gbs NULL or bytes below one block; AMP_ERR_NOMEM / AMP_ERR_CUDA otherwise.          */
amp_status amp_probe_hbm_read(long long bytes, double* gbs, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* AMP4D_AMP_H */

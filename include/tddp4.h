/*
 * tddp4.h -- C-ABI boundary of the B200-native time-dependent four-body amplitude likelihood.
 *
 * What it computes: the per-event time-dependent D0 -> K+ pi- pi+ pi- decay rate of arXiv:1702.06735
 * eq. (1) with the two amplitudes A_f, Abar_f modelled as coherent sums of
 * quasi-two-body decay chains, eq. (2), its Monte-Carlo normalisation over a
 * phase-space sample, the negative log-likelihood handed to a host-side minimiser
 * (PAPER.md lines 14, 18, 95), and the companion pseudo-event generator (phase-space generation followed
 * by accept/reject against the same rate).  Formulas the paper does not print
 * (spin factors, lineshapes, barrier factors, time integrals, Raubold-Lynch generation, Philox streams)
 * follow the readings O-1 .. O-9 of SURVEY.md 8(c), restated in DESIGN.md.
 *
 * Conventions
 *   - Units GeV and ps.  Metric (+,-,-,-).  Four-vectors are (E, px, py, pz).
 *   - Final-state order: 0 = K+, 1 = pi-, 2 = pi+, 3 = pi-.
 *   - Event layout is SoA fp64: p4[(4*particle + component) * ld + event], ld = row stride in doubles.
 *   - Every function returns TDDP4_OK (0) or a negative tddp4_status; no exception crosses the boundary;
 *     tddp4_last_error() gives a text for the last failure of that handle.
 *   - "host" / "device" on a pointer says where the memory must live.  The caller owns every buffer it
 *     passes; the handle owns only its internal caches.  Device buffers must belong to the CUDA device
 *     that was current at tddp4_create().
 *   - All work is enqueued on the handle's stream (tddp4_set_stream; default: a private non-blocking
 *     stream).  Calls that return a value to the host synchronise that stream; *_async calls do not.
 *   - A handle is not thread-safe; use one per host thread.
 *   - There is no CPU fallback: without a usable CUDA device tddp4_create() fails with TDDP4_ERR_CUDA.
 */
#ifndef TDDP4_H
#define TDDP4_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct tddp4 tddp4; /* opaque handle */

typedef enum {
  TDDP4_OK = 0,
  TDDP4_ERR_ARG = -1,       /* bad argument / model description                                  */
  TDDP4_ERR_CUDA = -2,      /* CUDA runtime error (text in tddp4_last_error)                     */
  TDDP4_ERR_CAPACITY = -3,  /* generate: more accepted events than `capacity` (counts are exact) */
  TDDP4_ERR_DOMAIN = -4,    /* a resonance pole mass is below its own decay threshold            */
  TDDP4_ERR_NONFINITE = -5, /* some P_i <= 0 or non-finite: *nll_out = +inf                       */
  TDDP4_ERR_STATE = -6      /* call order: events or parameters missing                          */
} tddp4_status;

/* limits of one model */
#define TDDP4_MAX_RES 16
#define TDDP4_MAX_TERMS 32
#define TDDP4_MAX_COUPLINGS 16

/* Spin-factor kinds.  The two topologies of PAPER.md Fig. 2 (lines 40-44):
 *   VV_*   : D -> R1 R2, R1 -> (perm[0] perm[1]), R2 -> (perm[2] perm[3]);   res = {R1, R2}
 *   AP_S   : D -> X perm[3], X -> V perm[2] (S-wave), V -> (perm[0] perm[1]); res = {X, V}, X axial
 *   TP_D   : same cascade, X a tensor, both X vertices in D-wave;            res = {X, V}
 *   NONRES : constant amplitude 1;                                           res = {-1, -1}          */
enum {
  TDDP4_SF_NONRES = 0, TDDP4_SF_VV_S = 1, TDDP4_SF_VV_P = 2, TDDP4_SF_VV_D = 3,
  TDDP4_SF_AP_S = 4, TDDP4_SF_TP_D = 5,
  TDDP4_SF_AP_D = 6   /* the AP_S cascade with X -> V perm[2] in D-wave: d_mu L2^{mu nu}(p_X, q_X) v_nu (the resonance
                       * entry of X then has L = 2); further building block in the sense of PAPER.md line 51          */
};
/* Lineshape kinds ("resonance lineshapes" are a class of building blocks; the paper names none):
 * 0 relativistic Breit-Wigner with mass-dependent width and Blatt-Weisskopf ratio (O-6);
 * 1 relativistic Breit-Wigner with constant width, T = 1 / (m0^2 - s - i m0 Gamma0).                               */
enum { TDDP4_LS_RUNNING = 0, TDDP4_LS_CONSTANT = 1 };

typedef struct {
  int L;         /* orbital angular momentum of the resonance's own decay: exponent 2L+1 of the running width
                    and order of its Blatt-Weisskopf factor (O-5, O-6).  m0, Gamma0 come via tddp4_set_params.
                    A state that decays in two partial waves is listed twice (one entry per L).              */
  int lineshape; /* TDDP4_LS_*                                                                                 */
  double r;      /* Blatt-Weisskopf radius of this resonance's own vertex, GeV^-1; 0: the model's r_res        */
} tddp4_res;

typedef struct {
  int spin_factor; /* TDDP4_SF_*                                                       */
  int res[2];      /* resonance indices, see above; -1 = none                          */
  int perm[4];     /* role -> final-state index; a permutation of 0..3                 */
  int coupling;    /* kappa(k): which complex coupling multiplies this chain, eq. (2); *
                    * Bose-symmetrised orderings share one coupling  */
} tddp4_term;

typedef struct {
  double m_parent;     /* nominal D0 mass; used by the generator only (event kinematics use p^2)     */
  double m_final[4];
  double r_res;        /* Blatt-Weisskopf radius of resonance vertices, GeV^-1                       */
  double r_parent;     /* ... of the D0 vertex                                                       */
  int n_res;
  const tddp4_res *res;    /* host [n_res]                                                           */
  int n_terms;
  const tddp4_term *terms; /* host [n_terms]                                                         */
  int n_couplings;         /* K_c; every coupling 0 .. K_c-1 must be used by at least one term               */
  double t_lo, t_hi;       /* decay-time window of the normalisation; t_hi = +INFINITY allowed       */
  int use_resolution;      /* 0: eq. (1) as printed; 1: per-event Gaussian sigma_t (O-8): the data *
                            * sample must be loaded with sigma_t > 0; P_i = R_i(t_i, sigma_i) / N_i(sigma_i);   *
                            * 2: time-integrated (decay time not measured): P_i = int_window R(p_i, t) dt / N,  *
                            * the data sample is loaded without t and sigma_t                                    */
} tddp4_model_desc;

/* ---- life cycle -------------------------------------------------------------------------------- */
/* Builds a handle on the current CUDA device from a host-side description (copied).  Recurring
 * lineshapes are de-duplicated into "instances" ("substituted by a link to a single
 * instance").                                                                                        */
int tddp4_create(const tddp4_model_desc *desc, tddp4 **out);
int tddp4_destroy(tddp4 *h);
/* cuda_stream: a cudaStream_t (0 = legacy default stream).  The handle does not own it.              */
int tddp4_set_stream(tddp4 *h, void *cuda_stream);
const char *tddp4_last_error(const tddp4 *h);
const char *tddp4_version(void);

/* ---- step 0/1: event store, kinematics + spin factors, once per event set ------------------------ */
/* which: 0 = data sample, 1 = normalisation sample.  p4: [16][ld] SoA as above (ld >= n); t: decay
 * times [n] (data; may be NULL for the normalisation sample); sigma_t: per-event resolution [n] or
 * NULL; weight: normalisation weights w_j [n] or NULL (= 1).  on_device = 0: host pointers, copied
 * with cudaMemcpyAsync; 1: device pointers, read once.  The call builds the parameter-independent
 * caches (invariant masses, lineshape shape functions, spin x barrier factors) and does not keep p4. */
int tddp4_load_events(tddp4 *h, int which, int64_t n, int64_t ld, const double *p4, const double *t,
                      const double *sigma_t, const double *weight, int on_device);

/* ---- per minimiser call -------------------------------------------------------------------------- */
/* c, cbar: host [K_c][2] (re, im) couplings of A_f and Abar_f (eq. 2); mass_width: host [n_res][2]
 * (m0, Gamma0); x, y mixing parameters, tau lifetime in ps (Gamma = 1/tau) of eq. (1).  Compares with
 * the previous values to find which lineshape instances, hence which coupling columns, are dirty.    */
int tddp4_set_params(tddp4 *h, const double *c, const double *cbar, const double *mass_width, double x,
                     double y, double tau);

/* NLL = -sum_i log( R_i / N ) over the data sample (steps 2-7).  nll_out: host.  prob_out: device [n]
 * or NULL; receives P_i = R_i / N.  Synchronous.  TDDP4_ERR_NONFINITE if some P_i <= 0 or non-finite. */
int tddp4_nll(tddp4 *h, double *nll_out, double *prob_out);
/* Pipelined form: enqueue the evaluation for the current parameters into result slot 0..63 and return;
 * tddp4_nll_result waits for that slot.  Parameters are captured at enqueue time.                    */
int tddp4_nll_async(tddp4 *h, int slot);
int tddp4_nll_result(tddp4 *h, int slot, double *nll_out);
/* The pieces of the last completed evaluation in `slot`, for sharded (multi-GPU) use and parity:
 * out[0] = sum_i log B_i, out[1] = sum_i t_i, out[2] = N (normalisation), out[3] = NLL, out[4] = number
 * of events with non-positive / non-finite rate.                                                     */
int tddp4_nll_parts(tddp4 *h, int slot, double out[5]);

/* NLL and its analytic gradient in one pass over the data sample (derived from eq. (1) and
 * eq. (2)).  grad_out: host [4 K_c + 2]:
 *   [2k], [2k+1]             d NLL / d Re c_k, d NLL / d Im c_k            (k < K_c)
 *   [2 K_c + 2k], [.. + 1]   d NLL / d Re cbar_k, d NLL / d Im cbar_k
 *   [4 K_c], [4 K_c + 1]     d NLL / dx, d NLL / dy
 * Masses, widths and tau are not differentiated.  Stale columns / Gram matrix / time rows are refreshed first.
 * Works in both modes (use_resolution = 0 and 1).  Synchronous.                                         */
int tddp4_nll_grad(tddp4 *h, double *nll_out, double *grad_out);

/* Batched form for independent parameter points (the 2 n_par points of a numerical gradient, a scan, a
 * replayed minimiser trajectory): equivalent to tddp4_set_params + tddp4_nll for each point in order, with all
 * evaluations enqueued back to back and ONE synchronisation at the end.  params: host [n_points][stride],
 * stride = tddp4_param_stride(h) = 4 K_c + 2 n_res + 3, one point laid out as c[K_c][2], cbar[K_c][2],
 * mass_width[n_res][2], x, y, tau.  nll_out: host [n_points]; status_out: host [n_points] or NULL, per-point
 * tddp4_status (a failed point gets NaN, or +inf for TDDP4_ERR_NONFINITE).  Returns the first non-OK status.
 * The handle is left holding the last valid point's parameters.                                        */
int tddp4_param_stride(const tddp4 *h);
int tddp4_nll_batch(tddp4 *h, int64_t n_points, const double *params, double *nll_out, int *status_out);

/* ---- step 6: normalisation through the Gram matrix ----------------------------------------------- */
/* G_sum[k][l] = sum_j w_j a_k(p_j) conj(a_l(p_j)) over THIS handle's normalisation sample for the
 * current masses/widths (recomputed if dirty); host [K_c][K_c][2]; *n_norm = its event count.         */
int tddp4_gram(tddp4 *h, double *G_sum, int64_t *n_norm);
/* How the Gram matrix is refreshed after a mass or width moved (the
 * normalisation pass dominates a fit).  mode 0 (default): one full pass over the static cache of the normalisation
 * sample, nothing of it stored.  mode 1: the library also keeps the sample's coupling columns (16 K_c bytes per event)
 * and, when the columns made stale since the last pass are few enough that reading the clean ones back (16 B each) and
 * rebuilding only the stale ones moves fewer bytes than a full pass, runs an incremental pass; otherwise a full pass that
 * re-stores the stale columns.  Either way G has the bits of a full pass.  mode -1 only queries.  incremental_passes
 * (host, may be NULL): number of incremental passes run so far.  Synchronises when the mode changes.              */
int tddp4_set_gram_mode(tddp4 *h, int mode, int64_t *incremental_passes);
/* Replace the Gram matrix used for N by G_sum / n_norm given by the caller (e.g. the all-reduced sum of
 * all ranks' matrices).  Stays in force until the masses/widths change again.                         */
int tddp4_gram_override(tddp4 *h, const double *G_sum, int64_t n_norm);
/* N for the current parameters from the Gram matrix in force; host out.                              */
int tddp4_norm(tddp4 *h, double *norm_out);

/* ---- event-sharded evaluation: the same exchange without a host round trip --------
 * One process per GPU holds a contiguous block of both samples.  Per call each rank enqueues
 *   tddp4_gram_enqueue   (only when a mass or width moved)  -> all-gather of 2 K_c^2 + 1 doubles -> tddp4_gram_reduce
 *   tddp4_nll_enqueue                                        -> all-gather of 8 doubles           -> sum in rank order
 * on the handle's stream; the collective (NCCL, the caller's) runs on that same stream between them, so nothing
 * synchronises until the gathered result words are read.
 * tddp4_gram_enqueue: G_dev device [2 K_c^2 + 1] receives this rank's Gram sums ([K_c][K_c][2]) followed by its
 *   normalisation event count as a double (refreshed first if stale; an override in force is dropped).
 * tddp4_gram_reduce: gathered_dev device [world][2 K_c^2 + 1]; the handle's Gram matrix becomes the sum over ranks,
 *   added in rank order by one kernel (same bits on every rank), normalised by n_norm_total.  Stays in force
 *   until the masses/widths change or the normalisation sample is reloaded.
 * tddp4_nll_enqueue: result_dev device [8]: words 0..4 as tddp4_nll_parts ([3] = this rank's NLL term
 *   Gamma sum t - sum log B + n log N with the Gram matrix in force), [5..7] unused.
 * tddp4_gram_state: *valid = the matrix in force matches the current masses/widths; *overridden = it came from
 *   tddp4_gram_override / tddp4_gram_reduce.                                                           */
int tddp4_gram_enqueue(tddp4 *h, double *G_dev);
int tddp4_gram_reduce(tddp4 *h, const double *gathered_dev, int world, int64_t n_norm_total);
int tddp4_nll_enqueue(tddp4 *h, double *result_dev);
int tddp4_gram_state(const tddp4 *h, int *valid, int *overridden);

/* ---- companion path: generation (G1-G6) ---------------------------------------------------------- */
/* Candidates first .. first+n_candidates-1 of Philox stream (seed, stream_id) are generated by
 * Raubold-Lynch with t ~ Exp(tau), weighted by w B (eq. 1 with the current parameters) and accepted
 * iff u E < w B.  Envelope E = envelope_scale * max of w B over candidates 0 .. n_pilot-1 of the same
 * stream; n_pilot = 0: E = envelope_scale.  Accepted events are written compacted, in candidate order:
 * out_p4 device [16][capacity] (row stride = capacity), out_t device [capacity], out_index device
 * [capacity] int64 candidate indices or NULL.  n_accepted, n_overflow (ratio above envelope; accepted),
 * envelope_out: host.  TDDP4_ERR_CAPACITY if n_accepted > capacity (first `capacity` are written).    */
int tddp4_generate(tddp4 *h, uint64_t seed, uint32_t stream_id, int64_t first, int64_t n_candidates,
                   int64_t n_pilot, double envelope_scale, int64_t capacity, double *out_p4, double *out_t,
                   int64_t *out_index, int64_t *n_accepted, int64_t *n_overflow, double *envelope_out);
/* Rigorous upper bound on the Raubold-Lynch weight w of this model's final state (host out): the product
 * of the three breakup momenta at their individual maxima.  With a constant-amplitude model, B = 2, so
 * tddp4_generate(n_pilot = 0, envelope_scale = 2 * bound) un-weights candidates to flat phase space.  */
int tddp4_weight_bound(const tddp4 *h, double *bound_out);
/* Raw candidates (no accept step) for parity: device out_p4 [16][n], out_t [n], out_w [n] (phase-space
 * weight), out_ratio [n] (w B), out_u [n] (accept uniform); any may be NULL.                          */
int tddp4_candidates(tddp4 *h, uint64_t seed, uint32_t stream_id, int64_t first, int64_t n, double *out_p4,
                     double *out_t, double *out_w, double *out_ratio, double *out_u);

/* ---- validation projections (Fig. 3) ---------------------------------------- */
/* The five observables the paper projects its generated samples on: m12, m34 (invariant masses of the pi+ pi- pair =
 * particles (2,3) and of the K+ pi- pair = particles (0,1)), cos12, cos34 (helicity cosines of the pi+ and of the K+ in
 * their pair's rest frame, with respect to the pair's flight direction in the D rest frame) and phi (angle between the
 * two decay planes in the D rest frame, in (-pi, pi]); the paper does not define them, DESIGN.md 3 gives the reading.
 * p4: device [16][ld] SoA, any frame.  ranges: host [5][2] (lo, hi) per observable; bin = floor((v - lo)/(hi - lo) *
 * n_bins), v == hi counts in the last bin, values outside are dropped.  hist_out: host [5][n_bins] counts.
 * values_dev: device [5][n] or NULL, the per-event observables.  n_bins <= 512.  Synchronous.           */
int tddp4_project(tddp4 *h, int64_t n, int64_t ld, const double *p4, int n_bins, const double *ranges, int64_t *hist_out,
                  double *values_dev);
/* tddp4_project for callers that may not allocate (code under CUDA-graph capture, serving loops, harnesses that forbid
 * cudaMalloc): the same kernel, the same observables and bin rule, but the histogram the kernel accumulates into is a
 * file-scope device array of the library, unsigned 64-bit [5][TDDP4_PROJECT_STATIC_MAX_BINS] = 20 KiB, which every GPU
 * that loads the library holds until the process exits.  The call allocates and frees nothing (no cudaMalloc, cudaFree
 * or allocating library routine) and does not synchronise: it enqueues, on the handle's stream, a clear of the array, the
 * kernel, and a device-to-device copy of the counts into hist_dev; the first call on a device also looks the array's
 * device address up (cudaGetSymbolAddress, once per device), so make one call before a capture begins.
 *   p4, n, ld, n_bins, ranges, values_dev: as tddp4_project.  hist_dev: DEVICE [5][n_bins] int64, the caller's; every
 *   element is written (it need not be cleared), valid once the stream has reached the end of the enqueued work.
 * n_bins > TDDP4_PROJECT_STATIC_MAX_BINS is rejected with TDDP4_ERR_ARG (text in tddp4_last_error); so is a call while
 * another device than the handle's is current.  ALL calls of a process on one GPU share the one array, whatever the
 * handle: each call clears it first (it keeps the previous call's counts), and two calls whose work overlaps on the GPU
 * (different streams, no dependency between them) race on it -- order them on one stream or with events.          */
#define TDDP4_PROJECT_STATIC_MAX_BINS 512
int tddp4_project_static(tddp4 *h, int64_t n, int64_t ld, const double *p4, int n_bins, const double *ranges,
                         int64_t *hist_dev, double *values_dev);

/* ---- inspection (per-layer parity, profiling) ---------------------------------------------------- */
enum {
  TDDP4_GET_S = 0,       /* invariant masses squared, [n_sys][n]                                     */
  TDDP4_GET_SHAPE = 1,   /* parameter-free lineshape shape g = q^(2L+1) F_L(z)^2 / sqrt(s), [n_inst][n] */
  TDDP4_GET_STATIC = 2,  /* spin factor x barrier factors per term, [n_terms][n] (caller's term order) */
  TDDP4_GET_COLUMNS = 3, /* coupling columns a_kappa, [K_c][n][2] (data sample, current parameters)   */
  TDDP4_GET_TERMS = 4    /* per-term amplitudes a_k, [n_terms][n][2], recomputed (caller's term order) */
};
/* Copies a cache of event set `which` into the caller's device buffer `out` (row stride n).          */
int tddp4_get(tddp4 *h, int which, int what, double *out);
/* Layout of the caches: systems (bit mask of final-state particles) and lineshape instances.  Arrays
 * must hold 16 resp. 32 ints.                                                                        */
int tddp4_layout(const tddp4 *h, int *n_sys, int *sys_mask, int *n_inst, int *inst_res, int *inst_sys,
                 int *inst_sub);

/* Per-kernel CUDA-event timing on the handle's stream.  kernel ids: */
enum {
  TDDP4_K_KIN = 0,       /* step 1 at load                                                            */
  TDDP4_K_COLUMNS = 1,   /* reserved (steps 2+3 alone are never launched: they are fused into COLNLL / GRAM)   */
  TDDP4_K_GRAM = 2,      /* steps 2+3+6 fused over the normalisation sample (fp64 tensor-core Gram)    */
  TDDP4_K_NLL = 3,       /* steps 4+5+7 over cached columns (coupling / x / y / tau-only call)         */
  TDDP4_K_GEN_RATIO = 4, TDDP4_K_GEN_EMIT = 5,
  TDDP4_K_COLNLL = 6,    /* steps 2+3+4+5+7 fused over the data sample (call after a mass/width move)  */
  TDDP4_K_TRES = 7,      /* resolution mode: per-event time rows (re-run when x, y or tau moved)               */
  TDDP4_K_GRAD = 8,      /* steps 4+5+7 and the analytic gradient in one pass over cached columns (tddp4_nll_grad) */
  TDDP4_K_COUNT = 9
};
int tddp4_profile(tddp4 *h, int enable);
/* total_ms, launches and (alg_bytes may be NULL) the algorithmic bytes of those launches -- the rows each launch
 * had to read and write, counted on the host from its dirty masks, DESIGN.md "Kernels" -- since the last reset,
 * for one kernel id; synchronises.                                                                     */
int tddp4_profile_read(tddp4 *h, int kernel_id, double *total_ms, int64_t *launches, double *alg_bytes);
int tddp4_profile_reset(tddp4 *h);
/* In-kernel duration of the coupling-only NLL kernel (8(a) rows 4+5+7) while profiling is on: per launch, the time on the
 * GPU's %globaltimer from the start of its earliest block to the moment its last block has written the result -- what the
 * kernel itself takes, without the launch gap a pair of CUDA events around an isolated launch also measures.  Host out:
 * the sum over launches since the last tddp4_profile_reset in microseconds and their number; synchronises.      */
int tddp4_profile_in_kernel(tddp4 *h, double *total_us, int64_t *launches);
/* The same for kernel_id = TDDP4_K_NLL (identical to the call above) or TDDP4_K_GRAD (the gradient kernel of tddp4_nll_grad
 * without resolution: earliest block start to the gradient written); any other id is TDDP4_ERR_ARG.                      */
int tddp4_profile_in_kernel_of(tddp4 *h, int kernel_id, double *total_us, int64_t *launches);
/* Number of kernels this handle has launched since creation (all kinds).                            */
int64_t tddp4_launch_count(const tddp4 *h);
/* Measured fp64 issue rate of this GPU: a dependent-free chain of DFMA instructions on every SM (the
 * denominator of the "alu"-bound fractions of the generator, kinematics and time-row kernels).  Host out:
 * fp64 instructions per second (one per lane; an FMA counts once).  Synchronous, ~1 ms.              */
int tddp4_fp64_peak(tddp4 *h, double *inst_per_s);
/* The branch-free fp64 primitives the kernels use where an IEEE division or square root would put a divergent slow path
 * into a hot loop (Breit-Wigner reciprocal, barrier factors, generator boosts; csrc/jit_shared.cuh), evaluated on arrays
 * for accuracy tests: what = 0 1/x, 1 sqrt(x), 2 1/sqrt(x), 3 x/y.  x, y (what = 3 only), out: device [n]; inputs must
 * be normal numbers (x > 0 for the roots).  Synchronous.                                                        */
int tddp4_math_probe(tddp4 *h, int what, int64_t n, const double *x, const double *y, double *out);
/* The CUDA source of a kernel the library specialises to a model and compiles at run time with NVRTC (the two fused
 * passes over the static caches: what = 0 the Gram pass, 8(a) rows 2+3+6; what = 1 the data pass after a mass/width move,
 * rows 2..5+7; the model's table of shared lineshape / spin-factor instances becomes compile-time
 * constants; what = 4 the candidate kernel of the generator, G1-G5), or of a header these include (what = 2
 * "jit_shared.cuh", 3 "nll_shared.cuh", 5 "tables.h", 6 "device_math.cuh"; desc may then be any valid model).  weighted: the event set carries a weight row; mode (what = 1): 0 full-range time functions, 1 small mixing
 * phases, 2 resolution / time-integrated rows; mode (what = 0): 0 plain pass, 1 pass that stores the columns, 2
 * incremental pass (tddp4_set_gram_mode).  Needs NO device: it is what tddp4_create hands to NVRTC, exposed so that
 * a build check can compile it.  Host buf of cap bytes (may be NULL with cap = 0); returns the size needed including the
 * terminating NUL (the text is written only if it fits), or a negative tddp4_status.                              */
int64_t tddp4_jit_source(const tddp4_model_desc *desc, int what, int weighted, int mode, char *buf, int64_t cap);

#ifdef __cplusplus
}
#endif
#endif /* TDDP4_H */

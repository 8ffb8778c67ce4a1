/* madme.h — C ABI of the B200 (sm_100a) matrix-element library (libmadme.so).
 *
 * The hot path of MadFlow-style event generation that arxiv 2211.14056 optimises
 * ("parallelized in the event axis"; §2: "spinors, vertices and
 * propagators" as device code behind one custom op, momenta in, |M|^2 out, no gradient),
 * with the entry points BASELINE.json:north_star lists: me_init, rambo_generate, me_eval,
 * vegas_iterate.  Every step of every call runs in hand-written CUDA kernels; there is NO CPU
 * fallback: on a machine without a CUDA device every compute call returns ME_ENODEV.
 *
 * Conventions common to all calls
 *   - return 0 on success, a negative ME_E* code otherwise; me_last_error() gives a thread-local
 *     message.  Nothing throws across the boundary.
 *   - "dev" pointers are device (HBM) pointers, 16-byte aligned; "host" pointers are host memory.
 *     The caller owns every data buffer and keeps it alive until the stream work completed.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  All calls are
 *     asynchronous on `stream`, except vegas_iterate / vegas_finish, which synchronise once to return their scalars.
 *   - a handle belongs to the device that was current in me_init (calls switch to it and back) and owns scratch
 *     that its vegas_* calls share: use one handle from ONE stream at a time (one handle per stream otherwise).
 *   - allocation: me_init and me_reserve allocate; no other call allocates, frees or synchronises behind the
 *     caller's back (vegas_integrand beyond the reserved size fails with ME_EINVAL).
 *   - units: GeV.  Momenta are (E, px, py, pz), metric (+,-,-,-); legs 0,1 are the incoming partons
 *     along +z / -z, legs 2.. the final state in the order of the process name.
 *   - fp64 throughout (BASELINE.json:metric), Philox words are uint32.
 */
#ifndef MADME_H
#define MADME_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

enum {
  ME_OK = 0,
  ME_EINVAL = -1,    /* null pointer, negative count, bad dimension, unaligned pointer */
  ME_EPROCESS = -2,  /* unknown process name */
  ME_ECUDA = -3,     /* a CUDA runtime call or kernel launch failed (message has the CUDA error) */
  ME_ENODEV = -4,    /* no CUDA device: this library has no CPU path */
  ME_EDIM = -5       /* grid / random-number dimension does not match process and ps_mode */
};

typedef struct me_handle me_handle; /* opaque, library-owned; created by me_init, released by me_free */

/* Fixed couplings, no running, no width in any propagator (reading R-A2). */
typedef struct {
  double alpha_s, alpha_em, m_top, w_top; /* w_top must be 0 (kept for layout compatibility) */
  double ptj_min, dr_min;                 /* cuts of BASELINE.json:configs[2,3]; <= 0 disables one */
} me_params;

/* Vegas grid (Lepage 1978, the paper's refs [7,8]; VegasFlow PAPER.md:29,35). */
typedef struct {
  int n_dim, n_bins;
  double* edges;  /* dev [n_dim][n_bins+1], caller-owned, refined in place */
  double alpha;   /* damping exponent (1.5 in config 4) */
  uint64_t seed;
  int iteration;  /* Philox counter word 3; incremented by vegas_iterate */
  int ps_mode;    /* 0 classic RAMBO (n_dim = 4 n_final), 1 RAMBO "on diet" (n_dim = 3 n_final - 4),
                     2 hadronic (vegas_* only; n_dim = 3 n_final - 2): the first two coordinates are the momentum fractions
                     x1, x2 weighted with a DECLARED toy gluon density 3 x^-1.2 (1-x)^5, sqrt_s is the hadronic energy,
                     the rest drives RAMBO on diet at sqrt(x1 x2) sqrt_s (no PDF grids exist here) */
} vegas_grid;

typedef struct {
  double integral, variance; /* this iteration: I_j [pb], sigma_j^2 */
  double sum_w, sum_w2;      /* sum f, sum f^2 over the n_ev events */
  long long n_pass;          /* events with f != 0 (passed the cuts) */
} vegas_result;

/* me_init — select the generated kernel of `process` and fix its parameters.
 * process: "epem_mupmum" (e+ e- -> mu- mu+), "gg_ttx", "gg_ttxg", "gg_ttxgg" (BASELINE.json:configs[0-3]), and the
 * quark-initiated channels of the paper's hadronic processes (Table 1), legs in the
 * order of the name: "qqx_ttx", "qqx_ttxg", "qqx_ttxgg" (q qbar -> t tbar + 0, 1, 2 gluons) and "qg_ttxq", "qg_ttxqg"
 * (q g -> t tbar q + 0, 1 gluons) with their charge conjugates "qxg_ttxqx", "qxg_ttxqxg" (qbar g -> t tbar qbar + 0, 1
 * gluons); q is one massless flavour; and "gg_ttxggg" (g g -> t tbar g g g, SURVEY.md 8(f) N2:
 * 1 240 diagrams, 120 colour flows, evaluated in two passes with the colour-flow vector in tensor memory).
 * Allocates the handle and the fixed-size device scratch of the Vegas path (reduction partials, the survivor staging
 * of the fused integrand: about 25 MB, independent of the event count). */
int me_init(const char* process, const me_params* params, me_handle** out);
void me_free(me_handle* h);
/* me_reserve — size the per-event scratch of vegas_integrand / vegas_iterate / vegas_unweight (the integrand values
 * and their packed bin indices, 32 bytes per event, plus 8 bytes per 256 events) for calls of up to max_events
 * events.  Grows only (a smaller request is a no-op); synchronises the device when it has to replace a buffer. */
int me_reserve(me_handle* h, long long max_events);
int me_n_external(const me_handle* h);
int me_n_final(const me_handle* h);
/* what: 0 Feynman diagrams, 1 colour-pure amplitude terms, 2 diagrams with a 4-gluon vertex, 3 colour flows,
 * 4 helicity combinations, 5 off-shell currents, 6 shared-memory bytes per event, 7 events (warps) per CTA,
 * 8 registers per thread of the me_eval kernel, 9 resident CTAs per SM, 10 SM count, 11 events reserved by
 * me_reserve, 12 the handle's device ordinal, 13 address of the per-event scratch (to check that calls do not
 * reallocate). */
long long me_info(const me_handle* h, int what);
/* nominal fp64 flops per event of the emitted program (real add or mul = 1, FMA = 2) */
double me_flops_per_event(const me_handle* h);

/* me_eval — steps a5-a10 of SURVEY.md §8(a): external wavefunctions, off-shell currents, closing
 * amplitudes, colour-flow vector J, J^dagger CF J, helicity sum, averages.
 * momenta: dev [n_ev][n_ext][4]; me2: dev [n_ev], GeV^(-2(n_final-2)).  Cuts are NOT applied here. */
int me_eval(me_handle* h, const double* momenta, double* me2, long long n_ev, void* stream);
/* as me_eval, additionally storing every helicity combination's contribution (already scaled by the
 * averaging factor): me2_hel dev [n_ev][2^n_ext], index h = sum_l b_l 2^l, b_l = 1 for helicity +1. */
int me_eval_helicities(me_handle* h, const double* momenta, double* me2_hel, long long n_ev, void* stream);

/* philox_uniform — step a1: Philox4x32-10, key = (seed lo, seed hi), counter = (event lo, event hi,
 * pair index d/2, iteration); u = ((w0 2^32 + w1) >> 11 + 1/2) 2^-53 in the OPEN interval (0,1).
 * rand: dev [n_ev][n_dim], event index = first_event + row. */
int philox_uniform(uint64_t seed, uint64_t iteration, long long first_event, int n_dim, double* rand,
                   long long n_ev, void* stream);

/* rambo_generate — step a3: uniforms -> momenta + phase-space weight (BASELINE.json:north_star).
 * rand: dev [n_ev][n_dim], n_dim = 4 n_final (ps_mode 0) or 3 n_final - 4 (ps_mode 1);
 * masses: HOST [n_final]; momenta: dev [n_ev][n_final+2][4] (incoming legs filled in);
 * weights: dev [n_ev], GeV^(2 n_final - 4).  n_final in 2..6. */
int rambo_generate(const double* rand, double sqrt_s, const double* masses, int n_final, int ps_mode,
                   double* momenta, double* weights, long long n_ev, void* stream);

/* apply_cuts — step a4: pass[ev] = 1 iff every final jet (gluon; also the massless final quark of q g -> t tbar q (g))
 * has pT > ptj_min and DeltaR > dr_min to every other final parton (true rapidity; strict).
 * is_gluon: HOST [n_final], 1 for the jets; pass: dev int32 [n_ev]. */
int apply_cuts(const double* momenta, int n_final, const int* is_gluon, double ptj_min, double dr_min,
               int* pass, long long n_ev, void* stream);

/* vegas_map — step a2 alone: y dev [n][n_dim] -> x dev [n][n_dim], jac dev [n], idx dev int32 [n][n_dim]. */
int vegas_map(const double* edges, int n_dim, int n_bins, const double* y, double* x, double* jac, int* idx,
              long long n, void* stream);
/* vegas_refine — step a12 alone: S dev [n_dim][n_bins] accumulated f^2; edges dev, refined in place. */
int vegas_refine(double* edges, int n_dim, int n_bins, const double* S, double alpha, void* stream);

/* vegas_integrand — steps a1-a11 fused for events [first_event, first_event + n_ev) of iteration
 * g->iteration: Philox -> Vegas map -> RAMBO -> cuts -> |M|^2 (skipped for cut events) ->
 * f = jac W_ps Theta me2 /(2 s) C, C = 0.3893793721e9 pb GeV^2; deterministic fixed-shape reduction.
 * sums: dev [3 + n_dim*n_bins] = (sum f, sum f^2, #f != 0, S_{d,i});  f_out: dev [n_ev] or NULL.
 * Does not refine; asynchronous. */
int vegas_integrand(me_handle* h, const vegas_grid* g, double sqrt_s, long long first_event, long long n_ev,
                    double* sums, double* f_out, void* stream);
/* vegas_iterate — one full iteration over events [0, n_ev): integrand, result, grid refinement in place
 * (all on the device), ++g->iteration.  result: HOST.  Synchronises `stream` once. */
int vegas_iterate(me_handle* h, vegas_grid* g, double sqrt_s, long long n_ev, vegas_result* result, void* stream);

/* vegas_combine — the one exchange of a sharded iteration: sums[j] = parts[0][j] + parts[1][j] + ...
 * in that FIXED order (reproducible whatever the arrival order).  parts: dev [n_parts][n_out], sums: dev [n_out]. */
int vegas_combine(const double* parts, int n_parts, int n_out, double* sums, void* stream);
/* vegas_finish — step 3 of SURVEY.md 8(c) G7 from the accumulated sums of n_total events:
 * I = sums[0]/N, sigma^2 = [sums[1]/N - I^2]/(N-1), n_pass = sums[2].  sums: dev [>= 3]; result: HOST.
 * Synchronises `stream` once. */
int vegas_finish(const double* sums, long long n_total, vegas_result* result, void* stream);

/* Unweighted events — the step behind the path.
 * vegas_max_weight: *w_max (dev [1]) = max_e f[e] over f dev [n_ev].
 * vegas_unweight: hit-or-miss on the weights f (dev [n_ev]) of events [first_event, first_event + n_ev) of iteration
 * `iteration`: event e is kept iff f > 0 and u_e w_max < f, u_e = the Philox uniform of counter (event lo, event hi,
 * 0x7fffffff, iteration), words 0-1 — a counter word no phase-space dimension uses, so the decision is independent
 * of the event's kinematics and reproducible under any sharding.  accepted: dev int64 [n_ev] receives the GLOBAL
 * indices of the kept events in ascending order; counts: dev int64 [2] = (number kept, number with f > w_max, which
 * are always kept and signal that w_max was too small). */
int vegas_max_weight(const double* f, long long n_ev, double* w_max, void* stream);
int vegas_unweight(me_handle* h, const double* f, long long n_ev, double w_max, uint64_t seed, uint64_t iteration,
                   long long first_event, long long* accepted, long long* counts, void* stream);
/* vegas_unweight_static — vegas_unweight for callers that cannot allocate (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): the same decision and the same output (accepted, counts as above), no handle,
 * no me_reserve.  The per-block counters live in a file-scope device array of fixed size instead of a cudaMalloc'ed
 * buffer: the call allocates and frees nothing and synchronises nothing.  Limits: n_ev <= VEGAS_UNWEIGHT_STATIC_MAX_EVENTS
 * per call (more: ME_EINVAL); every GPU that loads the library holds the array (128 KB) until exit; all calls on a device
 * share it, so calls that OVERLAP on the GPU (two streams, a graph replayed beside another call) race: one at a time
 * per device.  Runs on the CURRENT device.  vegas_unweight_static_init looks the array's device address up for the
 * current device (cudaGetSymbolAddress, once per device); the first vegas_unweight_static on a device does it itself,
 * so call the init beforehand where even that look-up is unwelcome (before a capture). */
#define VEGAS_UNWEIGHT_STATIC_MAX_EVENTS 4194304
int vegas_unweight_static_init(void);
int vegas_unweight_static(const double* f, long long n_ev, double w_max, uint64_t seed, uint64_t iteration,
                          long long first_event, long long* accepted, long long* counts, void* stream);
/* vegas_generate — the kinematics of LISTED events of iteration g->iteration on grid g (the grid the weights were
 * computed with, i.e. before its refinement): Philox -> Vegas map -> RAMBO for event_ids dev int64 [n].
 * momenta: dev [n][n_ext][4] (partonic centre-of-mass frame); weights: dev [n] = jac W_ps C/(2 s_hat) (times the
 * toy densities in ps_mode 2): the event weight without |M|^2 and cuts. */
int vegas_generate(me_handle* h, const vegas_grid* g, double sqrt_s, const long long* event_ids, long long n,
                   double* momenta, double* weights, void* stream);

/* fp64_peak_probe — a register-resident DFMA chain on every SM (8 independent accumulators per thread):
 * runs n_iter x 8 x 256 DFMA per thread on `stream`; returns the thread-DFMA count in *n_dfma (host).
 * The caller times it with CUDA events: this is the measured denominator of the fp64 roofline. */
int fp64_peak_probe(long long n_iter, double* sink /*dev [1]*/, double* n_dfma /*host*/, void* stream);

const char* me_last_error(void);

#ifdef __cplusplus
}
#endif
#endif

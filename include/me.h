/* =====================================================================================
 * me.h — C-ABI boundary of the B200-native tree-level matrix-element engine.
 *
 * What it computes.  For each phase-space point of one of five fixed processes the
 * library evaluates the tree-level matrix element "based on Feynman diagrams and
 * helicity amplitudes" (section 2), one event per GPU thread in
 * lockstep, in double, float or mixed precision, where mixed
 * means Feynman diagrams in double and "color algebra" in single precision (PAPER.md
 * line 81, section 3):
 *
 *     ME(p) = (1/D) * sum_{h good} sum_{sigma,tau} conj(J_sigma(p,h)) C_{sigma tau} J_tau(p,h)
 *
 * J = colour-flow amplitudes ("jamp"), C = colour matrix, D = averaging denominator
 * (the paper itself prints no formula — every reading is listed in
 * DESIGN.md).  The paper's interface is "batch of momenta in, batch of MEs out"
 * (PAPER.md line 41); the entry-point names are those of BASELINE.json `north_star`.
 *
 * Conventions: metric (+,-,-,-), GeV, p = (E,px,py,pz); the two
 * initial-state particles come first with their physical incoming momenta, final-state
 * particles are outgoing.  Particle order: e+ e- mu+ mu- / g g t t~ [g [g [g]]].
 * Helicity index ihel in [0, 2^npar): bit (npar-1-k) set <=> particle k has helicity +1.
 *
 * Pointers named d_* are DEVICE pointers, everything else is HOST memory.  The caller
 * owns every buffer it passes; the library owns me_ctx and its internal scratch.
 * No function throws or aborts; every function returns an me_status.
 *
 * Devices.  A context belongs to the CUDA device that was current at me_create: its tables, colour matrix and scratch live
 * there.  Every entry point that takes a context runs on that device; if another device is current at the call it is
 * switched for the duration of the call and restored on return.  Buffers passed in must be reachable from that device.
 * One process may hold contexts on several devices.
 *
 * Concurrency.  A context is NOT thread-safe: one host thread at a time per context (use one context per thread).  From
 * one thread, calls on one context may be issued on any streams: a call on another stream than the previous call of the same
 * context first waits (on the device, cudaStreamWaitEvent) for that call, because they share the context's scratch
 * (jamp staging of g g -> t t~ g g g, cached currents of ME_OPT_SHARE_CURRENTS, the workspace of me_filter_helicities /
 * me_select_helicity_color) and helicity lists.  Results are therefore correct on any mix of streams, but calls on ONE
 * context do not overlap on the GPU; to run several batches concurrently (several producers sharing
 * one GPU) create one context per stream.  me_set_helicities / me_filter_helicities wait for the context's previous call on
 * the host before they replace the lists.
 *
 * Alignment.  d_momenta, d_rnd: 16 bytes (what the vector loads need; cudaMalloc and torch give 256 or more); d_me, d_me_hel:
 * 8 bytes.  Anything less returns ME_EALIGN.
 * ===================================================================================== */
#ifndef PAPER_2303_18244_B200_ME_H
#define PAPER_2303_18244_B200_ME_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct me_ctx me_ctx; /* opaque; one per (process, parameters, device) */

typedef enum {
  ME_OK = 0,
  ME_EINVAL = 1,       /* null pointer, negative n, unknown enum value */
  ME_EPROCESS = 2,     /* unknown process id */
  ME_ENOTFILTERED = 3, /* me_compute before me_filter_helicities / me_set_helicities */
  ME_EALIGN = 4,       /* d_momenta / d_me not 16-byte aligned */
  ME_ENOMEM = 5,       /* host or device allocation failed */
  ME_ECUDA = 6,        /* a CUDA call failed; me_strerror(ME_ECUDA) names the last one */
  ME_ETOOLARGE = 7     /* me_compute_static: n beyond ME_STATIC_MAX_EVENTS; me_strerror(ME_ETOOLARGE) says by how much */
} me_status;

typedef enum {
  ME_EPEM_MUPMUM = 0, /* e+ e- -> mu+ mu-   (2 diagrams, 16 helicities, 1 colour)        */
  ME_GG_TTX = 1,      /* g g -> t t~        (3 diagrams, 16 helicities, 2 colour flows)  */
  ME_GG_TTXG = 2,     /* g g -> t t~ g      (16 diagrams, 32 helicities, 6 flows)        */
  ME_GG_TTXGG = 3,    /* g g -> t t~ g g    (123 diagrams, 64 helicities, 24 flows)      */
  ME_GG_TTXGGG = 4    /* g g -> t t~ g g g  (1240 diagrams, 128 helicities, 120 flows)   */
} me_process;

/* "double", "float" and "mixed" (diagrams FP64, colour algebra FP32). */
typedef enum { ME_FP64 = 0, ME_MIXED = 1, ME_FP32 = 2 } me_precision;

/* Standard-Model inputs (BASELINE.json configs): cfg 1 uses mz, wz, aewm1 (=1/alpha_EM),
 * sw2 (=sin^2 theta_W); the QCD processes use mt, alpha_s.  wt must be 0 (reading Q4). */
typedef struct {
  double mz, wz, aewm1, sw2;
  double mt, wt, alpha_s;
} me_sm_params;

typedef struct {
  int npar, ninitial, ndiagrams, ncomb, ncolor, color_denom, avg_denom;
  int page;                   /* P of the AoSoA momentum layout (events per page), 32       */
  int nkernels;               /* diagram kernels one me_compute pass launches per helicity chunk */
  int namplitudes;            /* amplitudes per helicity (a 4-gluon vertex yields three)    */
  double mass[8];             /* external masses in particle order, GeV                      */
  double flops_per_helicity[3]; /* ALGORITHMIC real flops per (event, helicity), by me_precision: every current,
                                   amplitude and colour-sum term evaluated exactly once */
  double flops_per_event_fixed[3]; /* helicity-independent flops per event (invariants, bases)   */
  double flops_executed_per_helicity[3]; /* flops the kernels actually issue (>= algorithmic: recomputation) */
  double flops_per_event_shared;  /* ME_OPT_SHARE_CURRENTS: ALGORITHMIC flops per event of the sharing kernel over the full helicity
                                     set (every current evaluated once per distinct helicity assignment of ITS OWN legs, in the walk
                                     order of the kernel), fixed part included; 0 where no such kernel exists                          */
  double flops_executed_per_event_shared; /* the same with what the sharing kernels actually issue (recomputation included)           */
} me_info;

/* Create a context for `process` on the current CUDA device.  Builds the colour matrix and
 * helicity tables on the device.  *out is untouched on failure.
 * Errors: ME_EINVAL (null), ME_EPROCESS, ME_EINVAL (wt != 0 or mt <= 0 for a QCD process), ME_ECUDA. */
me_status me_create(me_process process, const me_sm_params* params, me_ctx** out);

/* Frees the context and its device scratch.  Synchronises the device.  Null is ME_EINVAL. */
me_status me_destroy(me_ctx* ctx);

me_status me_get_info(const me_ctx* ctx, me_info* out);

/* Helicity filtering (reading Q7; BASELINE.json north_star
 * "me_filter_helicities(momenta, n)").  Evaluates, ALWAYS in FP64, every helicity combination
 * on the first n events of d_momenta; helicity h is "good" iff
 *     max_events  ME_h(evt) / sum_h' ME_h'(evt)  >  1e-12.
 * mask_out[w] bit b <=> helicity index 64*w+b is good.  The mask is stored in the context and
 * returned.  Synchronises `stream`.  n must be >= 1; the buffer must hold ceil(n/P) pages.  The per-helicity fractions are
 * reduced on the device (workspace of (ncomb + 1) n doubles owned by the context); only ncomb doubles reach the host.
 * d_momenta layout: see me_compute. */
me_status me_filter_helicities(me_ctx* ctx, const double* d_momenta, int64_t n,
                               uint64_t mask_out[2], int* ngood_out, void* stream);

/* Options.  ME_OPT_PARITY_PAIRING is off by default, ME_OPT_SHARE_CURRENTS is on by default.
 * ME_OPT_PARITY_PAIRING: for the pure-QCD processes |M_h|^2 = |M_{~h}|^2 where ~h flips
 * every helicity (parity invariance, tree level, real momenta), so me_compute evaluates one helicity of every good
 * pair and counts it twice: half the work, same number up to rounding (~1e-14).  Ignored for e+ e- -> mu+ mu- and
 * whenever the installed mask is not closed under h -> ~h.  me_compute_helicities is unaffected.
 * ME_OPT_SHARE_CURRENTS (second half: "sharing sub-tree currents across helicity
 * combinations"): a gluon sub-tree current depends only on the helicities of its own gluons, a one-gluon quark current on one
 * quark and one gluon helicity.  With the option on (the default), g g -> t t~ g g runs a kernel that walks the good helicities in a
 * reflected Gray order (quark helicities fastest) and re-evaluates a current only when one of ITS helicities changed since the
 * previous step; three-gluon sub-trees are parked in an L2-resident scratch owned by the context.  Same diagrams, same
 * amplitudes, same number up to rounding order (~1e-14).  g g -> t t~ g g g groups the helicities by their gluon helicities (one CTA
 * loops over the four quark-helicity assignments of a group): its last diagram kernel forms the colour-ordered four-gluon
 * currents once per group and needs no local jamp accumulators.  Ignored by the other processes.  me_info.flops_per_event_shared
 * is the algorithmic flop count with the option on.  me_compute_helicities / me_compute_jamps are unaffected. */
typedef enum { ME_OPT_PARITY_PAIRING = 0, ME_OPT_SHARE_CURRENTS = 1 } me_option;
me_status me_set_option(me_ctx* ctx, me_option option, int value);

/* Install a helicity mask without filtering (e.g. one returned by an earlier context). */
me_status me_set_helicities(me_ctx* ctx, const uint64_t mask[2]);

/* The hot path.  Asynchronous on `stream`
 * (a cudaStream_t passed as void*; null = default stream).  No host<->device copy, no
 * synchronisation (except a one-off scratch allocation for ME_GG_TTXGGG, and for ME_GG_TTXGG with
 * ME_OPT_SHARE_CURRENTS, the first time or when a later call needs more; the scratch is bounded whatever n is).
 * The result of an event does not depend on the batch it is in: a batch of any size, sliced or (ME_GG_TTXGG, small batches) with the
 * helicity list of an event block split over several thread blocks, gives every event the same bits.
 *   d_momenta : DEVICE, FP64 in every precision mode, AoSoA [ceil(n/P)][npar][4][P] with
 *               P = me_info.page and component order (E,px,py,pz); event e lives at page e/P,
 *               lane e%P.  The last page must be allocated in full; lanes >= n are read
 *               but their results discarded (they must hold finite numbers, e.g. a repeated event).
 *   d_me      : DEVICE, FP64 [n]; ME averaged over initial helicities/colours and divided by
 *               the identical-particle factor (avg_denom).  Non-finite values are not an error.
 * n = 0 is a no-op returning ME_OK.
 * Errors: ME_EINVAL, ME_ENOTFILTERED, ME_EALIGN, ME_ENOMEM, ME_ECUDA (launch failure). */
me_status me_compute(me_ctx* ctx, const double* d_momenta, int64_t n, me_precision precision,
                     double* d_me, void* stream);

/* The hot path for callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc):
 * g g -> t t~ g g only (ME_EPROCESS otherwise), at most ME_STATIC_MAX_EVENTS events per call.  Same arguments, layout and result as
 * me_compute with ME_OPT_SHARE_CURRENTS on (ME_OPT_PARITY_PAIRING is honoured), same kernel; the kernel's current cache (SURVEY.md section
 * 8(f) item 4: sub-tree currents parked across the helicity walk) is not the context's lazily allocated scratch but a file-scope
 * `static __device__` array of the library, 64 CTAs x 208 KB = 13 MiB, which every GPU that loads the library holds until exit.
 * The call makes no cudaMalloc / cudaFree and calls no allocating library routine; the first call on a device resolves the
 * array's device address (cudaGetSymbolAddress, once per device).  Asynchronous on `stream`, no synchronisation, no copy.
 * EVERY call on a device, from any context, uses the same array: calls that overlap on the GPU (different streams, threads or
 * contexts) race on it and give wrong results; calls on one stream, or otherwise ordered on the device, are safe.  The array keeps
 * the last call's contents; nothing in it has to start at zero (the first step of the helicity walk writes every vector it later
 * reads), so the call clears nothing.  It is independent of the context's own scratch and stream ordering (include "Concurrency").
 * n = 0 is a no-op.  Errors: ME_EINVAL, ME_EPROCESS, ME_ENOTFILTERED, ME_EALIGN, ME_ETOOLARGE (n > ME_STATIC_MAX_EVENTS; nothing is
 * launched), ME_ECUDA. */
#define ME_STATIC_MAX_EVENTS 8192
me_status me_compute_static(me_ctx* ctx, const double* d_momenta, int64_t n, me_precision precision,
                            double* d_me, void* stream);

/* The same computation with HOST buffers: the end-to-end call ("e2e"; the paper's
 * data flow "momenta in, matrix elements out", section 2, as seen from a host-side event generator).
 *   h_momenta : HOST, same AoSoA layout and padding rule as d_momenta; page-locked memory lets the
 *               copies overlap the computation (pageable memory is accepted, the copies then serialise).
 *   h_me      : HOST, FP64 [n].
 * The batch is cut in slices of 6 x 128 events per SM (whole waves of CTAs); slice k + 1 is copied to the device on an internal copy stream while slice k is computed, the
 * MEs of slice k return on a second copy stream; odd slices are computed on an internal stream so that
 * consecutive kernels overlap.  Two slice buffers per direction are owned by the context (allocated on
 * first use, freed by me_destroy).  Asynchronous like me_compute: work is ordered after what `stream` already holds,
 * and `stream` waits for the last device -> host copy, so synchronising `stream` makes h_me valid.
 * The buffers must stay untouched until then.  One call at a time per context.
 * Errors: as me_compute. */
me_status me_compute_host(me_ctx* ctx, const double* h_momenta, int64_t n, me_precision precision,
                          double* h_me, void* stream);

/* Same pass, but also returns the per-helicity colour-summed |M_h|^2 (not averaged) for ALL
 * ncomb helicities (masked ones evaluate too): d_me_hel is DEVICE FP64 [ncomb][n].
 * Used by the filter and by the parity tests.  d_me may be null.  Asynchronous on `stream`. */
me_status me_compute_helicities(me_ctx* ctx, const double* d_momenta, int64_t n,
                                me_precision precision, double* d_me, double* d_me_hel, void* stream);

/* Event-by-event random choice of a helicity and a leading-colour flow (section 5; SURVEY.md
 * section 8(f) item 2).  Per event two uniforms come from Philox4x32-10 with key = seed and counter
 * (event lo32, event hi32, 0x53454C45, 0), event = first_event + row: u1 = u53(w0,w1), u2 = u53(w2,w3) (mapping of
 * me_philox_uniform).  d_ihel[e] = helicity index drawn with probability ME_h / sum_h ME_h over the installed good
 * helicities; d_icol[e] = colour-flow index drawn with probability |J_s|^2 / sum_s |J_s|^2 at that helicity; both by
 * inverse CDF in index order with FP64 left-to-right sums (first k with cum_k >= u * total).  FP64 throughout; every
 * kernel stays in lockstep (the helicity enters as data).  d_ihel, d_icol: DEVICE int32 [n].  Asynchronous on `stream`
 * (the workspace, max(ncomb, 2 ncolor) x n doubles, is owned by the context and grown on first use: that one call
 * synchronises).  Errors as me_compute. */
me_status me_select_helicity_color(me_ctx* ctx, const double* d_momenta, int64_t n, uint64_t seed, uint64_t first_event,
                                   int32_t* d_ihel, int32_t* d_icol, void* stream);

/* Device-side cross-section sums and hit-or-miss unweighting ("hit-or-miss unweighting,
 * cross-section", line 45 the idea of offloading them).
 *   w_i = flux * d_weight[i] * d_me[i]   (flux = 1/(2 s) for a fixed-energy collision; d_weight from me_rambo)
 *   sums_out (HOST) = { sum_i w_i, sum_i w_i^2, max_i w_i }: sigma = sums[0]/n, its standard error from sums[1]
 *   d_accept[i] (DEVICE uint8 [n], nullable: the flags are then not stored, *naccept_out is still produced) = 1 iff u_i * wmax < w_i, with u_i = u53 of Philox4x32-10 at counter
 *   (event lo32, event hi32, 0x554E5754, 0), key = seed, event = first_event + i; wmax <= 0 selects the batch maximum;
 *   *naccept_out = number of accepted events.
 * Reductions are fixed-order trees without atomics (bit-identical run to run).  Allocates temporaries and
 * synchronises `stream`.  Errors: ME_EINVAL (n < 1, null, flux <= 0), ME_ENOMEM, ME_ECUDA. */
me_status me_unweight(const double* d_weight, const double* d_me, int64_t n, double flux, uint64_t seed, uint64_t first_event,
                      double wmax, double sums_out[3], uint8_t* d_accept, int64_t* naccept_out, void* stream);

/* Colour-flow amplitudes of one helicity (test hook for step a6): d_jamp is DEVICE FP64
 * [ncolor][2][n] (re, im), in units where the overall factor g_s^(npar-2) and a global
 * phase are stripped; QCD processes only. */
me_status me_compute_jamps(me_ctx* ctx, const double* d_momenta, int64_t n, int ihel,
                           double* d_jamp, void* stream);

/* Host copy of the colour matrix numerators (row-major [ncolor][ncolor], exact integers);
 * C = numerators / color_denom. */
me_status me_color_matrix(const me_ctx* ctx, double* numerators_out);

/* Counter-based RNG (reading Q14): Philox4x32-10 with
 * key = (seed lo32, seed hi32), counter = (event lo32, event hi32, k, j), k in [0,per_event),
 * j in {0,1}; the 8 output words of (k; j=0,1) give 4 uniforms
 *     u_i = ((w_2i >> 5) * 2^26 + (w_2i+1 >> 6) + 0.5) * 2^-53   in (0,1).
 * d_rnd: DEVICE FP64 [n][per_event][4]; event index = first_event + row.  Asynchronous. */
me_status me_philox_uniform(uint64_t seed, uint64_t first_event, int64_t n, int per_event,
                            double* d_rnd, void* stream);

/* RAMBO flat phase space (step a1, reading Q12) for the context's process at sqrt_s:
 * d_rnd [n][nfinal][4] -> d_momenta AoSoA (layout of me_compute, last page padded with copies
 * of event n-1), d_weight [n] (nullable) = phase-space weight in GeV^(2 nfinal - 4).
 * Massive final particles by xi rescaling (Newton).  Asynchronous. */
me_status me_rambo(const me_ctx* ctx, double sqrt_s, const double* d_rnd, int64_t n,
                   double* d_momenta, double* d_weight, void* stream);

/* Measured-peak microbenchmarks used by bench.py for the roofline denominator: run a
 * register-resident FMA-chain kernel (FP64 if fp64 != 0 else FP32) on the whole GPU and
 * return the achieved TFLOP/s in *tflops_out (2 flops per FMA).  Synchronises. */
me_status me_fma_peak(int fp64, double* tflops_out);

const char* me_strerror(me_status status);

#ifdef __cplusplus
}
#endif
#endif

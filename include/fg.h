/* fg.h — C ABI of the B200-native Monte-Carlo integrator for divergence-subtracted QED vertex graphs
 * without lepton loops (hot path of arXiv:1909.08015; PAPER.md = /root/reference/PAPER.md).
 *
 * One path: graph -> plan (host combinatorics + tables) -> fg_integrate (one sm_100a kernel pass
 * per precision rung: Philox -> Hepp-sector sample + pdf -> all forest terms of the integrand ->
 * conditioning check -> y = I/g -> compensated sums -> block reduce) -> mean, variance, counters.
 *
 * Conventions
 *  - every call returns int: 0 = FG_OK, negative = error code; fg_strerror(code) names it and
 *    fg_last_error_message() (thread-local) has the detail.  No exception crosses the ABI.
 *  - handles (fg_graph, fg_plan) are opaque, owned by the caller, released by *_destroy.
 *  - pointer arguments are HOST pointers unless the name ends in _dev; inputs are borrowed for the
 *    duration of the call only; outputs are written through caller-provided pointers.
 *  - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  Calls that return
 *    results to host memory synchronise that stream before returning.
 *  - there is NO CPU compute path: every entry point that evaluates anything launches CUDA kernels
 *    and fails with FG_E_CUDA when no device is usable.
 */
#ifndef FG_H_
#define FG_H_
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

#define FG_OK 0
#define FG_E_ARG -1       /* NULL / out-of-range argument */
#define FG_E_COUNT -2     /* need 2n electron + n photon lines on 2n+1 vertices, 1 <= n <= 5 */
#define FG_E_NOT_PATH -3  /* electron lines are not one simple open path v_0..v_2n (lepton loop or broken line) */
#define FG_E_VERTEX -4    /* a vertex without exactly one photon (internal or the external one) */
#define FG_E_NOT_1PI -5   /* an electron line not spanned by a photon: not 1PI / leg correction */
#define FG_E_LOOPS -6     /* n > 5 */
#define FG_E_CUDA -7      /* CUDA runtime error or no device */
#define FG_E_LIMIT -8     /* an internal table limit was exceeded */
#define FG_E_OPTS -9      /* invalid plan options */

typedef struct fg_graph fg_graph;
typedef struct fg_plan fg_plan;

/* Internal line of the graph.  kind 0 = electron, 1 = photon.  Vertices are numbered along the electron path:
 * electron line i (i = 1..2n) joins v_{i-1} and v_i.  The Feynman parameters z follow the canonical line order
 * "electron lines e_1..e_2n, then photons sorted by their lower end" (eq. (12)). */
typedef struct { int32_t u, v; int32_t kind; } fg_edge;

/* Build a graph from its internal lines and the vertex of the external photon. */
int fg_graph_create(const fg_edge* edges, int32_t n_edges, int32_t ext_photon_vertex, fg_graph** out);
void fg_graph_destroy(fg_graph*);

/* Gauge-invariant class (k, m, m') of a graph (Table I at 397-409): m and m' count the internal photons to
 * the left and to the right of the external photon along the electron path ("or vice versa": kmm[1] >= kmm[2]), k those
 * with their ends on opposite sides of it; k + m + m' = n.  kmm: three ints, written by the call.  Host only. */
int fg_graph_class(const fg_graph*, int32_t* kmm);

/* Plan options.  fg_plan_opts_default fills the Calc-2 constants of PAPER.md:370-377.
 *  C[4]      mixture weights C_1..C_4 of g = sum C_k g_k; must be >= 0 and sum to 1
 *  D         exponent scale of the third component
 *  merge_ext_lines  1: the two electron lines at the external-photon vertex share one variable, M = 3n-1
 *            (fn.12); 0: M = 3n
 *  deg_rule  0 = the built-in substitute rule R-Deg of DESIGN.md (the paper's own algorithm for Deg(s) is only in its Refs.
 *            [42], [32]: PAPER.md:250); any other value is refused with FG_E_OPTS until that algorithm is available
 *  deg_consts the six hand-chosen constants of that algorithm, eq. (15), in the order C_bigZ, C_bigF,
 *            C_add, C_subI, C_subSE, C_subO (defaults 0.256, 0.839, 0.786, 0.2, 0, 0.2); carried for the paper's rule, not
 *            used by rule 0
 *  deg_table optional host array of 2^M doubles overriding Deg(s); NULL = deg_rule
 *  rng       pseudorandom generator of the sample stream: 0 = Philox4x32-10 (Calc 2; counter = (sample id,
 *            call), key = seed), 1 = MRG32k3a (Calc 1; L'Ecuyer 1999): seed -> starting values
 *            1 + ((seed_lo | seed_hi) (i+1) + 12344) mod (m - 1), i.e. seed 0 is the reference implementation's 12345 x 6,
 *            and sample s owns outputs 32 s, 32 s + 1, ... of that sequence (jump by powers of the recurrence matrices)
 *  structure_only  fg_host_plan only: stop after subgraphs, forests, terms and the Deg/Z tables (no Dirac tables)
 *  rel_tol, abs_tol  a sample whose estimated round-off error exceeds max(rel_tol*|I|, abs_tol*g) is
 *            re-evaluated in double-double (abs_tol plays the role of sigma/4 in (18))
 *  err_factor safety factor K of the running error estimate K*2^-53*sum|terms| (0 = default 8)                                 */
typedef struct {
  double C[4];
  double D;
  int32_t merge_ext_lines;
  int32_t deg_rule;
  const double* deg_table;
  double rel_tol, abs_tol;
  double err_factor;
  double deg_consts[6];
  int32_t structure_only;
  int32_t rng;
} fg_plan_opts;
void fg_plan_opts_default(fg_plan_opts* o);

/* Host: UV-divergent subgraphs, forests, operator table, element instances, Dirac coefficient tables, Deg/Z
 * tables; then uploads them to `device`.  "fg_plan" in BASELINE.json. */
int fg_plan_create(const fg_graph*, const fg_plan_opts*, int32_t device, fg_plan** out);
void fg_plan_destroy(fg_plan*);

/* Changes the acceptance tolerances of an existing plan (e.g. after a pilot run has measured sigma). */
int fg_plan_set_tol(fg_plan*, double rel_tol, double abs_tol);

/* Per-kernel device timing (CUDA events on the launching stream, four per slab; nothing synchronises while the work is
 * enqueued: fg_plan_timing waits for the recorded events and folds them).  fg_plan_timing returns the milliseconds accumulated since fg_plan_profile:
 * ms3[0] double-precision pass (geometry + stream kernels), ms3[1] double-double and quad-double passes, ms3[2] final
 * reduction; and the kernels launched. */
int fg_plan_profile(fg_plan*, int32_t enable);
int fg_plan_timing(const fg_plan*, double* ms3, int64_t* launches);

/* Profiling builds only (-DFG_PHASE_PROF): warp-cycles (clock64, summed over all warps of the double-precision pass) spent in
 * 0 sampler, 1 element geometry, 2 tensor-core record groups, 3 static scalar groups, 4 dynamic groups, 5 ring wait + chunk
 * barrier, 6 node products, 7 forest sum + weights, 8 group dispatch / flush.  Returns 1 when the library was built with the
 * counters, 0 when not (cycles stay 0).  reset != 0 clears them. */
int fg_plan_phase_cycles(const fg_plan*, uint64_t* cycles16, int32_t reset);

typedef struct {
  int32_t n_loops, M;                 /* loops, number of Feynman variables */
  int32_t n_subgraphs, n_forests, n_terms;       /* UV-divergent subgraphs incl. G; forests; (F,G') terms */
  int32_t n_geoms, n_nums, n_nodes;   /* distinct element geometries, (geometry, operator) tables, value nodes */
  int64_t n_records, n_coefs, n_coefs_nonzero;   /* numerator stream: records, stored and non-zero coefficients */
  int64_t table_bytes;                /* device bytes of all plan tables */
  int64_t stream_bytes;               /* bytes of the numerator coefficient stream (subset of table_bytes) */
  double flops_per_sample;            /* algorithmic FP64 flops of a5-a7 + sampler (FMA = 2), non-zero coefs only */
  double exec_flops_per_sample;       /* flops the double-precision kernel actually executes per sample */
  double plan_seconds;                /* host time spent in fg_plan_create */
  int64_t wave_samples;               /* samples per wave of the double-precision pass (0 from fg_host_plan) */
} fg_plan_stats;
int fg_plan_info(const fg_plan*, fg_plan_stats* out);

/* Host-only planning (no device, no kernels): runs the whole planner and returns its statistics (table_bytes = 0),
 * the structure dump described below (subs: up to subs_cap rows of 4 ints; returns the ints written to `terms`) and
 * the Deg / Z_1 tables (2^M doubles each).  Any output pointer may be NULL.  For CPU tests of the host logic. */
int fg_host_plan(const fg_graph*, const fg_plan_opts*, fg_plan_stats* stats, int32_t* subs, int32_t subs_cap,
                 int32_t* terms, int32_t terms_cap, double* deg, double* Z1);

/* Host-only debug surface of the planner's Dirac algebra: the coefficient table of ONE Wick matching of ONE
 * element = the UV-divergent subgraph on the vertex interval [a,b] with the child subgraphs `kids` (n_kids pairs a,b) shrunk.
 * Slots are numbered in string order (from the outgoing end).  pairs: n_pairs matched slot pairs (i < j); qslot: the unmatched
 * slot that carries gamma^nu (operator A only) or -1; op: 0 = A, 1 = U, 2 = L, 3 = L - U; comp: 0 / 1 = u / v of a
 * self-energy element.  Output: gaps = the other unmatched slots (n_gaps of them), table[T] for every subset T of the gaps
 * (bit g of T: gap g carries gamma^0 A_j), INCLUDING the factor (-1/2)^n_pairs of the Wick contractions.
 * Returns the number of slots of the element, or a negative error code. */
int fg_host_dirac_table(const fg_graph*, int32_t a, int32_t b, const int32_t* kids, int32_t n_kids, int32_t op, int32_t comp,
                        const int32_t* pairs, int32_t n_pairs, int32_t qslot, double* table, int32_t table_cap, int32_t* gaps,
                        int32_t* n_gaps);

/* Structure dump for tests (expression (11)).
 *  subs: n_subgraphs rows (a, b, type 0 = self-energy / 1 = vertexlike, in_chain)
 *  terms: flat ints: sign, index of G', n_members, then (sub index, op) pairs, op 0=A 1=U 2=L 3=L-U.
 *  Returns the number of ints written to `terms`, or FG_E_LIMIT if cap is too small. */
int fg_plan_structure(const fg_plan*, int32_t* subs, int32_t* terms, int32_t terms_cap);
/* Copies Deg(s) and Z_1(s) (2^M doubles each; either may be NULL). */
int fg_plan_tables(const fg_plan*, double* deg, double* Z1);

typedef struct {
  double mean;            /* (16): sum y / N */
  double variance;        /* (17): sigma_down^2 = sum y^2 / N^2 - (sum y)^2 / N^3 */
  double sum_y[2];        /* double-double (hi, lo) */
  double sum_y2[2];
  uint64_t n_samples;
  uint64_t n_flagged;     /* samples re-evaluated in double-double (second rung) */
  uint64_t n_flagged2;    /* of those: samples re-evaluated again in quad-double (third rung) */
  uint64_t n_rejected;    /* samples that contributed 0: degenerate point, non-finite value, or not resolved by the
                             last (quad-double) rung */
  uint64_t n_pdf_big_exp; /* samples whose pdf left the double range, kept as x*2^j */
} fg_result;

/* Samples [0, n_samples) of the Philox stream `seed`.  Blocks until the result is on the host. */
int fg_integrate(const fg_plan*, uint64_t n_samples, uint64_t seed, void* stream, fg_result* out);
/* Samples [first_sample, first_sample + n_samples): sharding and checkpoint/resume. */
int fg_integrate_range(const fg_plan*, uint64_t first_sample, uint64_t n_samples, uint64_t seed, void* stream,
                       fg_result* out);
/* Asynchronous form: the result is left in device memory (`out_dev`, sizeof(fg_result) bytes, written by the
 * final reduction kernel on `stream`); no host synchronisation.
 * A plan owns ONE set of work buffers (wave tables, scratch, queues, partial sums): all integrations of a plan must be
 * enqueued on the same stream (they then run one after another), or be separated by a synchronisation; calls from several
 * host threads are serialised by a mutex inside the library, which does not lift that rule.  Use one plan per stream for
 * concurrent work. */
int fg_integrate_async(const fg_plan*, uint64_t first_sample, uint64_t n_samples, uint64_t seed, void* stream,
                       void* out_dev);
/* Exact combination of two shards (double-double sums add; mean/variance recomputed). */
int fg_result_merge(const fg_result* a, const fg_result* b, fg_result* out);

/* ---- several graphs at once: initialisation stage, acceptance rule (18), block scheduling, combination (19) ----------------
 * (PAPER.md:286, 290-294, 328-359).  A batch borrows its plans (they must outlive it).  Per graph it keeps the running sums of
 * everything folded so far, the next unused Philox sample id, t_j = seconds per sample, and abs_tol_j of (18).
 *  fg_batch_pilot   initialisation stage: n_pilot samples of every graph from sample id first_sample on (loose relative
 *                   tolerance 1e-6), measures t_j, then sets abs_tol_j = (1/4) sigma_j sqrt(sum sigma_l^2) / sum sigma_l on
 *                   every plan.  sigma_l = s_l / sqrt(N): N = target_samples per graph if > 0 (the tolerance the END of such a
 *                   run needs), else the samples folded so far (the paper's floating rule); rel_tol is the
 *                   relative part of the criterion from then on.
 *  fg_batch_next    draws the graph of the next block, p_j = (C_j / sqrt t_j) / sum_l (C_l / sqrt t_l), C_j = sigma_j sqrt N_j
 *                   = the per-sample standard deviation, with the uniform Philox4x32-10(key = sched_seed, counter = (block
 *                   index, 0, 0, 0)) words 0, 1; reserves block_samples sample ids of that graph.
 *  fg_batch_fold    adds a block result (and, if seconds > 0, a new measurement of t_j) to graph j and refreshes every abs_tol.
 *  fg_batch_run     n_blocks times: next, fg_plan_set_tol (18), fg_integrate_range, fold (one GPU; several ranks: dist.py).
 *  fg_batch_total   value = sum of the means, sigma_down by (19). */
typedef struct fg_batch fg_batch;
int fg_batch_create(fg_plan* const* plans, int32_t n_plans, fg_batch** out);
void fg_batch_destroy(fg_batch*);
int fg_batch_pilot(fg_batch*, uint64_t n_pilot, uint64_t seed, uint64_t first_sample, double target_samples, double rel_tol, void* stream);
int fg_batch_set_times(fg_batch*, const double* seconds_per_sample);
int fg_batch_probabilities(const fg_batch*, double* p);
int fg_batch_next(fg_batch*, uint64_t sched_seed, uint64_t block_samples, int32_t* graph, uint64_t* first_sample);
int fg_batch_fold(fg_batch*, int32_t graph, const fg_result* block, double seconds);
int fg_batch_run(fg_batch*, uint64_t n_blocks, uint64_t block_samples, uint64_t seed, uint64_t sched_seed, void* stream);
int fg_batch_result(const fg_batch*, int32_t graph, fg_result* out, double* abs_tol, double* seconds_per_sample);
int fg_batch_total(const fg_batch*, double* value, double* sigma_down, uint64_t* n_total);
/* Class sums (Table I): fg_batch_set_classes stores a class (k, m, m') for every graph of the batch (3 ints per
 * graph, e.g. from fg_graph_class; borrowed for the call); fg_batch_class_total returns the value (sum of the means) and
 * sigma_down by (19) of the graphs of one class and their number (0 graphs: value 0). */
int fg_batch_set_classes(fg_batch*, const int32_t* kmm_per_graph);
int fg_batch_class_total(const fg_batch*, const int32_t* kmm, double* value, double* sigma_down, int32_t* n_graphs);

/* ---- parity / debug surface (device kernels; outputs are HOST arrays, any may be NULL) -------------------
 * fg_sample_dump: for samples first..first+n-1: all Philox words (n * M * 4, call-major), mixture component (n),
 * ordering j_1..j_M (n*M), z (n*M), pdf mantissa in [0.5,1) and exponent (n each), bad flag (n). */
int fg_sample_dump(const fg_plan*, uint64_t first, uint64_t n, uint64_t seed, void* stream, uint32_t* philox_words,
                   int32_t* comp, uint8_t* orderings, double* z, double* pdf_mant, int32_t* pdf_exp, uint8_t* bad);
/* fg_eval_points: integrand at n given points (n*M doubles, on the simplex; n <= 2^24).  I = final value (double-double
 * or quad-double where flagged), I_double = plain double pass, err = the running error estimate of the first rung that ran.
 * flags: bit0 = re-evaluated in double-double, bit3 = re-evaluated again in quad-double, bit1 = non-finite value or
 * degenerate point, bit2 = not resolved by the last rung (estimated error of the quad-double value still above the
 * tolerance: the integrator lets such a sample contribute 0).
 * mode 0: as the integrator does (double -> double-double -> quad-double); 1: double only; 2: double-double for every
 * point, quad-double for what that leaves; 3: quad-double for every point. */
int fg_eval_points(const fg_plan*, const double* z, uint64_t n, int32_t mode, void* stream, double* I,
                   double* I_double, double* err, uint8_t* flags);
/* fg_sample_eval_dump: what the integrator computes per sample, for samples first..first+n-1:
 * I (final), y = I/g, flags as above. */
int fg_sample_eval_dump(const fg_plan*, uint64_t first, uint64_t n, uint64_t seed, void* stream, double* I, double* y,
                        uint8_t* flags);
/* ---- no-allocation entry point ---------------------------------------------------------------------------------------------
 * For callers that cannot call cudaMalloc (CUDA graph capture, serving loops, harnesses that forbid it).
 * fg_eval_points_dd_noalloc: the integrand at n points in double-double (the second rung for EVERY point, no further rung), like
 * fg_eval_points(mode 2) without its quad-double follow-up.  ALL pointers are DEVICE pointers owned by the caller:
 * z_dev n*M doubles (points on the simplex), I_dev n doubles, err_dev n doubles or NULL (error estimate), flags_dev n bytes
 * (bit1 = non-finite / degenerate, bit2 = not resolved by double-double at the plan's tolerance).  The call allocates nothing:
 * the per-block scratch of the kernel lives in a static device array of 32 MiB (held by every GPU that loads the library until
 * exit); plan tables and the plan's partial-sum buffer come from fg_plan_create.  Limits (fg_noalloc_limits): n <= 2^20, and the
 * plan's per-block scratch must fit the array (FG_E_LIMIT otherwise).  Asynchronous on `stream`; no host synchronisation.
 * Every call shares the array and the plan's buffers: calls (of this or of any other integration on the same plan, or of this
 * entry point on ANY plan of the same device) that overlap on the GPU race; enqueue them on one stream or synchronise between them.
 * fg_noalloc_setup(device) resolves the array's device address (cudaGetSymbolAddress, once per device); call it before a graph
 * capture; fg_eval_points_dd_noalloc does it itself on its first call for a device otherwise. */
int fg_noalloc_setup(int32_t device);
int fg_noalloc_limits(uint64_t* scratch_bytes, uint64_t* max_points);
int fg_eval_points_dd_noalloc(const fg_plan*, const double* z_dev, uint64_t n, void* stream, double* I_dev, double* err_dev,
                              uint8_t* flags_dev);

/* fg_dfma_peak: FP64-FMA micro-benchmark on the plan-independent device (the roofline denominator):
 * returns achieved TFLOP/s (FMA = 2) over `iters` dependent-chain steps x 8 chains per thread on all SMs. */
int fg_dfma_peak(int32_t device, int32_t iters, void* stream, double* tflops, double* ms);

/* fg_dmma_peak: the same for the FP64 tensor path (mma.sync m8n8k4 f64, 8 independent accumulator pairs per warp). */
int fg_dmma_peak(int32_t device, int32_t iters, void* stream, double* tflops, double* ms);

const char* fg_strerror(int code);
const char* fg_last_error_message(void);
const char* fg_version(void);

#ifdef __cplusplus
}
#endif
#endif

/*
 * vegas_b200.h -- C ABI of libvegas_b200.so: one Vegas iteration over a batch of events + the grid
 * refinement it feeds, on one NVIDIA B200 (sm_100a).
 *
 * What the calls compute is the data-parallel hot path of VegasFlow (Monte Carlo
 * integration by "importance sampling techniques from Vegas" on "adaptive grids", where "every iteration
 * informs the subsequent run"; user API PAPER.md:L72-L79: VegasFlow(n_dim, n_events,
 * events_limit) / compile(integrand) / run_integration(n_iter)).  The paper prints no equation; the
 * arithmetic is the reading S1-S7 / I0-I4 / R1-R17 of SURVEY.md section 8.c, restated in DESIGN.md.
 *
 * Conventions
 *   - Plain C, no torch / CUDA types.  Pointers are HOST pointers unless the name starts with dev_.
 *   - Every function returns an int status (VEGAS_OK = 0, negative = error) unless stated.  After an
 *     error vegas_last_error() returns a static, thread-local, NUL-terminated description.
 *   - The caller owns every buffer it passes.  `params` is copied at create.  `dev_workspace` (device
 *     memory, >= vegas_workspace_bytes(), 256-byte aligned) and `cuda_stream` (a cudaStream_t cast to
 *     void*, NULL = the legacy default stream) are borrowed and must outlive the context; the hot path
 *     allocates no device memory itself (every device buffer, the scratch of vegas_debug_events included, is a
 *     region of dev_workspace; the microbenchmark vegas_pipe_rate is the one exception, stated there); it allocates a few hundred bytes of pinned host memory for results.
 *   - A context is not thread-safe.  Calls that return results to host pointers are synchronous at
 *     return (they synchronise the stream); they enqueue asynchronously inside (no host sync between
 *     the launches of one iteration).
 *   - There is no CPU fallback: every step runs in CUDA kernels; without a CUDA device vegas_create
 *     fails with VEGAS_ECUDA.
 */
#ifndef VEGAS_B200_H
#define VEGAS_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct vegas_ctx vegas_ctx; /* opaque; created by vegas_create, freed by vegas_destroy */

enum {
    VEGAS_OK = 0,
    VEGAS_EINVAL = -1,       /* bad argument (range, NULL, wrong n_params) */
    VEGAS_ECUDA = -2,        /* a CUDA runtime call failed / no device */
    VEGAS_ENOMEM = -3,       /* workspace too small or host allocation failed */
    VEGAS_ESTATE = -4,       /* call order: e.g. vegas_refine before any vegas_iterate */
    VEGAS_EUNSUPPORTED = -5, /* no compiled kernel instance for (integrand_id, dim, precision); device is not sm_100 */
    VEGAS_EGRID = -6         /* grid not strictly increasing from 0 to 1; grid left unchanged */
};

/* Per-event arithmetic precision (uniform, map, Jacobian, integrand).  wf, (wf)^2, all sums, the
 * histogram, the refinement and the master edges are always fp64 (BASELINE.json configs[3]: "FP32
 * integrand with FP64 accumulation"; reading R14). */
enum { VEGAS_FP64 = 0, VEGAS_FP32_EVAL = 1,
       /* fp64 arithmetic throughout, but one 32-bit Philox word per coordinate instead of 52 bits of two words
        * (reading R3: "a 32-bit-per-coordinate variant ... as an extra, mirrored in the oracle and reported
        * separately"): u = r/2^32, coordinate k uses block k>>2, word k&3.  Halves the Philox work of the fp64
        * configurations; the estimates are those of a different, equally valid random stream.  Available for
        * gauss_sym, gauss_double, lo_2to2 and toy_sum. */
       VEGAS_FP64_U32 = 2 };

/* Built-in integrands (device functions chosen at compile time; BASELINE.json north_star "Integrand
 * evaluation") and their `params` (doubles):
 *   0 gauss_sym      {alpha, mu}                         f = prod_k exp(-(x_k-mu)^2/alpha^2)/(alpha sqrt(pi))   configs[0]
 *   1 gauss_double   {alpha, mu1, mu2}                   f = 1/2 [prod N(x_k;mu1,alpha) + prod N(x_k;mu2,alpha)]  configs[1],[2]
 *   2 genz_osc_peak  {phase_fraction, c_0 .. c_{dim-1}}  f = cos(2 pi phase + sum c_k x_k) prod 1/(c_k^-2+(x_k-1/2)^2), fp32   configs[3]
 *   3 lo_2to2        {sqrt_s, sqrt_shat_min, cos_cut, pdf_a, pdf_b=5}   synthetic LO 2->2, dim = 3          configs[4]
 *   4 toy_sum        {}                                  f = sum_k x_k
 */
enum { VEGAS_GAUSS_SYM = 0, VEGAS_GAUSS_DOUBLE = 1, VEGAS_GENZ_OSC_PEAK = 2, VEGAS_LO_2TO2 = 3, VEGAS_TOY_SUM = 4,
       VEGAS_USER = 5 /* run-time compiled user integrand: vegas_create_custom only */,
       VEGAS_LO_2TO2_TAB = 6 /* lo_2to2 with a tabulated PDF: params {sqrt_s, sqrt_shat_min, cos_cut} + vegas_set_table */ };

/* Device bytes the caller must provide to vegas_create for this (dim, nbins).  0 if out of range. */
size_t vegas_workspace_bytes(int dim, int nbins);

/* Create an integrator state: uniform grid (E[k][i] = i/nbins), iteration counter 0.
 * Mirrors VegasFlow(n_dim, ...) + compile(integrand): the integrand is selected
 * among the compiled instances instead of being traced.
 *   dim 1..32; nbins 2..4095 (fp64) / 2..511 (fp32) so that m*nbins is exact (S2).
 * Errors: VEGAS_EINVAL (ranges, NULL out, n_params mismatch, misaligned workspace), VEGAS_ENOMEM
 * (workspace_bytes too small), VEGAS_EUNSUPPORTED (no instance; a device other than sm_100: the library carries
 * sm_100a code only), VEGAS_ECUDA. */
int vegas_create(vegas_ctx** out, int dim, int nbins, int integrand_id, const double* params, int n_params,
                 int precision, void* dev_workspace, size_t workspace_bytes, void* cuda_stream);

/* User integrand, compiled at run time (the paper's `integrator.compile(integrand)`: the user
 * writes a function of the points in the unit hypercube).  `source` is a NUL-terminated
 * translation unit in the subset of C that is also valid CUDA device code and must define
 *     VEGAS_INTEGRAND double vegas_user_integrand(const double* x, int dim, const double* params)
 * (VEGAS_INTEGRAND expands to __device__ here; helper functions need the same prefix).  NVRTC compiles it for
 * sm_100a together with the library's own kernel templates (the headers next to the library, csrc/), without
 * fused-multiply-add contraction of the user's arithmetic, into the same iterate kernel the built-in integrands
 * use (run-time shaped: any dim <= 32, any nbins, fp64); everything else (grid, refine, run_integration, parity
 * hook) works as for vegas_create.  params (0..16 doubles) are copied.  precision: VEGAS_FP64 or VEGAS_FP64_U32.
 * On a compilation error the compiler log is available from vegas_last_error().
 * Errors: VEGAS_EINVAL (NULL source, ranges, > 16 params, precision), VEGAS_EUNSUPPORTED (NVRTC compilation
 * failed), VEGAS_ENOMEM, VEGAS_ECUDA. */
int vegas_create_custom(vegas_ctx** out, int dim, int nbins, const char* source, const double* params, int n_params,
                        int precision, void* dev_workspace, size_t workspace_bytes, void* cuda_stream);

/* lo_2to2_tab (PDF interpolation is part of the integrand in the paper's
 * workloads -- a synthetic table stands in for a PDF grid): the toy PDF g(x) of lo_2to2 is replaced by four-point
 * Lagrange (cubic) interpolation of `values[0..n-1]`, knots uniform in ln x: values[j] = g(tau^(1 - j/(n-1))),
 * tau = (sqrt_shat_min/sqrt_s)^2, so values[0] = g(tau), values[n-1] = g(1).  4 <= n <= 4096; copied into the
 * workspace.  vegas_iterate fails with VEGAS_ESTATE until a table is set.
 * Errors: VEGAS_EINVAL (NULL, n out of range, another integrand), VEGAS_ECUDA. */
int vegas_set_table(vegas_ctx* ctx, const double* values, int n);

/* One Vegas iteration (S1-S6): n_events events, global event index e in [0, n_events), cut into
 * ceil(n_events/events_per_launch) kernel launches (PAPER.md:L57-L65 `events_limit`; results do not
 * depend on it, reading R16).  Event e draws its point from Philox4x32-10 keyed by `seed` with counter
 * (e, iteration, coordinate block), maps it through the grid, evaluates the integrand, and the kernels
 * accumulate S1 = sum wf, S2 = sum (wf)^2 and H[k][bin_k] += (wf)^2.
 * When the iteration is cut into several launches they are dealt to internal non-blocking streams forked from and
 * joined to the context's stream (they are independent: global event index, reductions into H), so small launches
 * overlap; seen from the caller everything is ordered on the context's stream.
 *   integral = S1/n, error = sqrt(max(0,(S2/n - I^2)/(n-1))); hist (may be NULL) receives dim*nbins
 *   doubles, row-major [k][i].  The histogram also stays on the device for vegas_refine.
 * On success the iteration counter increments by one.  Non-finite results are returned as they are.
 * An iteration cut into 16 or more launches is captured once per (n_events, events_per_launch, seed, launch shape)
 * into a CUDA graph and replayed (vegas_use_cuda_graph(ctx, 0) turns that off): at small batches the host's launch
 * rate is otherwise the floor.  An iteration may have at most 2^20 launches.
 * Errors: VEGAS_EINVAL (n_events < 2, events_per_launch == 0 or so small that the iteration would need more than
 * 2^20 launches, NULL integral/error), VEGAS_ECUDA. */
int vegas_iterate(vegas_ctx* ctx, uint64_t n_events, uint64_t events_per_launch, uint64_t seed,
                  double* integral, double* error, double* hist);

/* Grid refinement (S7) from the histogram of the last vegas_iterate: 3-point smoothing, damping
 * ((1-r)/ln(1/r))^alpha, rebinning to equal damped weight; rebuilds the mapping table; clears H.
 * All-or-nothing over the dimensions: if any dimension's new edges are not strictly increasing the call returns
 * VEGAS_EGRID and the grid, the table AND the histogram stay as they were, so the caller may refine again (for
 * instance with another alpha); after a successful refinement the histogram is consumed (VEGAS_ESTATE until the
 * next vegas_iterate).  vegas_set_grid and vegas_reset also drop the histogram (it was sampled through another grid).
 * If an earlier vegas_refine_enqueue was rejected and not yet collected, this call still refines and then reports
 * that rejection as VEGAS_EGRID (last_error says which).
 * Errors: VEGAS_EINVAL (alpha < 0 or NaN), VEGAS_ESTATE (no histogram), VEGAS_EGRID, VEGAS_ECUDA. */
int vegas_refine(vegas_ctx* ctx, double alpha);

/* Asynchronous form of vegas_refine: enqueue only (no host synchronisation); the outcome of all refinements
 * enqueued since the last collect is read by vegas_refine_collect (VEGAS_EGRID if any of them was rejected --
 * each rejected one left its grid unchanged -- else VEGAS_OK), which synchronises the stream.  vegas_refine =
 * enqueue + collect.  vegas_iterate_enqueue + vegas_refine_enqueue make a whole step without a host round trip
 * (bench.py's device-timed region). */
int vegas_refine_enqueue(vegas_ctx* ctx, double alpha);
int vegas_refine_collect(vegas_ctx* ctx);

/* One whole step -- vegas_iterate_enqueue + vegas_refine_enqueue -- with the refinement FUSED into the iteration's
 * kernels: the CTA that finishes last over all launches of the iteration runs S6 and then S7 (all its warps, in
 * the shared memory the event loop no longer needs), commits the grid and clears the accumulators, so a step is one
 * kernel per launch and needs no memset and no separate refinement kernel (the latency of small iterations:
 * BASELINE.json configs[0]).  Same numbers as the two calls.  Asynchronous; afterwards vegas_iterate_collect (without
 * hist: it was consumed, and cleared even if the refinement was rejected), vegas_last_sums, vegas_last_npass and
 * vegas_refine_collect (the refinement's outcome) work as after the two calls.  vegas_run_integration replays this step
 * as a CUDA graph.  Falls back to the two kernels if the launch shape has less shared memory than one dimension's
 * refinement needs.
 * Errors: those of vegas_iterate_enqueue and vegas_refine_enqueue. */
int vegas_step_enqueue(vegas_ctx* ctx, uint64_t n_events, uint64_t events_per_launch, uint64_t seed, double alpha,
                       int* n_kernel_launches);

/* Device time (ms, CUDA events on the context's stream: memset + launches + finalize) of the iteration enqueued
 * `back` iterations ago (0 = the latest).  The last 64 iterations keep their events.  Synchronises on that
 * iteration's end event.  VEGAS_EINVAL if `back` is out of range. */
int vegas_iteration_kernel_ms(const vegas_ctx* ctx, int back, double* kernel_ms);

/* Master edges, fp64, dim*(nbins+1) doubles row-major [k][i].  set validates 0 = E0 < E1 < ... < EN = 1
 * (else VEGAS_EGRID, grid unchanged) and rebuilds the table with wd = E[i+1]-E[i] (S2). */
int vegas_get_grid(const vegas_ctx* ctx, double* edges);
int vegas_set_grid(vegas_ctx* ctx, const double* edges);

/* Uniform grid, iteration counter 0, histogram cleared. */
int vegas_reset(vegas_ctx* ctx);

/* The counter word fed to Philox as "iteration" (test hook; S1). */
int vegas_set_iteration(vegas_ctx* ctx, uint32_t iteration);
int vegas_get_iteration(const vegas_ctx* ctx, uint32_t* iteration);

/* Parity hook: S1-S4 for events first_event .. first_event+count-1 of the current iteration counter,
 * computed by the same device functions as vegas_iterate.  Any output pointer may be NULL.
 *   bins [count*dim] int32, x [count*dim] (fp32 values widened to double in fp32 mode), jac [count],
 *   f [count], wf [count] (= (double)J*(double)f), pass [count] (1 unless the integrand's cut rejected
 *   the event). */
int vegas_debug_events(vegas_ctx* ctx, uint64_t first_event, uint32_t count, uint64_t seed, int32_t* bins,
                       double* x, double* jac, double* f, double* wf, int32_t* pass);

/* S1, S2 of the last vegas_iterate and the device time of everything it enqueued (CUDA events on the
 * context's stream: all launches + finalize, excluding the result copy).  After a graph-replayed
 * vegas_run_integration kernel_ms is that run's average device time per step.  Any pointer may be NULL.
 * VEGAS_ESTATE before the first iterate. */
int vegas_last_sums(const vegas_ctx* ctx, double* S1, double* S2, double* kernel_ms);

/* Asynchronous form used for timing (bench.py): enqueue one iteration without reading results back
 * and without synchronising; results stay on the device until vegas_iterate_collect (same outputs as
 * vegas_iterate) which synchronises.  n_kernel_launches (may be NULL) receives how many kernels the
 * call enqueued. */
int vegas_iterate_enqueue(vegas_ctx* ctx, uint64_t n_events, uint64_t events_per_launch, uint64_t seed,
                          int* n_kernel_launches);
int vegas_iterate_collect(vegas_ctx* ctx, double* integral, double* error, double* hist);   /* hist after a successful
                                                      * vegas_refine: VEGAS_ESTATE (it was consumed) */

/* NEXT-2, multi-GPU sharding ("ensure that all GPUs ... receive a share"):
 * events are counter-indexed, so GPU g of G runs the events [first, first + count) of an iteration of n_total events
 * and the only exchange is one sum over the GPUs of the unreduced partials.
 *   vegas_iterate_shard_enqueue  S1-S5 for [first, first + count) (count may be 0), cut into launches like
 *                                vegas_iterate; leaves the shard's partial sums in the partials region; increments
 *                                the iteration counter; no host synchronisation.
 *   vegas_partials               device pointer and length (doubles) of that region, contiguous and 256-byte
 *                                aligned: {S1.hi, S1.lo, S2.hi, S2.lo, npass, 0, 0, 0, H[dim][nbins]} -- S1 = S1.hi +
 *                                S1.lo (a compensated pair), npass as a double.  The harness adds the regions of
 *                                all GPUs in place (torch.distributed.all_reduce(SUM) on a tensor view: one call of
 *                                8 + dim*nbins doubles per iteration, NCCL on GPUs), on the context's stream.
 *   vegas_finalize_enqueue       S6 from the (summed) region: I, sigma for n_total events; afterwards
 *                                vegas_iterate_collect / vegas_last_sums / vegas_last_npass / vegas_refine work as
 *                                after vegas_iterate, and every GPU refines to the identical grid.
 * Errors: VEGAS_EINVAL (range outside [0, n_total), n_total < 2, events_per_launch == 0), VEGAS_ESTATE (finalize
 * without a shard; collect/refine between shard and finalize), VEGAS_ECUDA. */
int vegas_iterate_shard_enqueue(vegas_ctx* ctx, uint64_t n_total, uint64_t first, uint64_t count,
                                uint64_t events_per_launch, uint64_t seed, int* n_kernel_launches);
int vegas_partials(const vegas_ctx* ctx, void** dev_partials, size_t* n_doubles);
int vegas_finalize_enqueue(vegas_ctx* ctx, uint64_t n_total);
/* vegas_finalize_enqueue + vegas_refine_enqueue(alpha) as ONE kernel (S6 by one thread beside the first steps of S7): the
 * tail of a sharded step after the all-reduce.  Same numbers as the two calls; afterwards vegas_iterate_collect (without
 * hist: it was consumed), vegas_last_sums, vegas_last_npass and vegas_refine_collect work as after them.
 * Errors: those of the two calls. */
int vegas_finalize_step_enqueue(vegas_ctx* ctx, uint64_t n_total, double alpha);

/* Test hook: load H (dim*nbins doubles >= 0, row-major [k][i], host) as if a vegas_iterate had produced it, so that
 * hand-made histograms reach the refinement kernel (the independent pins of S7).  Synchronises.
 * Errors: VEGAS_EINVAL (NULL, a negative or NaN cell), VEGAS_ECUDA. */
int vegas_set_histogram(vegas_ctx* ctx, const double* hist);

/* Launch-shape tuning knobs of the iterate kernel (the batch-size / occupancy study):
 * CTAs per SM and threads per CTA (0 = the kernel instance's default, 1 x 1024 for the instances tuned to the
 * BASELINE.json configurations and 2 x 512 for the generic ones; threads a multiple of 32, <= 1024), and
 * the number R of lane-indexed shared-memory histogram replicas (power of two 1..32; 0 = the largest
 * that fits).  Results do not depend on them beyond summation order.  VEGAS_EINVAL if the shape cannot
 * run (shared memory); ctas_per_sm is clamped to what the device can hold. */
int vegas_set_launch_shape(vegas_ctx* ctx, int ctas_per_sm, int threads_per_cta);
int vegas_set_hist_replicas(vegas_ctx* ctx, int replicas);
int vegas_get_launch_shape(const vegas_ctx* ctx, int* ctas_per_sm, int* threads_per_cta, int* hist_replicas,
                           size_t* smem_bytes);

/* Number of events of the last iteration whose integrand was not cut away (lo_2to2's cuts; equals
 * n_events for the other integrands).  VEGAS_ESTATE before the first iterate. */
int vegas_last_npass(const vegas_ctx* ctx, uint64_t* npass);

void vegas_destroy(vegas_ctx* ctx);

const char* vegas_last_error(void);

/* Library / device facts for reports: writes the SM count and the SM clock (kHz) of the device the
 * context runs on. */
int vegas_device_info(const vegas_ctx* ctx, int* sm_count, int* sm_clock_khz);

/* run_integration (PAPER.md:L79 `integrator.run_integration(n_iter, log_time=True)`, L88 "every iteration informs
 * the subsequent run"): n_warmup + n_iter times { vegas_iterate(n_events, events_per_launch, seed);
 * vegas_refine(alpha) }, then the classic Vegas combination of the last n_iter iterations (the warm-up ones only
 * adapt the grid; paper silent on the formula, reading R18 in DESIGN.md):
 *     w_i = 1/sigma_i^2,  mean = sum w_i I_i / sum w_i,  error = 1/sqrt(sum w_i),
 *     chi2_dof = sum w_i (I_i - mean)^2 / (n_iter - 1)           (0 when n_iter = 1)
 * Iterations with sigma_i = 0 (or not finite) carry no weight; if none has weight: mean = plain average, error = 0.
 * iter_integral / iter_error / iter_kernel_ms (each n_warmup + n_iter doubles, host, may be NULL) receive every
 * iteration's estimate and device time (the `log_time` of the paper's call).  A refine that fails with
 * VEGAS_EGRID leaves the grid as it was and the run goes on.  The per-iteration work runs in the kernels; the
 * combination is host arithmetic over n_iter numbers (vegas_combine_iterations, callable on its own, no GPU).
 * By default the whole step {memset, launches, finalize, refine, commit} is captured once into a CUDA graph and
 * replayed (the iteration counter then lives in device memory and the per-iteration (I, sigma) are logged on the
 * device together with a device time stamp; one host synchronisation per 64 iterations; iter_kernel_ms[i] is the
 * device time from the end of iteration i-1 -- for the first one, from the start of the run -- to the end of
 * iteration i, i.e. refinement i-1 + iteration i, read from %globaltimer).  Steps of one launch each are captured 16 to
 * a graph, their kernels linked by programmatic dependent launch (the next step's launch and shared-memory prologue run
 * under this step's tail; VEGAS_NO_PDL=1 in the environment switches that off).  vegas_use_cuda_graph(ctx, 0) selects the
 * plain loop of blocking calls (per-iteration times from CUDA events, refinement excluded) and also keeps
 * vegas_iterate from replaying graphs of many-launch iterations.  Both give the same numbers.
 * Errors: VEGAS_EINVAL (n_iter < 1, n_warmup < 0, NULL mean/error, iterate's argument errors), VEGAS_ECUDA. */
int vegas_use_cuda_graph(vegas_ctx* ctx, int enable);
int vegas_run_integration(vegas_ctx* ctx, int n_iter, int n_warmup, uint64_t n_events, uint64_t events_per_launch,
                          uint64_t seed, double alpha, double* mean, double* error, double* chi2_dof,
                          double* iter_integral, double* iter_error, double* iter_kernel_ms);
int vegas_combine_iterations(int n, const double* integral, const double* error, double* mean, double* comb_error,
                             double* chi2_dof);

/* Batch-size study / tuner (BASELINE.json north_star "Batching: the events-per-launch batch size is tuned on one
 * GPU, mirroring the paper's batch-size study", "finding the right batch size can make a
 * notable difference").  Times one iteration of n_events on the current grid for each of the n_candidates values
 * of events_per_launch (after one untimed warm-up iteration; CUDA events around memset + launches + finalize),
 * writes the times to ms[n_candidates] (host, may be NULL) and the fastest candidate to *best.  The grid and the
 * iteration counter are left as they were; the device histogram afterwards belongs to a tuning run, so
 * vegas_refine needs a fresh vegas_iterate (VEGAS_ESTATE otherwise).
 * Errors: VEGAS_EINVAL (NULL candidates/best, n_candidates < 1, a candidate of 0, n_events < 2), VEGAS_ECUDA. */
int vegas_tune_events_per_launch(vegas_ctx* ctx, uint64_t n_events, uint64_t seed, const uint64_t* candidates,
                                 int n_candidates, uint64_t* best, double* ms);

/* The launch geometry vegas_iterate uses when an iteration is cut into several launches (BASELINE.json configs[2], the
 * batch-size study of PAPER.md:L57-L65): the launches are dealt to `stream_lanes` internal streams
 * (min(launches, 128): the kernels a device runs concurrently) and each gets `ctas_per_launch` CTAs, the g that
 * minimises  ceil(L g / min(cta_slots, lanes g)) x (3 + events_per_launch / (g threads_per_cta))  -- the number of waves
 * the L launches' CTAs run in, times the length of a CTA in events per thread (3 = its fixed cost: zeroing and flushing
 * the shared histogram, staging the table, the launch).  One launch: all `cta_slots` CTAs (fewer only if there are not
 * 32 events for each).  When lanes x g CTAs do not cover the CTA slots (the device runs at most 128 kernels at a time:
 * launches of one CTA each on 148 SMs) every `extra_cta_every`-th launch gets one CTA more (0: none), aiming at 1.15 x
 * the slots in flight.  Pure host arithmetic: no device, no context.  `cta_slots` = CTAs resident on the device
 * (vegas_device_info: sm_count x ctas_per_sm of the launch shape).  Any output pointer may be NULL.
 * Errors: VEGAS_EINVAL (a zero argument, threads_per_cta outside 32..1024, cta_slots outside 1..2048, more than 2^20
 * launches). */
int vegas_plan_launches(uint64_t n_events, uint64_t events_per_launch, int threads_per_cta, int cta_slots, int* n_launches,
                        int* stream_lanes, int* ctas_per_launch, int* extra_cta_every);

/* Measured instruction throughput (thread-instructions per second over the whole GPU, current clocks) of
 * one SM pipe the hot path is bound by -- the denominators of the "alu" roofline bench.py reports
 * (BASELINE.json north_star: "fraction of the FP pipe roofline").  Each call runs a
 * few milliseconds of 8 independent dependency chains per thread at full occupancy on `cuda_stream`
 * (NULL = default stream) and synchronises.  No context needed -- and so no workspace: this benchmark call is the one
 * place where the library allocates device memory itself (cudaMalloc / cudaFree of 8 KB per SM, 2.4 MB on a B200, for the
 * chains' results); it is not part of the hot path.
 *   VEGAS_PIPE_DFMA            fp64 fused multiply-add   (peak FLOP/s = 2 x rate)
 *   VEGAS_PIPE_FFMA            fp32 fused multiply-add
 *   VEGAS_PIPE_IMAD_WIDE       32x32->64 integer multiply (two per Philox round)
 *   VEGAS_PIPE_LOP3            three-input logic op (two per Philox round)
 *   VEGAS_PIPE_SHARED_F64_ADD  fp64 atomicAdd on shared memory, lane-indexed replicas (R = 32), random cells
 * and, as evidence for the histogram design (none of them is a roofline denominator):
 *   VEGAS_PIPE_SHARED_F64_ADD_R8     the same update in the layout configs[3] is forced into (2000 cells, R = 8)
 *   VEGAS_PIPE_SHARED_F64_RMW_PLAIN  the non-atomic LDS.64, DADD, STS.64 a lane-and-warp-private word would allow
 *   VEGAS_PIPE_SHARED_U32_ADD        the native 32-bit integer shared-memory atomic add
 * and, as evidence for what the event loop's issue rate is bound by (same section):
 *   VEGAS_PIPE_DFMA_3REG             DFMA whose three source operands are three different registers (VEGAS_PIPE_DFMA
 *                                    repeats one; a polynomial step with its coefficient in a register is this form)
 *   VEGAS_PIPE_MIX_EVENT_LOOP        the event loop's ratio: 3 (IMAD.WIDE + LOP3), 2 IMAD, 5 DFMA, 5 LOP3 per group
 *                                    (the rate counts all 18 instructions of a group)
 * Errors: VEGAS_EINVAL (unknown pipe, NULL out), VEGAS_ECUDA. */
enum { VEGAS_PIPE_DFMA = 0, VEGAS_PIPE_FFMA = 1, VEGAS_PIPE_IMAD_WIDE = 2, VEGAS_PIPE_LOP3 = 3, VEGAS_PIPE_SHARED_F64_ADD = 4,
       VEGAS_PIPE_SHARED_F64_ADD_R8 = 5, VEGAS_PIPE_SHARED_F64_RMW_PLAIN = 6, VEGAS_PIPE_SHARED_U32_ADD = 7,
       VEGAS_PIPE_DFMA_3REG = 8, VEGAS_PIPE_MIX_EVENT_LOOP = 9 };
int vegas_pipe_rate(int pipe, void* cuda_stream, double* thread_instr_per_s);

/* Grid refinement (S7, as vegas_refine computes it) for callers that cannot give the library device memory.
 *
 * Every other call works in the workspace the caller allocated for vegas_create.  A caller that runs as a guest in
 * another program -- a plug-in, a framework callback, a custom operator: it receives device pointers to its inputs and
 * outputs, while the host program's memory pool already owns almost all of the GPU's memory -- has no allocator to ask:
 * its own cudaMalloc may fail for lack of free memory, and cudaMalloc / cudaFree hold up the whole device while the
 * host's streams are busy, which a step inside a pipelined loop must not do.  For them the working memory of the
 * refinement (candidate edges, a writable copy of the histogram, the rebuilt mapping table, outcome flags) is an array
 * compiled into the library.  This call needs no context, makes no cudaMalloc / cudaFree and calls no library routine
 * that allocates.
 *
 *   dev_edges     in   device, dim*(nbins+1) doubles, row-major [k][i]: the current grid, 0 = E0 < ... < EN = 1 per row
 *   dev_hist      in   device, dim*nbins doubles, row-major [k][i]: H of an iteration sampled through that grid
 *   dev_new_edges out  device, dim*(nbins+1) doubles: the refined grid -- bit-identical to what vegas_refine commits for
 *                      the same edges, histogram and alpha.  If the refinement is rejected (some dimension's new edges
 *                      not strictly increasing: vegas_refine's VEGAS_EGRID) it receives a copy of dev_edges.  A
 *                      dimension whose histogram sums to 0 keeps its edges.  May be the same buffer as dev_edges.
 *   dev_status    out  device, one int: 0 = refined, 1 = rejected
 * Inputs and outputs belong to the caller.  The call only enqueues one kernel on `cuda_stream` (NULL = the legacy
 * default stream) and returns; outputs are valid once the stream reaches that point.  The device that owns the stream
 * must be the current device.
 *
 * Limits and sharing -- read before use:
 *   - dim * (nbins + 1) <= VEGAS_STATIC_MAX_EDGES (8192; all BASELINE.json configurations are below 2100).  Larger grids
 *     are refused with VEGAS_EINVAL and a message naming the limit; they need vegas_create + vegas_refine.
 *   - The array is 4 * VEGAS_STATIC_MAX_EDGES doubles + 256 bytes, about 256 KB, and every GPU on which this library is
 *     loaded holds it from load until the process exits, whether or not this call is ever made.
 *   - There is ONE array per device.  Every call uses it, and it keeps the contents of the previous call; the kernel
 *     resets what has to start from zero (the outcome counters) and overwrites the rest before reading it.  Two calls
 *     whose kernels can run at the same time on one device (different streams, different host threads) race on it and
 *     give garbage: serialise them (same stream, or an event between them).
 *   - The first call on each device does a one-time set-up for that device (it asks the CUDA runtime for the array's
 *     device address -- cudaGetSymbolAddress -- and raises the kernel's shared-memory limit).  Make that first call
 *     outside any stream capture, e.g. once at start-up.
 * Errors: VEGAS_EINVAL (ranges, the size limit, alpha < 0 or NaN, a NULL or misaligned pointer), VEGAS_EUNSUPPORTED (a
 * device other than sm_100), VEGAS_ECUDA.  Reading: SURVEY 8.c S7; PAPER.md:L88 ("every iteration informs the
 * subsequent run"). */
#define VEGAS_STATIC_MAX_EDGES 8192
int vegas_refine_static_enqueue(int dim, int nbins, double alpha, const double* dev_edges, const double* dev_hist,
                                double* dev_new_edges, int* dev_status, void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* VEGAS_B200_H */

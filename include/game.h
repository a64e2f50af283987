/*
 * game.h -- C ABI of libgame.so, the B200-native (sm_100a) hot path of the GAME model of
 * arXiv:1211.5481 ("Genetic Algorithm Modeling with GPU Parallel Computing Technology"):
 * batched fitness evaluation of a whole GA population over the training patterns, plus the
 * per-generation GA operators, all on the device.
 *
 * Citations: "PAPER.md:<line>" is the paper text; "SURVEY 8(c) R<n>" / "DESIGN.md D<n>" are the
 * readings fixed where the paper is silent (DESIGN.md lists every one of them).
 *
 * Notation: P patterns, N features per pattern, d polynomial degree (Chebyshev)
 * or number of harmonics K (polytrigo, eq.(6)), G genes per chromosome, M chromosomes.
 *   G = N*d + 1 (Chebyshev)  or  N*2d + 1 (trig)      [DESIGN.md D1; eq.(5)]
 * Gene order: gene 0 = bias a_0; then one block per feature i = 0..N-1:
 *   Chebyshev: T_1(x_i) .. T_d(x_i);   trig: cos(1 x_i)..cos(d x_i), sin(1 x_i)..sin(d x_i)
 *   (the paper's [a_1..a_3, b_1..b_3]).
 *
 * Conventions
 *  - Every function returns int: GAME_OK (0) or a negative GAME_ERR_*.  No exceptions, no aborts,
 *    no printing.  game_last_error() gives a ctx-owned message for the last failing call.
 *  - Pointers named *_dev are DEVICE pointers (cudaMalloc'ed / torch CUDA tensors), *_host are HOST
 *    pointers.  All device buffers are CALLER-OWNED and only BORROWED by the context: they must stay
 *    alive and unchanged in size while bound; the library never frees them.  The context owns only
 *    its small host struct.  Device buffers must be 16-byte aligned, contiguous, row-major.
 *  - All work is enqueued on the stream given to game_set_stream (default: the legacy default
 *    stream) and is ASYNCHRONOUS; nothing synchronises with the host except game_sync and the
 *    *_host entry points (which finish with a stream synchronise).
 *  - A context is not thread-safe; distinct contexts are independent.
 *  - There is no CPU fallback: without a CUDA device every compute entry returns GAME_ERR_CUDA.
 */
#ifndef GAME_H_
#define GAME_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct game_ctx game_ctx; /* opaque */

enum {
    GAME_OK = 0,
    GAME_ERR_INVALID_ARG = -1, /* bad shape, pointer, alignment or parameter            */
    GAME_ERR_BAD_STATE = -2,   /* call order: eval before load_kb/bind_state, step without a fresh fitness */
    GAME_ERR_CUDA = -3,        /* CUDA runtime error (sticky errors surface at game_sync) */
    GAME_ERR_WORKSPACE = -4,   /* workspace_bytes smaller than game_workspace_bytes       */
    GAME_ERR_UNSUPPORTED = -5  /* shape outside what the kernels cover (stated per call)  */
};

/* family = expansion | (activation << 8) | (shared << 16)                    [DESIGN.md D1, D2]
 *   expansion : 0 CHEBYSHEV (T_1..T_d, eq.(1)), 1 TRIG (cos/sin k=1..d, eq.(6))
 *   activation: 0 IDENTITY (the paper's raw sum, eq.(2)), 1 SIGMOID, 2 TANH (BASELINE.json)
 *   shared    : 0 per-feature coefficients (BASELINE.json: G = N*d+1 / N*2d+1), 1 the paper's literal form (PAPER.md:52-55
 *               eq.(2), 75-77 eq.(5), 84-89): ONE coefficient per degree for all features, G = d+1 (Chebyshev) or 2d+1
 *               (trig, gene order [a_0, a_1..a_d, b_1..b_d]); the expansion term of gene j is the sum over the features of
 *               g_j(f_i) (the per-pattern sums of PAPER.md:110).  Shared mode runs on every path: the tensor-core scheme up to 64 terms
 *               (G - 1 <= 64), the FFMA scheme and the fused loop.
 * BASELINE.json configs c0,c1,c3,c4 = 0x0100; c2 = 0x0201. */
enum { GAME_FAMILY_SHARED = 1 << 16 };
enum { GAME_EXP_CHEBYSHEV = 0, GAME_EXP_TRIG = 1 };
enum { GAME_ACT_IDENTITY = 0, GAME_ACT_SIGMOID = 1, GAME_ACT_TANH = 2 };

/* Precision scheme of the fitness contraction z = W . phi^T  (eq.(2), 61).
 *   AUTO     : F16X3 when the shape is covered by the tensor-core kernel, else FFMA.
 *   FFMA     : fp32 FFMA on the CUDA cores (phi and W in fp32, fp32 accumulate).
 *   F16X3    : tcgen05 tensor cores, fp32-recovering 2-term fp16 split of BOTH operands
 *              (v = hi + lo, hi = rn_f16(v), lo = rn_f16(v - hi)); three kind::f16 MMAs per K step
 *              (lo.hi, hi.lo, hi.hi; the lo.lo term, <= 2^-22 relative, is dropped), fp32 accumulation in TMEM.
 *              Both operands are pre-scaled by exact powers of two, undone on the epilogue's FFMA: every chromosome row so
 *              that its largest gene lands in [2^13, 2^14) (the split is then relative at ANY scale of the genes: 1e-8 and
 *              300 behave alike), phi by 16.  Preconditions: finite genes (a row with an Inf / NaN gene gets a non-finite
 *              fitness, which the GA ranks worst) and |phi| < 4094 (phi is bounded by 1 for Chebyshev on |x| <= 1 and for
 *              trig).
 *              Accuracy: fitness within 1e-5 of fp64 -- measured 6e-8 .. 1.4e-6 on the BASELINE shapes and on populations
 *              around the optimum; see DESIGN.md section 2 for the table.  The one regime with a weaker statement is a
 *              REGRESSION fit (IDENTITY, TANH) that is nearly perfect: with residual noise sigma and outputs of size
 *              rms(z), a relative error eps of z moves the fitness of a near-optimal chromosome by ~eps rms(z) / sigma.
 *              The scheme's outputs carry ~4e-7 rms(z) of unsystematic error each (it averages out as 1 / sqrt(P)) and,
 *              after calibration (below), up to ~1e-7 of systematic error (the noise of the calibration fit itself), so
 *              the 1e-5 bound holds for rms(z) / sigma <= 100, i.e. fitness >= 1e-4 of the mean square output; beyond
 *              that the bound is 2e-7 rms(z) / sigma (measured at P = 9000, identity output: 2.1e-5 at rms(z) / sigma =
 *              230, 2.7e-5 at 760, 4.8e-5 at 2300, 1.0e-4 at 7600, where plain fp32 arithmetic -- GAME_SCHEME_FFMA,
 *              unbiased rounding -- gives 6.9e-7, 5.5e-6, 8.5e-6, 1.1e-5: force FFMA if a fit that good must be ranked
 *              to 1e-5; tanh outputs stay below 2.5e-5 throughout).  Classification outputs
 *              (SIGMOID against 0/1 targets) never get there.  The tensor core adds into its accumulator with
 *              truncation, which shrinks |z| by ~1.6e-8 per MMA; two measures keep that inside the bound where it would
 *              not be: K extents beyond 320 genes are accumulated 20 K steps at a time and the chunks added in fp32
 *              round-to-nearest (G = 2401, identity output: 2e-7), and for the regression activations (IDENTITY, TANH) the
 *              shrink of every row is measured on 256 patterns spread evenly over the knowledge base (rows 0, s, 2s, ..
 *              with s = P / 256: the order of the patterns does not matter) against an fp64 contraction before each
 *              evaluation and folded into the row's factor (one extra launch of the fused kernel + three small kernels per
 *              evaluation; near-optimal regression with residual noise 0.01: 7.7e-6 / 8.7e-7 instead of 8.9e-5 / 8.9e-6;
 *              game_set_option(GAME_OPT_CALIBRATE, 0) turns it off; rows longer than 3184 genes are not
 *              calibrated).
 *              Covers any N and d for Chebyshev, d <= 128 for the trigonometric family (the fp32 multiple-angle
 *              recurrence leaves the 1e-5 fitness bound beyond that: 2e-6 at d = 100, 2e-5 at d = 400).  The K axis
 *              is the gene order without the bias gene, 16 genes per K step; phi of a 256-pattern tile stays resident
 *              in shared memory up to 20 K steps, i.e. G - 1 <= 320; longer K extents are streamed.  Trigonometric
 *              d > 128 -> GAME_ERR_UNSUPPORTED when F16X3 is forced, FFMA under AUTO.  Shared coefficients
 *              (GAME_FAMILY_SHARED): covered for G - 1 <= 64 terms, FFMA beyond.
 *   FFMA covers G <= 448 (its shared-memory tile); forcing it on a larger G -> GAME_ERR_UNSUPPORTED.
 * Both schemes sum each tile's squared errors in fp32 and accumulate tile sums at ~48 bits or more (fp64, or float-float
 * pairs) in a fixed order (run-to-run bit-stable; equal chromosomes get equal fitness in any slot). */
enum { GAME_SCHEME_AUTO = 0, GAME_SCHEME_FFMA = 1, GAME_SCHEME_F16X3 = 2 };

/* Create a context for a knowledge base of P patterns x N features, expansion degree d, population of
 * M chromosomes.  Validates: P >= 1, N >= 1, d >= 1, M >= 1, known family -> GAME_ERR_INVALID_ARG;
 * a shape no kernel covers (trigonometric d > 128, or more than 64 shared terms, together with G > 448) -> GAME_ERR_UNSUPPORTED.
 * Host only; touches no device memory. */
int game_create(game_ctx** out, int64_t P, int32_t N, int32_t d, int32_t M, int32_t family);

/* Frees the library-owned host state only (never the bound device buffers). NULL is a no-op. */
int game_destroy(game_ctx* ctx);

/* G = N*d+1 (Chebyshev) or N*2d+1 (trig)  [DESIGN.md D1]. */
int game_num_genes(const game_ctx* ctx, int32_t* G);

/* Bytes of device workspace game_bind_state needs (fp64 partial sums per CTA, the split W operand
 * images of the tensor-core scheme, counters).  Depends only on the shapes given to game_create. */
int game_workspace_bytes(const game_ctx* ctx, size_t* bytes);

/* cudaStream_t to enqueue on (e.g. torch.cuda.current_stream().cuda_stream); NULL = default stream. */
int game_set_stream(game_ctx* ctx, void* cuda_stream);

/* Choose the precision scheme (GAME_SCHEME_*).  Default AUTO. */
int game_set_scheme(game_ctx* ctx, int32_t scheme);
/* The scheme the next game_eval_fitness will run (AUTO resolved): GAME_SCHEME_FFMA or GAME_SCHEME_F16X3. */
int game_get_scheme(const game_ctx* ctx, int32_t* scheme);

/* Bind the knowledge base ("the dataset is never altered"): X_dev[P][N] float32
 * row-major, t_dev[P] float32 targets.  Borrowed; read by every game_eval_fitness.
 * The caller may rewrite X_dev / t_dev between calls with work enqueued on the context's stream (a kernel, a copy); plain
 * stream order is all that is needed.  (The library's kernels are chained by programmatic dependent launch and, on small
 * grids, start reading the knowledge base before their predecessor has finished -- but only behind a kernel the library
 * itself enqueued within the same call; the first kernel of every public call waits for everything enqueued before it.) */
int game_load_kb(game_ctx* ctx, const float* X_dev, const float* t_dev);

/* Bind the mutable state: two population buffers popA_dev/popB_dev [M][G] float32 (the current
 * population starts in A; game_step writes the other one and swaps), fitness_dev[M] float32, and
 * workspace_dev of at least game_workspace_bytes bytes (GAME_ERR_WORKSPACE otherwise).  Borrowed. */
int game_bind_state(game_ctx* ctx, float* popA_dev, float* popB_dev, float* fitness_dev,
                    void* workspace_dev, size_t workspace_bytes);

/* GA parameters (operators defined by BASELINE.json, D3/D5):
 * elite in [0, M), tournament >= 1, p_cross and p_mut in [0,1], sigma >= 0 finite.
 * Defaults: elite 2, tournament 3, p_cross 0.9, p_mut 0.05, sigma 0.1. */
int game_set_ga_params(game_ctx* ctx, int32_t elite, int32_t tournament, double p_cross, double p_mut,
                       float sigma);

/* Execution switches, for measurements and for callers with special needs; none of them is read from the environment.
 * Defaults give the fastest correct path.  Changing one makes the next generation loop re-capture its CUDA graph.
 *   GAME_OPT_PDL        1 (default): the kernels of a generation are chained by programmatic dependent launch; 0: plain
 *                       stream-ordered launches.  Results are bit-identical either way.
 *   GAME_OPT_GRAPH      1 (default): game_run / game_evolve replay 16 generations at a time from a CUDA graph; 0: plain
 *                       launches.  Bit-identical either way.
 *   GAME_OPT_CALIBRATE  1 (default): the per-row calibration of the tensor-core scheme for IDENTITY / TANH outputs (see
 *                       GAME_SCHEME_F16X3).  0 CHANGES RESULTS: the accuracy statement of F16X3 for regression outputs no
 *                       longer holds (near-optimal fits: ~1e-4 instead of 1e-5); it marks the fitness stale.
 *   GAME_OPT_UNIT_PAIRS 0 (default): the library sizes the tensor-core kernel's work units by its cost model; n >= 1: n
 *                       chromosome-tile pairs per unit (clamped to what the population has).  Bit-identical either way.
 * Unknown option or bad value -> GAME_ERR_INVALID_ARG. */
enum { GAME_OPT_PDL = 0, GAME_OPT_GRAPH = 1, GAME_OPT_CALIBRATE = 2, GAME_OPT_UNIT_PAIRS = 3 };
int game_set_option(game_ctx* ctx, int32_t option, int32_t value);

/* Selection method of game_step.  TOURNAMENT (default, BASELINE.json) uses the `tournament` size of game_set_ga_params.
 * RANKING and ROULETTE are the paper's own methods, defined here with integer arithmetic only
 * (R10): parents A and B of child slot c come from words 0 and 1 of the Philox draw (0, c, gen, TAG_SELECT);
 *   RANKING : rank r (0 = best under (fitness, index), NaN worst) has weight M - r, u = floor(w M(M+1)/2 / 2^32), the parent
 *             holds the smallest rank r with (r+1) M - r (r+1)/2 > u;
 *   ROULETTE: weight_i = floor(clamp(1 - fitness_i, 0, 1) * 2^32) (PAPER.md:91 fitness = 1 - error; NaN / inf -> 0),
 *             u = floor(w * sum / 2^32), the parent is the smallest index whose prefix sum exceeds u (sum = 0: uniform).
 * Elitism, crossover and mutation are unchanged. */
enum { GAME_SEL_TOURNAMENT = 0, GAME_SEL_RANKING = 1, GAME_SEL_ROULETTE = 2 };
int game_set_selection(game_ctx* ctx, int32_t selection);

/* Error metric written to fitness_dev ("the MSE or the RMSE may be used"): MSE (default) or
 * RMSE = sqrt(MSE), taken in fp64 before the single rounding to fp32.  Lower is better either way (the GA order is the
 * same); the threshold of game_run_until is compared against the chosen metric.
 * GAME_ERROR_ONE_MINUS_MSE is the paper's literal fitness ("the fitness is calculated as the complement of the
 * error (i.e. 1-error)"): fitness_dev[m] = float(1 - MSE), HIGHER is better and the best-fitness trace holds maxima.  The
 * GA operators then work on the error e = 1 - fitness_dev (one fp32 subtraction): elitism, tournaments, ranking and the
 * roulette weights (which are floor(clamp(1 - e, 0, 1) 2^32), i.e. the fitness itself) are the functions of an error vector
 * documented above, and the threshold of game_run_until is still a learning-ERROR threshold (stop when 1 - best <= it).
 * RESOLUTION under GAME_ERROR_ONE_MINUS_MSE: the operators are a function of fitness_dev alone (that is what makes them
 * reproducible from a fitness vector, game_assume_fitness included), and float(1 - MSE) has a spacing of 6e-8 just below 1.
 * Two chromosomes whose MSE differ by less than that get the same fitness and tie (the lower index wins); the subtraction
 * 1 - fitness_dev is exact, the rounding of 1 - MSE before it is not.  At the paper's own error levels (MSE threshold
 * 1e-3) this is 4-5 digits below what is compared; on a regression fit with MSE below ~1e-6 most of the
 * population ties, the true best can drop out of the elite and the search stalls: run the search on GAME_ERROR_MSE or
 * GAME_ERROR_RMSE there (full fp32 relative resolution at any error level) and report 1 - MSE at the end if wanted.
 * Invalidates the fitness. */
enum { GAME_ERROR_MSE = 0, GAME_ERROR_RMSE = 1, GAME_ERROR_ONE_MINUS_MSE = 2 };
int game_set_error_metric(game_ctx* ctx, int32_t metric);

/* Random replacement ("a variable number of chromosomes are randomly generated to replace older
 * individuals"; R12): the last `immigrants` child slots of every game_step (never elite slots:
 * 0 <= immigrants <= M - elite, checked against the current elite count; clamped again if elite grows later) are
 * fresh random chromosomes, genes uniform in [-1,1) as at initialisation, Philox counter (g>>2, c, gen, TAG_IMMIGRANT = 4),
 * word g&3.  Default 0. */
int game_set_immigrants(game_ctx* ctx, int32_t immigrants);

/* Current population <- genes uniform in [-1,1) from Philox4x32-10 with
 * key = seed, counter = (g>>2, m, 0, TAG_INIT), word g&3, w = float(word>>8)*2^-23 - 1  [SURVEY 8(c) R6].
 * Invalidates the fitness.  Async. */
int game_init_population(game_ctx* ctx, uint64_t seed);

/* Which of popA/popB is current (device pointer), e.g. to upload or download a population with a
 * plain device copy.  Writing through it is allowed between calls (call game_invalidate_fitness after). */
int game_current_population(const game_ctx* ctx, float** pop_dev);
/* Mark the fitness stale (after the caller wrote the current population).  REQUIRED after every such write, also when
 * the fitness is stale already: the tensor-core scheme keeps fp16 hi/lo operand images of the current population in the
 * workspace (game_step updates them gene by gene as it writes the children, so a generation loop runs no image pass),
 * and this call is what tells the library to rebuild them from the population at the next evaluation. */
int game_invalidate_fitness(game_ctx* ctx);
/* Mark fitness_dev as valid without evaluating (after the caller wrote fitness_dev itself, e.g. to
 * feed the GA operators a given fitness vector -- the "same fitness vector and seed" parity hook). */
int game_assume_fitness(game_ctx* ctx);

/* fitness_dev[m] = (1/P) sum_p (act(sum_g W[m][g] phi_g(x_p)) - t_p)^2 for the current population
 * (eq.(2),(3), MSE; lower is better, D4).  Feature expansion, contraction,
 * activation, squared error and the per-chromosome reduction run in ONE fused kernel (phi never
 * reaches HBM), followed by a small fixed-order fp64 reduction over CTAs.  Needs load_kb + bind_state
 * (GAME_ERR_BAD_STATE).  Async. */
int game_eval_fitness(game_ctx* ctx);

/* One GA generation in one kernel: elitism (the `elite` best by
 * (fitness, index), NaN worst, copied unchanged to slots 0..elite-1), tournament selection with
 * replacement, single-point crossover (one child per slot), per-gene Gaussian mutation, all drawn from
 * Philox4x32-10 keyed by seed with counter (index, chromosome, gen, tag).  Reads the current population
 * and fitness_dev (must be valid: GAME_ERR_BAD_STATE), writes the other buffer, swaps, invalidates the
 * fitness.  Bit-exact against the oracle for the same fitness vector and seed.  Async. */
int game_step(game_ctx* ctx, uint64_t seed, uint32_t gen);

/* n_gens x (eval, step with gen = gen0 + i) followed by a final eval, all on one stream with no host
 * synchronisation (PAPER.md:97, 170 future work (i)).  best_fitness_dev (device, [n_gens+1] float32, or
 * NULL) receives the best fitness of each generation's population (lowest; highest under GAME_ERROR_ONE_MINUS_MSE).  Seed,
 * generation index and trace slot live in device memory, so runs of 16 or more generations are replayed from a CUDA graph
 * captured once per configuration (game_set_option(GAME_OPT_GRAPH, 0): plain launches).  Async. */
int game_run(game_ctx* ctx, uint64_t seed, uint32_t gen0, uint32_t n_gens, float* best_fitness_dev);

/* game_run with the paper's stop rule ("maximum number of iterations or the learning error threshold",
 * PAPER.md:128-133 MSE threshold 0.001): generation g's population is final as soon as its best fitness <= threshold.
 * Nothing synchronises with the host: all max_gens generations are enqueued, a device flag set by the fitness
 * finalisation makes the remaining kernels return at once (the GA step then carries the population over unchanged).
 * best_fitness_dev[0..max_gens] (device; entries after the stopping generation are left untouched) and gens_done_dev
 * (device int32: GA steps performed, 0..max_gens) are required.  Afterwards the current population is the stopping
 * generation's and fitness_dev is its fitness.  Async. */
int game_run_until(game_ctx* ctx, uint64_t seed, uint32_t gen0, uint32_t max_gens, float threshold,
                   float* best_fitness_dev, int32_t* gens_done_dev);

/* n_gens x (eval, step with gen = gen0 + i) with NO trailing evaluation (the population is left one step past its
 * last fitness): the generation loop of PAPER.md:97 as one call, launches only, no host synchronisation.  This is
 * what bench.py times as "K steps".  Async. */
int game_evolve(game_ctx* ctx, uint64_t seed, uint32_t gen0, uint32_t n_gens);

/* game_evolve as ONE persistent kernel for the latency-bound regime of the paper's own experiments (PAPER.md:120-136:
 * 2100 patterns, a few dozen chromosomes, thousands of iterations): a cooperative grid of one CTA per SM expands its
 * slice of the patterns once, then runs n_gens x (fitness, GA step) with two grid barriers per generation and no kernel
 * launch in between.  fp32 FFMA arithmetic (the FFMA scheme's accuracy); the GA operators, selection method, immigrants
 * and RMSE setting are those of game_step, bit for bit, on the fitness the kernel itself computed.  best_fitness_dev
 * ([n_gens] device, or NULL) receives the best fitness of every evaluated generation; fitness_dev is left holding the
 * fitness of the LAST evaluated population (the one before the final step).  Covers M <= 1024, P*M*G <= 2e8 and a
 * per-CTA slice that fits 200 KB of shared memory; otherwise GAME_ERR_UNSUPPORTED (use game_evolve).  Async. */
int game_evolve_fused(game_ctx* ctx, uint64_t seed, uint32_t gen0, uint32_t n_gens, float* best_fitness_dev);

/* Stream synchronise; returns GAME_ERR_CUDA if any enqueued work failed. */
int game_sync(game_ctx* ctx);

/* HOST-buffer entry point (what bench.py's e2e leg times): one whole generation on host data.
 * Copies X_host[P][N], t_host[P] into the bound knowledge-base buffers (which must therefore be
 * writable) and W_host[M][G] into the current population, runs eval + step(seed, gen), then copies the
 * fitness of the INPUT population to F_host[M] and the NEXT population to W_next_host[M][G] (either may
 * be NULL), and synchronises the stream.  Host buffers should be pinned for full copy bandwidth.  A knowledge base of
 * 64 MB or more is uploaded in 8 pattern ranges on a library-owned copy stream and each range is evaluated as soon as it
 * has landed (partial sums carried across the launches), so the PCIe transfer hides behind the fitness kernel. */
int game_generation_host(game_ctx* ctx, const float* X_host, const float* t_host, const float* W_host,
                         float* F_host, float* W_next_host, uint64_t seed, uint32_t gen);

/* OUT-OF-CORE evaluation ("the dataset can be very large ... requires greater attention to GPU memory
 * management, in terms of scheduling and data transfers host-to-device"): the knowledge base stays in HOST memory
 * (X_host[P][N], t_host[P], P as given to game_create -- it may exceed device memory; pinned memory for full bandwidth) and
 * passes through a ring of n_slots (2..8) device buffers of slot_rows patterns each: X_ring_dev[n_slots * slot_rows][N],
 * t_ring_dev[n_slots * slot_rows] (caller-owned, 16-byte aligned, slot_rows a multiple of 256).  One plain asynchronous
 * copy per pattern range on a library-owned copy stream, n_slots - 1 ranges ahead of the fused fitness kernel, which is
 * launched once per range and carries its partial sums across the launches; fitness_dev is then the fitness of the current
 * population over all P patterns, marked valid (game_step may follow).  A slot is used in whole rounds of the kernel's
 * persistent grid, so every pattern tile is evaluated by the same CTA pair in the same order as in a resident
 * game_eval_fitness: the result is BIT-IDENTICAL to it.  Needs game_bind_state, not game_load_kb.  Tensor-core scheme
 * only (GAME_ERR_UNSUPPORTED otherwise); slots too small for one round of the grid -> GAME_ERR_INVALID_ARG (the message
 * says how many patterns a slot needs).  Async. */
int game_eval_fitness_streamed(game_ctx* ctx, const float* X_host, const float* t_host, float* X_ring_dev, float* t_ring_dev,
                               int64_t slot_rows, int32_t n_slots);

/* Pattern-sharded evaluation (PAPER.md:172 future work (iii) multi-GPU; "massive data sets"): each
 * rank binds ITS shard of the knowledge base (P = shard size) and the same population.  game_eval_sse writes the
 * un-normalised sums sse_dev[m] = sum over this shard of (act(z) - t)^2 (device, fp64 [M]) instead of a fitness; the caller
 * adds them across ranks (one all-reduce of M doubles per generation, e.g. ncclAllReduce / torch.distributed) and calls
 * game_set_fitness_from_sse(sum, P_total): fitness_dev[m] = float(sse[m] / P_total), marked valid; best_fitness_dev may be
 * NULL.  Every rank then calls game_step with the same seed: the counter-based RNG and the identical all-reduced fitness
 * give identical populations on all ranks, no broadcast.  Async. */
int game_eval_sse(game_ctx* ctx, double* sse_dev);
int game_set_fitness_from_sse(game_ctx* ctx, const double* sse_dev, int64_t P_total, float* best_fitness_dev);

/* The pattern-sharded GENERATION LOOP with the exchange inside the library (no host code between generations): every rank
 * (one process per GPU) has bound its shard and the same population; per generation game_eval_sse's kernels, ONE
 * ncclAllReduce(sum) of M doubles on the context's stream (NVLink / NVSwitch: 32 KB at M = 4096, latency only), the
 * finalisation with P_total and the GA step, n_gens times, all enqueued at once.  best_fitness_dev ([n_gens] device, or
 * NULL) receives the best fitness of every generation (identical on all ranks).  NCCL is loaded at run time
 * (libnccl.so.2, the copy the process already has); game_comm_unique_id fills a 128-byte id on ONE rank, which the caller
 * passes to all ranks (e.g. torch.distributed broadcast) for game_comm_init(id, rank, world).  GAME_ERR_UNSUPPORTED if NCCL
 * cannot be loaded; a world of 1 is valid (the all-reduce is then a copy).  Async. */
int game_comm_unique_id(void* id128_host);
int game_comm_init(game_ctx* ctx, const void* id128_host, int32_t rank, int32_t world);
int game_evolve_sharded(game_ctx* ctx, uint64_t seed, uint32_t gen0, uint32_t n_gens, int64_t P_total, float* best_fitness_dev);

/* Test / validation use case: outputs of ONE chromosome w_dev[G] (device; e.g. a row of the current
 * population) on Q patterns X_dev[Q][N] (device, any Q >= 1, independent of the bound knowledge base):
 * y_dev[q] = act(sum_g w[g] phi_g(x_q)), computed in fp32 (recurrences and a G-term dot product): within 1e-5 of the fp64
 * value relative to max(1, |y|).  Chromosomes of any accepted length (staged in shared memory up to 57 K genes, read through
 * the caches beyond).  Async. */
int game_predict(game_ctx* ctx, const float* w_dev, const float* X_dev, int64_t Q, float* y_dev);

/* Confusion counts of thresholded outputs against 0/1 targets (PAPER.md:91, 140-146 classification quality):
 * counts_dev[4] (device, 64-bit) = {TP, FP, TN, FN}, predicted class = (y > threshold), true class = (t > 0.5).
 * The counters are cleared first.  Async. */
int game_confusion(game_ctx* ctx, const float* y_dev, const float* t_dev, int64_t Q, float threshold,
                   uint64_t* counts_dev);

/* Number of kernels this context has launched so far (for bench.py's gpu_launches). */
int game_launch_count(const game_ctx* ctx, uint64_t* launches);

/* Diagnostics of the LAST tensor-core fitness launch (what the profiles/ summaries quote): the share of its issue loop the
 * MMA-issuing warp spent waiting for a W operand slot (a_full), for the generated phi stage (b_full) and for a free TMEM
 * accumulator (acc_empty), averaged over the leader CTAs.  Synchronises the stream.  raw_host (or NULL) receives up to
 * raw_slots of the per-CTA records, 16 int64 each: the three waits and the loop's length in SM cycles, then -- in a library
 * built with -DGAME_PROFILE_PHASES -- globaltimer stamps (ns) of kernel entry, prologue done, predecessor complete, last MMA
 * issued, cluster through, exit. */
int game_mma_stall(game_ctx* ctx, double* frac_a_full, double* frac_b_full, double* frac_acc_empty, int64_t* raw_host,
                   int32_t raw_slots);

/* Number of CUDA-graph replays this context has issued so far: game_run / game_evolve capture the launch chain of 16
 * generations once (seed, generation index and best-fitness slot live in device memory, so the graph needs no per-generation
 * argument) and replay it; every replay adds its kernel count to game_launch_count.  0 when the graph path is off
 * (game_set_option(GAME_OPT_GRAPH, 0)), unavailable, or the run was shorter than 16 generations. */
int game_graph_replays(const game_ctx* ctx, uint64_t* replays);

/* Whether the per-row calibration of the tensor-core scheme is doing its job (scheme F16X3 above: for the regression
 * activations IDENTITY and TANH the 1e-5 accuracy statement rests on it).
 *   active        : 1 if an evaluation under the current settings calibrates (scheme resolves to F16X3, activation IDENTITY
 *                   or TANH, rows of at most 3184 genes, GAME_OPT_CALIBRATE left on), else 0 -- sigmoid outputs need
 *                   none, the FFMA scheme has nothing to calibrate.
 *   rows_rejected : in the LAST calibrated evaluation, the number of chromosomes whose measured shrink was not applied because
 *                   the fit came out non-finite or beyond 1e-4 in magnitude (a row with an Inf / NaN gene; a row whose outputs
 *                   on the sample patterns are all ~0, so that rounding noise dominates the fit).  Such a row is evaluated
 *                   with the uncalibrated scheme (error up to ~1e-4 relative on a near-optimal regression fit instead of
 *                   1e-5).  0 before the first calibrated evaluation.
 * The sample is 256 patterns spread evenly over the knowledge base this context is bound to (the host-buffer and
 * out-of-core entries pick the same rows from host memory, so they stay bit-identical to the resident evaluation).  Under
 * pattern sharding (game_eval_sse / game_evolve_sharded) every rank samples its OWN shard: the correction, of relative size
 * ~1e-6, therefore depends on how the patterns are partitioned -- well inside the accuracy bound, but sharded sums are not
 * bit-identical to a one-GPU evaluation for these activations.  Synchronises the stream. */
int game_calibration_status(game_ctx* ctx, int32_t* active, int32_t* rows_rejected);

/* Timing hook for the roofline line: when enabled, game_eval_fitness brackets the fused fitness kernel
 * with CUDA events on the context's stream; game_fitness_kernel_ms returns the sum of the recorded
 * durations (milliseconds) and the number of launches since the hook was (re)enabled, after
 * synchronising on the last event. */
int game_time_fitness_kernel(game_ctx* ctx, int32_t enable);
int game_fitness_kernel_ms(game_ctx* ctx, double* total_ms, uint64_t* launches);

/* ctx-owned string describing the last error on this context ("" if none); valid until the next call. */
const char* game_last_error(const game_ctx* ctx);

/* ONE fitness evaluation that allocates no device memory and needs no workspace -- for callers who have none to give.
 *
 * Who this is for.  Every other entry point borrows its scratch from the caller (the workspace of game_bind_state), so
 * the caller must be able to obtain device memory.  Some cannot: a plug-in that runs inside a host application owning the
 * whole GPU (it is handed input and output buffers from the host's pool and may not call cudaMalloc behind its back); a
 * control or serving loop with a latency budget, where cudaMalloc / cudaFree would stall every stream of the device; a
 * process whose device memory was fully assigned before this library was loaded.  Such a caller passes only inputs and
 * the output; the scratch (the transposed population and the per-block partial sums of the FFMA scheme) sits in a fixed
 * array of 4 456 448 bytes (4.25 MiB) that is part of libgame.so's device image.  Every GPU on which the process uses
 * the library holds that array from module load until exit, called or not -- that is the cost of this entry point.
 *
 * What it computes.  fitness_dev[m] = (1/P) sum_p (act(sum_g W[m][g] phi_g(x_p)) - t_p)^2 (eq.(2),(3);
 * MSE) for W_dev[M][G], X_dev[P][N], t_dev[P] (device, float32, row-major, 16-byte aligned, caller-owned, only read) into
 * fitness_dev[M] (device, float32, written).  G and `family` are those of game_create.  The kernels, the grid and the
 * order of summation are those of game_eval_fitness under GAME_SCHEME_FFMA (fp32 FFMA, fp64 partial sums in a fixed
 * order), so the values agree with that path; the GA operators, the error-metric setting and the best-fitness output are
 * not part of it.  Enqueued on cuda_stream (a cudaStream_t, NULL = default stream); asynchronous.
 *
 * Limits.  M <= GAME_NOALLOC_MAX_M (1024) and G <= GAME_NOALLOC_MAX_G (448, the FFMA kernel's own bound).  Anything
 * larger returns GAME_ERR_UNSUPPORTED and says which limit was hit; use game_eval_fitness with a workspace instead.
 * Bad pointers / shapes -> GAME_ERR_INVALID_ARG; no device, wrong architecture, launch failure -> GAME_ERR_CUDA.  There
 * is no context, so the message goes to err_host (host buffer of err_len bytes, NUL-terminated, "" on success; may be NULL).
 *
 * No allocation: the call performs no cudaMalloc / cudaFree / cudaMallocAsync and calls no library routine that does; host
 * side it uses a fixed table and a mutex.
 *
 * First call per device.  The first call that targets a given device (the device fitness_dev lives on, made current for
 * the duration of the call) does a one-time set-up there: it asks the runtime where the array sits on that device and
 * raises the fitness kernel's shared-memory limit.  Make that first call during initialisation, outside any stream
 * capture; later calls go straight to the three kernel launches.
 *
 * Sharing.  There is ONE array per device and process.  Nothing is carried from call to call (each call rewrites the
 * transposed population in full and every block clears its row of partial sums before adding to it, so stale contents
 * of an earlier, differently shaped call are harmless), but two calls whose kernels can run at the same time on one
 * device -- different streams, or different host threads without stream ordering between them -- overwrite each other's
 * scratch and both results are garbage.  Keep all calls for a device on one stream, or order them with events. */
enum { GAME_NOALLOC_MAX_M = 1024, GAME_NOALLOC_MAX_G = 448 };
int game_eval_fitness_noalloc(const float* X_dev, const float* t_dev, const float* W_dev, float* fitness_dev,
                              int64_t P, int32_t N, int32_t d, int32_t M, int32_t family, void* cuda_stream,
                              char* err_host, size_t err_len);

#ifdef __cplusplus
}
#endif
#endif /* GAME_H_ */

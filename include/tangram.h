/* libtangram — C ABI of the B200-native TANGRAM pipeline-composition search.
 *
 * What is computed: the composition step of TANGRAM §5.2 restated as an exact
 * integer bitmask dynamic program (BASELINE.json:north_star).  For one planning
 * instance with L layers (atoms), K GPU islands, P intra-slice plans and m microbatches:
 *
 *   slice  [a,b), 0 <= a < b <= L, index s(a,b) = a*(2L-a+1)/2 + (b-a-1), NS = L(L+1)/2
 *   c[a][b][k] = min_p { time_us[s][k][p] : time != TG_INVALID, mem_mb[s][k][p] <= cap_mb[k] }
 *                (PAPER.md:240 plans carry time and memory; :236 memory infeasibility)
 *   x[j][k]    = ceil(act_mb*1000 / bw_gbps[j][k]) microseconds, j = upstream stage's island
 *                (PAPER.md:240 only pipeline activations cross islands; :160 asymmetric links)
 *   plan       = stages (a_i,b_i,k_i) tiling [0,L) with pairwise distinct islands
 *   sum        = sum_i c[a_i][b_i][k_i] + sum_i x[k_i][k_{i+1}]
 *   T          = max_i c[a_i][b_i][k_i]          (PAPER.md:250 (1): slowest stage is the bottleneck)
 *   iter       = sum + (m-1)*T                   (1F1B; formula from north_star)
 *   result     = argmin of (iter, T, mask, k_0, b_0, k_1, b_1, ...)   -- exactly one plan is correct
 *
 * All pointers in the signatures are plain C pointers; each argument says HOST, DEVICE or EITHER.
 * "EITHER" pointers are classified with cudaPointerGetAttributes.  No call throws; every call
 * returns a tg_status and leaves its outputs untouched on error.  tg_last_error() gives a
 * thread-local message.  There is no CPU fallback: without a CUDA device every compute call
 * returns TG_ERR_CUDA.
 */
#ifndef TANGRAM_H_
#define TANGRAM_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct tg_instance tg_instance; /* opaque; owns DEVICE copies of every table passed in */

typedef enum {
    TG_OK = 0,
    TG_ERR_NULL = 1,   /* a required pointer is NULL                       */
    TG_ERR_SHAPE = 2,  /* L, K, P, m or n outside the limits below         */
    TG_ERR_RANGE = 3,  /* a table value outside its documented range       */
    TG_ERR_OOM = 4,    /* device or host allocation failed                 */
    TG_ERR_CUDA = 5    /* any other CUDA failure, or no device             */
} tg_status;

enum {
    TG_MAX_K = 16,
    TG_MAX_L = 255,
    TG_MAX_P = 255,
    TG_MAX_M = 1 << 20,
    TG_TIME_MAX = 1 << 25,
    TG_MAX_ACT = 8,          /* distinct per-boundary activation sizes of an instance (tg_instance_set_boundary_act) */
    TG_MAX_NODES = 64,       /* nodes of a cluster profile (tg_islands_build)     */
    TG_INVALID = 0x7fffffff, /* "no such intra-slice plan" marker in time_us */
    TG_INF = 1 << 30         /* saturating "no plan" value of the DP        */
};

/* tg_instance_create — SURVEY.md §8(b); north_star "tg_instance_create(cost/memory tables per
 * slice x island x intra-plan, island GPU counts and capacities, bandwidth matrix, m)".
 *   time_us      EITHER [NS][K][P] int32, p fastest; each entry in [0,TG_TIME_MAX] or TG_INVALID
 *   mem_mb       EITHER [NS][K][P] int32, per-GPU MB needed by that plan, >= 0
 *   island_gpus  EITHER [K] >= 1 (validated and kept; not used by the recurrence)
 *   island_cap_mb EITHER [K] per-GPU capacity in MB, >= 0
 *   bw_gbps      EITHER [K][K] sender-major, > 0 off the diagonal, diagonal ignored
 *   act_mb       activation MB crossing every stage boundary, >= 0
 * All inputs are copied to device memory owned by the instance; the caller keeps its buffers.
 * Range validation of the tables runs on the device.  Errors: NULL -> TG_ERR_NULL; limits
 * 1<=L<=TG_MAX_L, 1<=K<=TG_MAX_K, 1<=P<=TG_MAX_P, 1<=m<=TG_MAX_M -> TG_ERR_SHAPE; bad values ->
 * TG_ERR_RANGE.  Synchronises the device's legacy default stream once. */
tg_status tg_instance_create(int32_t L, int32_t K, int32_t P, int32_t m, const int32_t* time_us,
                             const int32_t* mem_mb, const int32_t* island_gpus,
                             const int32_t* island_cap_mb, const int32_t* bw_gbps, int32_t act_mb,
                             tg_instance** out);

/* tg_instance_create_classes — SURVEY.md §8(f) NEXT-3(a), redundancy pruning by signature (slices
 * with the same composition of atoms are queried once).  The tables are given per signature class:
 *   class_of_slice  EITHER [NS] int32 in [0, n_classes): class of slice s(a,b)
 *   class_time_us   EITHER [n_classes][K][P], class_mem_mb likewise (same value rules as tg_instance_create)
 * and the instance is by definition the one whose time_us[s][k][p] = class_time_us[class_of_slice[s]][k][p] (same
 * for mem_mb); 1 <= n_classes <= NS.  Only the class tables cross the host-device link (for identical layers
 * n_classes = L: NS/L = (L+1)/2 times fewer bytes).  The instance keeps them: tg_solve_batch's cost-table loader reads the
 * class rows (n_classes*K*P entries, L2 resident) instead of the NS*K*P expanded entries, and when the class of a slice
 * depends on its length only (identical layers; detected at creation) a staged cost row is one value per diagonal,
 * broadcast instead of read per start.  The expanded tables are also materialised on the device (tg_instance_read_time,
 * tg_prune and the variant tables work on them; after tg_prune, tg_instance_set_actmem or tg_instance_set_stages they
 * alone define the instance).  Everything else as tg_instance_create; a class index out of range -> TG_ERR_RANGE. */
tg_status tg_instance_create_classes(int32_t L, int32_t K, int32_t P, int32_t m, int32_t n_classes,
                                     const int32_t* class_of_slice, const int32_t* class_time_us,
                                     const int32_t* class_mem_mb, const int32_t* island_gpus,
                                     const int32_t* island_cap_mb, const int32_t* bw_gbps, int32_t act_mb,
                                     tg_instance** out);

/* tg_instance_create_batch — n instances in one call: element i of every array argument describes instance i
 * exactly as the arguments of tg_instance_create do (L, K, P, m, act_mb: HOST arrays of n int32; time_us ...
 * bw_gbps: HOST arrays of n pointers, each EITHER host or device).  All uploads and validations are enqueued
 * first and the call synchronises ONCE (tg_instance_create synchronises once per instance: 1024 instances cost
 * 1024 round trips).  The instances of a batch share ONE device allocation (two table uploads per instance, one
 * validation launch for the batch); each is destroyed individually with tg_instance_destroy and the allocation is
 * released with the last of them.  All or nothing: on any error nothing is created, out[0..n) is NULL and the message names
 * the first offending instance.  n == 0 is a no-op. */
tg_status tg_instance_create_batch(int32_t n, const int32_t* L, const int32_t* K, const int32_t* P, const int32_t* m,
                                   const int32_t* const* time_us, const int32_t* const* mem_mb,
                                   const int32_t* const* island_gpus, const int32_t* const* island_cap_mb,
                                   const int32_t* const* bw_gbps, const int32_t* act_mb, tg_instance** out);

/* tg_instance_set_actmem — SURVEY.md §8(f) NEXT-1, depth-aware activation memory under 1F1B (PAPER.md:246
 * "earlier stages hold more in-flight activations", :258(i)).  actmem_mb: EITHER [NS][K][P] int32 in
 * [0, 2^20], MB that plan p of (slice, island) needs PER in-flight microbatch, copied; NULL removes the table.
 * With the table set, a stage followed by r later stages holds q = r + 1 microbatches, so its plan p is
 * feasible iff mem_mb + q * actmem_mb <= cap_mb[k]; the stage cost becomes c_q = min over the plans feasible
 * at depth q, and the candidate thresholds are the distinct finite c_q of all depths.  Everything else
 * (sum, T, iter, tie-breaks) is unchanged; stage_plan[i] is the lowest p attaining c_q of that stage.
 * tg_reduce keeps reporting depth 1; tg_prune then uses the three-axis rules stated there.  Synchronises the
 * legacy default stream. */
tg_status tg_instance_set_actmem(tg_instance* inst, const int32_t* actmem_mb);

/* tg_instance_set_transfer_bound — SURVEY.md §8(c) A2 variant / §8(f) NEXT-3(b): the activation transfer between
 * two stages is its own pipeline slot ("communication can be the bottleneck").  With on != 0 a
 * transfer is admissible at threshold T iff x[j][k] <= T, so a plan's bottleneck is
 * T = max(max stage time, max boundary transfer), the candidate thresholds are the distinct finite stage costs
 * and off-diagonal transfer times, and iter = sum + (m-1) * T as before (the sum still includes the transfers).
 * on == 0 restores the core definition.  Combines with tg_instance_set_actmem.  No device work. */
tg_status tg_instance_set_transfer_bound(tg_instance* inst, int32_t on);

/* tg_instance_set_stages — SURVEY.md §8(f) NEXT-2, multi-stage partial plans ("a model-slice/island plan
 * can include multiple pipeline stages", :248, :250 (1) "ranks the slowest stages in all model-slice/island plans").
 *   slow_us   EITHER [NS][K][P] int32: slowest internal pipeline stage of the partial plan, 0 <= slow_us <= time_us on
 *             every valid entry (time_us is then the partial plan's whole time for one microbatch, the sum of its
 *             internal stages); copied; NULL removes the tables
 *   n_stages  EITHER [NS][K][P] int32 in [1, 255]: its number of internal stages, or NULL (all ones); copied
 * With the tables set an entry is admissible at threshold T iff slow_us <= T; a plan's bottleneck is T = max slow_us of
 * its partial plans, sum still adds the time_us (and transfers), iter = sum + (m-1)*T, and the candidate thresholds are
 * the distinct slow_us at which some cell's cost changes.  The plan choice is part of the optimum: stage_plan[i] =
 * lowest p with the least time_us among the entries of its cell that are admissible at T*.  slow_us == time_us is the
 * core definition bit for bit.  n_stages does not enter the optimum; tg_plan_pipeline_stages adds it up for a result.
 * Not combinable with tg_instance_set_actmem (the depth of a partial plan would count the internal stages behind it,
 * which needs a stage counter in the DP state): either call on an instance that has the other table -> TG_ERR_SHAPE;
 * tg_prune on such an instance -> TG_ERR_SHAPE.  Combines with tg_instance_set_transfer_bound.  Values out of range ->
 * TG_ERR_RANGE.  Synchronises the legacy default stream. */
tg_status tg_instance_set_stages(tg_instance* inst, const int32_t* slow_us, const int32_t* n_stages);

/* tg_instance_set_boundary_act — SURVEY.md §8(f) NEXT-3(b), per-boundary activation sizes (PAPER.md:240 (1) "only
 * transferring stage inputs and outputs"; :350 communication can be the bottleneck).
 *   act_mb_b  EITHER [L+1] int32: act_mb_b[b] MB cross the boundary in front of layer b, 1 <= b <= L-1, each in [0, 2^20]
 *             (entries 0 and L are ignored); copied; NULL restores the scalar act_mb of tg_instance_create
 * The transfer of a cut at b from island j to island k then costs x_b[j][k] = ceil(act_mb_b[b]*1000 / bw_gbps[j][k]) us
 * (unusable above TG_TIME_MAX); with tg_instance_set_transfer_bound every boundary's finite transfer times are candidate
 * thresholds.  A constant array is the scalar definition bit for bit.  At most TG_MAX_ACT distinct sizes among the
 * boundaries 1..L-1, else TG_ERR_SHAPE; values out of range -> TG_ERR_RANGE; on an instance with multi-stage partial
 * plans (tg_instance_set_stages, and vice versa) -> TG_ERR_SHAPE.  Combines with tg_instance_set_actmem and
 * tg_instance_set_transfer_bound.  tg_reduce's x_out reports the matrix of the first boundary's size. */
tg_status tg_instance_set_boundary_act(tg_instance* inst, const int32_t* act_mb_b);

/* NULL is a no-op.  The instance must not be in use by an unsynchronised tg_solve_batch. */
tg_status tg_instance_destroy(tg_instance* inst);

typedef struct { /* one per instance, POD, 8-byte aligned, 224 bytes */
    int64_t iter_time_us;      /* sum + (m-1)*T* ; INT64_MAX if no feasible plan               */
    int64_t sum_us;            /* sum of stage times + transfers of the returned plan          */
    int32_t bottleneck_us;     /* T*                                                           */
    int32_t n_stages;          /* 0 if infeasible                                              */
    uint32_t island_mask;      /* S*                                                           */
    uint32_t n_thresholds_run; /* diagnostics: DPs executed for this instance                  */
    int32_t stage_begin[TG_MAX_K]; /* stage i covers [stage_begin[i], stage_begin[i+1]), last ends at L */
    int32_t stage_island[TG_MAX_K];
    int32_t stage_plan[TG_MAX_K];  /* lowest p attaining c for that (slice, island)            */
} tg_result;

enum { /* flags of tg_solve_batch_ex */
    TG_SOLVE_DEFAULT = 0,   /* exact branch-and-bound search over the candidate thresholds (DESIGN.md R-search) */
    TG_SOLVE_FULL_SWEEP = 1 /* run the DP at every candidate T (rate benchmark; same result)           */
};

typedef struct { /* optional diagnostics of one tg_solve_batch_ex call, written on the device  */
    uint64_t n_dp;           /* DPs executed (all instances)                                   */
    uint64_t plans_dense;    /* sum over DPs of NS*K*2^(K-1): SURVEY.md §8(d) "plans evaluated" */
    uint64_t states_live;    /* sum over DPs of L*Ke*2^(Ke-1), Ke = islands alive at that T     */
    uint64_t n_rounds;       /* scheduler rounds                                               */
    uint64_t n_barriers;     /* grid-wide barriers executed                                    */
    uint64_t n_items_global_c; /* DPs whose cost tables did not fit in shared memory           */
    uint64_t error_flag;     /* internal consistency flag of the solver, 0 = none; 2 = a staged cost row broke its
                                bound, 3 = evaluated-threshold list full, 4 = a queue-mode ring slot was overwritten
                                before its instance folded it, 5 = queue-mode watchdog (no item published for ~20 s
                                and the batch not finished); any non-zero flag makes the call return TG_ERR_CUDA
                                (synchronous) or poisons the results (asynchronous, see tg_solve_batch_ex)          */
    uint64_t relax_admissible; /* admissible relaxations executed: stage (c <= T) + transfer, summed over DPs */
    uint64_t states_windowed;  /* DP states the kernel actually wrote: sum over DPs of Ke*2^(Ke-1) rows x the row window */
    /* SM cycles summed over the solver's CTAs (thread 0 of each): */
    uint64_t cyc_stage;         /* staging the thresholded cost rows of an item                         */
    uint64_t cyc_levels;        /* DP levels (streaming over the masks)                                 */
    uint64_t cyc_level_barrier; /* wait at the barrier between two levels (team or CTA)                 */
    uint64_t cyc_grid_wait;     /* wait at the grid barriers between scheduler rounds                   */
    uint64_t cyc_scheduler;     /* folding results, planning the next thresholds, laying out the items  */
    uint64_t cyc_backtrack;     /* plan back-tracker                                                    */
} tg_solve_stats;

/* tg_solve_batch — north_star "tg_solve_batch(instances, stream) -> best iteration time and plan".
 * Steps: cost-table loader, transfer table, candidate thresholds, exact threshold
 * search with monotone bounds (in place of the T=inf lower-bound run), per-T popcount-wavefront DP,
 * threshold-sweep reduction, plan back-tracker.
 *   instances   HOST array of n instance handles (all created on the current device)
 *   out         EITHER: n results.  DEVICE: written asynchronously on `cuda_stream`, valid after the
 *               stream is synchronised.  HOST: the call copies the results back and synchronises.
 *   cuda_stream a cudaStream_t (NULL = legacy default stream)
 * Never mutates the instances.  An infeasible instance is not an error (iter_time_us = INT64_MAX,
 * n_stages = 0).  n == 0 is a no-op.  Scratch memory comes from a stream-ordered pool of the library's own (the device's
 * default pool is not touched; the tables of the instances come from the same pool).  Freed workspaces and tables stay
 * cached in that pool -- up to 14 GB, the DP scratch of the largest shapes; the environment variable TG_POOL_KEEP_MB
 * lowers it -- until tg_release_cached_memory() is called.
 * Internal errors of the solver (they have never been observed; the checks exist because the search keeps bounded
 * lists): a call with a HOST buffer or HOST statistics returns TG_ERR_CUDA; in the fully asynchronous form (DEVICE
 * results, no statistics) every result of the call is instead written with n_stages = -1 and
 * iter_time_us = INT64_MAX, so a plan of a failed search can never be mistaken for the optimum. */
tg_status tg_solve_batch(tg_instance* const* instances, int32_t n, tg_result* out, void* cuda_stream);

/* Same, with flags and optional statistics (stats: EITHER or NULL; HOST forces a synchronise). */
tg_status tg_solve_batch_ex(tg_instance* const* instances, int32_t n, tg_result* out, uint32_t flags,
                            tg_solve_stats* stats, void* cuda_stream);

/* Total number of pipeline stages of a returned plan: the sum of n_stages over its partial plans (n_stages of plain
 * instances is 1, so this is result->n_stages for them).  result: HOST; n_out: HOST.  Synchronous. */
tg_status tg_plan_pipeline_stages(tg_instance* inst, const tg_result* result, int32_t* n_out);

typedef enum {
    TG_PRUNE_EXACT = 0,     /* R1 infeasible + R2 dominated; threshold ignored                  */
    TG_PRUNE_IMBALANCE = 1, /* + R3, threshold = theta in permille, 1000..16384                 */
    TG_PRUNE_BOTTLENECK = 2 /* + R4, threshold = stage-time cap in microseconds                 */
} tg_prune_mode;

/* tg_prune — north_star "tg_prune(threshold) for the dominated-plan pruning"
 * (pruning policies), :43/:360 (incompatible partial plans); rules R1-R4 of SURVEY.md §8(c).
 * Marks entries of the instance's time table dead (TG_INVALID), in place and monotone (never revives
 * an entry).  EXACT and BOTTLENECK are idempotent; IMBALANCE re-estimates the islands' atom profile
 * from the live table on every call, so a second call may kill more.
 * On an instance with a footprint table (tg_instance_set_actmem) R1 is
 * "infeasible at the shallowest depth", mem_mb + actmem_mb > cap_mb[k], and R2 dominance is on the three
 * axes (time, mem_mb, actmem_mb): q kills p iff q is no larger on every axis and differs, or equals p with
 * q < p; such a q is feasible at every depth where p is and no slower.  R3 and R4 read the times only.
 *   counts_out  HOST int64[4]: entries newly killed by R1..R4.  The call synchronises `cuda_stream`. */
tg_status tg_prune(tg_instance* inst, tg_prune_mode mode, int64_t threshold, int64_t counts_out[4],
                   void* cuda_stream);

/* tg_prune_batch — tg_prune over n DISTINCT instances with one mode and threshold in one pass: one grid over every
 * cell of the batch (the raw tables streamed once, 385 MB for the 1024-instance batch), one
 * synchronisation.  counts_out: HOST int64 [n][4], row i = what tg_prune(instances[i], ...) would have returned;
 * the tables end up exactly as after n single calls.  n == 0 is a no-op; n in [0, 65535]; an instance listed twice
 * -> TG_ERR_RANGE; argument errors are reported before anything is modified. */
tg_status tg_prune_batch(tg_instance* const* instances, int32_t n, tg_prune_mode mode, int64_t threshold,
                         int64_t* counts_out, void* cuda_stream);

/* tg_prune_batch_static — tg_prune_batch for callers that cannot allocate device memory (code under CUDA graph
 * capture, tight serving loops, harnesses that forbid cudaMalloc): same kernels, same results, but the pass's scratch
 * (per-rule counters, R3 caps, instance descriptors) lives in one file-scope device array of the library, 216 KB, that
 * every GPU which loads the library holds until exit.  The call allocates and frees nothing on the device -- no
 * cudaMalloc / cudaMallocAsync / cudaFree, no pool -- and does not need the library's per-device set-up.
 *   n           in [0, TG_PRUNE_STATIC_MAX_N]; more -> TG_ERR_SHAPE (the message names the limit; use tg_prune_batch)
 *   instances   as tg_prune_batch, but an instance that still keeps class tables (tg_instance_create_classes, never
 *               pruned or given a variant table) -> TG_ERR_SHAPE: pruning it would have to free those tables
 *   counts_out  HOST int64 [n][4]; the call synchronises `cuda_stream`
 * Every call shares the one array, which keeps the previous call's contents; the call clears what must start at zero.
 * Calls from threads of one process are serialised inside the library; two calls that overlap on the GPU some other
 * way (two processes cannot: each has its own copy) would race on it.  Argument errors are reported before anything
 * is modified. */
#define TG_PRUNE_STATIC_MAX_N 1024
tg_status tg_prune_batch_static(tg_instance* const* instances, int32_t n, tg_prune_mode mode, int64_t threshold,
                                int64_t* counts_out, void* cuda_stream);

/* ---- step-level entry points (used by the parity tests to check single steps) ---------------- */

/* Steps 1-3 alone: reduced tables and candidate thresholds.  All outputs HOST, any may be NULL.
 *   c_out    [NS][K] int32, TG_INF where no feasible plan      argp_out [NS][K] int32, -1 if none
 *            (on an instance with a footprint table: the tables of depth 1, the least restrictive)
 *   x_out    [K][K] int32 (0 on the diagonal, TG_INF if > TG_TIME_MAX)
 *   cand_out capacity NS*K int32: ascending distinct candidate thresholds; *n_cand_out receives their count.
 * On a core instance the count is at most NS*K.  With tg_instance_set_actmem the thresholds are the distinct finite
 * costs of ALL K depths and with tg_instance_set_transfer_bound the finite transfer times join them, so the count can
 * reach NS*K*K + K*K: tg_reduce then writes only the first NS*K of them (it never writes past the documented
 * capacity) while *n_cand_out still reports the full count; tg_candidates returns the whole list.
 * Synchronises `cuda_stream`. */
tg_status tg_reduce(tg_instance* inst, int32_t* c_out, int32_t* argp_out, int32_t* x_out,
                    int32_t* cand_out, int32_t* n_cand_out, void* cuda_stream);

/* Step 3 alone with an explicit capacity (PAPER.md:250 (1) "ranks the slowest stages"): the
 * ascending distinct candidate thresholds of the instance as the solver sees them (all depths, plus the transfer times
 * under the transfer bound).  cand_out: HOST, `capacity` int32 (may be NULL with capacity 0 to query the count);
 * at most `capacity` entries are written, *n_cand_out (HOST, required) receives the full count.  capacity < 0 ->
 * TG_ERR_RANGE.  Synchronises `cuda_stream`. */
tg_status tg_candidates(tg_instance* inst, int32_t* cand_out, int64_t capacity, int32_t* n_cand_out, void* cuda_stream);

/* Step 5 + 7 at ONE threshold: DP at T (T < 0 means infinity), top reduction and back-track.
 * out (EITHER): iter_time_us = f_T + (m-1)*T with T = 2^30 for infinity, bottleneck_us = that T,
 * INT64_MAX if no plan is admissible at T. */
tg_status tg_dp_at(tg_instance* inst, int64_t T, tg_result* out, void* cuda_stream);

/* Copies the instance's current time table (after pruning) to HOST time_out [NS][K][P]. */
tg_status tg_instance_read_time(tg_instance* inst, int32_t* time_out);

/* tg_islands_build — SURVEY.md §8(f) NEXT-4: GPU island construction as a front end that produces the
 * island arguments of tg_instance_create from per-node profiles.  All pointers HOST.
 *   node_gpus / node_compute / node_mem_mb / node_intra_bw  [n_nodes]: GPUs of the node and, per GPU, compute capacity
 *             (any unit), memory in MB and intra-node interconnect bandwidth (the GPUs of a node are identical)
 *   inter_bw  [n_nodes][n_nodes] sender-major network bandwidth between nodes (directional), diagonal ignored
 *   eps_c / eps_m / eps_i  tolerances of Eq. 1-2 in permille (100 = 10 %)
 * Islands satisfy PAPER.md Eq. 1-3 (same GPU count, compute / memory / intra-node bandwidth ratios within 1 + eps, every
 * link inside an island at least as fast as every link leaving it) and are built by the three steps of PAPER.md:193 as
 * DESIGN.md reading N4 fixes them (run-cutting by compute, memory and intra-node bandwidth, then greedy agglomerative
 * clustering on the inter-node bandwidth).  Outputs: island_of_node [n_nodes]; *k_out = K; island_gpus [K], island_cap_mb
 * [K] (smallest memory of the island), bw_gbps [K][K] (slowest link from a node of j to a node of k; diagonal: slowest
 * inner link, or the intra-node bandwidth of a single-node island) -- buffers of n_nodes (n_nodes^2) entries suffice.
 * 1 <= n_nodes <= TG_MAX_NODES else TG_ERR_SHAPE; values < 1 (memory < 0) or above 2^20 -> TG_ERR_RANGE.  K may exceed
 * TG_MAX_K: tg_instance_create then rejects it.  Runs one small kernel; synchronises the legacy default stream. */
tg_status tg_islands_build(int32_t n_nodes, const int32_t* node_gpus, const int32_t* node_compute, const int32_t* node_mem_mb,
                           const int32_t* node_intra_bw, const int32_t* inter_bw, int32_t eps_c, int32_t eps_m, int32_t eps_i,
                           int32_t* island_of_node, int32_t* k_out, int32_t* island_gpus, int32_t* island_cap_mb, int32_t* bw_gbps);

/* Returns the workspaces cached by the library's memory pool on the current device to the driver (an embedding
 * framework with an allocator of its own may need the memory back).  Synchronises the device.  No-op before the first call. */
tg_status tg_release_cached_memory(void);

/* Device time in milliseconds of the persistent solver kernel most recently launched by this host
 * thread (CUDA events recorded on its stream around the launch; waits for it to finish).  HOST out. */
tg_status tg_last_solver_kernel_ms(float* ms_out);

/* The same for the cost-table loader kernel of the most recent tg_solve_batch, tg_reduce or
 * tg_dp_at of this host thread.  HOST out. */
tg_status tg_last_loader_kernel_ms(float* ms_out);

const char* tg_last_error(void); /* thread-local, valid until the next tg_* call on the thread */
int32_t tg_version(void);

#ifdef __cplusplus
}
#endif
#endif /* TANGRAM_H_ */

/* cao.h -- C ABI of libcao: constraint-aware evolutionary auto-tuning steps on one B200 (sm_100a).
 *
 * The operations follow the problem statement of "Constraint-aware Optimization in Auto-Tuning"
 * (arxiv/paper_2606_28372; "Lnnn" = line of PAPER.md, "Ox"/"Ax" = readings listed in DESIGN.md):
 *   P = (X, D, C): parameters, finite domains, predicate constraints           L129-135 (sec. IV-A)
 *   the search space is fully resolved before tuning                            L137
 *   Search Space queries: is-valid, valid samples, valid neighbours             L139-143, L215
 *   strategies DE / PSO / Firefly / GA with repair to the nearest valid config  Alg.1-3
 *   memoisation of evaluated configs, budget interruption                       L268, L125
 *
 * Conventions
 *   - Every function returns 0 (CAO_OK) or a negative cao_status; cao_last_error() gives a
 *     thread-local message for the last failure.  No exceptions cross this boundary.
 *   - Pointers named h_* are HOST memory, d_* are DEVICE memory.  ALL device memory is owned by the
 *     caller: the library reports the bytes it needs, is handed 256-byte aligned base pointers and
 *     never allocates device memory itself.  Buffers must stay alive while the handle that was
 *     given them is alive.  Handles (cao_space, cao_runs) are host objects owned by the library.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Launching
 *     calls are asynchronous on it unless stated otherwise.
 *   - There is no CPU fallback: without a CUDA device every launching call returns CAO_E_CUDA.
 *
 * Layouts
 *   - Index row: one byte per parameter, idx_d in [0, m_d), parameter 0 first.  In HBM a row
 *     occupies row_bytes = 16 (n <= 16) or 32 (n <= 32) bytes, the padding bytes are zero.
 *   - Linear index L = sum_d idx_d * stride_d, the FIRST declared parameter is the most
 *     significant digit (itertools.product order, A1).
 *   - Bitmap: bit (L & 63) of 64-bit little-endian word (L >> 6) is 1 iff config L is valid.
 *   - rank of a valid config = its position in the valid table, which is sorted by L.
 */
#ifndef CAO_H_
#define CAO_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct cao_space cao_space;
typedef struct cao_runs cao_runs;

typedef enum {
    CAO_OK = 0,
    CAO_E_INVALID_ARG = -1,  /* null pointer, bad enum, malformed constraint program, ...        */
    CAO_E_STATE = -2,        /* call order violated (e.g. fill before count)                      */
    CAO_E_TOO_LARGE = -3,    /* n > 32, m_d > 256, N >= 2^40, V >= 2^32, pop > 1024               */
    CAO_E_EMPTY_SPACE = -4,  /* V == 0                                                            */
    CAO_E_POP_GT_VALID = -5, /* population larger than the number of valid configs               */
    CAO_E_WORKSPACE = -6,    /* misaligned / missing workspace                                    */
    CAO_E_CUDA = -7          /* a CUDA runtime call failed (message holds cudaGetErrorString)     */
} cao_status;

typedef enum { CAO_DE = 0, CAO_PSO = 1, CAO_FIREFLY = 2, CAO_GA = 3 } cao_algo;

/* Hyperparameters, defaults from Table IV (L368-393). */
typedef struct {
    float de_F, de_CR;               /* 0.7, 0.6 (best1bin)                          L372-375 */
    float pso_w, pso_c1, pso_c2;     /* 0.5, 3.0, 0.5                                L378-380 */
    float ff_B0, ff_gamma, ff_alpha; /* 1.0, 1.0, 0.2                                L383-385 */
    int32_t ga_mutation_chance;      /* 5 => mutate 1 child in 5                     L389, L393 */
    int32_t ga_beta_b;               /* 3: Beta(1,b) parent selection over the sorted rank (A18) */
} cao_hparams;

/* SURVEY 8(f) switches of a set of runs.  NULL / all-default = the north_star path (constraint-aware, unified repair
 * key, DE best1bin, GA single_point, uniform initial sample).  Any non-default field selects the phased pipeline.
 *   constraint_aware  1 (default); 0 = the paper's non-constraint-aware counterparts (L107, L272, L284): the initial
 *                     population is random in the Cartesian space, nothing is repaired, an invalid configuration is
 *                     not evaluated (no memo bit, no budget) and the strategy sees `penalty` instead       [NEXT-2, A33-A34]
 *   repair_mode       0 = argmin (Hamming, sum|didx|, L) for every algorithm (north_star; A4);
 *                     1 = the paper's own repairs: DE nearest by sum|didx| alone (L215, L270); PSO / Firefly Alg.2
 *                     (L225-247): first non-empty of the strictly-adjacent / adjacent / Hamming neighbour sets
 *                     (L139-143; A28), member nearest to the particle's continuous position (squared Euclidean distance,
 *                     fp32; A30); GA Alg.3 (L298-309): a random member of that set (draw stream 5, slot 0).  Ties: smallest
 *                     L (A5).  All three sets empty: the configuration stays invalid and is penalised     [NEXT-1]
 *   de_mutation       0 best1 (default), 1 rand1, 2 currenttobest1, 3 randtobest1, 4 best2, 5 rand2 (L219, L272; A29)
 *   de_crossover      0 binomial (default), 1 exponential (L272)
 *   ga_crossover      0 single_point (default), 1 two_point, 2 uniform, 3 disruptive_uniform (L288; A31)
 *   init_lhs          1 = DE's initial population by Latin Hypercube Sampling, repaired to valid (L223; A35)   [NEXT-3]
 *                     The LHS points are always repaired with the unified key (Hamming, sum|didx|, L), also when
 *                     repair_mode = 1 selects the paper's own repairs for the generations that follow.
 *   penalty           objective reported for an unevaluated invalid configuration, > 0 and finite (L107: 1e20)          */
typedef struct {
    int32_t constraint_aware, repair_mode, de_mutation, de_crossover, ga_crossover, init_lhs;
    float penalty;
    int32_t reserved;
} cao_variant;

/* Constraint programs: postfix (RPN) over int64, one int32 word per token (O1, A2, A3).
 * PUSH_PARAM is followed by the parameter number, PUSH_CONST by the low and the high 32 bits.
 * DIV/MOD truncate toward zero; a zero divisor makes the whole constraint false; ADD/SUB/MUL/NEG
 * saturate to +-2^62.  A constraint holds iff its result is non-zero. */
enum {
    CAO_OP_PUSH_PARAM = 1, CAO_OP_PUSH_CONST = 2,
    CAO_OP_ADD = 3, CAO_OP_SUB = 4, CAO_OP_MUL = 5, CAO_OP_DIV = 6, CAO_OP_MOD = 7, CAO_OP_NEG = 8,
    CAO_OP_MIN = 9, CAO_OP_MAX = 10,
    CAO_OP_LT = 11, CAO_OP_LE = 12, CAO_OP_GT = 13, CAO_OP_GE = 14, CAO_OP_EQ = 15, CAO_OP_NE = 16,
    CAO_OP_AND = 17, CAO_OP_OR = 18, CAO_OP_NOT = 19
};

/* ---------------------------------------------------------------- define P = (X, D, C), L129-135 */
/* An empty problem P = (X, D, C) (L129).  The handle is a host object owned by the library. */
int cao_space_create(cao_space** out);
void cao_space_destroy(cao_space* s);
/* L131-132: appends a variable x_i with its finite domain D_i: n_values (1..256) int64 values (copied).  Call order =
 * digit order (A1).  Errors: CAO_E_STATE after the build, CAO_E_TOO_LARGE beyond 32 parameters / 256 values. */
int cao_space_add_param(cao_space* s, const char* name, const int64_t* h_values, int32_t n_values);
/* L133: appends a constraint c_j, a predicate over a subset of the variables, as a postfix program (copied, validated:
 * known opcodes, stack depth 1 at the end, <= 32).  Errors: CAO_E_INVALID_ARG for a malformed program. */
int cao_space_add_constraint(cao_space* s, const int32_t* h_rpn, int32_t n_words);

/* ---------------------------------------------------------------- build the space (S1; L137)
 * build_mode: 0 = word-parallel (constraints with a small scope become bit tables, the bitmap is
 * the AND of table words), 1 = plain (every constraint is interpreted for every config).  Both
 * give identical results.  Set before build_workspace_bytes. */
int cao_space_set_build_mode(cao_space* s, int32_t mode);
int cao_space_build_workspace_bytes(cao_space* s, uint64_t* bitmap_bytes, uint64_t* scratch_bytes);
/* L143 ("Hamming: all parameters identical except one"), L215: highest Hamming level the generation step probes in the bitmap before it falls back to the table scan:
 * -1 (default) = cost model (level h is probed while (number of rows at distance h) * 60 <= V * scan cost),
 * 0..6 = fixed (clamped to 1 when the space has more than 368 Hamming-1 neighbours or 65536 neighbour pairs).  Call before build_count; probe_levels() reports the level in use after build_count. */
int cao_space_set_probe_levels(cao_space* s, int32_t levels);
int cao_space_probe_levels(const cao_space* s, int32_t* levels);
/* L137 ("determines all configurations in the search space before starting the tuning process"), O1.
 * Pass 1: validity bitmap + per-512-config counts, then the exclusive scan of the counts.
 * Synchronises `stream` once to return V in *h_V.  d_scratch may be released after build_fill. */
int cao_space_build_count(cao_space* s, void* d_bitmap, void* d_scratch, void* stream, uint64_t* h_V);
/* Bytes of d_table for build_fill (needs V, i.e. a completed build_count): rows + Ltab + rank directory + probe lists. */
int cao_space_table_bytes(const cao_space* s, uint64_t* bytes);
/* Pass 2: valid rows (V x row_bytes), Ltab (V linear indices: u32 when N <= 2^32, else u64 -- see
 * cao_space_ltab_bytes) and the rank directory, into d_table. */
int cao_space_build_fill(cao_space* s, void* d_table, void* stream);
/* Re-runs the whole of S1 (tables, bitmap, counts, scan, rows, Ltab, directory) into the buffers of the last
 * build, asynchronously and without any host round trip: the definition is unchanged, so V and the layout are
 * the ones build_count returned.  Needs a completed build_count + build_fill; d_scratch must still be alive. */
int cao_space_rebuild(cao_space* s, void* stream);
/* Table III's columns (L334-341): Cartesian size N, number of valid configurations V, dimensions n; row_bytes = 16 or 32. */
int cao_space_sizes(const cao_space* s, uint64_t* N, uint64_t* V, int32_t* n, int32_t* row_bytes);
/* Statistics of the last build / rebuild (synchronises `stream`; d_scratch must still be alive): h_out4 = {blocks of
 * B consecutive configs the index range is cut into, blocks that survived the tabled constraints and went on to the
 * residual ones (0 when there is no residual constraint), non-empty 512-config groups, B}. */
int cao_space_build_stats(const cao_space* s, void* stream, uint64_t* h_out4);
/* Bytes per Ltab entry: 4 when N <= 2^32 (every linear index fits 32 bits), else 8. */
int cao_space_ltab_bytes(const cao_space* s, int32_t* bytes);
/* Borrowed device views into the caller's buffers; rank_dir[i] = number of valid L < 512*i. */
int cao_space_views(const cao_space* s, const uint64_t** d_bitmap, const uint8_t** d_rows,
                    const void** d_Ltab, const uint32_t** d_rank_dir);

/* ---------------------------------------------------------------- Search Space queries (L139), batched
 * L139: "functionality to query whether a particular solution is valid": d_out[i] = 1 iff row i is a valid configuration
 * (0 for a row with an index outside its domain).  d_idx_rows: count rows of row_bytes bytes each (padding ignored). */
int cao_space_is_valid(const cao_space* s, const uint8_t* d_idx_rows, uint64_t count, uint8_t* d_out,
                       void* stream);
/* S5 standalone: d_rank_out[i] = rank of argmin (Hamming, sum |didx|, L) over the valid table; the
 * identity for valid rows (L143, L215, L270; O9).  d_key_out (optional, may be NULL) receives
 * ham << 45 | sad << 32 | rank.  probe_levels: 0 = table scan only; 1..6 = first test the neighbours
 * at Hamming distance <= that level in the bitmap (exact: Hamming is the primary key); any other value
 * (e.g. -1) = the level the library's cost model chose for this space.  All settings give identical
 * results.  Rows with an index outside its domain are legal inputs (A27: they are invalid, skip the probes and are
 * repaired by the scan over their byte values); padding bytes (positions >= n) are ignored.
 * d_scratch: cao_space_repair_scratch_bytes(count) bytes. */
int cao_space_repair_scratch_bytes(const cao_space* s, uint64_t count, uint64_t* bytes);
int cao_space_repair(const cao_space* s, const uint8_t* d_idx_rows, uint64_t count, uint32_t* d_rank_out,
                     uint64_t* d_key_out, int32_t probe_levels, void* d_scratch, void* stream);
/* cao_space_repair without a scratch argument, for callers that have no way to obtain device scratch at the moment of
 * the call.  Everywhere else in this header the caller brings the scratch, which in practice means a cudaMalloc or a
 * framework allocator somewhere up the call chain.  Some callers cannot do that: code that runs inside a memory pool's or
 * an allocator's own callback (allocating there would re-enter it), a plugin whose host hands it input and output buffers
 * and a stream but forbids allocation, a process whose whole device-memory budget was reserved up front by another
 * component, or a latency-bound loop in which a cudaMalloc (it can synchronise the whole device) is not acceptable.
 * For them the library carries its own scratch: one array inside its device image, CAO_REPAIR_NOALLOC_MAX_ROWS rows
 * large (3 MiB + 256 bytes).  Every GPU on which the library's kernels get loaded holds that array until the process
 * exits, whether or not this function is ever called.
 *   - Same inputs, outputs, probe_levels meaning and results as cao_space_repair (S5: L143, L215, L270; O9); the caller
 *     still owns d_idx_rows (16-byte aligned), d_rank_out and d_key_out (either may be NULL, not both).
 *   - count > CAO_REPAIR_NOALLOC_MAX_ROWS returns CAO_E_TOO_LARGE and launches nothing: split the batch, or use
 *     cao_space_repair.  count == 0 is a no-op.
 *   - The function calls no cudaMalloc, cudaFree or other allocating routine.  That includes the optional per-kernel
 *     timing, which creates CUDA events: while cao_profile_enable(1) is in force the call returns CAO_E_STATE.
 *   - The first call on each device looks up the array's address on that device (cudaGetSymbolAddress, with the device
 *     that holds the space's buffers current, as for every launching call) and remembers it.  Make that first call
 *     before any stream capture is begun on that device; later calls only enqueue an 8-byte memset and the kernels.
 *   - There is ONE array per device and every call uses it.  It still holds the previous call's data when the next one
 *     starts; the function clears the part that must start at zero (the worklist counters) and overwrites the rest
 *     before reading it, so back-to-back calls on one stream are independent.  Two calls whose kernels can overlap on
 *     the GPU -- different streams without an event between them, or several host threads -- race on the array and give
 *     wrong ranks: order them on one stream or with events.  That holds across cao_space handles too: the array belongs
 *     to the library, not to a space. */
#define CAO_REPAIR_NOALLOC_MAX_ROWS 65536
int cao_space_repair_noalloc(const cao_space* s, const uint8_t* d_idx_rows, uint64_t count, uint32_t* d_rank_out,
                             uint64_t* d_key_out, int32_t probe_levels, void* stream);
/* NEXT-1 standalone (L139-143, L215, L270, Alg.2, Alg.3): the paper's own repairs for `count` rows.
 * mode 1 = index distance: d_rank_out[i] = argmin (sum |didx|, L);  2 = Alg.2 with d_x: count x n fp32 continuous
 * positions (row-major);  3 = Alg.3 with d_w: count 32-bit draws (member number floor(w K / 2^32) of the first non-empty
 * neighbour set, ascending L).  Valid rows map to themselves.  d_rank_out[i] = 0xFFFFFFFF when every neighbour set is
 * empty; d_rule_out (optional) receives the set used (0/1/2, 3 = none, 255 = valid row or mode 1).  Rows must be
 * in-domain.  d_scratch: cao_space_repair_mode_scratch_bytes(count) bytes, 256-byte aligned. */
int cao_space_repair_mode_scratch_bytes(const cao_space* s, uint64_t count, uint64_t* bytes);
int cao_space_repair_mode(const cao_space* s, int32_t mode, const uint8_t* d_idx_rows, const float* d_x, const uint32_t* d_w,
                          uint64_t count, uint32_t* d_rank_out, uint8_t* d_rule_out, void* d_scratch, void* stream);
/* Objective table by rank: V floats, > 0 and finite (borrowed).  L357: the evaluation replays pre-measured values
 * (methodology of [29]); L268: evaluated configurations are memoised, so the evaluation is a lookup. */
int cao_space_set_objective(cao_space* s, const float* d_obj);

/* ---------------------------------------------------------------- runs (S2-S7)
 * n_runs independent simulated tuning runs of `algo`; run k uses RNG run index first_run + k, so
 * any partition of the run indices gives the same per-run results. */
int cao_runs_workspace_bytes(const cao_space* s, int32_t algo, int32_t pop, uint32_t n_runs,
                             uint32_t max_gens, uint64_t* bytes);
/* L139 / L282(i) ("generate a number of random samples of only valid solutions"), L125 (budget):
 * creates the runs and executes generation 0 (S2; O4) on `stream`.  budget_unique: unique
 * evaluations per run, 0 = unlimited (L125, A20).  max_gens: generation cap = trajectory rows - 1. */
int cao_runs_create(const cao_space* s, int32_t algo, const cao_hparams* hp, uint32_t n_runs,
                    uint32_t first_run, int32_t pop, uint32_t budget_unique, uint32_t max_gens,
                    uint64_t seed, void* d_workspace, void* stream, cao_runs** out);
/* The same with the SURVEY 8(f) switches (var == NULL: defaults = cao_runs_create).  The workspace of a non-default
 * variant is larger: size it with cao_runs_workspace_bytes_ex.  Errors: CAO_E_INVALID_ARG for an unknown switch value,
 * init_lhs with an algorithm other than DE or with constraint_aware = 0, a DE population smaller than donors + 1. */
int cao_runs_workspace_bytes_ex(const cao_space* s, int32_t algo, const cao_variant* var, int32_t pop, uint32_t n_runs,
                                uint32_t max_gens, uint64_t* bytes);
int cao_runs_create_ex(const cao_space* s, int32_t algo, const cao_hparams* hp, const cao_variant* var, uint32_t n_runs,
                       uint32_t first_run, int32_t pop, uint32_t budget_unique, uint32_t max_gens, uint64_t seed,
                       void* d_workspace, void* stream, cao_runs** out);
void cao_runs_destroy(cao_runs* r);
/* How cao_runs_step executes: 1 = one fused persistent kernel (a warp group per run, population state in shared
 * memory for all the requested generations); 0 = phased, per generation k_op -> k_probe23 -> k_scan -> k_finish over
 * all runs (better when many candidates need the table scan).  Identical results.  The default is chosen at create:
 * fused unless the estimated share of invalid candidates that fall through the bitmap probes to the table scan,
 * exp(-V/N * rows within the probed Hamming levels), exceeds 1 % (configs[3]-like sparse spaces) or the population
 * does not fit the shared memory of one SM.  cao_runs_mode reports the mode in use. */
int cao_runs_mode(const cao_runs* r, int32_t* mode);
int cao_runs_set_mode(cao_runs* r, int32_t mode);
/* Fused mode only: threads per run as a multiple of the population rounded up to 32.  0 (default) = automatic: while the
 * runs of a launch fill only part of the GPU, a run gets more lanes (Firefly: four lanes per firefly; the others: twice the
 * threads for the cooperative neighbour probes and scans); 1, 2, 4 = fixed (4 = Firefly's four-lane operator, 16-byte
 * rows only; a width that does not apply falls back to 1).  Identical results at every width (O3: draws are addressed,
 * never consumed in order).  Call before the first fused cao_runs_step. */
int cao_runs_set_fused_width(cao_runs* r, int32_t width);
int cao_runs_fused_width(const cao_runs* r, int32_t* width);
/* One batched generation of every run, n_generations times: operator (Alg.1 L147-213 DE; L276-282 PSO; L284 Firefly;
 * L286-292 GA), snap (L280), validity (L139), repair (L215, L270, Alg.2-3), evaluation with memoisation (L268), selection
 * and budget test (L125, A20).  Stops recording at max_gens.  Asynchronous. */
int cao_runs_step(cao_runs* r, uint32_t n_generations, void* stream);
/* Eq.1 (L115): best configuration found so far per run (minimisation, O0), with its unique-evaluation count (L268) and the
 * generations executed.  Copies to DEVICE arrays of n_runs elements each (any may be NULL). */
int cao_runs_best(const cao_runs* r, float* d_best_f, uint32_t* d_best_rank, uint32_t* d_uniq,
                  uint32_t* d_gens_done, void* stream);
/* The "performance over time" of Fig. 3-4 (L395-403) in simulated mode, time = unique evaluations.
 * Borrowed: trajectory [gen][run] of packed {f32 best_f, u32 best_rank, u32 uniq}, gens 0..generation. */
int cao_runs_trajectory(const cao_runs* r, const void** d_traj, uint32_t* gens_recorded);
/* Parity taps of the last stepped generation, [run][ind]: post-snap pre-repair rows (row_bytes each),
 * validity flag, rank after repair, rank evaluated, f, accept flag, and [run] active flag. */
int cao_runs_debug_last(const cao_runs* r, const uint8_t** d_postsnap_rows, const uint8_t** d_valid,
                        const uint32_t** d_repaired_rank, const uint32_t** d_eval_rank, const float** d_f,
                        const uint8_t** d_accept, const uint8_t** d_active);
/* NEXT-1 tap of the last stepped generation, [run][ind]: neighbour rule that repaired the candidate (0 strictly-adjacent,
 * 1 adjacent, 2 Hamming), 3 = every set empty, 255 = not applicable (valid candidate, or another repair mode). */
int cao_runs_debug_rule(const cao_runs* r, const uint8_t** d_rule);
/* Raw population state, borrowed.  SURVEY 8(b) sketched one blob (`const void** d_state, uint64_t* bytes`); the arrays have
 * different element types and only some exist per algorithm, so this call takes a selector instead.  which: 0 idx rows [run][ind][row_bytes] u8, 1 rank [run][ind] u32,
 * 2 f [run][ind] f32, 3 x, 4 v, 5 pbest [run][dim][ind] f32 (dimension-major), 6 pbest_f [run][ind]. */
int cao_runs_debug_state(const cao_runs* r, int32_t which, const void** d_ptr, uint64_t* bytes);
/* Counters since create (synchronises `stream`): candidates whose post-snap row was invalid,
 * candidates that needed the table scan, candidates evaluated. */
int cao_runs_counters(const cao_runs* r, void* stream, uint64_t* n_repaired, uint64_t* n_scanned,
                      uint64_t* n_evaluated);
/* All thirty-two 64-bit statistics words since create (synchronises `stream`): 0 n_repaired, 1 n_scanned (candidates
 * that needed the table scan), 2 n_evaluated; fused mode only: 3 candidates that went to the Hamming-2 probe, 4 ...
 * beyond it, 5 invalid candidates resolved by the previous generation's memo, 6 ... by the per-run repair cache
 * (L268: memoisation); 7 n_penalised: candidates that stayed invalid and received the static penalty instead of an
 * evaluation (NEXT-1 / NEXT-2 variants only, L107; they are included in word 2); 8-13 clock cycles of thread 0 of every group in operator / tail / probe-2 /
 * deeper probes / scan / finish, 14-15 slowest run and most scan cycles in one run (only in builds with
 * -DCAO_GEN_STATS, else 0); 16-24 candidates of the stepped generations by Hamming distance of their repair
 * (16 = valid, 17 = Hamming 1, ..., 24 = eight or more; L143, L215); 25-31 reserved. */
int cao_runs_stats(const cao_runs* r, void* stream, uint64_t* h_out32);
/* NEXT-4 (Eq.2; A36): performance score of a set of runs against the calculated random-search baseline
 * B(t) = expected minimum of t draws without replacement from the V objective values (fp64).
 *   cao_space_sort_objective: d_sorted = the objective table in ascending order (V floats; d_scratch: the next power of
 *                             two >= V floats).  CAO_E_TOO_LARGE when V > 2^31.
 *   cao_space_baseline:       d_B[q] = B(d_t[q]) for S sampling points (unique-evaluation counts, clamped to 1..V).
 *   cao_runs_score:           d_per_t[q] = mean over the runs of (B - best_r(t)) / (B - f_opt), best_r(t) = best-so-far at
 *                             the last recorded generation whose unique-evaluation count is <= t (generation 0 if none;
 *                             the worst objective if nothing valid was evaluated); where B(t) = f_opt (t >= V, or a constant
 *                             table) the term is 1 for a run that holds the optimum, else 0; d_score[0] = their mean over q.
 *                             d_scratch: S * n_runs doubles.  Bit-identical to the oracle (same fp64 operation order). */
int cao_space_sort_objective(const cao_space* s, float* d_sorted, void* d_scratch, void* stream);
int cao_space_baseline(const cao_space* s, const float* d_sorted, const uint64_t* d_t, uint32_t S, double* d_B, void* stream);
int cao_runs_score(const cao_runs* r, const float* d_sorted, const uint64_t* d_t, const double* d_B, uint32_t S,
                   double* d_per_t, double* d_score, void* d_scratch, void* stream);
/* Kernels launched by this library in this process so far (bench.py's gpu_launches). */
uint64_t cao_launch_count(void);

/* Optional device timing per kernel class (bench.py's roofline): while enabled, every launch is bracketed by
 * CUDA events on its stream.  enable(1) clears the totals.  read() synchronises the recorded events and
 * returns the summed milliseconds and the launch count of class `cls`: 0 k_build_tables + k_inner_lut, 1 k_enum,
 * 2 count scan, 3 k_fill, 4 k_init, 5 k_op, 6 k_scan, 7 k_finish, 8 queries, 9 k_probe23, 10 k_gen, 11 k_residual,
 * 12 k_keys + k_masks, 13 k_res_prefix + k_res_class_table; name() gives the kernel names ("" beyond the last class). */
int cao_profile_enable(int32_t on);
int cao_profile_read(int32_t cls, double* h_ms_total, uint64_t* h_launches);
const char* cao_profile_name(int32_t cls);

/* Device self-tests for the parity of the arithmetic primitives (O3, O5-O7): out[i] from in[i]. */
int cao_test_philox(const uint32_t* d_ctr_key /* count x 6 */, uint32_t* d_out /* count x 4 */,
                    uint64_t count, void* stream);
/* The same inputs through cuRAND's device function curand_Philox4x32_10: a second, independent pin of the generator. */
int cao_test_curand_philox(const uint32_t* d_ctr_key /* count x 6 */, uint32_t* d_out /* count x 4 */,
                           uint64_t count, void* stream);
int cao_test_exp_neg(const float* d_z, float* d_out, uint64_t count, void* stream);
/* Integer-issue microbenchmark (the denominator of bench.py's "alu" roofline for the repair scan):
 * n_ctas x 256 threads, each runs `iters` x 8 independent chains of one instruction kind: 0 IMAD (mad.lo.u32),
 * 1 LOP3, 2 VABSDIFF4 (with accumulate), 3 POPC, 4 IADD, 5 IDP.4A (dp4a with accumulate).  d_out: n_ctas * 256 words.  The caller times it. */
int cao_test_int_peak(int32_t kind, uint32_t iters, uint32_t n_ctas, uint32_t* d_out, void* stream);

const char* cao_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* CAO_H_ */

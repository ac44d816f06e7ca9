// cao_runs_kernels.cuh -- S2-S4, S6, S7: batched generation step over many independent runs
// (Alg.1, Alg.3; O4-O8, O10 in DESIGN.md).
//
// One CTA per run, one thread per individual.  A generation is three launches:
//   k_op     operator (DE / PSO / Firefly / GA) -> snap -> linear index -> bitmap test -> Hamming-1 probe;
//            candidates that still have no rank go to the scan worklist
//   k_scan   (cao_repair_kernels.cuh) brute-force nearest-valid for the worklist
//   k_finish rank -> objective -> per-run dedup bitmap -> selection / state update -> best-so-far -> trajectory
// Every random number is addressed by (seed, run, generation, individual, stream, slot) (O3).
#pragma once
#include "cao_host.h"
#include "cao_repair_kernels.cuh"

#define CAO_RCACHE 256                                  // direct-mapped entries per run
__device__ __forceinline__ uint32_t rcache_slot(uint64_t L) { return (uint32_t)((L * 0x9E3779B97F4A7C15ull) >> 56); }

struct RunsMeta {
    uint32_t R, first_run, P, budget, max_gens, dedup_words;
    int32_t algo, probe_levels;
    uint64_t seed;
    cao_hparams hp;
    // taps of the last generation, [run][ind]
    uint8_t* cand; unsigned long long* key; uint8_t* valid; uint32_t* rep_rank; uint32_t* eval_rank; float* tap_f;
    uint8_t* accept; uint8_t* active;
    // population state
    uint8_t* idx; uint32_t* rank; float* f; float* x; float* v; float* pb; float* pbf;
    uint32_t* dedup;                                   // [run][dedup_words]
    uint32_t* uniq; uint32_t* gens_done; uint32_t* stagn; uint32_t* best_rank; float* best_f;
    uint32_t* traj;                                    // [gen][run]{f32 bits, rank, uniq}
    uint32_t* wl; uint32_t* wl_count;                  // candidates without a valid Hamming-1 neighbour
    uint32_t* wl2; uint32_t* wl2_count;                // ... and none up to the probed level: table scan
    ulonglong2* rcache;                                // [run][CAO_RCACHE] {L, key}: repairs at Hamming >= 2 already resolved (fused mode)
    uint32_t* ticket;                                  // [2] run ticket + finished-group counter of the fused kernel (self re-arming)
    unsigned long long* counters;                      // n_repaired, n_scanned, n_evaluated
    // SURVEY 8(f) variants (include/cao.h cao_variant); var_on = any non-default switch (phased pipeline only)
    cao_variant var;
    int32_t var_on;
    uint8_t* rule;                                     // NEXT-1 tap [run][ind]: neighbour rule used (0/1/2), 3 none, 255 n/a
    unsigned long long* key3;                          // Alg.2: [slot][3] per-rule minimum of (dist^2 bits << 32 | rank)
    uint32_t* cnt3;                                    // Alg.3: [slot][3] members per rule
    const uint8_t* present;                            // [dim][256]: the value index occurs in some valid configuration (A28)
};
#define CAO_RANK_NONE 0xFFFFFFFFu
__device__ __forceinline__ int de_donor_count(int mut) { return mut == 0 || mut == 2 ? 2 : mut == 1 || mut == 3 ? 3 : mut == 4 ? 4 : 5; }

// Shared scratch of the per-run CTAs.
struct RunShared {
    unsigned long long best;                           // (f bits << 32 | rank) of the best-so-far
    unsigned long long aux;                            // PSO: (pbest_f bits << 32 | i) of gbest
    uint32_t n_new, flag, n_inv;
};

// ---------------------------------------------------------------------------------------------
// O10: evaluate rank rk for run k: objective lookup, memoisation bit, best-so-far (block-level, order-free).
__device__ __forceinline__ float evaluate(const SpaceMeta& sm, const RunsMeta& rm, uint32_t k, uint32_t rk, RunShared* sh) {
    if (rk == CAO_RANK_NONE) {                          // NEXT-1 / NEXT-2 (A33): the configuration stayed invalid -> static penalty,
        atomicAdd(&rm.counters[7], 1ull);               // nothing memoised or counted (L107, L135, L284)
        return rm.var.penalty;
    }
    float f = __ldg(&sm.obj[rk]);
    uint32_t bit = 1u << (rk & 31);
    uint32_t old = atomicOr(&rm.dedup[(uint64_t)k * rm.dedup_words + (rk >> 5)], bit);
    if (!(old & bit)) atomicAdd(&sh->n_new, 1u);
    atomicMin(&sh->best, ((unsigned long long)fbits(f) << 32) | rk);
    return f;
}
__device__ __forceinline__ void eval_begin(const RunsMeta& rm, uint32_t k, RunShared* sh) {     // thread 0, before a sync
    uint32_t br = rm.best_rank[k];
    // nothing valid evaluated yet: no key at all, so that the FIRST valid evaluation is recorded whatever its value -- also an
    // objective at or above the penalty (the contract is only "> 0 and finite"); eval_end reports (penalty, no rank) meanwhile (A33)
    sh->best = br == 0xFFFFFFFFu ? ~0ull : (((unsigned long long)fbits(rm.best_f[k]) << 32) | br);
    sh->n_new = 0; sh->flag = 0; sh->aux = ~0ull;
}
__device__ __forceinline__ void eval_end(const RunsMeta& rm, uint32_t k, uint32_t g, RunShared* sh) {   // thread 0, after a sync
    uint32_t u = rm.uniq[k] + sh->n_new;
    rm.uniq[k] = u;
    const unsigned long long best = sh->best == ~0ull ? (((unsigned long long)fbits(rm.var.penalty) << 32) | 0xFFFFFFFFu) : sh->best;
    rm.best_f[k] = __uint_as_float((uint32_t)(best >> 32));
    rm.best_rank[k] = (uint32_t)best;
    uint32_t* t = rm.traj + ((uint64_t)g * rm.R + k) * 3;
    t[0] = (uint32_t)(best >> 32); t[1] = (uint32_t)best; t[2] = u;
}

// O4: P distinct valid ranks, uniform with linear probing; fills the population and evaluates it.
// Block-uniform call; s_r holds P words.  Ends with a __syncthreads().
template <int ALGO, int ROWW>
__device__ void init_population(const SpaceMeta& sm, const RunsMeta& rm, uint32_t k, uint32_t g, uint32_t stream,
                                uint32_t* s_r, RunShared* sh) {
    const uint32_t i = threadIdx.x, P = rm.P, run = rm.first_run + k;
    Draws dr(rm.seed, run, g, i, stream);
    // A35: with init_lhs the rank of individual i is the repaired LHS point (k_lhs_points + the repair pipeline left it in
    // rm.key); the stagnation re-init stays uniform (L266 "reinitialized randomly")
    const bool lhs = rm.var.init_lhs && stream == S_INIT;
    if (i < P) s_r[i] = lhs ? (uint32_t)rm.key[(uint64_t)k * P + i] : below(dr(0), sm.V);
    __syncthreads();
    bool dup = false;
    if (i < P) { uint32_t me = s_r[i]; for (uint32_t j = 0; j < i; ++j) dup |= (s_r[j] == me); }
    if (__syncthreads_or(dup)) {
        if (i == 0) {                                   // the sequential definition, rare
            for (uint32_t a = 0; a < P; ++a) {
                uint32_t r = s_r[a];
                for (;;) {
                    bool taken = false;
                    for (uint32_t j = 0; j < a; ++j) if (s_r[j] == r) { taken = true; break; }
                    if (!taken) break;
                    r = r + 1 == sm.V ? 0 : r + 1;
                }
                s_r[a] = r;
            }
        }
        __syncthreads();
    }
    if (i < P) {
        const uint32_t rk = s_r[i];
        const uint64_t q = (uint64_t)k * P + i;
        uint32_t w[ROWW];
        load_row<ROWW>(sm.rows + (uint64_t)rk * (ROWW * 4), w);
        float f = evaluate(sm, rm, k, rk, sh);
        rm.rank[q] = rk; rm.f[q] = f;
        if (ALGO == CAO_DE || ALGO == CAO_GA) {
            store_row<ROWW>(rm.idx + q * (ROWW * 4), w);
        } else {
#pragma unroll
            for (int d = 0; d < ROWW * 4; ++d) {
                if (d < sm.n) {
                    const uint64_t e = ((uint64_t)k * sm.n + d) * P + i;
                    float xd = coord_M(sm.M, (int)((w[d >> 2] >> ((d & 3) * 8)) & 0xFFu));
                    rm.x[e] = xd;
                    if (ALGO == CAO_PSO) {
                        float hi = coord_M(sm.M, (int)sm.m[d] - 1);
                        float c = __fsub_rn(u01(dr(1 + d)), 0.5f);
                        rm.v[e] = __fmul_rn(c, hi);
                        rm.pb[e] = xd;
                    }
                }
            }
            if (ALGO == CAO_PSO) rm.pbf[q] = f;
        }
    }
    __syncthreads();
}

// NEXT-2 (L272, L284; A34): the non-constraint-aware initial population is random in the Cartesian space and is not
// repaired: DE / GA idx_d = below(draw(slot 1+n+d), m_d); PSO / Firefly x_d = u01(draw(slot 1+n+d)) * hi_d (PSO velocity as
// in O4).  Invalid members hold rank CAO_RANK_NONE and the penalty.  Block-uniform call, ends with a __syncthreads().
template <int ALGO, int ROWW>
__device__ void init_population_unaware(const SpaceMeta& sm, const RunsMeta& rm, uint32_t k, uint32_t g, uint32_t stream, RunShared* sh) {
    const uint32_t i = threadIdx.x, P = rm.P, run = rm.first_run + k;
    const int n = sm.n;
    if (i < P) {
        Draws dr(rm.seed, run, g, i, stream);
        const uint64_t q = (uint64_t)k * P + i;
        uint32_t w[ROWW];
#pragma unroll
        for (int z = 0; z < ROWW; ++z) w[z] = 0;
        float vel[ROWW * 4];
        if (ALGO == CAO_PSO) {                                          // slots ascend: velocities (1+d) first, then positions
#pragma unroll
            for (int d = 0; d < ROWW * 4; ++d) if (d < n) vel[d] = __fmul_rn(__fsub_rn(u01(dr(1 + d)), 0.5f), coord_M(sm.M, (int)sm.m[d] - 1));
        }
#pragma unroll
        for (int d = 0; d < ROWW * 4; ++d) {
            if (d < n) {
                const uint32_t wd = dr(1 + n + d);
                uint32_t kd;
                if (ALGO == CAO_DE || ALGO == CAO_GA) kd = below(wd, (uint32_t)sm.m[d]);
                else {
                    const float hi = coord_M(sm.M, (int)sm.m[d] - 1);
                    const float xd = __fmul_rn(u01(wd), hi);
                    const uint64_t e = ((uint64_t)k * n + d) * P + i;
                    rm.x[e] = xd;
                    kd = (uint32_t)snap_M(sm.M, (int)sm.m[d], xd);
                    if (ALGO == CAO_PSO) { rm.v[e] = vel[d]; rm.pb[e] = xd; }
                }
                w[d >> 2] |= kd << ((d & 3) * 8);
            }
        }
        const uint64_t L = row_lin<ROWW>(sm, w);
        const uint32_t rk = bit_test(sm.bitmap, L) ? rank_of(sm, L) : CAO_RANK_NONE;
        const float f = evaluate(sm, rm, k, rk, sh);
        rm.rank[q] = rk; rm.f[q] = f;
        if (ALGO == CAO_DE || ALGO == CAO_GA) store_row<ROWW>(rm.idx + q * (ROWW * 4), w);
        if (ALGO == CAO_PSO) rm.pbf[q] = f;
    }
    __syncthreads();
}

// NEXT-3 (L223; A35): Latin Hypercube points of generation 0, one CTA per run, thread = individual: per dimension the
// stratum of individual i is the rank of its draw(slot 1+d) among the P draws (ties by individual), the point inside the
// stratum u01(draw(slot 1+n+d)).  The rows go to the candidate taps and through the ordinary repair pipeline (unified key).
template <int ROWW> __device__ __forceinline__ void candidate_tail(const SpaceMeta&, const RunsMeta&, uint64_t, const uint32_t (&)[ROWW],
                                                                   uint32_t*, uint32_t*, bool, RunShared&, bool, bool = false);
template <int ROWW>
__global__ void __launch_bounds__(1024) k_lhs_points(const __grid_constant__ SpaceMeta sm, const __grid_constant__ RunsMeta rm) {
    extern __shared__ uint32_t s_dyn[];                                 // P draws of the current dimension
    __shared__ RunShared sh;
    const uint32_t k = blockIdx.x, i = threadIdx.x, P = rm.P, run = rm.first_run + k;
    const int n = sm.n;
    uint32_t w[ROWW];
#pragma unroll
    for (int z = 0; z < ROWW; ++z) w[z] = 0;
    if (i == 0) sh.n_inv = 0;
    uint32_t strat[ROWW * 4];
    Draws dr(rm.seed, run, 0, i, S_INIT);
    for (int d = 0; d < n; ++d) {
        const uint32_t mine = i < P ? dr(1 + d) : 0;
        __syncthreads();
        if (i < P) s_dyn[i] = mine;
        __syncthreads();
        uint32_t perm = 0;
        if (i < P) for (uint32_t j = 0; j < P; ++j) { const uint32_t o = s_dyn[j]; perm += (o < mine) || (o == mine && j < i); }
        strat[d] = perm;
    }
    if (i < P) {
        for (int d = 0; d < n; ++d) {
            float t = __fadd_rn((float)strat[d], u01(dr(1 + n + d)));
            t = __fmul_rn(t, (float)sm.m[d]);
            t = __fdiv_rn(t, (float)P);
            int kd = (int)floorf(t);
            kd = min(kd, (int)sm.m[d] - 1);
            w[d >> 2] |= (uint32_t)kd << ((d & 3) * 8);
        }
    }
    __syncthreads();
    if (i < P) candidate_tail<ROWW>(sm, rm, (uint64_t)k * P + i, w, rm.wl, rm.wl_count, rm.probe_levels < 2, sh, false, true);
}

// Generation 0 (S2).
template <int ALGO, int ROWW>
__global__ void __launch_bounds__(1024) k_init(const __grid_constant__ SpaceMeta sm, const __grid_constant__ RunsMeta rm) {
    extern __shared__ uint32_t s_dyn[];
    __shared__ RunShared sh;
    const uint32_t k = blockIdx.x;
    if (threadIdx.x == 0) eval_begin(rm, k, &sh);
    __syncthreads();
    if (rm.var.constraint_aware) init_population<ALGO, ROWW>(sm, rm, k, 0, S_INIT, s_dyn, &sh);
    else init_population_unaware<ALGO, ROWW>(sm, rm, k, 0, S_INIT, &sh);
    if (threadIdx.x == 0) {
        eval_end(rm, k, 0, &sh);
        atomicAdd(&rm.counters[2], (unsigned long long)rm.P);
        if (rm.var.init_lhs && k == 0) { *rm.wl_count = 0; *rm.wl2_count = 0; }      // the LHS repair pass is done
    }
}

// ---------------------------------------------------------------------------------------------
// S4 + first half of S5 for the candidate held in w: store, validity, probe, worklist.
template <int ROWW>
__device__ __forceinline__ void candidate_tail(const SpaceMeta& sm, const RunsMeta& rm, uint64_t slot, const uint32_t (&w)[ROWW],
                                               uint32_t* wl, uint32_t* wl_count, bool count_scans, RunShared& sh, bool use_cache,
                                               bool unified) {
    if (!unified && (!rm.var.constraint_aware || rm.var.repair_mode == 1)) {
        // NEXT-2: no repair at all.  NEXT-1: every invalid candidate goes to the paper's own repair (cao_var_kernels.cuh),
        // which is not a function of the row alone (Alg.2 reads the position, Alg.3 draws), so nothing is memoised.
        store_row<ROWW>(rm.cand + slot * (ROWW * 4), w);
        const uint64_t L = row_lin<ROWW>(sm, w);
        const bool valid = bit_test(sm.bitmap, L);
        rm.key[slot] = valid ? make_key(0, 0, rank_of(sm, L)) : CAO_KEY_NONE;
        rm.valid[slot] = valid ? 1 : 0;
        rm.rule[slot] = 255;
        if (!valid) {
            atomicAdd(&sh.n_inv, 1u);
            if (rm.var.constraint_aware) {
                if (rm.algo == CAO_PSO || rm.algo == CAO_FIREFLY) { rm.key3[slot * 3] = ~0ull; rm.key3[slot * 3 + 1] = ~0ull; rm.key3[slot * 3 + 2] = ~0ull; }
                if (rm.algo == CAO_GA) { rm.cnt3[slot * 3] = 0; rm.cnt3[slot * 3 + 1] = 0; rm.cnt3[slot * 3 + 2] = 0; }
                worklist_push(rm.wl2, rm.wl2_count, (uint32_t)slot);
                atomicAdd(&rm.counters[1], 1ull);
            }
        }
        return;
    }
    // Repair is a pure function of the row: if this individual produced the same post-snap row in the generation
    // before (a particle that stopped moving, a repeated trial), last generation's key is still in the taps.
    uint32_t prev[ROWW];
    load_row_rw<ROWW>(rm.cand + slot * (ROWW * 4), prev);
    const uint64_t prev_key = rm.key[slot];
    bool same = prev_key != CAO_KEY_NONE;
#pragma unroll
    for (int z = 0; z < ROWW; ++z) same = same && prev[z] == w[z];
    bool valid;
    uint64_t key;
    if (same) {
        key = prev_key; valid = (key >> 45) == 0;
    } else {
        store_row<ROWW>(rm.cand + slot * (ROWW * 4), w);
        key = validate_probe<ROWW>(sm, w, rm.probe_levels >= 1, valid);
        if (key == CAO_KEY_NONE && use_cache) {                         // memoised repair of this run (L268 in spirit): exact,
            const uint64_t L = row_lin<ROWW>(sm, w);                    // repair(c) depends on c only
            const ulonglong2 e = rm.rcache[(slot / rm.P) * CAO_RCACHE + rcache_slot(L)];
            if (e.x == L) key = e.y;
        }
        rm.key[slot] = key;
    }
    rm.valid[slot] = valid ? 1 : 0;
    if (!valid) atomicAdd(&sh.n_inv, 1u);                               // flushed once per run and generation
    if (key == CAO_KEY_NONE) {
        worklist_push(wl, wl_count, (uint32_t)slot);
        if (count_scans) atomicAdd(&rm.counters[1], 1ull);               // straight to the scan
    }
}

#define ROW_BYTE(w, d) (((w)[(d) >> 2] >> (((d) & 3) * 8)) & 0xFFu)

// S3 + S4 for an ACTIVE run k (block-uniform call, contains barriers).  Unresolved candidates go to (wl, wl_count).
template <int ALGO, int ROWW>
__device__ __forceinline__ void gen_op(const SpaceMeta& sm, const RunsMeta& rm, uint32_t k, uint32_t g, uint32_t* s_dyn,
                                       RunShared& sh, uint32_t* wl, uint32_t* wl_count, bool count_scans, bool use_cache) {
    const uint32_t i = threadIdx.x, P = rm.P, run = rm.first_run + k;
    const int n = sm.n;
    const uint64_t q = (uint64_t)k * P + i;
    uint64_t qt = q;                                                    // slot of the candidate this thread produces (Firefly remaps)
    uint32_t w[ROWW];
#pragma unroll
    for (int z = 0; z < ROWW; ++z) w[z] = 0;
    Draws dr(rm.seed, run, g, i, S_OP);
    if (i == 0) sh.n_inv = 0;
    __syncthreads();

    if (ALGO == CAO_DE) {                                               // O5: best1bin on indices; NEXT-3 operators (A29)
        if (i < P) {
            const int mut = rm.var.de_mutation, nd = de_donor_count(mut);
            // nd distinct donors from X \ {x_i}: donor z = below(draw(z), P-1-z) mapped past i and the earlier donors in
            // ascending order (nd = 2: exactly O5's a, b)
            uint32_t don[5], taken[6];
            taken[0] = i;
            for (int z = 0; z < nd; ++z) {
                uint32_t a = below(dr(z), P - 1 - z);
                for (int t = 0; t <= z; ++t) if (a >= taken[t]) a += 1;
                int pos = z + 1;                                        // keep `taken` ascending
                while (pos > 0 && taken[pos - 1] > a) { taken[pos] = taken[pos - 1]; --pos; }
                taken[pos] = a;
                don[z] = a;
            }
            const uint32_t jrand = below(dr(nd), (uint32_t)n);
            uint32_t wd[5][ROWW], wx[ROWW], wbest[ROWW];
#pragma unroll
            for (int z = 0; z < 5; ++z)
                if (z < nd) load_row_rw<ROWW>(rm.idx + ((uint64_t)k * P + don[z]) * (ROWW * 4), wd[z]);
            load_row_rw<ROWW>(rm.idx + q * (ROWW * 4), wx);
            const uint32_t br = rm.best_rank[k];
            // best-so-far at generation start (A6); while nothing valid has been evaluated (NEXT-2 only): individual 0 (A34)
            if (br == CAO_RANK_NONE) load_row_rw<ROWW>(rm.idx + (uint64_t)k * P * (ROWW * 4), wbest);
            else load_row<ROWW>(sm.rows + (uint64_t)br * (ROWW * 4), wbest);
            uint32_t wv[ROWW];
#pragma unroll
            for (int z = 0; z < ROWW; ++z) wv[z] = 0;
#pragma unroll
            for (int d = 0; d < ROWW * 4; ++d) {
                if (d < n) {
                    const int top = (int)sm.m[d] - 1, xi = (int)ROW_BYTE(wx, d), bs = (int)ROW_BYTE(wbest, d);
                    int r0 = (int)ROW_BYTE(wd[0], d), r1 = (int)ROW_BYTE(wd[1], d), r2 = 0, r3 = 0, r4 = 0;
                    if (nd > 2) r2 = (int)ROW_BYTE(wd[2], d);
                    if (nd > 3) r3 = (int)ROW_BYTE(wd[3], d);
                    if (nd > 4) r4 = (int)ROW_BYTE(wd[4], d);
                    int vd;
                    if (mut == 0) vd = de_mutate_index(rm.hp.de_F, bs, r0, r1, top);
                    else {
                        int base, p1, q1, p2 = 0, q2 = 0; bool two = true;
                        switch (mut) {
                            case 1: base = r0; p1 = r1; q1 = r2; two = false; break;
                            case 2: base = xi; p1 = bs; q1 = xi; p2 = r0; q2 = r1; break;
                            case 3: base = r0; p1 = bs; q1 = r0; p2 = r1; q2 = r2; break;
                            case 4: base = bs; p1 = r0; q1 = r1; p2 = r2; q2 = r3; break;
                            default: base = r0; p1 = r1; q1 = r2; p2 = r3; q2 = r4; break;
                        }
                        float mf = __fadd_rn((float)base, __fmul_rn(rm.hp.de_F, (float)(p1 - q1)));
                        if (two) mf = __fadd_rn(mf, __fmul_rn(rm.hp.de_F, (float)(p2 - q2)));
                        vd = __float2int_rn(mf);
                        vd = min(max(vd, 0), top);
                    }
                    wv[d >> 2] |= (uint32_t)vd << ((d & 3) * 8);
                }
            }
            if (rm.var.de_crossover == 0) {                             // Alg.1: binomial
#pragma unroll
                for (int d = 0; d < ROWW * 4; ++d) {
                    if (d < n) {
                        const float rr = u01(dr(nd + 1 + d));
                        const uint32_t ud = (rr < rm.hp.de_CR || (uint32_t)d == jrand) ? ROW_BYTE(wv, d) : ROW_BYTE(wx, d);
                        w[d >> 2] |= ud << ((d & 3) * 8);
                    }
                }
            } else {                                                    // exponential (L272): one cyclic run of genes from j_rand
                uint32_t takem = 0;                                     // bit d: gene d comes from the mutant
                int d = (int)jrand, c = 0;
                do { takem |= 1u << d; d = d + 1 == n ? 0 : d + 1; ++c; } while (c < n && u01(dr(nd + 1 + c)) < rm.hp.de_CR);
#pragma unroll
                for (int e = 0; e < ROWW * 4; ++e)
                    if (e < n) w[e >> 2] |= (((takem >> e) & 1u) ? ROW_BYTE(wv, e) : ROW_BYTE(wx, e)) << ((e & 3) * 8);
            }
        }
    } else if (ALGO == CAO_GA) {                                        // O8: sorted population, Beta(1,b) parents, crossover
        uint64_t* s_L = (uint64_t*)s_dyn;                               // P linear indices (members may be invalid rows: NEXT-1/2)
        uint32_t* s_f = (uint32_t*)(s_L + P);                           // P objective bit patterns
        uint32_t* s_order = s_f + P;                                    // P
        if (i < P) {
            uint32_t wm[ROWW];
            load_row_rw<ROWW>(rm.idx + q * (ROWW * 4), wm);
            s_L[i] = row_lin<ROWW>(sm, wm); s_f[i] = fbits(rm.f[q]);
        }
        __syncthreads();
        if (i < P) {                                                    // L288: sorted by cost; ties by (L, i)
            const uint64_t myL = s_L[i]; const uint32_t myf = s_f[i];
            uint32_t pos = 0;
            for (uint32_t j = 0; j < P; ++j) {
                const uint64_t oL = s_L[j]; const uint32_t of = s_f[j];
                pos += (of < myf) || (of == myf && (oL < myL || (oL == myL && j < i)));
            }
            s_order[pos] = i;
        }
        __syncthreads();
        if (i < P) {
            const uint32_t B = (uint32_t)rm.hp.ga_beta_b;
            uint32_t sa = P, sb = P;
            for (uint32_t z = 0; z < B; ++z) sa = min(sa, below(dr(z), P));
            for (uint32_t z = 0; z < B; ++z) sb = min(sb, below(dr(B + z), P));
            if (sb == sa) sb = sa + 1 == P ? 0 : sa + 1;
            uint32_t wa[ROWW], wb[ROWW];
            load_row_rw<ROWW>(rm.idx + ((uint64_t)k * P + s_order[sa]) * (ROWW * 4), wa);
            load_row_rw<ROWW>(rm.idx + ((uint64_t)k * P + s_order[sb]) * (ROWW * 4), wb);
            uint32_t fromb = 0;                                         // bit d: gene d comes from parent B
            const int xo = rm.var.ga_crossover;
            if (xo == 0) {                                              // single point (Table IV)
                const int cut = n > 1 ? 1 + (int)below(dr(2 * B), (uint32_t)(n - 1)) : 1;
                for (int d = cut; d < n; ++d) fromb |= 1u << d;
            } else if (xo == 1) {                                       // two point (L288; A31): B between the two cuts
                const uint32_t c1 = below(dr(2 * B), (uint32_t)n + 1), c2 = below(dr(2 * B + 1), (uint32_t)n + 1);
                const uint32_t lo = min(c1, c2), hi = max(c1, c2);
                for (uint32_t d = lo; d < hi; ++d) fromb |= 1u << d;
            } else if (xo == 2) {                                       // uniform (L288)
                for (int d = 0; d < n; ++d) if (below(dr(2 * B + d), 2u) != 0) fromb |= 1u << d;
            } else {                                                    // disruptive uniform (L288; A31): at least half of the
                uint32_t diff = 0;                                      // differing genes come from B
#pragma unroll
                for (int d = 0; d < ROWW * 4; ++d) if (d < n && ROW_BYTE(wa, d) != ROW_BYTE(wb, d)) diff |= 1u << d;
                const int D = __popc(diff);
                int need = (D + 1) / 2, rem = D;
                for (int d = 0; d < n; ++d) {
                    if (!((diff >> d) & 1u)) continue;
                    const bool coin = below(dr(2 * B + d), 2u) == 1;
                    if (coin || need >= rem) { fromb |= 1u << d; if (need > 0) --need; }
                    --rem;
                }
            }
#pragma unroll
            for (int d = 0; d < ROWW * 4; ++d)
                if (d < n) w[d >> 2] |= (((fromb >> d) & 1u) ? ROW_BYTE(wb, d) : ROW_BYTE(wa, d)) << ((d & 3) * 8);
        }
    } else if (ALGO == CAO_PSO) {                                       // O6
        if (i == 0) sh.aux = ~0ull;
        __syncthreads();
        if (i < P) atomicMin(&sh.aux, ((unsigned long long)fbits(rm.pbf[q]) << 32) | i);
        __syncthreads();
        const uint32_t gb = (uint32_t)sh.aux;
        if (i < P) {
#pragma unroll
            for (int d = 0; d < ROWW * 4; ++d) {
                if (d < n) {
                    const uint64_t e = ((uint64_t)k * n + d) * P + i;
                    const float hi = coord_M(sm.M, (int)sm.m[d] - 1);
                    float r1 = u01(dr(2 * d)), r2 = u01(dr(2 * d + 1));
                    float xq = rm.x[e], pbq = rm.pb[e], gbq = rm.pb[((uint64_t)k * n + d) * P + gb];
                    float a = __fmul_rn(rm.hp.pso_c1, r1);
                    float b = __fsub_rn(pbq, xq);
                    float t1 = __fmul_rn(a, b);
                    float c = __fmul_rn(rm.hp.pso_c2, r2);
                    float ee = __fsub_rn(gbq, xq);
                    float t2 = __fmul_rn(c, ee);
                    float vv = __fmul_rn(rm.hp.pso_w, rm.v[e]);
                    vv = __fadd_rn(vv, t1);
                    vv = __fadd_rn(vv, t2);
                    float xx = __fadd_rn(xq, vv);
                    xx = clamp_pos(xx, hi);
                    rm.v[e] = vv; rm.x[e] = xx;
                    w[d >> 2] |= (uint32_t)snap_M(sm.M, (int)sm.m[d], xx) << ((d & 3) * 8);
                }
            }
        }
    } else {                                                            // O7: Firefly (Yang's rule, synchronous)
        float* s_xo = (float*)s_dyn;                                    // [j][d]
        float* s_fo = s_xo + (size_t)P * n;                             // [j]
        uint32_t* s_ord = (uint32_t*)(s_fo + P);                        // [brightness rank] -> firefly
        for (uint32_t e = i; e < P * (uint32_t)n; e += blockDim.x) {
            uint32_t j = e / n, d = e - j * n;
            s_xo[e] = rm.x[((uint64_t)k * n + d) * P + j];
        }
        if (i < P) s_fo[i] = rm.f[q];
        __syncthreads();
        // Thread i takes the firefly of brightness RANK i (ties by index), not firefly i: a warp then holds fireflies of
        // similar brightness, so for most attractors j its lanes agree on "j is brighter" -- whole warps skip the attractors
        // dimmer than all their fireflies instead of idling half their lanes.  The update of a firefly does not depend on
        // which thread computes it (draws are addressed by the firefly's index).
        if (i < P) {
            const float fme = s_fo[i];
            uint32_t pos = 0;
            for (uint32_t j = 0; j < P; ++j) { const float fj = s_fo[j]; pos += (fj < fme) || (fj == fme && j < i); }
            s_ord[pos] = i;
        }
        __syncthreads();
        if (i < P) {
            const uint32_t me = s_ord[i];
            qt = (uint64_t)k * P + me;
            float xi[ROWW * 4];
#pragma unroll
            for (int d = 0; d < ROWW * 4; ++d) xi[d] = d < n ? s_xo[me * n + d] : 0.0f;
            const float fi = s_fo[me];
            for (uint32_t j = 0; j < P; ++j) {
                if (!(s_fo[j] < fi)) continue;                          // only brighter (cheaper) fireflies attract
                const float* xj = s_xo + (size_t)j * n;
                float r2 = 0.0f;
#pragma unroll
                for (int d = 0; d < ROWW * 4; ++d)
                    if (d < n) { float df = __fsub_rn(xj[d], xi[d]); r2 = __fadd_rn(r2, __fmul_rn(df, df)); }
                float beta = __fmul_rn(rm.hp.ff_B0, exp_neg_spec(__fmul_rn(rm.hp.ff_gamma, r2)));
                // the n noise draws of this j are slots j*n .. j*n+n-1: all their Philox blocks are computed up
                // front as independent chains, then word (o + d) is picked with selects (o = first slot & 3)
                const uint32_t s0 = j * (uint32_t)n, b0 = s0 >> 2, o = s0 & 3;
                uint32_t nw[(ROWW + 1) * 4];
                {   // interleaved chains (the warp that holds the dimmest fireflies runs alone at the end of the launch:
                    // its latency, not the issue rate, decides the kernel time)
                    const uint32_t nblk = (o + (uint32_t)n + 3) >> 2;   // blocks that hold slots o .. o+n-1
                    const uint32_t k0 = (uint32_t)rm.seed, k1 = (uint32_t)(rm.seed >> 32);
                    uint4 q[ROWW + 1];
#pragma unroll
                    for (int z = 0; z < ROWW + 1; ++z) q[z] = make_uint4(0, 0, 0, 0);
                    constexpr int K1 = ROWW == 4 ? 4 : 5;
                    {
                        uint4 qa[K1];
                        philox4x32_10_multi<K1>(make_uint4(run, g, me, (S_OP << 24) | b0), k0, k1, qa);
#pragma unroll
                        for (int z = 0; z < K1; ++z) q[z] = qa[z];
                    }
                    if (nblk > (uint32_t)K1) {
                        if (ROWW == 4 || nblk == (uint32_t)K1 + 1) q[K1] = philox4x32_10(make_uint4(run, g, me, (S_OP << 24) | (b0 + K1)), k0, k1);
                        else {
                            uint4 qb4[4];
                            philox4x32_10_multi<4>(make_uint4(run, g, me, (S_OP << 24) | (b0 + K1)), k0, k1, qb4);
#pragma unroll
                            for (int z = 0; z < 4; ++z) if (K1 + z < ROWW + 1) q[K1 + z] = qb4[z];
                        }
                    }
#pragma unroll
                    for (int z = 0; z < ROWW + 1; ++z) { nw[z * 4] = q[z].x; nw[z * 4 + 1] = q[z].y; nw[z * 4 + 2] = q[z].z; nw[z * 4 + 3] = q[z].w; }
                }
#pragma unroll
                for (int d = 0; d < ROWW * 4; ++d) {
                    if (d < n) {
                        const uint32_t lo = (o & 1) ? nw[d + 1] : nw[d], hi = (o & 1) ? nw[d + 3] : nw[d + 2];
                        const uint32_t word = (o & 2) ? hi : lo;
                        float df = __fsub_rn(xj[d], xi[d]);
                        xi[d] = __fadd_rn(xi[d], __fmul_rn(beta, df));
                        float e = __fsub_rn(u01(word), 0.5f);
                        xi[d] = __fadd_rn(xi[d], __fmul_rn(rm.hp.ff_alpha, e));
                    }
                }
            }
#pragma unroll
            for (int d = 0; d < ROWW * 4; ++d) {
                if (d < n) {
                    float xx = clamp_pos(xi[d], coord_M(sm.M, (int)sm.m[d] - 1));
                    rm.x[((uint64_t)k * n + d) * P + me] = xx;
                    w[d >> 2] |= (uint32_t)snap_M(sm.M, (int)sm.m[d], xx) << ((d & 3) * 8);
                }
            }
        }
    }
    if (i < P) candidate_tail<ROWW>(sm, rm, qt, w, wl, wl_count, count_scans, sh, use_cache);
    __syncthreads();
    if (i == 0 && sh.n_inv) atomicAdd(&rm.counters[0], (unsigned long long)sh.n_inv);
}

// MAXT: 256 (populations up to 256: the register budget is not capped at 64) or 1024.
template <int ALGO, int ROWW, int MAXT>
__global__ void __launch_bounds__(MAXT) k_op(const __grid_constant__ SpaceMeta sm, const __grid_constant__ RunsMeta rm, uint32_t g) {
    extern __shared__ uint32_t s_dyn[];
    __shared__ RunShared sh;
    const uint32_t k = blockIdx.x;
    const bool active = rm.budget == 0 || rm.uniq[k] < rm.budget;       // O10 (g <= max_gens is enforced by the host)
    if (threadIdx.x == 0) rm.active[k] = active ? 1 : 0;
    if (!active) return;
    gen_op<ALGO, ROWW>(sm, rm, k, g, s_dyn, sh, rm.wl, rm.wl_count, rm.probe_levels < 2, false);
}

// ---------------------------------------------------------------------------------------------
// S6 + S7 after the repair scan.
__device__ __forceinline__ void frozen_row(const RunsMeta& rm, uint32_t k, uint32_t g) {      // thread 0: the row repeats (O10)
    uint32_t* t = rm.traj + ((uint64_t)g * rm.R + k) * 3;
    t[0] = fbits(rm.best_f[k]); t[1] = rm.best_rank[k]; t[2] = rm.uniq[k];
}

// S6 + S7 for an ACTIVE run k once every candidate has its repair key (block-uniform call, contains barriers).
template <int ALGO, int ROWW>
__device__ __forceinline__ void gen_finish(const SpaceMeta& sm, const RunsMeta& rm, uint32_t k, uint32_t g, uint32_t* s_dyn,
                                           RunShared& sh) {
    const uint32_t i = threadIdx.x, P = rm.P, run = rm.first_run + k;
    const int n = sm.n;
    if (i == 0) eval_begin(rm, k, &sh);
    __syncthreads();
    const uint64_t q = (uint64_t)k * P + i;
    uint32_t rk = 0; float f = 0.0f;
    if (!rm.var_on) {                                                   // statistics: Hamming distance of every repair
        const uint32_t h = i < P ? min((uint32_t)(rm.key[q] >> 45), 8u) : 31u;
        const uint32_t peers = __match_any_sync(0xFFFFFFFFu, h);
        if (i < P && (i & 31) == (uint32_t)(__ffs(peers) - 1)) atomicAdd(&rm.counters[16 + h], (unsigned long long)__popc(peers));
    }
    uint32_t cur[ROWW];                                                 // DE / GA: the row the individual holds after S5
#pragma unroll
    for (int z = 0; z < ROWW; ++z) cur[z] = 0;
    if (i < P) {
        rk = (uint32_t)rm.key[q];                                       // CAO_KEY_NONE -> CAO_RANK_NONE: the candidate stayed invalid
        if (rm.var.constraint_aware && rm.var.repair_mode == 1 && !rm.valid[q] && (ALGO == CAO_PSO || ALGO == CAO_FIREFLY)) {
            // Alg.2: the first non-empty neighbour set; its member nearest to the particle (k_scan_nb)
            uint32_t rule = 3;
            rk = CAO_RANK_NONE;
            for (int c = 2; c >= 0; --c) { const unsigned long long e = rm.key3[q * 3 + c]; if (e != ~0ull) { rule = (uint32_t)c; rk = (uint32_t)e; } }
            rm.rule[q] = (uint8_t)rule;
        }
        rm.rep_rank[q] = rk;
        if (ALGO == CAO_DE || ALGO == CAO_GA) {
            if (rk == CAO_RANK_NONE) load_row_rw<ROWW>(rm.cand + q * (ROWW * 4), cur);
            else load_row<ROWW>(sm.rows + (uint64_t)rk * (ROWW * 4), cur);
        }
        if (ALGO == CAO_GA) {                                           // L290, L311, L393: 1-in-X mutation after repair
            Draws dm(rm.seed, run, g, i, S_MUT);
            if (below(dm(0), (uint32_t)rm.hp.ga_mutation_chance) == 0) {
                const uint64_t L = row_lin<ROWW>(sm, cur);
                if (rm.var.constraint_aware) {
                    uint32_t K = 0;                                     // valid Hamming-1 neighbours, (d asc, value asc)
#pragma unroll
                    for (int d = 0; d < ROWW * 4; ++d) {
                        if (d < n) {
                            const int c = (int)ROW_BYTE(cur, d);
                            for (int val = 0; val < (int)sm.m[d]; ++val)
                                if (val != c && bit_test(sm.bitmap, L + (int64_t)(val - c) * (int64_t)sm.stride[d])) ++K;
                        }
                    }
                    if (K) {
                        uint32_t pick = below(dm(1), K), seen = 0;
                        uint64_t Lp = L; bool done = false;
#pragma unroll
                        for (int d = 0; d < ROWW * 4; ++d) {
                            if (d < n && !done) {
                                const int c = (int)ROW_BYTE(cur, d);
                                for (int val = 0; val < (int)sm.m[d] && !done; ++val) {
                                    if (val == c) continue;
                                    uint64_t L2 = L + (int64_t)(val - c) * (int64_t)sm.stride[d];
                                    if (bit_test(sm.bitmap, L2)) { if (seen == pick) { Lp = L2; done = true; } ++seen; }
                                }
                            }
                        }
                        rk = rank_of(sm, Lp);
                        load_row<ROWW>(sm.rows + (uint64_t)rk * (ROWW * 4), cur);
                    }
                } else {                                                // NEXT-2 (L309): one parameter gets a different value, if any
                    const uint32_t dmut = below(dm(1), (uint32_t)n), md = sm.m[dmut];
                    if (md > 1) {
                        uint32_t cd = 0;
#pragma unroll
                        for (int d = 0; d < ROWW * 4; ++d) if ((uint32_t)d == dmut) cd = ROW_BYTE(cur, d);
                        uint32_t val = below(dm(2), md - 1);
                        if (val >= cd) val += 1;
#pragma unroll
                        for (int z = 0; z < ROWW; ++z)
                            if ((uint32_t)z == (dmut >> 2)) cur[z] = (cur[z] & ~(0xFFu << ((dmut & 3) * 8))) | (val << ((dmut & 3) * 8));
                        const uint64_t Lm = L + (int64_t)((int)val - (int)cd) * (int64_t)sm.stride[dmut];
                        rk = bit_test(sm.bitmap, Lm) ? rank_of(sm, Lm) : CAO_RANK_NONE;
                    }
                }
            }
        }
        f = evaluate(sm, rm, k, rk, &sh);
        rm.eval_rank[q] = rk; rm.tap_f[q] = f;
    }

    if (ALGO == CAO_DE) {                                               // Alg.1; A7 (membership by linear index:
        uint64_t* s_old = (uint64_t*)s_dyn;                             // members may be invalid rows under NEXT-1 / NEXT-2)
        uint64_t* s_u = s_old + P;                                      // P trials
        uint64_t myL = 0;
        if (i < P) {
            uint32_t wo[ROWW];
            load_row_rw<ROWW>(rm.idx + q * (ROWW * 4), wo);
            s_old[i] = row_lin<ROWW>(sm, wo);
            myL = row_lin<ROWW>(sm, cur); s_u[i] = myL;
        }
        __syncthreads();
        bool acc = false;
        if (i < P) {
            acc = f <= rm.f[q];
            for (uint32_t j = 0; j < P && acc; ++j) if (s_old[j] == myL) acc = false;
            for (uint32_t j = 0; j < i && acc; ++j) if (s_u[j] == myL) acc = false;
            rm.accept[q] = acc ? 1 : 0;
        }
        const int any = __syncthreads_or(acc);
        if (acc) {
            store_row<ROWW>(rm.idx + q * (ROWW * 4), cur);
            rm.f[q] = f; rm.rank[q] = rk;
        }
        // L266: nothing accepted in two consecutive generations -> re-initialise (evaluated in this step)
        const uint32_t st = any ? 0 : rm.stagn[k] + 1;
        __syncthreads();
        if (st == 2) {
            if (rm.var.constraint_aware) init_population<CAO_DE, ROWW>(sm, rm, k, g, S_REINIT, (uint32_t*)s_dyn, &sh);
            else init_population_unaware<CAO_DE, ROWW>(sm, rm, k, g, S_REINIT, &sh);
            if (i == 0) atomicAdd(&rm.counters[2], (unsigned long long)P);
        }
        if (i == 0) rm.stagn[k] = st == 2 ? 0 : st;
    } else if (ALGO == CAO_GA) {                                        // L288: the children replace the population
        if (i < P) {
            store_row<ROWW>(rm.idx + q * (ROWW * 4), cur);
            rm.f[q] = f; rm.rank[q] = rk; rm.accept[q] = 0;
        }
    } else if (ALGO == CAO_PSO) {                                       // L282: repair affects the evaluation only
        if (i < P) {
            rm.f[q] = f; rm.rank[q] = rk;
            const bool improved = f < rm.pbf[q];                        // strict (A13)
            rm.accept[q] = improved ? 1 : 0;
            if (improved) {
                rm.pbf[q] = f;
                for (int d = 0; d < n; ++d) { const uint64_t e = ((uint64_t)k * n + d) * P + i; rm.pb[e] = rm.x[e]; }
            }
        }
    } else {
        if (i < P) { rm.f[q] = f; rm.rank[q] = rk; rm.accept[q] = 0; }
    }
    __syncthreads();
    if (i == 0) {
        eval_end(rm, k, g, &sh);
        rm.gens_done[k] += 1;
        atomicAdd(&rm.counters[2], (unsigned long long)P);
    }
}

template <int ALGO, int ROWW>
__global__ void __launch_bounds__(1024) k_finish(const __grid_constant__ SpaceMeta sm, const __grid_constant__ RunsMeta rm, uint32_t g) {
    extern __shared__ uint32_t s_dyn[];
    __shared__ RunShared sh;
    const uint32_t k = blockIdx.x;
    if (k == 0 && threadIdx.x == 0) { *rm.wl_count = 0; *rm.wl2_count = 0; }       // the scan of this generation is done
    if (!rm.active[k]) { if (threadIdx.x == 0) frozen_row(rm, k, g); return; }
    gen_finish<ALGO, ROWW>(sm, rm, k, g, s_dyn, sh);
}

#define GEN_NB 4                                          // candidates per batch of the in-group table scan (cao_gen_kernels.cuh)

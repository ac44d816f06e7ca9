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
};

// Shared scratch of the per-run CTAs.
struct RunShared {
    unsigned long long best;                           // (f bits << 32 | rank) of the best-so-far
    unsigned long long aux;                            // PSO: (pbest_f bits << 32 | i) of gbest
    uint32_t n_new, flag, n_inv;
};

// ---------------------------------------------------------------------------------------------
// O10: evaluate rank rk for run k: objective lookup, memoisation bit, best-so-far (block-level, order-free).
__device__ __forceinline__ float evaluate(const SpaceMeta& sm, const RunsMeta& rm, uint32_t k, uint32_t rk, RunShared* sh) {
    float f = __ldg(&sm.obj[rk]);
    uint32_t bit = 1u << (rk & 31);
    uint32_t old = atomicOr(&rm.dedup[(uint64_t)k * rm.dedup_words + (rk >> 5)], bit);
    if (!(old & bit)) atomicAdd(&sh->n_new, 1u);
    atomicMin(&sh->best, ((unsigned long long)fbits(f) << 32) | rk);
    return f;
}
__device__ __forceinline__ void eval_begin(const RunsMeta& rm, uint32_t k, RunShared* sh) {     // thread 0, before a sync
    uint32_t br = rm.best_rank[k];
    sh->best = br == 0xFFFFFFFFu ? ~0ull : (((unsigned long long)fbits(rm.best_f[k]) << 32) | br);
    sh->n_new = 0; sh->flag = 0; sh->aux = ~0ull;
}
__device__ __forceinline__ void eval_end(const RunsMeta& rm, uint32_t k, uint32_t g, RunShared* sh) {   // thread 0, after a sync
    uint32_t u = rm.uniq[k] + sh->n_new;
    rm.uniq[k] = u;
    rm.best_f[k] = __uint_as_float((uint32_t)(sh->best >> 32));
    rm.best_rank[k] = (uint32_t)sh->best;
    uint32_t* t = rm.traj + ((uint64_t)g * rm.R + k) * 3;
    t[0] = (uint32_t)(sh->best >> 32); t[1] = (uint32_t)sh->best; t[2] = u;
}

// O4: P distinct valid ranks, uniform with linear probing; fills the population and evaluates it.
// Block-uniform call; s_r holds P words.  Ends with a __syncthreads().
template <int ALGO, int ROWW>
__device__ void init_population(const SpaceMeta& sm, const RunsMeta& rm, uint32_t k, uint32_t g, uint32_t stream,
                                uint32_t* s_r, RunShared* sh) {
    const uint32_t i = threadIdx.x, P = rm.P, run = rm.first_run + k;
    Draws dr(rm.seed, run, g, i, stream);
    if (i < P) s_r[i] = below(dr(0), sm.V);
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

// Generation 0 (S2).
template <int ALGO, int ROWW>
__global__ void __launch_bounds__(1024) k_init(const __grid_constant__ SpaceMeta sm, const __grid_constant__ RunsMeta rm) {
    extern __shared__ uint32_t s_dyn[];
    __shared__ RunShared sh;
    const uint32_t k = blockIdx.x;
    if (threadIdx.x == 0) eval_begin(rm, k, &sh);
    __syncthreads();
    init_population<ALGO, ROWW>(sm, rm, k, 0, S_INIT, s_dyn, &sh);
    if (threadIdx.x == 0) {
        eval_end(rm, k, 0, &sh);
        atomicAdd(&rm.counters[2], (unsigned long long)rm.P);
    }
}

// ---------------------------------------------------------------------------------------------
// S4 + first half of S5 for the candidate held in w: store, validity, probe, worklist.
template <int ROWW>
__device__ __forceinline__ void candidate_tail(const SpaceMeta& sm, const RunsMeta& rm, uint64_t slot, const uint32_t (&w)[ROWW],
                                               uint32_t* wl, uint32_t* wl_count, bool count_scans, RunShared& sh, bool use_cache) {
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
    uint32_t w[ROWW];
#pragma unroll
    for (int z = 0; z < ROWW; ++z) w[z] = 0;
    Draws dr(rm.seed, run, g, i, S_OP);
    if (i == 0) sh.n_inv = 0;
    __syncthreads();

    if (ALGO == CAO_DE) {                                               // O5: best1bin on indices
        if (i < P) {
            uint32_t a = below(dr(0), P - 1); if (a >= i) a += 1;
            uint32_t b = below(dr(1), P - 2);
            uint32_t lo = min(i, a), hi = max(i, a);
            if (b >= lo) b += 1;
            if (b >= hi) b += 1;
            uint32_t jrand = below(dr(2), (uint32_t)n);
            uint32_t wa[ROWW], wb[ROWW], wx[ROWW], wbest[ROWW];
            load_row_rw<ROWW>(rm.idx + ((uint64_t)k * P + a) * (ROWW * 4), wa);
            load_row_rw<ROWW>(rm.idx + ((uint64_t)k * P + b) * (ROWW * 4), wb);
            load_row_rw<ROWW>(rm.idx + q * (ROWW * 4), wx);
            load_row<ROWW>(sm.rows + (uint64_t)rm.best_rank[k] * (ROWW * 4), wbest);
#pragma unroll
            for (int d = 0; d < ROWW * 4; ++d) {
                if (d < n) {
                    int vd = de_mutate_index(rm.hp.de_F, (int)ROW_BYTE(wbest, d), (int)ROW_BYTE(wa, d), (int)ROW_BYTE(wb, d),
                                             (int)sm.m[d] - 1);
                    float rr = u01(dr(3 + d));
                    uint32_t ud = (rr < rm.hp.de_CR || (uint32_t)d == jrand) ? (uint32_t)vd : ROW_BYTE(wx, d);
                    w[d >> 2] |= ud << ((d & 3) * 8);
                }
            }
        }
    } else if (ALGO == CAO_GA) {                                        // O8: sorted population, Beta(1,b) parents, single point
        unsigned long long* s_key = (unsigned long long*)s_dyn;         // P keys
        uint32_t* s_order = (uint32_t*)(s_key + P);                     // P
        if (i < P) s_key[i] = ((unsigned long long)fbits(rm.f[q]) << 32) | rm.rank[q];
        __syncthreads();
        if (i < P) {
            unsigned long long me = s_key[i];
            uint32_t pos = 0;
            for (uint32_t j = 0; j < P; ++j) { unsigned long long o = s_key[j]; pos += (o < me) || (o == me && j < i); }
            s_order[pos] = i;
        }
        __syncthreads();
        if (i < P) {
            const uint32_t B = (uint32_t)rm.hp.ga_beta_b;
            uint32_t sa = P, sb = P;
            for (uint32_t z = 0; z < B; ++z) sa = min(sa, below(dr(z), P));
            for (uint32_t z = 0; z < B; ++z) sb = min(sb, below(dr(B + z), P));
            if (sb == sa) sb = sa + 1 == P ? 0 : sa + 1;
            int cut = n > 1 ? 1 + (int)below(dr(2 * B), (uint32_t)(n - 1)) : 1;
            uint32_t wa[ROWW], wb[ROWW];
            load_row_rw<ROWW>(rm.idx + ((uint64_t)k * P + s_order[sa]) * (ROWW * 4), wa);
            load_row_rw<ROWW>(rm.idx + ((uint64_t)k * P + s_order[sb]) * (ROWW * 4), wb);
#pragma unroll
            for (int d = 0; d < ROWW * 4; ++d)
                if (d < n) w[d >> 2] |= (d < cut ? ROW_BYTE(wa, d) : ROW_BYTE(wb, d)) << ((d & 3) * 8);
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
        for (uint32_t e = i; e < P * (uint32_t)n; e += blockDim.x) {
            uint32_t j = e / n, d = e - j * n;
            s_xo[e] = rm.x[((uint64_t)k * n + d) * P + j];
        }
        if (i < P) s_fo[i] = rm.f[q];
        __syncthreads();
        if (i < P) {
            float xi[ROWW * 4];
#pragma unroll
            for (int d = 0; d < ROWW * 4; ++d) xi[d] = d < n ? s_xo[i * n + d] : 0.0f;
            const float fi = s_fo[i];
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
#pragma unroll
                for (int qb = 0; qb < ROWW + 1; ++qb) {
                    uint4 rr = make_uint4(0, 0, 0, 0);
                    if ((uint32_t)(qb * 4) < o + (uint32_t)n)
                        rr = philox4x32_10(make_uint4(run, g, i, (S_OP << 24) | (b0 + qb)), (uint32_t)rm.seed, (uint32_t)(rm.seed >> 32));
                    nw[qb * 4] = rr.x; nw[qb * 4 + 1] = rr.y; nw[qb * 4 + 2] = rr.z; nw[qb * 4 + 3] = rr.w;
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
                    rm.x[((uint64_t)k * n + d) * P + i] = xx;
                    w[d >> 2] |= (uint32_t)snap_M(sm.M, (int)sm.m[d], xx) << ((d & 3) * 8);
                }
            }
        }
    }
    if (i < P) candidate_tail<ROWW>(sm, rm, q, w, wl, wl_count, count_scans, sh, use_cache);
    __syncthreads();
    if (i == 0 && sh.n_inv) atomicAdd(&rm.counters[0], (unsigned long long)sh.n_inv);
}

template <int ALGO, int ROWW>
__global__ void __launch_bounds__(1024) k_op(const __grid_constant__ SpaceMeta sm, const __grid_constant__ RunsMeta rm, uint32_t g) {
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
    {                                                                   // statistics: Hamming distance of every repair
        const uint32_t h = i < P ? min((uint32_t)(rm.key[q] >> 45), 8u) : 31u;
        const uint32_t peers = __match_any_sync(0xFFFFFFFFu, h);
        if (i < P && (i & 31) == (uint32_t)(__ffs(peers) - 1)) atomicAdd(&rm.counters[16 + h], (unsigned long long)__popc(peers));
    }
    if (i < P) {
        rk = (uint32_t)rm.key[q];
        rm.rep_rank[q] = rk;
        if (ALGO == CAO_GA) {                                           // L290, L311, L393: 1-in-X mutation after repair
            Draws dm(rm.seed, run, g, i, S_MUT);
            if (below(dm(0), (uint32_t)rm.hp.ga_mutation_chance) == 0) {
                uint32_t cur[ROWW];
                load_row<ROWW>(sm.rows + (uint64_t)rk * (ROWW * 4), cur);
                const uint64_t L = row_lin<ROWW>(sm, cur);
                uint32_t K = 0;                                         // valid Hamming-1 neighbours, (d asc, value asc)
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
                }
            }
        }
        f = evaluate(sm, rm, k, rk, &sh);
        rm.eval_rank[q] = rk; rm.tap_f[q] = f;
    }

    if (ALGO == CAO_DE) {                                               // Alg.1; A7
        uint32_t* s_old = s_dyn;                                        // P old ranks
        uint32_t* s_u = s_dyn + P;                                      // P trial ranks
        if (i < P) { s_old[i] = rm.rank[q]; s_u[i] = rk; }
        __syncthreads();
        bool acc = false;
        if (i < P) {
            acc = f <= rm.f[q];
            for (uint32_t j = 0; j < P && acc; ++j) if (s_old[j] == rk) acc = false;
            for (uint32_t j = 0; j < i && acc; ++j) if (s_u[j] == rk) acc = false;
            rm.accept[q] = acc ? 1 : 0;
        }
        const int any = __syncthreads_or(acc);
        if (acc) {
            uint32_t row[ROWW];
            load_row<ROWW>(sm.rows + (uint64_t)rk * (ROWW * 4), row);
            store_row<ROWW>(rm.idx + q * (ROWW * 4), row);
            rm.f[q] = f; rm.rank[q] = rk;
        }
        // L266: nothing accepted in two consecutive generations -> re-initialise (evaluated in this step)
        const uint32_t st = any ? 0 : rm.stagn[k] + 1;
        __syncthreads();
        if (st == 2) {
            init_population<CAO_DE, ROWW>(sm, rm, k, g, S_REINIT, s_dyn, &sh);
            if (i == 0) atomicAdd(&rm.counters[2], (unsigned long long)P);
        }
        if (i == 0) rm.stagn[k] = st == 2 ? 0 : st;
    } else if (ALGO == CAO_GA) {                                        // L288: the children replace the population
        if (i < P) {
            uint32_t row[ROWW];
            load_row<ROWW>(sm.rows + (uint64_t)rk * (ROWW * 4), row);
            store_row<ROWW>(rm.idx + q * (ROWW * 4), row);
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

// cao_gen_kernels.cuh -- fused persistent generation kernel (S3-S7 for all requested generations in ONE launch).
// PAPER.md Alg.1 L147-213 (DE), L276-282 (PSO), L284 (Firefly), L286-292 + Alg.3 L298-311 (GA), L268 (memoisation),
// L125 (budget); readings O4-O10 / A6-A20 in DESIGN.md.
//
// Execution model: a GROUP of G = roundup32(P) threads owns one run; a CTA holds several groups (8 one-warp groups
// at P <= 32).  Groups are independent: they synchronise with __syncwarp() (G = 32) or a named barrier (G > 32),
// never with __syncthreads().  A group pulls run indices from a global ticket counter until none are left, so a slow
// run (a table scan, a Hamming-3 probe) delays nobody else and short runs (budget reached) free their slot at once.
// The whole population state of the run (index rows / positions, velocities, personal bests, f, rank), the repair
// memo of the previous generation and all scratch live in the group's slice of shared memory for the duration of the
// call; global memory sees the state once on entry and once on exit.  Per generation only the trajectory row, the
// per-run dedup bits (HBM, atomicOr) and the read-only space tables (bitmap, directory, rows, objective) are touched.
#pragma once
#include "cao_runs_kernels.cuh"

#include "cao_gen_layout.h"

struct GrpShared {                   // first words of every group slice
    unsigned long long best;         // (f bits << 32 | rank) of the best-so-far
    unsigned long long aux;          // PSO: (pbest_f bits << 32 | i) of gbest; probe: level minimum
    uint32_t run, uniq, stagn, n_new, flag, nwl, bestrow_rank, gens;
    uint32_t n_inv, n_scan, n_eval, n_p2, n_p3, n_memo, n_rc, pad;   // statistics of this run in this launch
    unsigned long long cyc[6];       // CAO_GEN_STATS builds: clock cycles in operator / tail / probe-2 / probe-3 / scan / finish
    uint32_t hist[16];               // repaired candidates by Hamming distance of the repair (0 = valid, ..., 8 = eight or more)
};
#ifdef CAO_GEN_STATS
#define CAO_TICK(slot) do { if (g.t == 0) { const long long now_ = clock64(); gs->cyc[slot] += (unsigned long long)(now_ - t_mark); t_mark = now_; } } while (0)
#else
#define CAO_TICK(slot) do { } while (0)
#endif
static_assert(sizeof(GrpShared) == GRP_SHARED_WORDS * 4, "GrpShared layout");

// CTA-wide tables in shared memory (built once per CTA in the kernel prologue).
struct CtaTabs {
    const uint16_t* nb;              // Hamming-1 neighbour list: d << 8 | k, k = 0 .. m_d - 2, sorted by (d, k)
    const uint64_t* stride;          // stride[d]
    const float* hi;                 // coord(m_d - 1) (O6)
    const uint32_t* pairs;           // pair list of the Hamming >= 2 probes (shared or global memory)
    uint32_t NB;
};

// Validity and rank of linear index L in ONE round trip: the directory entry and the 64-byte bitmap block of L are
// loaded together; the rank is only meaningful when the bit is set.
static __device__ __noinline__ uint32_t valid_rank(const uint64_t* __restrict__ bitmap, const uint32_t* __restrict__ dir, uint64_t L,
                                                   uint32_t* valid) {
    const uint32_t wi = (uint32_t)(L >> 6) & 7u;
    const ulonglong2* blk = (const ulonglong2*)(bitmap + ((L >> 6) & ~7ull));
    uint32_t r = __ldg(&dir[L >> CAO_DIR_SHIFT]);
    const ulonglong2 v0 = __ldg(&blk[0]), v1 = __ldg(&blk[1]), v2 = __ldg(&blk[2]), v3 = __ldg(&blk[3]);
    const uint64_t wd[8] = {v0.x, v0.y, v1.x, v1.y, v2.x, v2.y, v3.x, v3.y};
    const uint64_t below_mask = (1ull << (L & 63)) - 1ull;
    uint64_t mine = 0;
#pragma unroll
    for (uint32_t q = 0; q < 8; ++q) {
        r += q < wi ? __popcll(wd[q]) : 0;
        mine = q == wi ? wd[q] : mine;
    }
    r += __popcll(mine & below_mask);
    *valid = (uint32_t)((mine >> (L & 63)) & 1ull);
    return r;
}

// Group-cooperative Hamming-1 probe (exact: Hamming is the primary key, |delta| the secondary, L the third).  The
// `nopen` open candidates (list ol, linear indices Lc, rows8 = the group's candidate rows, RB bytes each) times their NB
// neighbours form one flat index space that the threads stride over, four independent bit tests in flight each.  A hit
// goes to the LOW WORD of hkey[candidate] with a native 32-bit shared-memory atomicMin on |delta| << 8 | ord (a 64-bit
// shared atomicMin is a compare-and-swap loop).  ord orders the neighbours of one candidate that share |delta| = s exactly
// like their linear indices L' = L -+ s * stride_d: the negative steps first (larger stride = smaller dimension first:
// ord = d), then the positive steps (smaller stride first: ord = 63 - d); h1_decode rebuilds (|delta|, L').  hkey[.] must
// hold ~0 on entry.  The caller synchronises afterwards.
template <int RB>
__device__ __forceinline__ void probe_h1_flat(const Grp& g, const uint64_t* __restrict__ bitmap, const CtaTabs& tb, const uint8_t* rows8,
                                              const uint32_t* ol, const uint64_t* Lc, unsigned long long* hkey, uint32_t nopen) {
    const uint32_t NB = tb.NB, total = nopen * NB;
    uint32_t jj = g.t / NB, t = g.t - jj * NB;
    const uint32_t sj = g.G / NB, st = g.G - sj * NB;
    uint32_t* hk32 = (uint32_t*)hkey;
    for (uint32_t q0 = g.t; q0 < total; q0 += 4 * g.G) {
        uint32_t kv[4], who[4]; bool bit[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const bool live = q0 + u * g.G < total;
            const uint32_t i2 = ol[live ? jj : 0], e = tb.nb[live ? t : 0], d = e >> 8, kq = e & 255u, cd = rows8[(size_t)i2 * RB + d];
            const int dv = (int)(kq + (kq >= cd)) - (int)cd;
            kv[u] = ((uint32_t)abs(dv) << 8) | (dv < 0 ? d : 63u - d); who[u] = i2;
            bit[u] = bit_test(bitmap, Lc[i2] + (int64_t)dv * (int64_t)tb.stride[d]) && live;
            t += st; jj += sj;
            if (t >= NB) { t -= NB; ++jj; }
        }
#pragma unroll
        for (int u = 0; u < 4; ++u)
            if (bit[u]) atomicMin(&hk32[2 * who[u]], kv[u]);
    }
}
// (|delta|, L') of the winning neighbour from the reduced word m != ~0 of a candidate with linear index L.
__device__ __forceinline__ uint64_t h1_decode(const CtaTabs& tb, uint32_t m, uint64_t L, uint32_t* sad) {
    const uint32_t sdv = m >> 8, ord = m & 63u, d = ord < 32u ? ord : 63u - ord;
    const uint64_t step = (uint64_t)sdv * tb.stride[d];
    *sad = sdv;
    return ord < 32u ? L - step : L + step;
}

// Group-cooperative brute-force scan of the whole valid table for up to NB candidates (rows in shared memory); the
// table rows come straight from L2, coalesced, RU rows in flight per thread.  s_key[b] must be ~0 on entry; on exit it
// holds ham << 45 | sad << 32 | rank.  Ends with a barrier.
template <int ROWW, int NB>
static __device__ __noinline__ void scan_grp(const Grp g, const uint8_t* __restrict__ rows, uint32_t V, const uint32_t* s_cw, int nb,
                                             unsigned long long* s_key) {
    uint32_t c[NB][ROWW];
#pragma unroll
    for (int b = 0; b < NB; ++b)
#pragma unroll
        for (int k = 0; k < ROWW; ++k) c[b][k] = b < nb ? s_cw[b * ROWW + k] : 0;
    uint64_t best[NB];
#pragma unroll
    for (int b = 0; b < NB; ++b) best[b] = ~0ull;
    constexpr int RU = ROWW == 4 ? 4 : 2;
    for (uint32_t r0 = g.t; r0 < V; r0 += RU * g.G) {
        uint32_t v[RU][ROWW];
#pragma unroll
        for (int u = 0; u < RU; ++u) {
            const uint32_t r = r0 + u * g.G;
            load_row<ROWW>(rows + (uint64_t)(r < V ? r : r0) * (ROWW * 4), v[u]);
        }
#pragma unroll
        for (int u = 0; u < RU; ++u) {
            const uint32_t r = r0 + u * g.G;
            if (r >= V) break;
#pragma unroll
            for (int b = 0; b < NB; ++b) {
                uint32_t sad = 0, ham = 0;
#pragma unroll
                for (int k = 0; k < ROWW; ++k) {
                    sad = sad4_acc(c[b][k], v[u][k], sad);
                    const uint32_t x = c[b][k] ^ v[u][k];
                    ham += __popc((((x & 0x7f7f7f7fu) + 0x7f7f7f7fu) | x) & 0x80808080u);
                }
                const uint64_t key = ((uint64_t)((ham << 13) + sad) << 32) | r;
                best[b] = key < best[b] ? key : best[b];
            }
        }
    }
#pragma unroll
    for (int b = 0; b < NB; ++b) {
        const uint64_t m = warp_min_key(best[b]);
        if ((g.t & 31) == 0 && b < nb) atomicMin(&s_key[b], (unsigned long long)m);
    }
    g.sync();
}

// ---------------------------------------------------------------------------------------------
// The group's view of its shared-memory slice.
struct GrpMem {
    GrpShared* gs;
    uint32_t* rank; float* f; uint32_t* idx; float* x; float* v; float* pb; float* pbf;
    uint32_t* cand; unsigned long long* key; uint32_t* scr; uint32_t* wl; uint32_t* cw; unsigned long long* skey;
    uint32_t* bestrow; uint64_t* Lc; uint32_t* aux4; uint64_t* ptab;
    __device__ __forceinline__ GrpMem(uint32_t* S, const GenLayout& l)
        : gs((GrpShared*)S), rank(S + l.rank), f((float*)(S + l.f)), idx(S + l.idx), x((float*)(S + l.x)), v((float*)(S + l.v)),
          pb((float*)(S + l.pb)), pbf((float*)(S + l.pbf)), cand(S + l.cand), key((unsigned long long*)(S + l.key)),
          scr(S + l.scr), wl(S + l.wl), cw(S + l.cw), skey((unsigned long long*)(S + l.skey)), bestrow(S + l.bestrow),
          Lc((uint64_t*)(S + l.Lc)), aux4(S + l.aux4), ptab((uint64_t*)(S + l.ptab)) {}
};

// O10: evaluate rank rk for run k.  Returns f; *is_new = this evaluation set the run's memo bit (L268).
__device__ __forceinline__ float evaluate_v2(const SpaceMeta& sm, const RunsMeta& rm, uint32_t k, uint32_t rk, bool& is_new) {
    const float f = __ldg(&sm.obj[rk]);
    const uint32_t bit = 1u << (rk & 31);
    const uint32_t old = atomicOr(&rm.dedup[(uint64_t)k * rm.dedup_words + (rk >> 5)], bit);
    is_new = !(old & bit);
    return f;
}
// Folds the evaluations of one phase into the group's counters: new memo bits and best-so-far (order-free).
__device__ __forceinline__ void fold_eval(const Grp& g, GrpShared* gs, bool has, bool is_new, float f, uint32_t rk) {
    const uint32_t nn = __popc(__ballot_sync(0xFFFFFFFFu, has && is_new));
    const uint64_t m = warp_min_key(has ? (((uint64_t)fbits(f) << 32) | rk) : ~0ull);
    if ((g.t & 31) == 0) {
        if (g.G == 32) {                                                // a single warp owns the slice: no atomics needed
            gs->n_new += nn;
            if (m < gs->best) gs->best = m;
        } else {
            if (nn) atomicAdd(&gs->n_new, nn);
            if (m != ~0ull) atomicMin(&gs->best, (unsigned long long)m);
        }
    }
}

// O4 inside the fused kernel (DE stagnation re-initialisation, L266): P distinct valid ranks, uniform with linear
// probing; fills the shared-memory population and evaluates it.  Group-uniform call, ends with a barrier.
template <int ROWW>
static __device__ __noinline__ void reinit_de_grp(const Grp g, const SpaceMeta& sm, const RunsMeta& rm, GrpMem& S, uint32_t k, uint32_t gen) {
    const uint32_t i = g.t, P = rm.P, run = rm.first_run + k;
    uint32_t* s_r = S.scr;
    Draws dr(rm.seed, run, gen, i, S_REINIT);
    if (i < P) s_r[i] = below(dr(0), sm.V);
    g.sync();
    bool dup = false;
    if (i < P) { const uint32_t me = s_r[i]; for (uint32_t j = 0; j < i; ++j) dup |= (s_r[j] == me); }
    if (g.sync_or(dup)) {
        if (i == 0) {                                                   // the sequential definition, rare
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
        g.sync();
    }
    bool is_new = false; float f = 0.0f; uint32_t rk = 0;
    if (i < P) {
        rk = s_r[i];
        uint32_t w[ROWW];
        load_row<ROWW>(sm.rows + (uint64_t)rk * (ROWW * 4), w);
        f = evaluate_v2(sm, rm, k, rk, is_new);
        S.rank[i] = rk; S.f[i] = f;
#pragma unroll
        for (int z = 0; z < ROWW; ++z) S.idx[i * ROWW + z] = w[z];
    }
    fold_eval(g, S.gs, i < P, is_new, f, rk);
    g.sync();
}

// ---------------------------------------------------------------------------------------------
// State transfer between the group's shared-memory slice and the caller's workspace (layouts of cao_runs_debug_state).
template <int ALGO, int ROWW>
__device__ __forceinline__ void load_state(const Grp& g, const SpaceMeta& sm, const RunsMeta& rm, GrpMem& S, uint32_t k) {
    const uint32_t P = rm.P, n = (uint32_t)sm.n;
    const uint64_t q0 = (uint64_t)k * P;
    for (uint32_t i = g.t; i < P; i += g.G) {
        S.rank[i] = rm.rank[q0 + i]; S.f[i] = rm.f[q0 + i];
        S.key[i] = CAO_KEY_NONE;                                         // the memo starts empty (it is only a shortcut)
        if (ALGO == CAO_PSO) S.pbf[i] = rm.pbf[q0 + i];
    }
    for (uint32_t e = g.t; e < P * ROWW; e += g.G) S.cand[e] = 0;       // padding bytes of the candidate rows stay zero
    if (ALGO == CAO_DE || ALGO == CAO_GA) {
        const uint32_t* src = (const uint32_t*)(rm.idx + q0 * (ROWW * 4));
        for (uint32_t e = g.t; e < P * ROWW; e += g.G) S.idx[e] = src[e];
    } else {
        const uint64_t e0 = (uint64_t)k * n * P;
        for (uint32_t e = g.t; e < n * P; e += g.G) {
            if (ALGO == CAO_PSO) { S.x[e] = rm.x[e0 + e]; S.v[e] = rm.v[e0 + e]; S.pb[e] = rm.pb[e0 + e]; }
            else { const uint32_t d = e / P, j = e - d * P; S.x[j * n + d] = rm.x[e0 + e]; }     // Firefly: [j][d] in shared memory
        }
    }
    if (g.t == 0) {
        GrpShared* gs = S.gs;
        const uint32_t br = rm.best_rank[k];
        gs->best = br == 0xFFFFFFFFu ? ~0ull : (((unsigned long long)fbits(rm.best_f[k]) << 32) | br);
        gs->uniq = rm.uniq[k]; gs->stagn = rm.stagn[k]; gs->bestrow_rank = 0xFFFFFFFFu;
        gs->n_inv = 0; gs->n_scan = 0; gs->n_eval = 0; gs->gens = 0;
        gs->n_p2 = 0; gs->n_p3 = 0; gs->n_memo = 0; gs->n_rc = 0;
        for (int z = 0; z < 6; ++z) gs->cyc[z] = 0;
        for (int z = 0; z < 16; ++z) gs->hist[z] = 0;
    }
    g.sync();
}
template <int ALGO, int ROWW>
__device__ __forceinline__ void store_state(const Grp& g, const SpaceMeta& sm, const RunsMeta& rm, GrpMem& S, uint32_t k) {
    const uint32_t P = rm.P, n = (uint32_t)sm.n;
    const uint64_t q0 = (uint64_t)k * P;
    for (uint32_t i = g.t; i < P; i += g.G) {
        rm.rank[q0 + i] = S.rank[i]; rm.f[q0 + i] = S.f[i];
        if (ALGO == CAO_PSO) rm.pbf[q0 + i] = S.pbf[i];
    }
    if (ALGO == CAO_DE || ALGO == CAO_GA) {
        uint32_t* dst = (uint32_t*)(rm.idx + q0 * (ROWW * 4));
        for (uint32_t e = g.t; e < P * ROWW; e += g.G) dst[e] = S.idx[e];
    } else {
        const uint64_t e0 = (uint64_t)k * n * P;
        for (uint32_t e = g.t; e < n * P; e += g.G) {
            if (ALGO == CAO_PSO) { rm.x[e0 + e] = S.x[e]; rm.v[e0 + e] = S.v[e]; rm.pb[e0 + e] = S.pb[e]; }
            else { const uint32_t d = e / P, j = e - d * P; rm.x[e0 + e] = S.x[j * n + d]; }
        }
    }
    if (g.t == 0) {
        const GrpShared* gs = S.gs;
        rm.uniq[k] = gs->uniq; rm.stagn[k] = gs->stagn;
        rm.best_f[k] = __uint_as_float((uint32_t)(gs->best >> 32)); rm.best_rank[k] = (uint32_t)gs->best;
        rm.gens_done[k] += gs->gens;
        if (gs->n_inv) atomicAdd(&rm.counters[0], (unsigned long long)gs->n_inv);
        if (gs->n_scan) atomicAdd(&rm.counters[1], (unsigned long long)gs->n_scan);
        if (gs->n_eval) atomicAdd(&rm.counters[2], (unsigned long long)gs->n_eval);
        if (gs->n_p2) atomicAdd(&rm.counters[3], (unsigned long long)gs->n_p2);
        if (gs->n_p3) atomicAdd(&rm.counters[4], (unsigned long long)gs->n_p3);
        if (gs->n_memo) atomicAdd(&rm.counters[5], (unsigned long long)gs->n_memo);
        if (gs->n_rc) atomicAdd(&rm.counters[6], (unsigned long long)gs->n_rc);
        for (int z = 0; z < 9; ++z) if (gs->hist[z]) atomicAdd(&rm.counters[16 + z], (unsigned long long)gs->hist[z]);
#ifdef CAO_GEN_STATS
        unsigned long long tot = 0;
        for (int z = 0; z < 6; ++z) { atomicAdd(&rm.counters[8 + z], gs->cyc[z]); tot += gs->cyc[z]; }
        atomicMax(&rm.counters[14], tot);                               // slowest run (cycles)
#ifdef CAO_GEN_STATS_PRINT
        if (tot > CAO_GEN_STATS_PRINT)
            printf("run %u cyc %llu: op %llu tail %llu p2 %llu p3 %llu scan %llu fin %llu | inv %u p2n %u p3n %u memo %u rc %u\n", k, tot,
                   gs->cyc[0], gs->cyc[1], gs->cyc[2], gs->cyc[3], gs->cyc[4], gs->cyc[5], gs->n_inv, gs->n_p2, gs->n_p3, gs->n_memo, gs->n_rc);
#endif
        atomicMax(&rm.counters[15], gs->cyc[4]);                        // most scan cycles in one run
#endif
    }
}

// ---------------------------------------------------------------------------------------------
// One generation `gen` of run k, state in shared memory.  last = write the parity taps of this generation.
// Dimension loops are runtime loops over bytes in shared memory (compact code: the kernel is bound by instruction
// issue and instruction fetch, not by memory).
template <int ALGO, int ROWW, bool WIDE>
__device__ __forceinline__ void generation(const Grp& g, const SpaceMeta& sm, const ProbeMeta& pm, const CtaTabs& tb,
                                           const RunsMeta& rm, GrpMem& S, uint32_t k, uint32_t gen, bool last) {
    constexpr int RB = ROWW * 4;
    const uint32_t i = g.t, P = rm.P, run = rm.first_run + k;
    const int n = sm.n;
    const bool has = i < P;
    GrpShared* gs = S.gs;
    uint8_t* cand8 = (uint8_t*)S.cand + (size_t)i * RB;                 // this thread's candidate row
    const uint8_t* idx8 = (const uint8_t*)S.idx;
    Draws dr(rm.seed, run, gen, i, S_OP);
    if (i == 0) { gs->n_new = 0; gs->nwl = 0; gs->aux = ~0ull; gs->flag = 0; }
#ifdef CAO_GEN_STATS
    long long t_mark = clock64();
#endif
    // memo of the previous generation: repair is a pure function of the row, so a candidate that repeats keeps its key
    uint64_t L = 0;
    bool same = has && S.key[has ? i : 0] != CAO_KEY_NONE;
#define PUT_DIM(d, ud)                                                                     \
    do {                                                                                   \
        const uint32_t ud_ = (ud);                                                         \
        same = same && cand8[d] == ud_;                                                    \
        cand8[d] = (uint8_t)ud_;                                                           \
        L += (uint64_t)ud_ * sm.stride[d];                                                 \
    } while (0)

    // ---- S3: operator
    if (ALGO == CAO_DE) {                                               // O5: best1bin on indices
        const uint32_t br = (uint32_t)gs->best;                         // best-so-far at generation start (A6)
        if (gs->bestrow_rank != br) {                                   // group-uniform
            g.sync();
            if (i < ROWW) S.bestrow[i] = ((const uint32_t*)(sm.rows + (uint64_t)br * RB))[i];
            if (i == 0) gs->bestrow_rank = br;
        }
        g.sync();
        if (has) {
            uint32_t a = below(dr(0), P - 1); if (a >= i) a += 1;
            uint32_t b = below(dr(1), P - 2);
            const uint32_t lo = min(i, a), hi = max(i, a);
            if (b >= lo) b += 1;
            if (b >= hi) b += 1;
            const uint32_t jrand = below(dr(2), (uint32_t)n);
            const uint8_t* ra = idx8 + (size_t)a * RB; const uint8_t* rb = idx8 + (size_t)b * RB;
            const uint8_t* rx = idx8 + (size_t)i * RB; const uint8_t* rbest = (const uint8_t*)S.bestrow;
#pragma unroll 2
            for (int d = 0; d < n; ++d) {
                const int vd = de_mutate_index(rm.hp.de_F, (int)rbest[d], (int)ra[d], (int)rb[d], (int)sm.m[d] - 1);
                const float rr = u01(dr(3 + d));
                PUT_DIM(d, (rr < rm.hp.de_CR || (uint32_t)d == jrand) ? (uint32_t)vd : (uint32_t)rx[d]);
            }
        }
    } else if (ALGO == CAO_GA) {                                        // O8: sorted population, Beta(1,b) parents, single point
        unsigned long long* s_key = (unsigned long long*)S.scr;         // P keys
        uint32_t* s_order = S.scr + 2 * P;                              // P
        g.sync();
        if (has) s_key[i] = ((unsigned long long)fbits(S.f[i]) << 32) | S.rank[i];
        g.sync();
        if (g.G == 32) {
            // One warp: position = keys below mine + equal keys in lower lanes (one MATCH for all the ties, so the loop
            // is a bare 64-bit less-than).  Equal keys are identical configurations: their order is immaterial anyway.
            const unsigned long long me = has ? s_key[i] : ~0ull - i;
            const uint32_t ties = __match_any_sync(0xFFFFFFFFu, me);
            if (has) {
                uint32_t pos = (uint32_t)__popc(ties & ((1u << i) - 1u));
                for (uint32_t j = 0; j < P; ++j) pos += s_key[j] < me;
                s_order[pos] = i;
            }
        } else if (has) {
            const unsigned long long me = s_key[i];
            uint32_t pos = 0;
            for (uint32_t j = 0; j < P; ++j) { const unsigned long long o = s_key[j]; pos += (o < me) || (o == me && j < i); }
            s_order[pos] = i;
        }
        g.sync();
        if (has) {
            const uint32_t B = (uint32_t)rm.hp.ga_beta_b;
            uint32_t sa = P, sb = P;
            for (uint32_t z = 0; z < B; ++z) sa = min(sa, below(dr(z), P));
            for (uint32_t z = 0; z < B; ++z) sb = min(sb, below(dr(B + z), P));
            if (sb == sa) sb = sa + 1 == P ? 0 : sa + 1;
            const int cut = n > 1 ? 1 + (int)below(dr(2 * B), (uint32_t)(n - 1)) : 1;
            // the child is assembled a word at a time (bytes below the cut from A, the rest from B), compared with last
            // generation's candidate and stored as words; only the linear index walks the dimensions
            const uint32_t* wa = S.idx + (size_t)s_order[sa] * ROWW; const uint32_t* wb = S.idx + (size_t)s_order[sb] * ROWW;
            uint32_t* cw = S.cand + (size_t)i * ROWW;
#pragma unroll
            for (int z = 0; z < ROWW; ++z) {
                const int nb_a = min(max(cut - 4 * z, 0), 4);                    // bytes of this word that come from A
                const uint32_t ma = nb_a >= 4 ? 0xFFFFFFFFu : ((1u << (8 * nb_a)) - 1u);
                const uint32_t cwz = (wa[z] & ma) | (wb[z] & ~ma);
                same = same && cw[z] == cwz;
                cw[z] = cwz;
            }
            for (int d = 0; d < n; ++d) L += (uint64_t)cand8[d] * tb.stride[d];
        }
        g.sync();                                                       // every parent row is read before the population is replaced
    } else if (ALGO == CAO_PSO) {                                       // O6
        g.sync();
        grp_min_key(g, has ? (((uint64_t)fbits(S.pbf[i]) << 32) | i) : ~0ull, &gs->aux);
        const uint32_t gb = (uint32_t)gs->aux;                          // gbest = pbest of argmin (pbest_f, i) at generation start
        if (has) {
            const float fM = (float)(sm.M - 1);
#pragma unroll 2
            for (int d = 0; d < n; ++d) {
                const uint32_t e = d * P + i;
                const float r1 = u01(dr(2 * d)), r2 = u01(dr(2 * d + 1));
                const float xq = S.x[e], pbq = S.pb[e], gbq = S.pb[d * P + gb];
                const float a = __fmul_rn(rm.hp.pso_c1, r1);
                const float b = __fsub_rn(pbq, xq);
                const float t1 = __fmul_rn(a, b);
                const float c = __fmul_rn(rm.hp.pso_c2, r2);
                const float ee = __fsub_rn(gbq, xq);
                const float t2 = __fmul_rn(c, ee);
                float vv = __fmul_rn(rm.hp.pso_w, S.v[e]);
                vv = __fadd_rn(vv, t1);
                vv = __fadd_rn(vv, t2);
                float xx = __fadd_rn(xq, vv);
                xx = clamp_pos(xx, tb.hi[d]);
                S.v[e] = vv; S.x[e] = xx;
                int kq = __float2int_rn(__fmul_rn(xx, fM));             // snap (O6, A11)
                kq = min(max(kq, 0), (int)sm.m[d] - 1);
                PUT_DIM(d, (uint32_t)kq);
            }
        }
    } else if (ROWW == 4 && WIDE) {                                     // O7: Firefly, FOUR LANES PER FIREFLY (underfilled GPU)
        // A lone warp per run is bound by the dependent chain r2 -> exp -> update of every attractor j.  Here lanes 4f..4f+3
        // share firefly f: lane `part` owns dimensions 4 part .. 4 part + 3, computes ONE Philox block per attractor instead
        // of five, and only the r2 sum is replicated: the 16 squared differences are gathered by shuffles and added in
        // dimension order, so every lane holds the oracle's r2 bit for bit.  The positions are exchanged through S.x.
        g.sync();
        const uint32_t ff = g.t >> 2, part = g.t & 3, lane_base = (g.t & 31u) & ~3u;
        const bool hasw = ff < P;
        float xi4[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) { const int d = (int)part * 4 + q; xi4[q] = (hasw && d < n) ? S.x[ff * n + d] : 0.0f; }
        const float fme = hasw ? S.f[ff] : 0.0f;
        for (uint32_t j = 0; j < P; ++j) {
            const bool brighter = hasw && S.f[j] < fme;
            if (!__any_sync(0xFFFFFFFFu, brighter)) continue;
            const float* xj = S.x + (size_t)j * n;
            float xj4[4], sq[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const int d = (int)part * 4 + q;
                xj4[q] = d < n ? xj[d] : 0.0f;
                const float df = __fsub_rn(xj4[q], xi4[q]);
                sq[q] = __fmul_rn(df, df);
            }
            // this lane's Philox block of the attractor's noise draws (slots j*n .. j*n+n-1); the next lane's block supplies
            // the words that spill over when the first slot is not block-aligned
            const uint32_t s0 = j * (uint32_t)n, o = s0 & 3;
            uint4 blk = philox4x32_10(make_uint4(run, gen, ff, (S_OP << 24) | ((s0 >> 2) + part)), (uint32_t)rm.seed, (uint32_t)(rm.seed >> 32));
            uint32_t nx = __shfl_down_sync(0xFFFFFFFFu, blk.x, 1), ny = __shfl_down_sync(0xFFFFFFFFu, blk.y, 1),
                     nz = __shfl_down_sync(0xFFFFFFFFu, blk.z, 1);
            if (o + (uint32_t)n > 16u) {                                // group-uniform: the last lane needs a fifth block
                if (part == 3) {
                    const uint4 b5 = philox4x32_10(make_uint4(run, gen, ff, (S_OP << 24) | ((s0 >> 2) + 4)), (uint32_t)rm.seed, (uint32_t)(rm.seed >> 32));
                    nx = b5.x; ny = b5.y; nz = b5.z;
                }
            }
            float r2 = 0.0f;                                            // sum over d = 0 .. 15 in order (padding adds +0)
#pragma unroll
            for (int pp = 0; pp < 4; ++pp)
#pragma unroll
                for (int q = 0; q < 4; ++q) r2 = __fadd_rn(r2, __shfl_sync(0xFFFFFFFFu, sq[q], lane_base + pp));
            const float beta = __fmul_rn(rm.hp.ff_B0, exp_neg_spec(__fmul_rn(rm.hp.ff_gamma, r2)));
            uint32_t w4[4];
            if (o == 0) { w4[0] = blk.x; w4[1] = blk.y; w4[2] = blk.z; w4[3] = blk.w; }
            else if (o == 1) { w4[0] = blk.y; w4[1] = blk.z; w4[2] = blk.w; w4[3] = nx; }
            else if (o == 2) { w4[0] = blk.z; w4[1] = blk.w; w4[2] = nx; w4[3] = ny; }
            else { w4[0] = blk.w; w4[1] = nx; w4[2] = ny; w4[3] = nz; }
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const int d = (int)part * 4 + q;
                const float df = __fsub_rn(xj4[q], xi4[q]);
                float tq = __fadd_rn(xi4[q], __fmul_rn(beta, df));
                const float e = __fsub_rn(u01(w4[q]), 0.5f);
                tq = __fadd_rn(tq, __fmul_rn(rm.hp.ff_alpha, e));
                xi4[q] = (brighter && d < n) ? tq : xi4[q];
            }
        }
        g.sync();                                                       // all start-of-generation positions are consumed
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int d = (int)part * 4 + q;
            if (hasw && d < n) S.x[ff * n + d] = clamp_pos(xi4[q], tb.hi[d]);
        }
        g.sync();
        if (has) {
            const float fM = (float)(sm.M - 1);
            for (int d = 0; d < n; ++d) {
                int kq = __float2int_rn(__fmul_rn(S.x[i * n + d], fM));
                kq = min(max(kq, 0), (int)sm.m[d] - 1);
                PUT_DIM(d, (uint32_t)kq);
            }
        }
    } else {                                                            // O7: Firefly (Yang's rule, synchronous)
        g.sync();
        float xi[RB];
        if (has) {
#pragma unroll
            for (int d = 0; d < RB; ++d) xi[d] = d < n ? S.x[i * n + d] : 0.0f;
        }
        const float fi = has ? S.f[i] : 0.0f;
        for (uint32_t j = 0; j < P; ++j) {
            const bool brighter = has && S.f[j] < fi;                   // only brighter (cheaper) fireflies attract
            if (!__any_sync(0xFFFFFFFFu, brighter)) continue;           // warp-uniform: draws are addressed by slot, skipping is free
            const float* xj = S.x + (size_t)j * n;
            // the n noise draws of this j are slots j*n .. j*n+n-1: all their Philox blocks at once (independent chains),
            // then one specialised update per alignment o = first slot & 3, so every word is a fixed register
            const uint32_t s0 = j * (uint32_t)n, o = s0 & 3;
            uint32_t nw[(ROWW + 1) * 4];
            {
                uint4 q5[ROWW + 1];
                if (ROWW == 4) {                                        // four blocks cover slots o .. o+15; the fifth only when o + n > 16
                    uint4 q4[4];
                    philox4x32_10_multi<4>(make_uint4(run, gen, i, (S_OP << 24) | (s0 >> 2)), (uint32_t)rm.seed, (uint32_t)(rm.seed >> 32), q4);
#pragma unroll
                    for (int z = 0; z < 4; ++z) q5[z] = q4[z];
                    q5[4] = make_uint4(0, 0, 0, 0);
                    if (o + (uint32_t)n > 16u)                          // warp-uniform
                        q5[4] = philox4x32_10(make_uint4(run, gen, i, (S_OP << 24) | ((s0 >> 2) + 4)), (uint32_t)rm.seed, (uint32_t)(rm.seed >> 32));
                } else {
                    uint4 qa[5], qb[4];
                    philox4x32_10_multi<5>(make_uint4(run, gen, i, (S_OP << 24) | (s0 >> 2)), (uint32_t)rm.seed, (uint32_t)(rm.seed >> 32), qa);
                    philox4x32_10_multi<4>(make_uint4(run, gen, i, (S_OP << 24) | ((s0 >> 2) + 5)), (uint32_t)rm.seed, (uint32_t)(rm.seed >> 32), qb);
#pragma unroll
                    for (int z = 0; z < 5; ++z) q5[z] = qa[z];
#pragma unroll
                    for (int z = 0; z < 4; ++z) q5[(5 + z) % (ROWW + 1)] = qb[z];
                }
#pragma unroll
                for (int z = 0; z < ROWW + 1; ++z) { nw[4 * z] = q5[z].x; nw[4 * z + 1] = q5[z].y; nw[4 * z + 2] = q5[z].z; nw[4 * z + 3] = q5[z].w; }
            }
            if (ROWW == 4) {
                // Narrow rows: all 16 dimension slots are computed unconditionally (straight-line code, xi in registers).  A
                // padding slot d >= n holds xj = xi = +0: it adds +0 to r2 (exact) and its update is discarded by the select.
                float xjv[RB];
#pragma unroll
                for (int d = 0; d < RB; ++d) xjv[d] = d < n ? xj[d] : 0.0f;
                float r2 = 0.0f;
#pragma unroll
                for (int d = 0; d < RB; ++d) { const float df = __fsub_rn(xjv[d], xi[d]); r2 = __fadd_rn(r2, __fmul_rn(df, df)); }
                const float beta = __fmul_rn(rm.hp.ff_B0, exp_neg_spec(__fmul_rn(rm.hp.ff_gamma, r2)));
#define FF_UPDATE_FLAT(O)                                                                    \
                _Pragma("unroll")                                                            \
                for (int d = 0; d < RB; ++d) {                                               \
                    const float df = __fsub_rn(xjv[d], xi[d]);                               \
                    float tq = __fadd_rn(xi[d], __fmul_rn(beta, df));                        \
                    const float e = __fsub_rn(u01(nw[d + (O)]), 0.5f);                       \
                    tq = __fadd_rn(tq, __fmul_rn(rm.hp.ff_alpha, e));                        \
                    xi[d] = (brighter && d < n) ? tq : xi[d];                                \
                }
                if (o == 0) { FF_UPDATE_FLAT(0) } else if (o == 1) { FF_UPDATE_FLAT(1) } else if (o == 2) { FF_UPDATE_FLAT(2) } else { FF_UPDATE_FLAT(3) }
#undef FF_UPDATE_FLAT
            } else {
                float r2 = 0.0f;
#pragma unroll
                for (int d = 0; d < RB; ++d)
                    if (d < n) { const float df = __fsub_rn(xj[d], xi[d]); r2 = __fadd_rn(r2, __fmul_rn(df, df)); }
                const float beta = __fmul_rn(rm.hp.ff_B0, exp_neg_spec(__fmul_rn(rm.hp.ff_gamma, r2)));
#define FF_UPDATE(O)                                                                         \
                _Pragma("unroll")                                                            \
                for (int d = 0; d < RB; ++d) {                                               \
                    if (d < n) {                                                             \
                        const float df = __fsub_rn(xj[d], xi[d]);                            \
                        float tq = __fadd_rn(xi[d], __fmul_rn(beta, df));                    \
                        const float e = __fsub_rn(u01(nw[d + (O)]), 0.5f);                   \
                        tq = __fadd_rn(tq, __fmul_rn(rm.hp.ff_alpha, e));                    \
                        xi[d] = brighter ? tq : xi[d];                                       \
                    }                                                                        \
                }
                if (o == 0) { FF_UPDATE(0) } else if (o == 1) { FF_UPDATE(1) } else if (o == 2) { FF_UPDATE(2) } else { FF_UPDATE(3) }
#undef FF_UPDATE
            }
        }
        g.sync();                                                       // all start-of-generation positions are consumed
        if (has) {
            const float fM = (float)(sm.M - 1);
#pragma unroll
            for (int d = 0; d < RB; ++d) {
                if (d < n) {
                    const float xx = clamp_pos(xi[d], tb.hi[d]);
                    S.x[i * n + d] = xx;
                    int kq = __float2int_rn(__fmul_rn(xx, fM));
                    kq = min(max(kq, 0), (int)sm.m[d] - 1);
                    PUT_DIM(d, (uint32_t)kq);
                }
            }
        }
    }
#undef PUT_DIM
    CAO_TICK(0);

    // ---- S4 + first part of S5: validity, warp-cooperative Hamming-1 probe, per-run repair cache
    uint64_t key = CAO_KEY_NONE;
    uint32_t valid = 0;
    if (has) {
        if (same) {
            key = S.key[i]; valid = (key >> 45) == 0;
        } else {
            const uint32_t rk0 = valid_rank(sm.bitmap, sm.dir, L, &valid);   // operator outputs are in-domain by construction
            if (valid) key = make_key(0, 0, rk0);
        }
    }
    const bool open = has && !same && !valid;
    if (pm.levels >= 1) {
        unsigned long long* hkey = (unsigned long long*)S.aux4;
        uint32_t* ol = S.scr;
        const uint32_t pos = grp_push(open, &gs->flag, g.G == 32);
        if (open) { ol[pos] = i; S.Lc[i] = L; hkey[i] = ~0ull; }
        g.sync();                                                       // candidate rows, list and linear indices are visible
        const uint32_t nopen = gs->flag;
        if (nopen) {
            probe_h1_flat<RB>(g, sm.bitmap, tb, (const uint8_t*)S.cand, ol, S.Lc, hkey, nopen);
            g.sync();
            if (open) {
                const uint32_t hit = (uint32_t)hkey[i];
                if (hit != 0xFFFFFFFFu) {
                    uint32_t dummy, sadv;
                    const uint64_t Lh = h1_decode(tb, hit, L, &sadv);
                    key = make_key(1u, sadv, valid_rank(sm.bitmap, sm.dir, Lh, &dummy));
                }
            }
        }
    }
    bool rc_hit = false;
    if (open && key == CAO_KEY_NONE) {                                  // memoised repairs of this run (L268 in spirit)
        const ulonglong2 e = rm.rcache[(uint64_t)k * CAO_RCACHE + rcache_slot(L)];
        if (e.x == L) { key = e.y; rc_hit = true; }
    }
    if (has && !same) S.key[i] = key;
    {
        const uint32_t pos = grp_push(has && key == CAO_KEY_NONE, &gs->nwl, g.G == 32);
        if (has && key == CAO_KEY_NONE) S.wl[pos] = i;
        const uint32_t ninv = __popc(__ballot_sync(0xFFFFFFFFu, has && !valid));
        const uint32_t nmemo = __popc(__ballot_sync(0xFFFFFFFFu, has && same && !valid));
        const uint32_t nrc = __popc(__ballot_sync(0xFFFFFFFFu, rc_hit));
        if ((i & 31) == 0) {
            if (g.G == 32) { gs->n_inv += ninv; gs->n_memo += nmemo; gs->n_rc += nrc; }
            else {
                if (ninv) atomicAdd(&gs->n_inv, ninv);
                if (nmemo) atomicAdd(&gs->n_memo, nmemo);
                if (nrc) atomicAdd(&gs->n_rc, nrc);
            }
        }
    }
    g.sync();
    CAO_TICK(1);

    // ---- rest of S5: the few unresolved candidates, by the whole group (Hamming-2/3 probes, then the table scan)
    const uint32_t nwl = gs->nwl;
    if (nwl) {
        uint32_t nscan = 0;
        if (pm.levels >= 2) {
            for (uint32_t fq = 0; fq < nwl; ++fq) {
                const uint32_t slot = S.wl[fq];
                const uint8_t* c = (const uint8_t*)S.cand + (size_t)slot * RB;
                if (i == 0) gs->aux = ~0ull;
                g.sync();
                const int found = probe_levels_grp(g, sm.bitmap, tb.stride, pm, tb.nb, tb.pairs, c, S.Lc[slot], S.ptab, &gs->aux);
                if (found == 2) CAO_TICK(2); else CAO_TICK(3);
                if (i == 0) {
                    gs->n_p2 += 1; gs->n_p3 += found != 2 && pm.levels >= 3;   // went to the Hamming-2 probe / beyond it
                    if (found) {
                        const uint64_t best = gs->aux;
                        uint32_t dummy;
                        const uint64_t kk = make_key((uint32_t)found, (uint32_t)(best >> 40),
                                                     valid_rank(sm.bitmap, sm.dir, best & ((1ull << 40) - 1), &dummy));
                        S.key[slot] = kk;
                        const uint64_t Lc = S.Lc[slot];
                        rm.rcache[(uint64_t)k * CAO_RCACHE + rcache_slot(Lc)] = make_ulonglong2(Lc, kk);
                    } else {
                        S.wl[nscan] = slot;                             // nscan <= fq: compacts in place
                    }
                }
                if (!found) ++nscan;
                g.sync();
            }
        } else {
            nscan = nwl;
        }
        for (uint32_t f0 = 0; f0 < nscan; f0 += GEN_NB) {
            const uint32_t nb = min((uint32_t)GEN_NB, nscan - f0);
            for (uint32_t e = i; e < nb * ROWW; e += g.G) S.cw[e] = S.cand[S.wl[f0 + e / ROWW] * ROWW + e % ROWW];
            if (i < GEN_NB) S.skey[i] = ~0ull;
            g.sync();
            scan_grp<ROWW, GEN_NB>(g, sm.rows, sm.V, S.cw, (int)nb, S.skey);
            if (i == 0) {                                               // one writer: cache entries are never torn
                for (uint32_t b = 0; b < nb; ++b) {
                    const uint64_t kk = S.skey[b];
                    S.key[S.wl[f0 + b]] = kk;
                    uint64_t Lc = 0;
                    for (int d = 0; d < n; ++d) Lc += (uint64_t)((const uint8_t*)(S.cw + b * ROWW))[d] * tb.stride[d];
                    rm.rcache[(uint64_t)k * CAO_RCACHE + rcache_slot(Lc)] = make_ulonglong2(Lc, kk);
                }
            }
            g.sync();
        }
        if (i == 0 && nscan) gs->n_scan += nscan;
        key = has ? S.key[i] : key;
        CAO_TICK(4);
    }

    {                                                                   // statistics: Hamming distance of every repair
        const uint32_t h = has ? min((uint32_t)(key >> 45), 8u) : 31u;
        const uint32_t peers = __match_any_sync(0xFFFFFFFFu, h);
        if (has && (i & 31) == (uint32_t)(__ffs(peers) - 1)) {
            if (g.G == 32) gs->hist[h] += (uint32_t)__popc(peers);      // distinct leaders write distinct entries
            else atomicAdd(&gs->hist[h], (uint32_t)__popc(peers));
        }
    }
    // ---- S6 + S7
    uint32_t rk = (uint32_t)key;
    const uint32_t rep = rk;
    float f = 0.0f; bool is_new = false;
    if (ALGO == CAO_GA) {                                               // L288: the children replace the population ...
        uint64_t Lr = 0;
        if (has) {
            uint32_t row[ROWW];
            load_row<ROWW>(sm.rows + (uint64_t)rk * RB, row);
            Lr = ltab_at(sm, rk);
#pragma unroll
            for (int z = 0; z < ROWW; ++z) S.idx[i * ROWW + z] = row[z];
        }
        // ... after the 1-in-X mutation into a uniformly drawn valid Hamming-1 neighbour (L290, L311, L393), listed in
        // (dimension ascending, value ascending) order = neighbour-list order.  All neighbours of all mutating children
        // are tested in one flat pass (bit masks in shared memory), then each child picks its own.
        Draws dm(rm.seed, run, gen, i, S_MUT);
        const bool mutate = has && below(dm(0), (uint32_t)rm.hp.ga_mutation_chance) == 0;
        uint64_t Lnew = ~0ull;
        const uint32_t MW = (tb.NB + 31) >> 5;                          // mask words per child
        if (MW <= 4) {
            uint32_t* ol = S.scr; uint32_t* mm = S.aux4;
            if (i == 0) gs->flag = 0;
            g.sync();
            const uint32_t pos = grp_push(mutate, &gs->flag, g.G == 32);
            if (mutate) {
                ol[pos] = i; S.Lc[i] = Lr;
                for (uint32_t w = 0; w < MW; ++w) mm[i * 4 + w] = 0;
            }
            g.sync();
            const uint32_t nmut = gs->flag, NB = tb.NB, total = nmut * NB;
            if (nmut) {
                uint32_t jj = g.t / NB, t = g.t - jj * NB;
                const uint32_t sj = g.G / NB, st = g.G - sj * NB;
                for (uint32_t q0 = g.t; q0 < total; q0 += 4 * g.G) {
                    uint32_t who[4], tt[4]; bool bit[4];
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const bool live = q0 + u * g.G < total;
                        const uint32_t i2 = ol[live ? jj : 0], tq = live ? t : 0, e = tb.nb[tq], d = e >> 8, kq = e & 255u;
                        const uint32_t cd = idx8[(size_t)i2 * RB + d];
                        const int dv = (int)(kq + (kq >= cd)) - (int)cd;
                        who[u] = i2; tt[u] = tq;
                        bit[u] = bit_test(sm.bitmap, S.Lc[i2] + (int64_t)dv * (int64_t)tb.stride[d]) && live;
                        t += st; jj += sj;
                        if (t >= NB) { t -= NB; ++jj; }
                    }
#pragma unroll
                    for (int u = 0; u < 4; ++u) if (bit[u]) atomicOr(&mm[who[u] * 4 + (tt[u] >> 5)], 1u << (tt[u] & 31));
                }
                g.sync();
                if (mutate) {
                    uint32_t K = 0;
                    for (uint32_t w = 0; w < MW; ++w) K += __popc(mm[i * 4 + w]);
                    if (K) {
                        uint32_t pick = below(dm(1), K), w = 0;
                        for (; w < MW; ++w) { const uint32_t c2 = __popc(mm[i * 4 + w]); if (pick < c2) break; pick -= c2; }
                        const uint32_t t2 = w * 32 + (uint32_t)kth_set_bit32(mm[i * 4 + w], pick);
                        const uint32_t e = tb.nb[t2], d = e >> 8, kq = e & 255u, cd = idx8[(size_t)i * RB + d];
                        const int dv = (int)(kq + (kq >= cd)) - (int)cd;
                        Lnew = Lr + (int64_t)dv * (int64_t)tb.stride[d];
                    }
                }
            }
        } else {                                                        // very wide spaces: one child at a time, two passes
            uint32_t todo = __ballot_sync(0xFFFFFFFFu, mutate);
            const uint32_t lane = i & 31;
            if (todo) __syncwarp();
            while (todo) {
                const int j = __ffs(todo) - 1;
                todo &= todo - 1;
                const uint64_t Lj = __shfl_sync(0xFFFFFFFFu, Lr, j);
                const uint8_t* c = idx8 + (size_t)((i & ~31u) + j) * RB;
                uint32_t K = 0;
                for (uint32_t t0 = 0; t0 < tb.NB; t0 += 32) {           // pass 1: count
                    const uint32_t t = t0 + lane;
                    bool bit = false;
                    if (t < tb.NB) {
                        const uint32_t e = tb.nb[t], d = e >> 8, kq = e & 255u, cd = c[d];
                        const int dv = (int)(kq + (kq >= cd)) - (int)cd;
                        bit = bit_test(sm.bitmap, Lj + (int64_t)dv * (int64_t)tb.stride[d]);
                    }
                    K += __popc(__ballot_sync(0xFFFFFFFFu, bit));
                }
                if (K) {
                    uint32_t pick = below(__shfl_sync(0xFFFFFFFFu, dm(1), j), K);
                    for (uint32_t t0 = 0; t0 < tb.NB; t0 += 32) {       // pass 2: the pick-th valid neighbour
                        const uint32_t t = t0 + lane;
                        bool bit = false; uint64_t Lp = 0;
                        if (t < tb.NB) {
                            const uint32_t e = tb.nb[t], d = e >> 8, kq = e & 255u, cd = c[d];
                            const int dv = (int)(kq + (kq >= cd)) - (int)cd;
                            Lp = Lj + (int64_t)dv * (int64_t)tb.stride[d];
                            bit = bit_test(sm.bitmap, Lp);
                        }
                        const uint32_t bal = __ballot_sync(0xFFFFFFFFu, bit);
                        const uint32_t cnt = __popc(bal);
                        if (pick < cnt) {
                            const int src = kth_set_bit32(bal, pick);
                            const uint64_t Lsel = __shfl_sync(0xFFFFFFFFu, Lp, src);
                            if ((int)lane == j) Lnew = Lsel;
                            break;
                        }
                        pick -= cnt;
                    }
                }
            }
        }
        if (has) {
            if (Lnew != ~0ull) {
                uint32_t dummy;
                rk = valid_rank(sm.bitmap, sm.dir, Lnew, &dummy);
                uint32_t row[ROWW];
                load_row<ROWW>(sm.rows + (uint64_t)rk * RB, row);
#pragma unroll
                for (int z = 0; z < ROWW; ++z) S.idx[i * ROWW + z] = row[z];
            }
            f = evaluate_v2(sm, rm, k, rk, is_new);
            S.f[i] = f; S.rank[i] = rk;
        }
        fold_eval(g, gs, has, is_new, f, rk);
    } else {
        uint32_t row[ROWW];
        if (has) {
            f = evaluate_v2(sm, rm, k, rk, is_new);
            if (ALGO == CAO_DE) load_row<ROWW>(sm.rows + (uint64_t)rk * RB, row);   // speculative: only accepted trials keep it
        }
        fold_eval(g, gs, has, is_new, f, rk);
        if (ALGO == CAO_DE) {                                           // Alg.1; A7
            uint32_t* s_u = S.scr;                                      // P trial ranks; S.rank = old ranks
            if (has) s_u[i] = rk;
            g.sync();
            bool acc = false;
            if (g.G == 32) {                                            // one warp: compare through shuffles, no divergence
                const uint32_t old = has ? S.rank[i] : 0xFFFFFFFFu;
                bool member = false;
                for (uint32_t j = 0; j < P; ++j) member |= __shfl_sync(0xFFFFFFFFu, old, j) == rk;
                const uint32_t twins = __match_any_sync(0xFFFFFFFFu, has ? rk : 0xFFFFFFFFu - i);   // lanes with the same trial
                acc = has && f <= S.f[i] && !member && (twins & ((1u << i) - 1u)) == 0;
            } else if (has) {
                acc = f <= S.f[i];
                for (uint32_t j = 0; j < P && acc; ++j) if (S.rank[j] == rk) acc = false;
                for (uint32_t j = 0; j < i && acc; ++j) if (s_u[j] == rk) acc = false;
            }
            const bool any = g.sync_or(acc);                            // barrier: all membership tests done before the updates
            if (acc) {
#pragma unroll
                for (int z = 0; z < ROWW; ++z) S.idx[i * ROWW + z] = row[z];
                S.f[i] = f; S.rank[i] = rk;
            }
            if (last && has) rm.accept[(uint64_t)k * P + i] = acc ? 1 : 0;
            // L266: nothing accepted in two consecutive generations -> re-initialise (evaluated in this step)
            const uint32_t st = any ? 0 : gs->stagn + 1;
            g.sync();
            if (st == 2) {
                reinit_de_grp<ROWW>(g, sm, rm, S, k, gen);
                if (i == 0) gs->n_eval += P;
            }
            if (i == 0) gs->stagn = st == 2 ? 0 : st;
        } else if (ALGO == CAO_PSO) {                                   // L282: repair affects the evaluation only
            if (has) {
                S.f[i] = f; S.rank[i] = rk;
                const bool acc = f < S.pbf[i];                          // strict (A13)
                if (acc) {
                    S.pbf[i] = f;
                    for (int d = 0; d < n; ++d) S.pb[d * P + i] = S.x[d * P + i];
                }
                if (last) rm.accept[(uint64_t)k * P + i] = acc ? 1 : 0;
            }
        } else {
            if (has) { S.f[i] = f; S.rank[i] = rk; }
        }
    }
    if (last && has) {                                                  // parity taps of the last stepped generation
        const uint64_t q = (uint64_t)k * P + i;
        uint4* dst = (uint4*)(rm.cand + q * RB);
        dst[0] = make_uint4(S.cand[i * ROWW], S.cand[i * ROWW + 1], S.cand[i * ROWW + 2], S.cand[i * ROWW + 3]);
        if (ROWW == 8) dst[1] = make_uint4(S.cand[i * ROWW + 4], S.cand[i * ROWW + 5], S.cand[i * ROWW + 6], S.cand[i * ROWW + 7]);
        rm.key[q] = key; rm.valid[q] = (key >> 45) == 0 ? 1 : 0; rm.rep_rank[q] = rep; rm.eval_rank[q] = rk; rm.tap_f[q] = f;
        if (ALGO == CAO_GA || ALGO == CAO_FIREFLY) rm.accept[q] = 0;
    }
    g.sync();
    CAO_TICK(5);
    if (i == 0) {                                                       // O10: trajectory row
        const uint32_t u = gs->uniq + gs->n_new;
        gs->uniq = u; gs->gens += 1; gs->n_eval += P;
        uint32_t* t = rm.traj + ((uint64_t)gen * rm.R + k) * 3;
        t[0] = (uint32_t)(gs->best >> 32); t[1] = (uint32_t)gs->best; t[2] = u;
    }
    g.sync();
}

// ---------------------------------------------------------------------------------------------
template <int ALGO, int ROWW, int MAXT, bool WIDE = false>
// Resident CTAs per SM (register budget), measured on the 10^5-run sweep: PSO and Firefly keep their per-dimension state and
// Philox chains in registers and run 8 % faster with 128 registers x 2 CTAs than with 80 x 3 (which spills ~140 bytes per
// thread); DE and GA are 8 % / 4 % faster with 3 CTAs.  64 registers x 4 CTAs lost everywhere (spills).
// WIDE (Firefly, four lanes per firefly, its own instantiation): the per-lane state is four dimensions and one Philox block, so
// it keeps the 3-CTA budget.
__global__ void __launch_bounds__(MAXT, MAXT == 256 ? (((ALGO == CAO_PSO || ALGO == CAO_FIREFLY) && !WIDE) ? 2 : 3) : 1)
k_gen(const __grid_constant__ SpaceMeta sm, const __grid_constant__ ProbeMeta pm, const __grid_constant__ RunsMeta rm,
      const __grid_constant__ GenLayout lay, uint32_t g_first, uint32_t n_gens) {
    extern __shared__ __align__(16) uint32_t s_dyn[];
    // CTA-wide tables: strides, upper coordinates, Hamming-1 neighbour list, and (when they fit) the probe target / pair lists
    CtaTabs tb;
    {
        uint64_t* s_stride = (uint64_t*)s_dyn;                          // CAO_MAX_DIMS
        float* s_hi = (float*)(s_dyn + 2 * CAO_MAX_DIMS);               // CAO_MAX_DIMS
        uint16_t* s_nb = (uint16_t*)(s_dyn + 3 * CAO_MAX_DIMS);         // lay.nb_words words
        uint32_t* s_pairs = s_dyn + 3 * CAO_MAX_DIMS + lay.nb_words;
        if (threadIdx.x < (uint32_t)sm.n) {
            const uint32_t d = threadIdx.x;
            s_stride[d] = sm.stride[d];
            s_hi[d] = coord_M(sm.M, (int)sm.m[d] - 1);
            uint32_t off = 0;
            for (uint32_t e = 0; e < d; ++e) off += sm.m[e] - 1u;
            for (uint32_t kq = 0; kq + 1 < sm.m[d]; ++kq) s_nb[off + kq] = (uint16_t)(d << 8 | kq);
        }
        tb.nb = s_nb; tb.stride = s_stride; tb.hi = s_hi; tb.NB = lay.NB;
        tb.pairs = pm.pairs;
        if (lay.probe_in_smem) {
            for (uint32_t e = threadIdx.x; e < pm.C2; e += blockDim.x) s_pairs[e] = __ldg(&pm.pairs[e]);
            tb.pairs = s_pairs;
        }
        __syncthreads();
    }
    const Grp g{threadIdx.x % lay.G, lay.G, threadIdx.x / lay.G};
    GrpMem S(s_dyn + lay.cta_words + g.id * lay.words, lay);
    GrpShared* gs = S.gs;
    const uint32_t g_last = g_first + n_gens;
    for (;;) {
        if (g.t == 0) gs->run = atomicAdd(rm.ticket, 1u);
        g.sync();
        const uint32_t k = gs->run;
        if (k >= rm.R) break;
        load_state<ALGO, ROWW>(g, sm, rm, S, k);
        uint32_t gen = g_first + 1;
#pragma unroll 1
        for (; gen <= g_last; ++gen) {
            const bool active = rm.budget == 0 || gs->uniq < rm.budget;  // O10 (gen <= max_gens is enforced by the host)
            if (!active) break;
            generation<ALGO, ROWW, WIDE>(g, sm, pm, tb, rm, S, k, gen, gen == g_last);
        }
        // a run that reached its budget stays frozen: its trajectory row repeats (O10)
        for (uint32_t q = gen + g.t; q <= g_last; q += g.G) {
            uint32_t* t = rm.traj + ((uint64_t)q * rm.R + k) * 3;
            t[0] = (uint32_t)(gs->best >> 32); t[1] = (uint32_t)gs->best; t[2] = gs->uniq;
        }
        if (g.t == 0) rm.active[k] = gen > g_last ? 1 : 0;               // was the last stepped generation executed?
        store_state<ALGO, ROWW>(g, sm, rm, S, k);
        g.sync();
    }
    // the last group to leave re-arms the ticket counter for the next launch
    if (g.t == 0) {
        __threadfence();
        const uint32_t d = atomicAdd(rm.ticket + 1, 1u);
        if (d + 1 == gridDim.x * lay.NG) { atomicExch(rm.ticket + 1, 0u); atomicExch(rm.ticket, 0u); }
    }
}

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
    uint32_t n_inv, n_scan, n_eval, pad;
};
static_assert(sizeof(GrpShared) == GRP_SHARED_WORDS * 4, "GrpShared layout");

struct Grp {
    uint32_t t, G, id;               // thread within the group, group size, group within the CTA
    __device__ __forceinline__ void sync() const {
        if (G == 32) __syncwarp();
        else asm volatile("bar.sync %0, %1;" ::"r"(id + 1), "r"(G) : "memory");
    }
    __device__ __forceinline__ bool sync_or(bool p) const {
        if (G == 32) return __any_sync(0xFFFFFFFFu, p);
        uint32_t r;
        asm volatile("{\n\t.reg .pred p, q;\n\tsetp.ne.u32 p, %1, 0;\n\tbar.red.or.pred q, %2, %3, p;\n\tselp.u32 %0, 1, 0, q;\n\t}"
                     : "=r"(r) : "r"((uint32_t)p), "r"(id + 1), "r"(G) : "memory");
        return r != 0;
    }
};

// Minimum of a 64-bit key over the warp: two REDUX on the halves (the high half decides, then the low half among the
// lanes that hold the minimal high half).
__device__ __forceinline__ uint64_t warp_min_key(uint64_t v) {
    const uint32_t hi = (uint32_t)(v >> 32), lo = (uint32_t)v;
    const uint32_t mh = __reduce_min_sync(0xFFFFFFFFu, hi);
    const uint32_t ml = __reduce_min_sync(0xFFFFFFFFu, hi == mh ? lo : 0xFFFFFFFFu);
    return ((uint64_t)mh << 32) | ml;
}
// Group-wide minimum into *slot (which must hold ~0 / a running minimum visible to the group); ends with a barrier.
__device__ __forceinline__ void grp_min_key(const Grp& g, uint64_t v, unsigned long long* slot) {
    const uint64_t m = warp_min_key(v);
    if ((g.t & 31) == 0 && m != ~0ull) atomicMin(slot, (unsigned long long)m);
    g.sync();
}

// Validity and rank of linear index L in ONE round trip: the directory entry and the 64-byte bitmap block of L are
// loaded together; the rank is only meaningful when the bit is set.
__device__ __forceinline__ uint32_t valid_rank(const SpaceMeta& sm, uint64_t L, bool& valid) {
    const uint32_t wi = (uint32_t)(L >> 6) & 7u;
    const ulonglong2* blk = (const ulonglong2*)(sm.bitmap + ((L >> 6) & ~7ull));
    uint32_t r = __ldg(&sm.dir[L >> CAO_DIR_SHIFT]);
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
    valid = (mine >> (L & 63)) & 1ull;
    return r;
}

// Hamming-1 probe of an invalid in-domain row (exact: Hamming is the primary key, |delta| the secondary, L the third):
// level |delta| = 1, 2, ... until a level has a valid neighbour.  All bit tests of a level are independent loads.
template <int ROWW>
__device__ __forceinline__ uint64_t probe_h1_v2(const SpaceMeta& sm, const uint32_t (&w)[ROWW], uint64_t L) {
    for (int delta = 1; delta < sm.M; ++delta) {
        uint64_t bestL = ~0ull;
        if (delta <= 2) {
            uint64_t cand[ROWW * 8];
            bool hit[ROWW * 8];
#pragma unroll
            for (int d = 0; d < ROWW * 4; ++d) {
                const int c = (int)ROW_BYTE(w, d);
                const uint64_t step = d < sm.n ? (uint64_t)delta * sm.stride[d] : 0;
                const bool okm = d < sm.n && c >= delta, okp = d < sm.n && c + delta < (int)sm.m[d];
                cand[2 * d] = okm ? L - step : L;  cand[2 * d + 1] = okp ? L + step : L;
                hit[2 * d] = okm;                  hit[2 * d + 1] = okp;
            }
#pragma unroll
            for (int e = 0; e < ROWW * 8; ++e) hit[e] = hit[e] && bit_test(sm.bitmap, cand[e]);
#pragma unroll
            for (int e = 0; e < ROWW * 8; ++e) if (hit[e] && cand[e] < bestL) bestL = cand[e];
        } else {                                                        // few dimensions are this wide
            for (int d = 0; d < sm.n; ++d) {
                if ((int)sm.m[d] <= delta) continue;
                const int c = (int)ROW_BYTE(w, d);
                const uint64_t step = (uint64_t)delta * sm.stride[d];
                if (c >= delta && bit_test(sm.bitmap, L - step) && L - step < bestL) bestL = L - step;
                if (c + delta < (int)sm.m[d] && bit_test(sm.bitmap, L + step) && L + step < bestL) bestL = L + step;
            }
        }
        if (bestL != ~0ull) return make_key(1u, (uint32_t)delta, rank_of(sm, bestL));
    }
    return CAO_KEY_NONE;
}

// ---------------------------------------------------------------------------------------------
// Group-cooperative Hamming-2/3 probe of ONE candidate (row in shared memory, s_cw).  *slot must be ~0 and visible to
// the group on entry.  Returns the level that found a valid neighbour (0 = none), group-uniform, and leaves
// (sad << 40 | L') in *slot.  tgt / pairs may point to shared or global memory.
template <int ROWW>
__device__ __forceinline__ int probe23_grp(const Grp& g, const SpaceMeta& sm, const ProbeMeta& pm, const uint16_t* tgt,
                                           const uint32_t* pairs, const uint32_t* s_cw, unsigned long long* slot) {
    const uint8_t* c = (const uint8_t*)s_cw;
    const uint32_t T = pm.T, C2 = pm.C2;
    uint64_t L = 0;
    for (int d = 0; d < sm.n; ++d) L += (uint64_t)c[d] * sm.stride[d];
    for (int level = 2; level <= pm.levels; ++level) {
        uint64_t best = ~0ull;
        for (uint32_t q = g.t; q < C2; q += g.G) {
            const uint32_t pr = pairs[q];
            const uint32_t e1 = tgt[pr & 0xFFFFu], e2 = tgt[pr >> 16];
            const uint32_t d1 = e1 >> 8, d2 = e2 >> 8;
            const int dv1 = (int)(e1 & 255) - (int)c[d1], dv2 = (int)(e2 & 255) - (int)c[d2];
            if (dv1 == 0 || dv2 == 0) continue;
            const uint64_t L2 = L + (int64_t)dv1 * (int64_t)sm.stride[d1] + (int64_t)dv2 * (int64_t)sm.stride[d2];
            const uint32_t s2 = (uint32_t)(abs(dv1) + abs(dv2));
            if (level == 2) {
                if (bit_test(sm.bitmap, L2)) { uint64_t k = ((uint64_t)s2 << 40) | L2; best = k < best ? k : best; }
            } else {
#pragma unroll 8
                for (uint32_t t3 = pm.dim_first[d2 + 1]; t3 < T; ++t3) {
                    const uint32_t e3 = tgt[t3], d3 = e3 >> 8;
                    const int dv3 = (int)(e3 & 255) - (int)c[d3];
                    const uint64_t L3 = L2 + (int64_t)dv3 * (int64_t)sm.stride[d3];
                    const bool bit3 = bit_test(sm.bitmap, L3);              // unconditional: dv3 == 0 re-reads L2 (a legal index)
                    if (dv3 != 0 && bit3) { uint64_t k = ((uint64_t)(s2 + (uint32_t)abs(dv3)) << 40) | L3; best = k < best ? k : best; }
                }
            }
        }
        grp_min_key(g, best, slot);                                     // barrier inside
        const bool found = *slot != ~0ull;
        g.sync();                                                       // everyone has read the slot before the next level writes it
        if (found) return level;
    }
    return 0;
}

// Group-cooperative brute-force scan of the whole valid table for up to NB candidates (rows in shared memory); the
// table rows come straight from L2, coalesced, RU rows in flight per thread.  s_key[b] must be ~0 on entry; on exit it
// holds ham << 45 | sad << 32 | rank.  Ends with a barrier.
template <int ROWW, int NB>
__device__ __forceinline__ void scan_grp(const Grp& g, const SpaceMeta& sm, const uint32_t* s_cw, int nb, unsigned long long* s_key) {
    uint32_t c[NB][ROWW];
#pragma unroll
    for (int b = 0; b < NB; ++b)
#pragma unroll
        for (int k = 0; k < ROWW; ++k) c[b][k] = b < nb ? s_cw[b * ROWW + k] : 0;
    uint64_t best[NB];
#pragma unroll
    for (int b = 0; b < NB; ++b) best[b] = ~0ull;
    constexpr int RU = ROWW == 4 ? 8 : 4;
    for (uint32_t r0 = g.t; r0 < sm.V; r0 += RU * g.G) {
        uint32_t v[RU][ROWW];
#pragma unroll
        for (int u = 0; u < RU; ++u) {
            const uint32_t r = r0 + u * g.G;
            load_row<ROWW>(sm.rows + (uint64_t)(r < sm.V ? r : r0) * (ROWW * 4), v[u]);
        }
#pragma unroll
        for (int u = 0; u < RU; ++u) {
            const uint32_t r = r0 + u * g.G;
            if (r >= sm.V) break;
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
    uint32_t* bestrow;
    __device__ __forceinline__ GrpMem(uint32_t* S, const GenLayout& l)
        : gs((GrpShared*)S), rank(S + l.rank), f((float*)(S + l.f)), idx(S + l.idx), x((float*)(S + l.x)), v((float*)(S + l.v)),
          pb((float*)(S + l.pb)), pbf((float*)(S + l.pbf)), cand(S + l.cand), key((unsigned long long*)(S + l.key)),
          scr(S + l.scr), wl(S + l.wl), cw(S + l.cw), skey((unsigned long long*)(S + l.skey)), bestrow(S + l.bestrow) {}
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
        if (nn) atomicAdd(&gs->n_new, nn);
        if (m != ~0ull) atomicMin(&gs->best, (unsigned long long)m);
    }
}

// O4 inside the fused kernel (DE stagnation re-initialisation, L266): P distinct valid ranks, uniform with linear
// probing; fills the shared-memory population and evaluates it.  Group-uniform call, ends with a barrier.
template <int ROWW>
__device__ void reinit_de_grp(const Grp& g, const SpaceMeta& sm, const RunsMeta& rm, GrpMem& S, uint32_t k, uint32_t gen) {
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
    }
}

// ---------------------------------------------------------------------------------------------
// One generation g of run k, state in shared memory.  last = write the parity taps of this generation.
template <int ALGO, int ROWW>
__device__ __forceinline__ void generation(const Grp& g, const SpaceMeta& sm, const ProbeMeta& pm, const uint16_t* tgt,
                                           const uint32_t* pairs, const RunsMeta& rm, GrpMem& S, uint32_t k, uint32_t gen, bool last) {
    const uint32_t i = g.t, P = rm.P, run = rm.first_run + k;
    const int n = sm.n;
    GrpShared* gs = S.gs;
    uint32_t w[ROWW];
#pragma unroll
    for (int z = 0; z < ROWW; ++z) w[z] = 0;
    Draws dr(rm.seed, run, gen, i, S_OP);
    if (i == 0) { gs->n_new = 0; gs->nwl = 0; gs->aux = ~0ull; }

    // ---- S3: operator
    if (ALGO == CAO_DE) {                                               // O5: best1bin on indices
        const uint32_t br = (uint32_t)gs->best;                         // best-so-far at generation start (A6)
        if (gs->bestrow_rank != br) {                                   // group-uniform
            g.sync();
            if (i < ROWW) S.bestrow[i] = ((const uint32_t*)(sm.rows + (uint64_t)br * (ROWW * 4)))[i];
            if (i == 0) gs->bestrow_rank = br;
        }
        g.sync();
        if (i < P) {
            uint32_t a = below(dr(0), P - 1); if (a >= i) a += 1;
            uint32_t b = below(dr(1), P - 2);
            const uint32_t lo = min(i, a), hi = max(i, a);
            if (b >= lo) b += 1;
            if (b >= hi) b += 1;
            const uint32_t jrand = below(dr(2), (uint32_t)n);
            uint32_t wa[ROWW], wb[ROWW], wx[ROWW], wbest[ROWW];
#pragma unroll
            for (int z = 0; z < ROWW; ++z) { wa[z] = S.idx[a * ROWW + z]; wb[z] = S.idx[b * ROWW + z]; wx[z] = S.idx[i * ROWW + z]; wbest[z] = S.bestrow[z]; }
#pragma unroll
            for (int d = 0; d < ROWW * 4; ++d) {
                if (d < n) {
                    const int vd = de_mutate_index(rm.hp.de_F, (int)ROW_BYTE(wbest, d), (int)ROW_BYTE(wa, d), (int)ROW_BYTE(wb, d),
                                                   (int)sm.m[d] - 1);
                    const float rr = u01(dr(3 + d));
                    const uint32_t ud = (rr < rm.hp.de_CR || (uint32_t)d == jrand) ? (uint32_t)vd : ROW_BYTE(wx, d);
                    w[d >> 2] |= ud << ((d & 3) * 8);
                }
            }
        }
    } else if (ALGO == CAO_GA) {                                        // O8: sorted population, Beta(1,b) parents, single point
        unsigned long long* s_key = (unsigned long long*)S.scr;         // P keys
        uint32_t* s_order = S.scr + 2 * P;                              // P
        g.sync();
        if (i < P) s_key[i] = ((unsigned long long)fbits(S.f[i]) << 32) | S.rank[i];
        g.sync();
        if (i < P) {
            const unsigned long long me = s_key[i];
            uint32_t pos = 0;
            for (uint32_t j = 0; j < P; ++j) { const unsigned long long o = s_key[j]; pos += (o < me) || (o == me && j < i); }
            s_order[pos] = i;
        }
        g.sync();
        if (i < P) {
            const uint32_t B = (uint32_t)rm.hp.ga_beta_b;
            uint32_t sa = P, sb = P;
            for (uint32_t z = 0; z < B; ++z) sa = min(sa, below(dr(z), P));
            for (uint32_t z = 0; z < B; ++z) sb = min(sb, below(dr(B + z), P));
            if (sb == sa) sb = sa + 1 == P ? 0 : sa + 1;
            const int cut = n > 1 ? 1 + (int)below(dr(2 * B), (uint32_t)(n - 1)) : 1;
            const uint32_t pa = s_order[sa], pbq = s_order[sb];
            uint32_t wa[ROWW], wb[ROWW];
#pragma unroll
            for (int z = 0; z < ROWW; ++z) { wa[z] = S.idx[pa * ROWW + z]; wb[z] = S.idx[pbq * ROWW + z]; }
#pragma unroll
            for (int d = 0; d < ROWW * 4; ++d)
                if (d < n) w[d >> 2] |= (d < cut ? ROW_BYTE(wa, d) : ROW_BYTE(wb, d)) << ((d & 3) * 8);
        }
        g.sync();                                                       // every parent row is read before the population is replaced
    } else if (ALGO == CAO_PSO) {                                       // O6
        g.sync();
        grp_min_key(g, i < P ? (((uint64_t)fbits(S.pbf[i]) << 32) | i) : ~0ull, &gs->aux);
        const uint32_t gb = (uint32_t)gs->aux;
        float gbest[ROWW * 4];
#pragma unroll
        for (int d = 0; d < ROWW * 4; ++d) gbest[d] = d < n ? S.pb[d * P + gb] : 0.0f;
        g.sync();                                                       // gbest is read before any pbest moves (finish phase)
        if (i < P) {
#pragma unroll
            for (int d = 0; d < ROWW * 4; ++d) {
                if (d < n) {
                    const uint32_t e = d * P + i;
                    const float hi = coord_M(sm.M, (int)sm.m[d] - 1);
                    const float r1 = u01(dr(2 * d)), r2 = u01(dr(2 * d + 1));
                    const float xq = S.x[e], pbq = S.pb[e];
                    const float a = __fmul_rn(rm.hp.pso_c1, r1);
                    const float b = __fsub_rn(pbq, xq);
                    const float t1 = __fmul_rn(a, b);
                    const float c = __fmul_rn(rm.hp.pso_c2, r2);
                    const float ee = __fsub_rn(gbest[d], xq);
                    const float t2 = __fmul_rn(c, ee);
                    float vv = __fmul_rn(rm.hp.pso_w, S.v[e]);
                    vv = __fadd_rn(vv, t1);
                    vv = __fadd_rn(vv, t2);
                    float xx = __fadd_rn(xq, vv);
                    xx = clamp_pos(xx, hi);
                    S.v[e] = vv; S.x[e] = xx;
                    w[d >> 2] |= (uint32_t)snap_M(sm.M, (int)sm.m[d], xx) << ((d & 3) * 8);
                }
            }
        }
    } else {                                                            // O7: Firefly (Yang's rule, synchronous)
        g.sync();
        float xi[ROWW * 4];
        if (i < P) {
#pragma unroll
            for (int d = 0; d < ROWW * 4; ++d) xi[d] = d < n ? S.x[i * n + d] : 0.0f;
            const float fi = S.f[i];
            for (uint32_t j = 0; j < P; ++j) {
                if (!(S.f[j] < fi)) continue;                           // only brighter (cheaper) fireflies attract
                const float* xj = S.x + (size_t)j * n;
                float r2 = 0.0f;
#pragma unroll
                for (int d = 0; d < ROWW * 4; ++d)
                    if (d < n) { const float df = __fsub_rn(xj[d], xi[d]); r2 = __fadd_rn(r2, __fmul_rn(df, df)); }
                const float beta = __fmul_rn(rm.hp.ff_B0, exp_neg_spec(__fmul_rn(rm.hp.ff_gamma, r2)));
                // the n noise draws of this j are slots j*n .. j*n+n-1: their Philox blocks are computed up front as
                // independent chains, then word (o + d) is picked with selects (o = first slot & 3)
                const uint32_t s0 = j * (uint32_t)n, b0 = s0 >> 2, o = s0 & 3;
                uint32_t nw[(ROWW + 1) * 4];
#pragma unroll
                for (int qb = 0; qb < ROWW + 1; ++qb) {
                    uint4 rr = make_uint4(0, 0, 0, 0);
                    if ((uint32_t)(qb * 4) < o + (uint32_t)n)
                        rr = philox4x32_10(make_uint4(run, gen, i, (S_OP << 24) | (b0 + qb)), (uint32_t)rm.seed, (uint32_t)(rm.seed >> 32));
                    nw[qb * 4] = rr.x; nw[qb * 4 + 1] = rr.y; nw[qb * 4 + 2] = rr.z; nw[qb * 4 + 3] = rr.w;
                }
#pragma unroll
                for (int d = 0; d < ROWW * 4; ++d) {
                    if (d < n) {
                        const uint32_t lo = (o & 1) ? nw[d + 1] : nw[d], hi = (o & 1) ? nw[d + 3] : nw[d + 2];
                        const uint32_t word = (o & 2) ? hi : lo;
                        const float df = __fsub_rn(xj[d], xi[d]);
                        xi[d] = __fadd_rn(xi[d], __fmul_rn(beta, df));
                        const float e = __fsub_rn(u01(word), 0.5f);
                        xi[d] = __fadd_rn(xi[d], __fmul_rn(rm.hp.ff_alpha, e));
                    }
                }
            }
#pragma unroll
            for (int d = 0; d < ROWW * 4; ++d) {
                if (d < n) {
                    xi[d] = clamp_pos(xi[d], coord_M(sm.M, (int)sm.m[d] - 1));
                    w[d >> 2] |= (uint32_t)snap_M(sm.M, (int)sm.m[d], xi[d]) << ((d & 3) * 8);
                }
            }
        }
        g.sync();                                                       // all start-of-generation positions are consumed
        if (i < P) {
#pragma unroll
            for (int d = 0; d < ROWW * 4; ++d) if (d < n) S.x[i * n + d] = xi[d];
        }
    }

    // ---- S4 + first part of S5: memo of the previous generation, validity, Hamming-1 probe, per-run repair cache
    uint64_t key = CAO_KEY_NONE;
    bool valid = false;
    uint64_t L = 0;
    if (i < P) {
        const uint64_t prev_key = S.key[i];
        bool same = prev_key != CAO_KEY_NONE;
#pragma unroll
        for (int z = 0; z < ROWW; ++z) same = same && S.cand[i * ROWW + z] == w[z];
        if (same) {
            key = prev_key; valid = (key >> 45) == 0;
        } else {
#pragma unroll
            for (int z = 0; z < ROWW; ++z) S.cand[i * ROWW + z] = w[z];
            L = row_lin<ROWW>(sm, w);                                   // operator outputs are in-domain by construction
            const uint32_t rk0 = valid_rank(sm, L, valid);
            if (valid) key = make_key(0, 0, rk0);
            else {
                if (pm.levels >= 1) key = probe_h1_v2<ROWW>(sm, w, L);
                if (key == CAO_KEY_NONE) {                              // memoised repairs of this run (L268 in spirit)
                    const ulonglong2 e = rm.rcache[(uint64_t)k * CAO_RCACHE + rcache_slot(L)];
                    if (e.x == L) key = e.y;
                }
            }
            S.key[i] = key;
        }
        if (key == CAO_KEY_NONE) S.wl[atomicAdd(&gs->nwl, 1u)] = i;
    }
    {
        const uint32_t ninv = __popc(__ballot_sync(0xFFFFFFFFu, i < P && !valid));
        if ((i & 31) == 0 && ninv) atomicAdd(&gs->n_inv, ninv);
    }
    g.sync();

    // ---- rest of S5: the few unresolved candidates, by the whole group (Hamming-2/3 probes, then the table scan)
    const uint32_t nwl = gs->nwl;
    if (nwl) {
        uint32_t nscan = 0;
        if (pm.levels >= 2) {
            for (uint32_t fq = 0; fq < nwl; ++fq) {
                const uint32_t slot = S.wl[fq];
                if (i < ROWW) S.cw[i] = S.cand[slot * ROWW + i];
                if (i == 0) gs->aux = ~0ull;
                g.sync();
                const int found = probe23_grp<ROWW>(g, sm, pm, tgt, pairs, S.cw, &gs->aux);
                if (i == 0) {
                    if (found) {
                        const uint64_t best = gs->aux;
                        const uint64_t kk = make_key((uint32_t)found, (uint32_t)(best >> 40), rank_of(sm, best & ((1ull << 40) - 1)));
                        S.key[slot] = kk;
                        uint64_t Lc = 0;
                        for (int d = 0; d < n; ++d) Lc += (uint64_t)((const uint8_t*)S.cw)[d] * sm.stride[d];
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
            if (nb == 1) scan_grp<ROWW, 1>(g, sm, S.cw, 1, S.skey);
            else scan_grp<ROWW, GEN_NB>(g, sm, S.cw, (int)nb, S.skey);
            if (i == 0) {                                               // one writer: cache entries are never torn
                for (uint32_t b = 0; b < nb; ++b) {
                    const uint64_t kk = S.skey[b];
                    S.key[S.wl[f0 + b]] = kk;
                    uint64_t Lc = 0;
                    for (int d = 0; d < n; ++d) Lc += (uint64_t)((const uint8_t*)(S.cw + b * ROWW))[d] * sm.stride[d];
                    rm.rcache[(uint64_t)k * CAO_RCACHE + rcache_slot(Lc)] = make_ulonglong2(Lc, kk);
                }
            }
            g.sync();
        }
        if (i == 0 && nscan) gs->n_scan += nscan;
        key = i < P ? S.key[i] : key;
    }

    // ---- S6 + S7
    uint32_t rk = (uint32_t)key;
    const uint32_t rep = rk;
    float f = 0.0f; bool is_new = false;
    uint32_t row[ROWW];
    if (i < P) {
        if (ALGO == CAO_GA) {                                           // L290, L311, L393: 1-in-X mutation after repair
            Draws dm(rm.seed, run, gen, i, S_MUT);
            if (below(dm(0), (uint32_t)rm.hp.ga_mutation_chance) == 0) {
                uint32_t cur[ROWW];
                load_row<ROWW>(sm.rows + (uint64_t)rk * (ROWW * 4), cur);
                const uint64_t Lr = row_lin<ROWW>(sm, cur);
                uint32_t K = 0;                                         // valid Hamming-1 neighbours, (d asc, value asc)
#pragma unroll
                for (int d = 0; d < ROWW * 4; ++d) {
                    if (d < n) {
                        const int c = (int)ROW_BYTE(cur, d);
                        for (int val = 0; val < (int)sm.m[d]; ++val)
                            if (val != c && bit_test(sm.bitmap, Lr + (int64_t)(val - c) * (int64_t)sm.stride[d])) ++K;
                    }
                }
                if (K) {
                    const uint32_t pick = below(dm(1), K); uint32_t seen = 0;
                    uint64_t Lp = Lr; bool done = false;
#pragma unroll
                    for (int d = 0; d < ROWW * 4; ++d) {
                        if (d < n && !done) {
                            const int c = (int)ROW_BYTE(cur, d);
                            for (int val = 0; val < (int)sm.m[d] && !done; ++val) {
                                if (val == c) continue;
                                const uint64_t L2 = Lr + (int64_t)(val - c) * (int64_t)sm.stride[d];
                                if (bit_test(sm.bitmap, L2)) { if (seen == pick) { Lp = L2; done = true; } ++seen; }
                            }
                        }
                    }
                    rk = rank_of(sm, Lp);
                }
            }
        }
        f = evaluate_v2(sm, rm, k, rk, is_new);
        if (ALGO == CAO_DE || ALGO == CAO_GA) load_row<ROWW>(sm.rows + (uint64_t)rk * (ROWW * 4), row);   // speculative for DE
    }
    fold_eval(g, gs, i < P, is_new, f, rk);

    bool acc = false;
    if (ALGO == CAO_DE) {                                               // Alg.1; A7
        uint32_t* s_u = S.scr;                                          // P trial ranks; S.rank = old ranks
        if (i < P) s_u[i] = rk;
        g.sync();
        if (i < P) {
            acc = f <= S.f[i];
            for (uint32_t j = 0; j < P && acc; ++j) if (S.rank[j] == rk) acc = false;
            for (uint32_t j = 0; j < i && acc; ++j) if (s_u[j] == rk) acc = false;
        }
        const bool any = g.sync_or(acc);                                // barrier: all membership tests done before the updates
        if (acc) {
#pragma unroll
            for (int z = 0; z < ROWW; ++z) S.idx[i * ROWW + z] = row[z];
            S.f[i] = f; S.rank[i] = rk;
        }
        // L266: nothing accepted in two consecutive generations -> re-initialise (evaluated in this step)
        const uint32_t st = any ? 0 : gs->stagn + 1;
        g.sync();
        if (st == 2) {
            reinit_de_grp<ROWW>(g, sm, rm, S, k, gen);
            if (i == 0) gs->n_eval += P;
        }
        if (i == 0) gs->stagn = st == 2 ? 0 : st;
    } else if (ALGO == CAO_GA) {                                        // L288: the children replace the population
        if (i < P) {
#pragma unroll
            for (int z = 0; z < ROWW; ++z) S.idx[i * ROWW + z] = row[z];
            S.f[i] = f; S.rank[i] = rk;
        }
    } else if (ALGO == CAO_PSO) {                                       // L282: repair affects the evaluation only
        if (i < P) {
            S.f[i] = f; S.rank[i] = rk;
            acc = f < S.pbf[i];                                         // strict (A13)
            if (acc) {
                S.pbf[i] = f;
                for (int d = 0; d < n; ++d) S.pb[d * P + i] = S.x[d * P + i];
            }
        }
    } else {
        if (i < P) { S.f[i] = f; S.rank[i] = rk; }
    }
    if (last && i < P) {                                                // parity taps of the last stepped generation
        const uint64_t q = (uint64_t)k * P + i;
        uint4* dst = (uint4*)(rm.cand + q * (ROWW * 4));
        dst[0] = make_uint4(S.cand[i * ROWW], S.cand[i * ROWW + 1], S.cand[i * ROWW + 2], S.cand[i * ROWW + 3]);
        if (ROWW == 8) dst[1] = make_uint4(S.cand[i * ROWW + 4], S.cand[i * ROWW + 5], S.cand[i * ROWW + 6], S.cand[i * ROWW + 7]);
        rm.key[q] = key; rm.valid[q] = (key >> 45) == 0 ? 1 : 0; rm.rep_rank[q] = rep; rm.eval_rank[q] = rk; rm.tap_f[q] = f;
        rm.accept[q] = acc ? 1 : 0;
    }
    g.sync();
    if (i == 0) {                                                       // O10: trajectory row
        const uint32_t u = gs->uniq + gs->n_new;
        gs->uniq = u; gs->gens += 1; gs->n_eval += P;
        uint32_t* t = rm.traj + ((uint64_t)gen * rm.R + k) * 3;
        t[0] = (uint32_t)(gs->best >> 32); t[1] = (uint32_t)gs->best; t[2] = u;
    }
    g.sync();
}

// ---------------------------------------------------------------------------------------------
template <int ALGO, int ROWW, int MAXT>
__global__ void __launch_bounds__(MAXT) k_gen(const __grid_constant__ SpaceMeta sm, const __grid_constant__ ProbeMeta pm,
                                              const __grid_constant__ RunsMeta rm, const __grid_constant__ GenLayout lay,
                                              uint32_t g_first, uint32_t n_gens) {
    extern __shared__ __align__(16) uint32_t s_dyn[];
    // probe target / pair lists: CTA-wide copy in shared memory when they fit
    const uint16_t* tgt = pm.tgt; const uint32_t* pairs = pm.pairs;
    if (lay.cta_words) {
        uint32_t* s_pairs = s_dyn;
        uint16_t* s_tgt = (uint16_t*)(s_dyn + pm.C2);
        for (uint32_t e = threadIdx.x; e < pm.C2; e += blockDim.x) s_pairs[e] = __ldg(&pm.pairs[e]);
        for (uint32_t e = threadIdx.x; e < pm.T; e += blockDim.x) s_tgt[e] = __ldg(&pm.tgt[e]);
        tgt = s_tgt; pairs = s_pairs;
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
        for (; gen <= g_last; ++gen) {
            const bool active = rm.budget == 0 || gs->uniq < rm.budget;  // O10 (gen <= max_gens is enforced by the host)
            if (!active) break;
            generation<ALGO, ROWW>(g, sm, pm, tgt, pairs, rm, S, k, gen, gen == g_last);
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

// cao_enum_kernels.cuh -- S1: search-space construction (O1).
//
// The Cartesian index range is cut into blocks of B consecutive configs (B = product of the trailing digits t..n-1,
// the smallest such product >= 256).  A constraint whose outer scope is small becomes a bit table: one B-bit row per
// combination of its outer scope digits, plus one FLAG byte per row (row has any bit).  The bitmap of a block is the
// AND of one row per tabled constraint.  Pruning is hierarchical and exact: a block dies at the first constraint whose
// row flag is zero, before any mask word is read -- so every outer prefix that violates a constraint on outer digits
// costs a few byte lookups and writes nothing (the bitmap is zero-filled by a memset that overlaps the table build).
// Constraints too wide for a table ("residual"; all of them in plain mode) are interpreted only for the configs that
// survive the AND, one warp per surviving block, the outer-only prefix of the program once per block.
#pragma once
#include "cao_host.h"

// Tabled descriptor: {toff_lo, toff_hi, foff, n_outer, (digit, cstride) x n_outer, prog_off, prog_len, rows,
//                     n_inner, Ci, (digit, istride) x n_inner}.
#define TD_TOFF 0
#define TD_FOFF 2
#define TD_NO 3
#define TD_OUT 4

// All constraint tables in one launch: blockIdx.y = tabled constraint; a CTA takes groups of RPC rows.
// Phase A: one thread per (row, combination of the INNER scope digits) interprets the program (the inner pattern of a
// row depends on those digits only); results go to shared memory.  Phase B: one thread per (row, inner pattern) looks
// its combination up (s_ci: pattern -> combination, computed once per CTA) and a warp ballot assembles 32 patterns
// into one half word of the row; the row flag is the OR of its half words.
__global__ void __launch_bounds__(256) k_build_tables(const __grid_constant__ SpaceMeta sm, const int64_t* __restrict__ dom,
                                                      const int32_t* __restrict__ desc, uint64_t* tables, uint8_t* flags,
                                                      uint64_t B, uint32_t Wb, int32_t t, uint32_t ci_cap) {
    extern __shared__ uint8_t s_dyn8[];
    uint16_t* s_ci = (uint16_t*)s_dyn8;                                 // ci_cap entries (0 = no lookup table: decode per thread)
    uint8_t* s_ev = s_dyn8 + 2 * (size_t)ci_cap;                        // RPC x Ci results
    __shared__ uint32_t s_any[64];                                      // per row of the pass: any bit set
    const int32_t* ds = desc + desc[blockIdx.y];
    const uint64_t toff = (uint32_t)ds[TD_TOFF] | ((uint64_t)(uint32_t)ds[TD_TOFF + 1] << 32);
    const uint32_t foff = (uint32_t)ds[TD_FOFF];
    const int no = ds[TD_NO];
    const int32_t* prog = desc + ds[TD_OUT + 2 * no];
    const int nw = ds[TD_OUT + 1 + 2 * no];
    const uint32_t rows = (uint32_t)ds[TD_OUT + 2 + 2 * no];
    const int ni = ds[TD_OUT + 3 + 2 * no];
    const uint32_t Ci = (uint32_t)ds[TD_OUT + 4 + 2 * no];
    const int32_t* din = ds + TD_OUT + 5 + 2 * no;
    const uint32_t per_row = Wb * 64;
    const bool lut = ci_cap >= B;
    if (lut) {
        for (uint32_t p = threadIdx.x; p < B; p += blockDim.x) {
            uint32_t q = p, c = 0;
            for (int d = sm.n - 1; d >= t; --d) {                       // inner digits of p, least significant first
                const uint32_t m = sm.m[d], idx = q % m; q /= m;
                for (int k = 0; k < ni; ++k) if (din[2 * k] == d) c += idx * (uint32_t)din[2 * k + 1];
            }
            s_ci[p] = (uint16_t)c;
        }
    }
    // rows per CTA pass: at most 256 program runs (phase A), 2048 patterns (phase B, 8 per thread) and 64 rows
    const uint32_t RPC = max(1u, min(min(Ci >= 256 ? 1u : 256u / Ci, 2048u / per_row), 64u));
    uint32_t* out32 = (uint32_t*)(tables + toff);
    for (uint32_t row0 = blockIdx.x * RPC; row0 < rows; row0 += gridDim.x * RPC) {
        const uint32_t nr = min(RPC, rows - row0);
        __syncthreads();
        if (threadIdx.x < 64) s_any[threadIdx.x] = 0;
        for (uint32_t e = threadIdx.x; e < nr * Ci; e += blockDim.x) {  // phase A
            const uint32_t rr = e / Ci, c = e - rr * Ci, row = row0 + rr;
            int64_t x[CAO_MAX_DIMS];
            for (int d = 0; d < sm.n; ++d) x[d] = dom[d * 256];
            for (int k = 0; k < no; ++k) {
                const int d = ds[TD_OUT + 2 * k];
                x[d] = dom[d * 256 + (row / (uint32_t)ds[TD_OUT + 1 + 2 * k]) % sm.m[d]];
            }
            for (int k = 0; k < ni; ++k) {
                const int d = din[2 * k];
                x[d] = dom[d * 256 + (c / (uint32_t)din[2 * k + 1]) % sm.m[d]];
            }
            s_ev[e] = (uint8_t)eval_program(prog, nw, x);
        }
        __syncthreads();
        for (uint32_t e = threadIdx.x; e < nr * per_row; e += blockDim.x) {     // phase B; per_row is a multiple of 64
            const uint32_t rr = e / per_row, p = e - rr * per_row;
            int ok = 0;
            if (p < B) {
                uint32_t c = 0;
                if (lut) c = s_ci[p];
                else {
                    uint32_t q = p;
                    for (int d = sm.n - 1; d >= t; --d) {
                        const uint32_t m = sm.m[d], idx = q % m; q /= m;
                        for (int k = 0; k < ni; ++k) if (din[2 * k] == d) c += idx * (uint32_t)din[2 * k + 1];
                    }
                }
                ok = s_ev[rr * Ci + c];
            }
            const uint32_t word = __ballot_sync(0xFFFFFFFFu, ok);
            if ((threadIdx.x & 31) == 0) {
                out32[((uint64_t)(row0 + rr) * per_row + p) >> 5] = word;
                if (word) s_any[rr] = 1;
            }
        }
        __syncthreads();
        if (threadIdx.x < nr) flags[foff + row0 + threadIdx.x] = (uint8_t)s_any[threadIdx.x];
    }
}

// Inner lookup table for pass 2: the index bytes of the inner digits of every pattern p < B, already at their byte
// positions inside the packed row (ROWW words per pattern; the outer bytes are zero).
__global__ void __launch_bounds__(256) k_inner_lut(const __grid_constant__ SpaceMeta sm, uint32_t* lut, uint64_t B, int32_t t, int roww) {
    const uint32_t p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= B) return;
    uint32_t w[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    uint32_t q = p;
    for (int d = sm.n - 1; d >= t; --d) {
        const uint32_t m = sm.m[d], idx = q % m; q /= m;
        w[d >> 2] |= idx << ((d & 3) * 8);
    }
    for (int z = 0; z < roww; ++z) lut[(size_t)p * roww + z] = w[z];
}

// ---------------------------------------------------------------------------------------------
// Pass 1a.  Every thread walks CH consecutive blocks with an odometer over the outer digits (one mixed-radix decode per
// thread, then increments).  Per block: row flags of the tabled constraints in turn (exit at the first zero), then the
// AND of the rows word by word; non-zero words go to the zero-filled bitmap with atomicOr (a block's first and last
// word are shared with its neighbours when B is not a multiple of 64).  Without residual constraints the popcounts of
// the words are added to the per-512 counts here; with them the surviving blocks are listed for pass 1b instead.
__global__ void __launch_bounds__(256) k_enum(const __grid_constant__ SpaceMeta sm, const __grid_constant__ EnumArgs a) {
    extern __shared__ uint32_t s_key[];                                 // [n_tab][blockDim] row index per tabled constraint
    const uint32_t tid = threadIdx.x, bd = blockDim.x;
    uint8_t* dig = (uint8_t*)(s_key + (size_t)a.n_tab * bd) + tid;      // [t][blockDim] outer digits of this thread's block
    const uint64_t o0 = ((uint64_t)blockIdx.x * bd + tid) * a.CH;
    if (o0 >= a.n_blocks) return;
    {
        uint64_t q = o0;
        for (int d = a.t - 1; d >= 0; --d) {
            const uint32_t m = sm.m[d]; uint32_t idx = 0;
            if (m > 1) { const uint64_t q2 = div_magic(q, sm.magic[d]); idx = (uint32_t)(q - q2 * m); q = q2; }
            dig[d * bd] = (uint8_t)idx;
        }
    }
    const uint32_t tail_bits = (uint32_t)(a.B - (uint64_t)(a.Wb - 1) * 64);      // 1..64 bits in the last word
    const uint64_t tail_mask = tail_bits == 64 ? ~0ull : ((1ull << tail_bits) - 1ull);
    for (uint32_t it = 0; it < a.CH; ++it) {
        const uint64_t o = o0 + it;
        if (o >= a.n_blocks) break;
        bool alive = true;
        for (int c = 0; c < a.n_tab && alive; ++c) {
            const int32_t* ds = a.desc + __ldg(&a.desc[c]);
            const int no = __ldg(&ds[TD_NO]);
            uint32_t k = 0;
            for (int e = 0; e < no; ++e) k += (uint32_t)dig[__ldg(&ds[TD_OUT + 2 * e]) * bd] * (uint32_t)__ldg(&ds[TD_OUT + 1 + 2 * e]);
            s_key[c * bd + tid] = k;
            alive = __ldg(&a.flags[(uint32_t)__ldg(&ds[TD_FOFF]) + k]) != 0;
        }
        if (alive) {
            const uint64_t g0 = o * a.B;                                // first global bit of the block
            const uint32_t sh = (uint32_t)(g0 & 63);
            uint64_t any = 0;
            for (uint32_t j = 0; j < a.Wb; ++j) {
                uint64_t w = j + 1 == a.Wb ? tail_mask : ~0ull;
                for (int c = 0; c < a.n_tab && w; ++c) {
                    const int32_t* ds = a.desc + __ldg(&a.desc[c]);
                    const uint64_t toff = (uint32_t)__ldg(&ds[TD_TOFF]) | ((uint64_t)(uint32_t)__ldg(&ds[TD_TOFF + 1]) << 32);
                    w &= __ldg(&a.tables[toff + (uint64_t)s_key[c * bd + tid] * a.Wb + j]);
                }
                if (!w) continue;
                any |= w;
                const uint64_t gw = (g0 >> 6) + j;
                const uint64_t lo = w << sh, hi = sh ? w >> (64 - sh) : 0;
                if (lo) { atomicOr((unsigned long long*)&a.bitmap[gw], (unsigned long long)lo); if (!a.n_res) atomicAdd(&a.cnt[gw >> 3], (uint32_t)__popcll(lo)); }
                if (hi) { atomicOr((unsigned long long*)&a.bitmap[gw + 1], (unsigned long long)hi); if (!a.n_res) atomicAdd(&a.cnt[(gw + 1) >> 3], (uint32_t)__popcll(hi)); }
            }
            if (any && a.n_res) a.live[atomicAdd(a.live_count, 1u)] = (uint32_t)o;    // n_blocks < 2^32 (N < 2^40, B >= 256 unless one block)
        }
        for (int d = a.t - 1; d >= 0; --d) {                            // odometer: next block
            const uint32_t v = dig[d * bd] + 1u;
            if (v < sm.m[d]) { dig[d * bd] = (uint8_t)v; break; }
            dig[d * bd] = 0;
        }
    }
}

// Pass 1b: residual constraints (too wide for a table, or plain mode), one warp per surviving block.  The program
// prefix that reads only outer digits runs once per block; the lanes share the surviving bits of each bitmap word of
// the block (k-th-set-bit selection), clear the ones whose suffix fails (atomicAnd on this block's bits only) and add
// the popcount of the survivors to the per-512 counts.
__global__ void __launch_bounds__(256) k_residual(const __grid_constant__ SpaceMeta sm, const __grid_constant__ EnumArgs a) {
    const uint32_t lane = threadIdx.x & 31;
    const uint32_t nlive = *a.live_count;
    const uint64_t wid = ((uint64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = ((uint64_t)gridDim.x * blockDim.x) >> 5;
    for (uint64_t li = wid; li < nlive; li += nwarps) {
        const uint64_t o = a.live[li];
        int64_t x[CAO_MAX_DIMS];
        {
            uint64_t q = o;
            for (int d = a.t - 1; d >= 0; --d) {
                const uint32_t m = sm.m[d]; uint32_t idx = 0;
                if (m > 1) { const uint64_t q2 = div_magic(q, sm.magic[d]); idx = (uint32_t)(q - q2 * m); q = q2; }
                x[d] = a.dom[d * 256 + idx];
            }
        }
        const uint64_t g0 = o * a.B, g1 = g0 + a.B;                     // global bit range of the block
        const uint64_t w0 = g0 >> 6, w1 = (g1 + 63) >> 6;
        for (uint64_t gw = w0; gw < w1; ++gw) {
            // this block's bits inside global word gw
            const uint64_t lo_bit = gw << 6;
            uint64_t own = ~0ull;
            if (lo_bit < g0) own &= ~0ull << (g0 - lo_bit);
            if (lo_bit + 64 > g1) own &= ~0ull >> (lo_bit + 64 - g1);
            uint64_t word = __ldcg(&a.bitmap[gw]) & own;                // written by k_enum (L2)
            for (int r = 0; r < a.n_res && word; ++r) {
                const int32_t* ds = a.desc + __ldg(&a.desc[a.n_tab + r]);
                const int nw = __ldg(&ds[0]);
                int64_t st0[CAO_MAX_STACK];
                int pc0 = 0, sp0 = 0;
                const int pre = eval_core(ds + 1, nw, x, 0, st0, 0, a.t, &pc0, &sp0);       // block-uniform
                if (pre == 1) continue;                                                    // holds for the whole block
                uint64_t kill = 0;
                if (pre == 0) kill = word;
                else {
                    const uint32_t c = __popcll(word);
                    for (uint32_t k = lane; k < c; k += 32) {
                        const int bit = kth_set_bit64(word, k);
                        uint64_t p = lo_bit + bit - g0;                 // pattern inside the block
                        for (int d = sm.n - 1; d >= a.t; --d) {
                            const uint32_t m = sm.m[d]; uint32_t idx = 0;
                            if (m > 1) { const uint64_t p2 = div_magic(p, sm.magic[d]); idx = (uint32_t)(p - p2 * m); p = p2; }
                            x[d] = a.dom[d * 256 + idx];
                        }
                        int64_t st[CAO_MAX_STACK];
                        for (int z = 0; z < sp0; ++z) st[z] = st0[z];
                        int u0, u1;
                        if (!eval_core(ds + 1, nw, x, pc0, st, sp0, -1, &u0, &u1)) kill |= 1ull << bit;
                    }
                    const uint32_t klo = __reduce_or_sync(0xFFFFFFFFu, (uint32_t)kill);
                    const uint32_t khi = __reduce_or_sync(0xFFFFFFFFu, (uint32_t)(kill >> 32));
                    kill = ((uint64_t)khi << 32) | klo;
                }
                word &= ~kill;
                if (kill && lane == 0) atomicAnd((unsigned long long*)&a.bitmap[gw], (unsigned long long)~kill);
            }
            if (word && lane == 0) atomicAdd(&a.cnt[gw >> 3], (uint32_t)__popcll(word));
        }
    }
}

// ---------------------------------------------------------------------------------------------
// Exclusive scan of the per-512 counts in two launches.  k_cnt_reduce: per-chunk sums; the last CTA to finish scans
// them in place (exclusive) and writes V.  k_cnt_apply (pass 2): directory = chunk offset + scan inside the chunk, and
// the list of non-empty groups for k_fill.
#define SCAN_CHUNK 4096                                  // entries per CTA (256 threads x 16)
__global__ void __launch_bounds__(256) k_cnt_reduce(const uint32_t* __restrict__ cnt, uint64_t nd, uint32_t* part, uint64_t n_part,
                                                    uint32_t* ticket, uint64_t* V_out) {
    __shared__ uint32_t ws[8];
    __shared__ uint64_t wl[8];
    __shared__ bool s_last;
    __shared__ uint64_t carry_s;
    uint64_t base = (uint64_t)blockIdx.x * SCAN_CHUNK + threadIdx.x * 16;
    uint32_t s = 0;
    for (int k = 0; k < 16; ++k) if (base + k < nd) s += cnt[base + k];
    for (int o = 16; o; o >>= 1) s += __shfl_xor_sync(0xFFFFFFFFu, s, o);
    if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t t = 0; for (int k = 0; k < 8; ++k) t += ws[k];
        part[blockIdx.x] = t;
        __threadfence();
        s_last = atomicAdd(ticket, 1u) + 1 == gridDim.x;
        carry_s = 0;
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    for (uint64_t b0 = 0; b0 < n_part; b0 += 256) {                     // the last CTA: exclusive scan of the chunk sums
        const uint64_t i = b0 + threadIdx.x;
        const uint64_t v = i < n_part ? __ldcg(&part[i]) : 0;
        uint64_t inc = v;
        for (int o = 1; o < 32; o <<= 1) { uint64_t t = __shfl_up_sync(0xFFFFFFFFu, inc, o); if ((threadIdx.x & 31) >= o) inc += t; }
        if ((threadIdx.x & 31) == 31) wl[threadIdx.x >> 5] = inc;
        __syncthreads();
        uint64_t off = carry_s;
        for (uint32_t k = 0; k < (threadIdx.x >> 5); ++k) off += wl[k];
        if (i < n_part) part[i] = (uint32_t)(off + inc - v);             // V < 2^32 is checked on the host
        __syncthreads();
        if (threadIdx.x == 255) carry_s = off + inc;
        __syncthreads();
    }
    if (threadIdx.x == 0) { *V_out = carry_s; *ticket = 0; }
}
// nd counts the trailing zero entry too, so the last directory entry receives the total.
__global__ void __launch_bounds__(256) k_cnt_apply(const uint32_t* __restrict__ cnt, uint64_t nd, const uint32_t* __restrict__ part,
                                                   uint32_t* dir, uint32_t* groups, uint32_t* group_count) {
    __shared__ uint32_t ws[8];
    uint64_t base = (uint64_t)blockIdx.x * SCAN_CHUNK + threadIdx.x * 16;
    uint32_t v[16], s = 0;
    for (int k = 0; k < 16; ++k) { v[k] = (base + k < nd) ? cnt[base + k] : 0; s += v[k]; }
    uint32_t inc = s;
    for (int o = 1; o < 32; o <<= 1) { uint32_t t = __shfl_up_sync(0xFFFFFFFFu, inc, o); if ((threadIdx.x & 31) >= o) inc += t; }
    if ((threadIdx.x & 31) == 31) ws[threadIdx.x >> 5] = inc;
    __syncthreads();
    uint32_t off = part[blockIdx.x];
    for (uint32_t k = 0; k < (threadIdx.x >> 5); ++k) off += ws[k];
    off += inc - s;
    // non-empty groups of this thread go to the list (warp-aggregated append; the order is irrelevant)
    uint32_t mine = 0;
    for (int k = 0; k < 16; ++k) mine += v[k] != 0;
    uint32_t incl = mine;
    for (int o = 1; o < 32; o <<= 1) { uint32_t t = __shfl_up_sync(0xFFFFFFFFu, incl, o); if ((threadIdx.x & 31) >= o) incl += t; }
    const uint32_t total = __shfl_sync(0xFFFFFFFFu, incl, 31);
    uint32_t gbase = 0;
    if ((threadIdx.x & 31) == 0 && total) gbase = atomicAdd(group_count, total);
    gbase = __shfl_sync(0xFFFFFFFFu, gbase, 0) + incl - mine;
    for (int k = 0; k < 16; ++k) {
        if (base + k < nd) dir[base + k] = off;
        off += v[k];
        if (v[k]) groups[gbase++] = (uint32_t)(base + k);
    }
}

// cao_enum_kernels.cuh -- S1: search-space construction (O1).
//
// The Cartesian index range is cut into blocks of B consecutive configs (B = product of the trailing
// digits t..n-1).  A constraint whose scope is small is turned into a bit table indexed by its outer
// scope digits; each row holds the B-bit validity pattern over the inner digits.  The bitmap of a block
// is the AND of one row per constraint; constraints too wide for a table ("residual") are interpreted
// only for the configs that survive the AND.  In plain mode every constraint is residual.
#pragma once
#include "cao_host.h"

// All constraint tables in one launch: blockIdx.y = tabled constraint; a CTA takes groups of RPC rows.
// Phase A: one thread per (row, combination of the INNER scope digits) interprets the program (the inner pattern
// of a row depends on those digits only); results go to shared memory.  Phase B: one thread per (row, inner
// pattern) looks its combination up and a warp ballot assembles 32 patterns into one half word of the row.
// Tabled descriptor: {toff_lo, toff_hi, n_outer, (digit, cstride) x n_outer, prog_off, prog_len, rows,
//                     n_inner, Ci, (digit, istride) x n_inner}.
__global__ void __launch_bounds__(256) k_build_tables(const __grid_constant__ SpaceMeta sm, const int64_t* __restrict__ dom,
                                                      const int32_t* __restrict__ desc, uint64_t* tables, uint64_t B,
                                                      uint32_t Wb, int32_t t) {
    extern __shared__ uint8_t s_ev[];                                   // RPC x Ci results
    const int32_t* ds = desc + desc[blockIdx.y];
    const uint64_t toff = (uint32_t)ds[0] | ((uint64_t)(uint32_t)ds[1] << 32);
    const int no = ds[2];
    const int32_t* prog = desc + ds[3 + 2 * no];
    const int nw = ds[4 + 2 * no];
    const uint32_t rows = (uint32_t)ds[5 + 2 * no];
    const int ni = ds[6 + 2 * no];
    const uint32_t Ci = (uint32_t)ds[7 + 2 * no];
    const int32_t* din = ds + 8 + 2 * no;
    const uint32_t per_row = Wb * 64;
    // rows per CTA pass: at most 256 program runs (phase A) and 2048 patterns (phase B, 8 per thread)
    const uint32_t RPC = max(1u, min(Ci >= 256 ? 1u : 256u / Ci, 2048u / per_row));
    uint32_t* out32 = (uint32_t*)(tables + toff);
    for (uint32_t row0 = blockIdx.x * RPC; row0 < rows; row0 += gridDim.x * RPC) {
        const uint32_t nr = min(RPC, rows - row0);
        __syncthreads();
        for (uint32_t e = threadIdx.x; e < nr * Ci; e += blockDim.x) {  // phase A
            const uint32_t rr = e / Ci, c = e - rr * Ci, row = row0 + rr;
            int64_t x[CAO_MAX_DIMS];
            for (int d = 0; d < sm.n; ++d) x[d] = dom[d * 256];
            for (int k = 0; k < no; ++k) {
                const int d = ds[3 + 2 * k];
                x[d] = dom[d * 256 + (row / (uint32_t)ds[4 + 2 * k]) % sm.m[d]];
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
                uint32_t q = p, c = 0;
                for (int d = sm.n - 1; d >= t; --d) {                   // inner digits of p, least significant first
                    const uint32_t m = sm.m[d], idx = q % m; q /= m;
                    for (int k = 0; k < ni; ++k) if (din[2 * k] == d) c += idx * (uint32_t)din[2 * k + 1];
                }
                ok = s_ev[rr * Ci + c];
            }
            const uint32_t word = __ballot_sync(0xFFFFFFFFu, ok);
            if ((threadIdx.x & 31) == 0) out32[((uint64_t)(row0 + rr) * per_row + p) >> 5] = word;
        }
    }
}

// Value classes of a residual constraint (residual descriptor r: {nw, words...}).
// k_res_prefix: one thread per block of configs runs the program up to its first inner parameter; the single
// stack value left is the block's class key, entered into a small open-addressing table with atomicCAS.
__global__ void __launch_bounds__(256) k_res_prefix(const __grid_constant__ SpaceMeta sm, const int64_t* __restrict__ dom,
                                                    const int32_t* __restrict__ desc, int r, const ResClassArgs rc,
                                                    uint64_t n_blocks, int32_t t) {
    const uint64_t o = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (o >= n_blocks) return;
    const int32_t* ds = desc + desc[r];
    int64_t x[CAO_MAX_DIMS];
    uint64_t q = o;
    for (int d = t - 1; d >= 0; --d) {
        const uint32_t m = sm.m[d]; uint32_t idx = 0;
        if (m > 1) { const uint64_t q2 = div_magic(q, sm.magic[d]); idx = (uint32_t)(q - q2 * m); q = q2; }
        x[d] = dom[d * 256 + idx];
    }
    int64_t st[CAO_MAX_STACK];
    int pc0 = 0, sp0 = 0;
    const int pre = eval_core(ds + 1, ds[0], x, 0, st, 0, t, &pc0, &sp0);
    uint32_t cls = CAO_CLS_FALSE;                                       // a zero divisor in the prefix: all false
    if (pre == 2) {
        const long long key = st[0];
        uint32_t h = (uint32_t)(((uint64_t)key * 0x9E3779B97F4A7C15ull) >> 40) & (CAO_HS - 1);
        cls = CAO_CLS_OVERFLOW;
        for (int probe = 0; probe < 64; ++probe) {
            const long long old = atomicCAS((unsigned long long*)&rc.keys[h], (unsigned long long)CAO_CLS_EMPTY, (unsigned long long)key);
            if (old == CAO_CLS_EMPTY || old == key) { cls = h; break; }
            h = (h + 1) & (CAO_HS - 1);
        }
        if (cls == CAO_CLS_OVERFLOW) *rc.overflow = 1;
    }
    rc.blk_class[o] = cls;
}
// k_res_class_table: one thread per (hash slot, inner pattern) resumes the program from the class key.
__global__ void __launch_bounds__(256) k_res_class_table(const __grid_constant__ SpaceMeta sm, const int64_t* __restrict__ dom,
                                                         const int32_t* __restrict__ desc, int r, const ResClassArgs rc,
                                                         uint64_t B, uint32_t Wb, int32_t t) {
    const uint64_t gid = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const uint32_t per_row = Wb * 64;
    if (gid >= (uint64_t)CAO_HS * per_row) return;                      // whole warps: the bound is a multiple of 64
    const uint32_t slot = (uint32_t)(gid / per_row), p = (uint32_t)(gid - (uint64_t)slot * per_row);
    const long long key = rc.keys[slot];
    int ok = 0;
    if (key != CAO_CLS_EMPTY && p < B) {
        const int32_t* ds = desc + desc[r];
        int64_t x[CAO_MAX_DIMS];
        for (int d = 0; d < sm.n; ++d) x[d] = dom[d * 256];
        uint32_t q = p;
        for (int d = sm.n - 1; d >= t; --d) { const uint32_t m = sm.m[d]; x[d] = dom[d * 256 + q % m]; q /= m; }
        int64_t st[CAO_MAX_STACK];
        st[0] = key;
        int u0, u1;
        ok = eval_core(ds + 1, ds[0], x, rc.pc0, st, 1, -1, &u0, &u1);
    }
    const uint32_t word = __ballot_sync(0xFFFFFFFFu, ok);
    if ((threadIdx.x & 31) == 0) ((uint32_t*)rc.table)[gid >> 5] = word;
}

__device__ __forceinline__ uint64_t get64(const uint64_t* mk, uint32_t r, uint32_t Wb) {
    uint32_t j = r >> 6, s = r & 63;
    if (j >= Wb) return 0;
    uint64_t v = mk[j] >> s;
    if (s && j + 1 < Wb) v |= mk[j + 1] << (64 - s);
    return v;
}

// Pass 1.  desc layout: [0..n_tab) offsets of tabled descriptors {toff_lo, toff_hi, n_outer, (digit, cstride)*},
// [n_tab..n_tab+n_res) offsets of residual descriptors {nw, words*}.
__global__ void __launch_bounds__(256) k_enum_pass1(const __grid_constant__ SpaceMeta sm,
                                                    const __grid_constant__ EnumArgs a) {
    extern __shared__ uint64_t smem64[];
    uint64_t* masks = smem64;
    uint8_t* od = (uint8_t*)(masks + (size_t)(a.nb + 1) * a.Wb);
    const uint32_t tid = threadIdx.x, bd = blockDim.x;
    const uint64_t o0 = (uint64_t)blockIdx.x * a.nb;
    const uint32_t tail_bits = (uint32_t)(a.B - (uint64_t)(a.Wb - 1) * 64);      // 1..64 bits in the last word
    for (uint32_t i = tid; i <= a.nb; i += bd) {
        uint64_t o = o0 + i;
        uint64_t* mk = masks + (size_t)i * a.Wb;
        if (o >= a.n_blocks) { for (uint32_t j = 0; j < a.Wb; ++j) mk[j] = 0; continue; }
        uint64_t q = o;
        for (int d = a.t - 1; d >= 0; --d) {
            uint32_t m = sm.m[d];
            uint32_t idx = 0;
            if (m > 1) { uint64_t q2 = div_magic(q, sm.magic[d]); idx = (uint32_t)(q - q2 * m); q = q2; }
            od[d * bd + tid] = (uint8_t)idx;
        }
        for (uint32_t j = 0; j + 1 < a.Wb; ++j) mk[j] = ~0ull;
        mk[a.Wb - 1] = tail_bits == 64 ? ~0ull : ((1ull << tail_bits) - 1ull);
        uint64_t any = 1;
        for (int c = 0; c < a.n_tab && any; ++c) {
            const int32_t* ds = a.desc + __ldg(&a.desc[c]);
            uint64_t toff = (uint32_t)__ldg(&ds[0]) | ((uint64_t)(uint32_t)__ldg(&ds[1]) << 32);
            int no = __ldg(&ds[2]);
            uint64_t k = 0;
            for (int e = 0; e < no; ++e) k += (uint64_t)od[__ldg(&ds[3 + 2 * e]) * bd + tid] * (uint32_t)__ldg(&ds[4 + 2 * e]);
            const uint64_t* tab = a.tables + toff + k * a.Wb;
            any = 0;
            for (uint32_t j = 0; j < a.Wb; ++j) { uint64_t v = mk[j] & __ldg(&tab[j]); mk[j] = v; any |= v; }
        }
        for (int c = 0; c < a.n_rc && any; ++c) {                       // residual constraints with value classes
            if (__ldg(a.rc[c].overflow)) continue;                      // (handled in phase 1b)
            const uint32_t cls = __ldg(&a.rc[c].blk_class[o]);
            any = 0;
            if (cls == CAO_CLS_FALSE) { for (uint32_t j = 0; j < a.Wb; ++j) mk[j] = 0; }
            else {
                const uint64_t* tab = a.rc[c].table + (uint64_t)cls * a.Wb;
                for (uint32_t j = 0; j < a.Wb; ++j) { uint64_t v = mk[j] & __ldg(&tab[j]); mk[j] = v; any |= v; }
            }
        }
    }
    // Phase 1b: residual constraints (too wide for a table, or plain mode).  One warp per block of configs: the
    // program prefix that reads only outer digits runs once per block, the lanes then share the surviving bits
    // of each mask word (warp-level compaction by k-th-set-bit selection) and clear the ones that fail.
    bool need_1b = a.n_res > a.n_rc;
    for (int c = 0; c < a.n_rc; ++c) need_1b = need_1b || __ldg(a.rc[c].overflow) != 0;
    if (need_1b) {
        __syncthreads();
        const uint32_t lane = tid & 31, warp = tid >> 5, nwarp = bd >> 5;
        for (uint32_t i = warp; i <= a.nb; i += nwarp) {
            const uint64_t o = o0 + i;
            if (o >= a.n_blocks) continue;
            uint64_t* mk = masks + (size_t)i * a.Wb;
            uint64_t anyb = 0;
            for (uint32_t j = lane; j < a.Wb; j += 32) anyb |= mk[j];
            if (!__any_sync(0xFFFFFFFFu, anyb != 0)) continue;
            int64_t x[CAO_MAX_DIMS];
            {
                uint64_t q = o;
                for (int d = a.t - 1; d >= 0; --d) {
                    const uint32_t m = sm.m[d]; uint32_t idx = 0;
                    if (m > 1) { const uint64_t q2 = div_magic(q, sm.magic[d]); idx = (uint32_t)(q - q2 * m); q = q2; }
                    x[d] = a.dom[d * 256 + idx];
                }
            }
            for (int r = 0; r < a.n_res; ++r) {
                if (r < a.n_rc && !__ldg(a.rc[r].overflow)) continue;  // already applied through its classes
                const int32_t* ds = a.desc + __ldg(&a.desc[a.n_tab + r]);
                const int nw = __ldg(&ds[0]);
                int64_t st0[CAO_MAX_STACK];
                int pc0 = 0, sp0 = 0;
                const int pre = eval_core(ds + 1, nw, x, 0, st0, 0, a.t, &pc0, &sp0);       // block-uniform
                if (pre == 1) continue;                                                    // holds for the whole block
                if (pre == 0) { for (uint32_t j = lane; j < a.Wb; j += 32) mk[j] = 0; __syncwarp(); break; }
                for (uint32_t j = 0; j < a.Wb; ++j) {
                    const uint64_t word = mk[j];
                    const uint32_t c = __popcll(word);
                    uint64_t kill = 0;
                    for (uint32_t k = lane; k < c; k += 32) {
                        const int bit = kth_set_bit64(word, k);
                        uint64_t p = (uint64_t)j * 64 + bit;
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
                    __syncwarp();
                    if (lane == 0 && (klo | khi)) mk[j] = word & ~(((uint64_t)khi << 32) | klo);
                    __syncwarp();
                }
            }
        }
    }
    __syncthreads();
    // Phase 2: re-align the block masks to 64-bit words of the global bitmap (coalesced stores).
    const uint64_t g0 = o0 * a.B;
    uint64_t o1 = o0 + a.nb; if (o1 > a.n_blocks) o1 = a.n_blocks;
    const uint64_t g1 = o1 * a.B;                       // == N for the last CTA
    const uint64_t w_first = (g0 + 63) >> 6, w_end = (g1 + 63) >> 6;
    for (uint64_t w = w_first + tid; w < w_end; w += bd) {
        uint64_t rel = (w << 6) - g0;
        uint64_t i = a.B > 1 ? div_magic(rel, a.magicB) : rel;
        uint32_t r = (uint32_t)(rel - i * a.B);
        uint64_t val = get64(masks + i * a.Wb, r, a.Wb);
        uint64_t avail = a.B - r;
        // B >= 64 whenever there is more than one block, so at most one following block contributes
        if (avail < 64) val |= get64(masks + (i + 1) * a.Wb, 0, a.Wb) << avail;
        a.bitmap[w] = val;
        if (val) atomicAdd(&a.cnt[w >> 3], (uint32_t)__popcll(val));
    }
}

// ---------------------------------------------------------------------------------------------
// Exclusive scan of the per-512 counts (three small launches; the data is N/128 bytes).
#define SCAN_CHUNK 4096                                  // entries per CTA (256 threads x 16)
__global__ void __launch_bounds__(256) k_scan_reduce(const uint32_t* __restrict__ cnt, uint64_t nd, uint32_t* part) {
    __shared__ uint32_t ws[8];
    uint64_t base = (uint64_t)blockIdx.x * SCAN_CHUNK + threadIdx.x * 16;
    uint32_t s = 0;
    for (int k = 0; k < 16; ++k) if (base + k < nd) s += cnt[base + k];
    for (int o = 16; o; o >>= 1) s += __shfl_xor_sync(0xFFFFFFFFu, s, o);
    if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) { uint32_t t = 0; for (int k = 0; k < 8; ++k) t += ws[k]; part[blockIdx.x] = t; }
}
// One CTA: exclusive scan of the partials in place; total (= V) to *V_out as u64 (overflow of u32 is detected on the host).
__global__ void __launch_bounds__(1024) k_scan_partials(uint32_t* part, uint64_t n_part, uint64_t* V_out) {
    __shared__ uint64_t ws[32];
    __shared__ uint64_t carry_s;
    if (threadIdx.x == 0) carry_s = 0;
    __syncthreads();
    for (uint64_t base = 0; base < n_part; base += 1024) {
        uint64_t i = base + threadIdx.x;
        uint64_t v = i < n_part ? part[i] : 0, s = v;
        for (int o = 1; o < 32; o <<= 1) { uint64_t t = __shfl_up_sync(0xFFFFFFFFu, s, o); if ((threadIdx.x & 31) >= o) s += t; }
        if ((threadIdx.x & 31) == 31) ws[threadIdx.x >> 5] = s;
        __syncthreads();
        if (threadIdx.x < 32) {
            uint64_t t = ws[threadIdx.x], u = t;
            for (int o = 1; o < 32; o <<= 1) { uint64_t z = __shfl_up_sync(0xFFFFFFFFu, u, o); if (threadIdx.x >= o) u += z; }
            ws[threadIdx.x] = u - t;
        }
        __syncthreads();
        uint64_t excl = carry_s + ws[threadIdx.x >> 5] + s - v;
        if (i < n_part) part[i] = (uint32_t)excl;
        __syncthreads();
        if (threadIdx.x == 1023) carry_s = excl + v;
        __syncthreads();
    }
    if (threadIdx.x == 0) *V_out = carry_s;
}
// In-place exclusive scan of each chunk plus the chunk offset.  nd here counts the trailing zero entry
// too, so the last entry receives the total.
__global__ void __launch_bounds__(256) k_scan_apply(uint32_t* cnt, uint64_t nd, const uint32_t* __restrict__ part) {
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
    for (int k = 0; k < 16; ++k) { if (base + k < nd) cnt[base + k] = off; off += v[k]; }
}

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
    // rows per CTA pass: at most 256 program runs (phase A, the slow part: one interpreter run per thread), 8192
    // patterns (phase B, 32 cheap lookups per thread) and 64 rows
    const uint32_t RPC = max(1u, min(min(Ci >= 256 ? 1u : 256u / Ci, 8192u / per_row), 64u));
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
// The descriptor words (a few hundred to a few thousand) are staged in shared memory by every CTA of pass 1: the
// kernels chase pointers through them for every block, and a chain of dependent global loads is what bounds them.
__device__ __forceinline__ const int32_t* stage_desc(const EnumArgs& a, int32_t* s_desc) {
    if (!a.desc_in_smem) return a.desc;
    for (uint32_t e = threadIdx.x; e < a.desc_words; e += blockDim.x) s_desc[e] = __ldg(&a.desc[e]);
    __syncthreads();
    return s_desc;
}
// Outer digits of block o.
__device__ __forceinline__ void decode_outer(const SpaceMeta& sm, int t, uint64_t o, uint8_t* dig, uint32_t stride) {
    uint64_t q = o;
    for (int d = t - 1; d >= 0; --d) {
        const uint32_t m = sm.m[d]; uint32_t idx = 0;
        if (m > 1) { const uint64_t q2 = div_magic(q, sm.magic[d]); idx = (uint32_t)(q - q2 * m); q = q2; }
        dig[d * stride] = (uint8_t)idx;
    }
}
__device__ __forceinline__ uint32_t table_key(const int32_t* ds, const uint8_t* dig, uint32_t stride) {
    const int no = ds[TD_NO];
    uint32_t k = 0;
    for (int e = 0; e < no; ++e) k += (uint32_t)dig[ds[TD_OUT + 2 * e] * stride] * (uint32_t)ds[TD_OUT + 1 + 2 * e];
    return k;
}

// Pass 1a: which blocks survive the tabled constraints?  Every thread owns a CHUNK of CH consecutive blocks = all
// combinations of the last k outer digits under one prefix of the others (CH = product of those k digits, chosen on the
// host).  The tabled constraints are sorted: first the n_inv "chunk-invariant" ones, whose outer scope does not touch
// the last k digits -- their row flags are tested ONCE per chunk and a failing prefix kills all CH blocks at once
// (hierarchical pruning: on a sparse space nearly every chunk ends here, after a few byte loads) -- then the others,
// per block, four independent byte loads at a time.  Survivors go to the live list together with their table row
// indices (keys), first into shared memory, then with one global atomic per CTA.  Nothing else is touched.
__global__ void __launch_bounds__(256) k_enum(const __grid_constant__ SpaceMeta sm, const __grid_constant__ EnumArgs a) {
    extern __shared__ int32_t s_enum[];
    const uint32_t tid = threadIdx.x, bd = blockDim.x;
    const int32_t* desc = stage_desc(a, s_enum);
    uint8_t* dig = (uint8_t*)(s_enum + (a.desc_in_smem ? a.desc_words : 0)) + tid;      // [t][blockDim]
    uint32_t* s_list = (uint32_t*)(s_enum + (a.desc_in_smem ? a.desc_words : 0)) + ((size_t)bd * max(1, a.t) + 3) / 4;   // [bd * CH]
    __shared__ uint32_t s_n, s_base;
    if (tid == 0) s_n = 0;
    __syncthreads();
    const uint64_t o0 = ((uint64_t)blockIdx.x * bd + tid) * a.CH;
    const bool mine = o0 < a.n_blocks;
    bool chunk_alive = mine;
    if (mine) {
        decode_outer(sm, a.t, o0, dig, bd);
        for (int c0 = 0; c0 < a.n_inv && chunk_alive; c0 += 4) {        // chunk-invariant constraints: once per CH blocks
            uint8_t f[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                f[u] = 1;
                if (c0 + u < a.n_inv) {
                    const int32_t* ds = desc + desc[c0 + u];
                    f[u] = __ldg(&a.flags[(uint32_t)ds[TD_FOFF] + table_key(ds, dig, bd)]);
                }
            }
            chunk_alive = f[0] && f[1] && f[2] && f[3];
        }
    }
    if (__syncthreads_or(chunk_alive)) {
        for (uint32_t it = 0; it < a.CH; ++it) {
            const uint64_t o = o0 + it;
            bool alive = chunk_alive && o < a.n_blocks;
            for (int c0 = a.n_inv; c0 < a.n_tab && alive; c0 += 4) {
                uint8_t f[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    f[u] = 1;
                    if (c0 + u < a.n_tab) {
                        const int32_t* ds = desc + desc[c0 + u];
                        f[u] = __ldg(&a.flags[(uint32_t)ds[TD_FOFF] + table_key(ds, dig, bd)]);
                    }
                }
                alive = f[0] && f[1] && f[2] && f[3];
            }
            const uint32_t bal = __ballot_sync(0xFFFFFFFFu, alive);
            if (bal) {                                                  // the CTA collects its survivors in shared memory
                uint32_t base = 0;
                if ((tid & 31) == 0) base = atomicAdd(&s_n, (uint32_t)__popc(bal));
                base = __shfl_sync(0xFFFFFFFFu, base, 0);
                if (alive) s_list[base + __popc(bal & ((1u << (tid & 31)) - 1u))] = (uint32_t)o;   // n_blocks < 2^32
            }
            if (chunk_alive) {
                for (int d = a.t - 1; d >= 0; --d) {                    // odometer: next block
                    const uint32_t v = dig[d * bd] + 1u;
                    if (v < sm.m[d]) { dig[d * bd] = (uint8_t)v; break; }
                    dig[d * bd] = 0;
                }
            }
        }
    }
    __syncthreads();
    const uint32_t n = s_n;
    if (tid == 0 && n) s_base = atomicAdd(a.live_count, n);             // one global atomic per CTA
    __syncthreads();
    for (uint32_t e = tid; e < n; e += bd) a.live[s_base + e] = s_list[e];
}

// Table row indices (keys) of every live block, one thread per block (the survivors cluster in a few CTAs of k_enum, so
// this is a separate, balanced pass): k_masks then reads keys instead of decoding the block for every mask word.
__global__ void __launch_bounds__(256) k_keys(const __grid_constant__ SpaceMeta sm, const __grid_constant__ EnumArgs a) {
    extern __shared__ int32_t s_enum[];
    const uint32_t tid = threadIdx.x, bd = blockDim.x;
    const int32_t* desc = stage_desc(a, s_enum);
    uint8_t* dig = (uint8_t*)(s_enum + (a.desc_in_smem ? a.desc_words : 0)) + tid;
    const uint32_t nlive = *a.live_count;
    for (uint32_t li = blockIdx.x * bd + tid; li < nlive; li += gridDim.x * bd) {
        decode_outer(sm, a.t, a.live[li], dig, bd);
        for (int c = 0; c < a.n_tab; ++c) a.keys[(uint64_t)li * a.n_tab + c] = table_key(desc + desc[c], dig, bd);
    }
}

// Pass 1b: one thread per (live block, word of its mask): AND of one row word per tabled constraint (independent
// loads), non-zero words go to the zero-filled bitmap with atomicOr (a block's first and last word are shared with its
// neighbours when B is not a multiple of 64).  Without residual constraints the popcounts are added to the per-512
// counts here.
__global__ void __launch_bounds__(256) k_masks(const __grid_constant__ SpaceMeta sm, const __grid_constant__ EnumArgs a) {
    extern __shared__ int32_t s_enum[];
    const uint32_t tid = threadIdx.x, bd = blockDim.x;
    const int32_t* desc = stage_desc(a, s_enum);
    uint8_t* dig = (uint8_t*)(s_enum + (a.desc_in_smem ? a.desc_words : 0)) + tid;
    const uint32_t nlive = *a.live_count;
    const uint64_t total = (uint64_t)nlive * a.Wb;
    const uint32_t tail_bits = (uint32_t)(a.B - (uint64_t)(a.Wb - 1) * 64);      // 1..64 bits in the last word
    for (uint64_t e = (uint64_t)blockIdx.x * bd + tid; e < total; e += (uint64_t)gridDim.x * bd) {
        const uint32_t li = (uint32_t)(e / a.Wb), j = (uint32_t)(e - (uint64_t)li * a.Wb);
        const uint64_t o = a.live[li];
        if (!a.keys) decode_outer(sm, a.t, o, dig, bd);
        uint64_t w = (j + 1 == a.Wb && tail_bits < 64) ? ((1ull << tail_bits) - 1ull) : ~0ull;
        for (int c0 = 0; c0 < a.n_tab && w; c0 += 4) {
            uint64_t r[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                r[u] = ~0ull;
                if (c0 + u < a.n_tab) {
                    const int32_t* ds = desc + desc[c0 + u];
                    const uint64_t toff = (uint32_t)ds[TD_TOFF] | ((uint64_t)(uint32_t)ds[TD_TOFF + 1] << 32);
                    const uint32_t key = a.keys ? a.keys[(uint64_t)li * a.n_tab + c0 + u] : table_key(ds, dig, bd);
                    r[u] = __ldg(&a.tables[toff + (uint64_t)key * a.Wb + j]);
                }
            }
            w &= r[0] & r[1] & r[2] & r[3];
        }
        if (!w) continue;
        const uint64_t g0 = o * a.B;                                    // first global bit of the block
        const uint32_t sh = (uint32_t)(g0 & 63);
        const uint64_t gw = (g0 >> 6) + j;
        const uint64_t lo = w << sh, hi = sh ? w >> (64 - sh) : 0;
        if (lo) { atomicOr((unsigned long long*)&a.bitmap[gw], (unsigned long long)lo); if (!a.n_res) atomicAdd(&a.cnt[gw >> 3], (uint32_t)__popcll(lo)); }
        if (hi) { atomicOr((unsigned long long*)&a.bitmap[gw + 1], (unsigned long long)hi); if (!a.n_res) atomicAdd(&a.cnt[(gw + 1) >> 3], (uint32_t)__popcll(hi)); }
    }
}

// Pass 1c (only with residual constraints: too wide for a table, or plain mode), over the LIVE blocks only.
// k_res_prefix: one thread per (live block, residual constraint) runs the program prefix that reads only outer digits
// and stores where it stopped: status 0 = the constraint is false for the whole block, 1 = true for the whole block,
// 2 = resume at (pc, sp) with the stored stack (up to CAO_RES_STACK values), 3 = stack too deep to store (k_residual
// re-runs the prefix).
// Value classes: if the prefix leaves exactly ONE stack value and the rest of the program reads inner parameters only
// (decided on the host: a.rc_of[r] >= 0), the constraint depends on the outer digits through that value alone.  The
// value is entered into a 4096-slot open-addressing table (atomicCAS, one attempt per distinct value per warp); the
// slot is the block's class.  k_res_class_table then resumes the program once per (class, inner pattern) and k_residual
// ANDs the class mask into the block -- instead of interpreting the suffix for every surviving config of every block.
// Exact: same program, same operands, same order.  More than 4096 values: overflow flag, per-config path.
#define CAO_RES_STACK 3
#define CAO_HS 4096
#define CAO_CLS_EMPTY ((long long)0x8080808080808080ll)   // below -2^62: never a saturated value
#define CAO_CLS_NONE 0xFFFFFFFFu
struct ResPrefix { int32_t status, pc, sp; uint32_t cls; long long st[CAO_RES_STACK]; };
__global__ void __launch_bounds__(256) k_res_prefix(const __grid_constant__ SpaceMeta sm, const __grid_constant__ EnumArgs a, ResPrefix* out) {
    extern __shared__ int32_t s_enum[];
    const int32_t* desc = stage_desc(a, s_enum);
    const uint32_t nlive = *a.live_count, lane = threadIdx.x & 31;
    const uint64_t total = (uint64_t)nlive * a.n_res;
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t e0 = (uint64_t)blockIdx.x * blockDim.x; e0 < total; e0 += stride) {      // whole warps iterate together
        const uint64_t e = e0 + threadIdx.x;
        const bool valid = e < total;
        const uint32_t li = valid ? (uint32_t)(e / a.n_res) : 0, r = valid ? (uint32_t)(e - (uint64_t)li * a.n_res) : 0;
        ResPrefix p;
        p.status = 1; p.pc = 0; p.sp = 0; p.cls = CAO_CLS_NONE;
        for (int z = 0; z < CAO_RES_STACK; ++z) p.st[z] = 0;
        if (valid) {
            uint8_t dig[CAO_MAX_DIMS];
            decode_outer(sm, a.t, a.live[li], dig, 1);
            int64_t x[CAO_MAX_DIMS];
            for (int d = 0; d < a.t; ++d) x[d] = a.dom[d * 256 + dig[d]];
            const int32_t* ds = desc + desc[a.n_tab + r];
            int64_t st0[CAO_MAX_STACK];
            int pc0 = 0, sp0 = 0;
            const int pre = eval_core(ds + 1, ds[0], x, 0, st0, 0, a.t, &pc0, &sp0);
            p.status = pre == 2 && sp0 > CAO_RES_STACK ? 3 : pre; p.pc = pc0; p.sp = sp0;
            for (int z = 0; z < CAO_RES_STACK; ++z) p.st[z] = z < sp0 ? st0[z] : 0;
        }
        const int rc = valid ? a.rc_of[r] : -1;
        const bool wants = rc >= 0 && p.status == 2 && !*a.rc[rc >= 0 ? rc : 0].overflow;
        const long long key = wants ? p.st[0] : (long long)lane;        // lanes without a class never match a real key by accident:
        const uint32_t peers = __match_any_sync(0xFFFFFFFFu, (unsigned long long)key) &   // ... they also differ in `wants`
                               __match_any_sync(0xFFFFFFFFu, wants ? rc : -1 - (int)lane);
        uint32_t cls = CAO_CLS_NONE;
        if (wants && lane == (uint32_t)(__ffs(peers) - 1)) {            // one insertion per distinct (constraint, value) per warp
            long long* keys = a.rc[rc].keys;
            uint32_t h = (uint32_t)(((uint64_t)key * 0x9E3779B97F4A7C15ull) >> 40) & (CAO_HS - 1);
            for (int probe = 0; probe < 64; ++probe) {
                const long long old = atomicCAS((unsigned long long*)&keys[h], (unsigned long long)CAO_CLS_EMPTY, (unsigned long long)key);
                if (old == CAO_CLS_EMPTY || old == key) { cls = h; break; }
                h = (h + 1) & (CAO_HS - 1);
            }
            if (cls == CAO_CLS_NONE) *a.rc[rc].overflow = 1;
        }
        cls = __shfl_sync(0xFFFFFFFFu, cls, __ffs(peers) - 1);
        if (wants) p.cls = cls;
        if (valid) out[e] = p;
    }
}
// k_res_class_table: one thread per (class constraint, used hash slot, inner pattern) resumes the program from the class
// key.  Every CTA first compacts the used slots (a few dozen of 4096) into the same slot-ordered list in shared memory --
// warp w reads slots [512 w, 512 w + 512) with 16 coalesced loads in flight, ballots, one barrier for the eight warp
// counts -- so that the (used slot, 32 patterns) items can be dealt evenly to all the warps of the grid.
__global__ void __launch_bounds__(256) k_res_class_table(const __grid_constant__ SpaceMeta sm, const __grid_constant__ EnumArgs a) {
    __shared__ uint16_t s_used[CAO_HS];
    __shared__ uint32_t s_cnt[8];
    const uint32_t lane = threadIdx.x & 31, wl = threadIdx.x >> 5;
    const uint32_t wid = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = (gridDim.x * blockDim.x) >> 5;
    const int rc = blockIdx.y;
    const long long* __restrict__ keys = a.rc[rc].keys;
    uint32_t bal[CAO_HS / 256], mine = 0;
    {
        long long kv[CAO_HS / 256];
#pragma unroll
        for (int it = 0; it < CAO_HS / 256; ++it) kv[it] = keys[wl * (CAO_HS / 8) + it * 32 + lane];
#pragma unroll
        for (int it = 0; it < CAO_HS / 256; ++it) { bal[it] = __ballot_sync(0xFFFFFFFFu, kv[it] != CAO_CLS_EMPTY); mine += (uint32_t)__popc(bal[it]); }
    }
    if (lane == 0) s_cnt[wl] = mine;
    __syncthreads();
    uint32_t base = 0, n_used = 0;
    for (uint32_t k = 0; k < 8; ++k) { if (k < wl) base += s_cnt[k]; n_used += s_cnt[k]; }
#pragma unroll
    for (int it = 0; it < CAO_HS / 256; ++it) {
        if ((bal[it] >> lane) & 1u) s_used[base + __popc(bal[it] & ((1u << lane) - 1u))] = (uint16_t)(wl * (CAO_HS / 8) + it * 32 + lane);
        base += (uint32_t)__popc(bal[it]);
    }
    __syncthreads();
    const int32_t* ds = a.desc + a.desc[a.n_tab + a.rc[rc].r];
    const uint32_t per_row = a.Wb * 64;
    const uint32_t chunks = per_row >> 5;                               // 32 patterns per warp item
    for (uint32_t item = wid; item < n_used * chunks; item += nwarps) {
        const uint32_t slot = s_used[item / chunks], p0 = (item % chunks) << 5;
        const long long key = keys[slot];
        const uint32_t p = p0 + lane;
        int ok = 0;
        if (p < a.B) {
            int64_t x[CAO_MAX_DIMS];
            for (int d = 0; d < sm.n; ++d) x[d] = a.dom[d * 256];
            uint32_t q = p;
            for (int d = sm.n - 1; d >= a.t; --d) { const uint32_t m = sm.m[d]; x[d] = a.dom[d * 256 + q % m]; q /= m; }
            int64_t st[CAO_MAX_STACK];
            st[0] = key;
            int u0, u1;
            ok = eval_core(ds + 1, ds[0], x, a.rc[rc].pc0, st, 1, -1, &u0, &u1);
        }
        const uint32_t word = __ballot_sync(0xFFFFFFFFu, ok);
        if (lane == 0) ((uint32_t*)a.rc[rc].table)[((uint64_t)slot * per_row + p0) >> 5] = word;
    }
}

// 64 bits of a B-bit mask (Wb words) starting at bit position rel (may be negative or run past the end: zeros).
__device__ __forceinline__ uint64_t mask_bits(const uint64_t* __restrict__ mk, int64_t rel, uint32_t Wb) {
    uint64_t v = 0;
    if (rel <= -64 || rel >= (int64_t)Wb * 64) return 0;
    if (rel < 0) return __ldg(&mk[0]) << (uint32_t)(-rel);
    const uint32_t j = (uint32_t)(rel >> 6), s = (uint32_t)(rel & 63);
    v = __ldg(&mk[j]) >> s;
    if (s && j + 1 < Wb) v |= __ldg(&mk[j + 1]) << (64 - s);
    return v;
}

// k_residual: one warp per live block, one lane per bitmap word of the block.  Class constraints: AND of the class mask.
// Other residual constraints: the set bits left in the block (a handful on sparse spaces) are numbered across the words;
// the lanes take them 32 at a time and resume every such program from its stored prefix.  Failing bits are cleared with
// atomicAnd (this block's bits only); the survivors are added to the per-512 counts.
__global__ void __launch_bounds__(256) k_residual(const __grid_constant__ SpaceMeta sm, const __grid_constant__ EnumArgs a,
                                                  const ResPrefix* __restrict__ pre) {
    extern __shared__ int32_t s_enum[];
    const int32_t* desc = stage_desc(a, s_enum);
    const uint32_t lane = threadIdx.x & 31;
    const uint32_t nlive = *a.live_count;
    const uint64_t wid = ((uint64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = ((uint64_t)gridDim.x * blockDim.x) >> 5;
    for (uint64_t li = wid; li < nlive; li += nwarps) {
        const uint64_t o = a.live[li];
        const uint64_t g0 = o * a.B, g1 = g0 + a.B;                     // global bit range of the block
        const uint64_t w0 = g0 >> 6, w1 = (g1 + 63) >> 6;
        bool dead = false, generic = false;
        for (int r = 0; r < a.n_res; ++r) {
            const ResPrefix& q = pre[li * a.n_res + r];
            dead = dead || q.status == 0;
            generic = generic || (q.status >= 2 && q.cls == CAO_CLS_NONE);
        }
        int64_t x[CAO_MAX_DIMS];
        if (generic && !dead) {
            uint8_t dig[CAO_MAX_DIMS];
            decode_outer(sm, a.t, o, dig, 1);
            for (int d = 0; d < a.t; ++d) x[d] = a.dom[d * 256 + dig[d]];
        }
        for (uint64_t wb = w0; wb < w1; wb += 32) {                     // 32 bitmap words per pass, one per lane
            const uint64_t gw = wb + lane;
            uint64_t own = 0;
            if (gw < w1) {
                own = ~0ull;
                const uint64_t lo_bit = gw << 6;
                if (lo_bit < g0) own &= ~0ull << (g0 - lo_bit);
                if (lo_bit + 64 > g1) own &= ~0ull >> (lo_bit + 64 - g1);
            }
            const uint64_t orig = own ? (__ldcg(&a.bitmap[gw]) & own) : 0;    // written by k_masks (L2)
            uint64_t word = dead ? 0 : orig;
            for (int r = 0; r < a.n_res && word; ++r) {                 // class constraints: one mask word per lane
                const ResPrefix& q = pre[li * a.n_res + r];
                if (q.status != 2 || q.cls == CAO_CLS_NONE) continue;
                const uint64_t* tab = a.rc[a.rc_of[r]].table + (uint64_t)q.cls * a.Wb;
                word &= mask_bits(tab, (int64_t)(gw << 6) - (int64_t)g0, a.Wb);
            }
            if (generic && !dead) {
                const uint64_t snap = word;                             // the numbering of the set bits is fixed here
                const uint32_t pc = __popcll(word);
                uint32_t inc = pc;
#pragma unroll
                for (int s = 1; s < 32; s <<= 1) { const uint32_t v = __shfl_up_sync(0xFFFFFFFFu, inc, s); if (lane >= (uint32_t)s) inc += v; }
                const uint32_t tot = __shfl_sync(0xFFFFFFFFu, inc, 31), excl = inc - pc;
                for (uint32_t k0 = 0; k0 < tot; k0 += 32) {             // the k-th set bit of the pass goes to lane k - k0
                    const uint32_t k = k0 + lane;
                    uint32_t src = 0;                                   // owner word = last lane whose exclusive offset is <= k
#pragma unroll
                    for (int step = 16; step; step >>= 1) {
                        const uint32_t c = src + step;
                        const uint32_t oc = __shfl_sync(0xFFFFFFFFu, excl, c & 31);
                        if (c < 32 && oc <= k) src = c;
                    }
                    const uint64_t sw = __shfl_sync(0xFFFFFFFFu, snap, src);
                    const uint32_t se = __shfl_sync(0xFFFFFFFFu, excl, src);
                    bool fail = false; int bit = 0;
                    if (k < tot) {
                        bit = kth_set_bit64(sw, k - se);
                        uint64_t p = ((wb + src) << 6) + bit - g0;      // pattern inside the block
                        for (int d = sm.n - 1; d >= a.t; --d) {
                            const uint32_t m = sm.m[d]; uint32_t idx = 0;
                            if (m > 1) { const uint64_t p2 = div_magic(p, sm.magic[d]); idx = (uint32_t)(p - p2 * m); p = p2; }
                            x[d] = a.dom[d * 256 + idx];
                        }
                        for (int r = 0; r < a.n_res && !fail; ++r) {
                            const ResPrefix& q = pre[li * a.n_res + r];
                            if (q.status < 2 || q.cls != CAO_CLS_NONE) continue;
                            const int32_t* ds = desc + desc[a.n_tab + r];
                            int64_t st[CAO_MAX_STACK];
                            int u0, u1, pc0 = 0, sp0 = 0;
                            if (q.status == 2) { pc0 = q.pc; sp0 = q.sp; for (int z = 0; z < CAO_RES_STACK; ++z) st[z] = q.st[z]; }
                            fail = !eval_core(ds + 1, ds[0], x, pc0, st, sp0, -1, &u0, &u1);
                        }
                    }
                    // every lane hands its verdict to the lane that owns the word
                    for (uint32_t l2 = 0; l2 < 32; ++l2) {
                        const uint32_t s2 = __shfl_sync(0xFFFFFFFFu, src, l2);
                        const int b2 = __shfl_sync(0xFFFFFFFFu, bit, l2);
                        const bool f2 = __shfl_sync(0xFFFFFFFFu, (int)(fail && k < tot), l2) != 0;
                        if (f2 && s2 == lane) word &= ~(1ull << b2);
                    }
                }
            }
            const uint64_t kill = orig & ~word;
            if (kill) atomicAnd((unsigned long long*)&a.bitmap[gw], (unsigned long long)~kill);
            if (word) atomicAdd(&a.cnt[gw >> 3], (uint32_t)__popcll(word));
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
    if (base + 16 <= nd) {                                              // four independent 128-bit loads (the buffer is 256-byte aligned)
        const uint4* q = (const uint4*)(cnt + base);
        const uint4 a0 = q[0], a1 = q[1], a2 = q[2], a3 = q[3];
        s = a0.x + a0.y + a0.z + a0.w + a1.x + a1.y + a1.z + a1.w + a2.x + a2.y + a2.z + a2.w + a3.x + a3.y + a3.z + a3.w;
    } else {
        for (int k = 0; k < 16; ++k) if (base + k < nd) s += cnt[base + k];
    }
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
    if (base + 16 <= nd) {
        const uint4* q = (const uint4*)(cnt + base);
        const uint4 a0 = q[0], a1 = q[1], a2 = q[2], a3 = q[3];
        v[0] = a0.x; v[1] = a0.y; v[2] = a0.z; v[3] = a0.w; v[4] = a1.x; v[5] = a1.y; v[6] = a1.z; v[7] = a1.w;
        v[8] = a2.x; v[9] = a2.y; v[10] = a2.z; v[11] = a2.w; v[12] = a3.x; v[13] = a3.y; v[14] = a3.z; v[15] = a3.w;
    } else {
        for (int k = 0; k < 16; ++k) v[k] = (base + k < nd) ? cnt[base + k] : 0;
    }
    for (int k = 0; k < 16; ++k) s += v[k];
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

// Single-pass variant for cao_space_rebuild (the table address is known, so the two halves need no host round trip between
// them): decoupled look-back over the chunk sums.  CTAs take chunk numbers from a ticket (so every predecessor has started),
// publish state[b] = flag << 62 | value (flag 1: the chunk's own sum, 2: the inclusive prefix) and walk back over their
// predecessors until they meet an inclusive prefix.  state[] and the ticket must be zero on entry.  Same outputs as
// k_cnt_reduce + k_cnt_apply: directory, list of non-empty groups, V.
__global__ void __launch_bounds__(256) k_cnt_scan1(const uint32_t* __restrict__ cnt, uint64_t nd, unsigned long long* state, uint32_t* ticket,
                                                   uint32_t* dir, uint32_t* groups, uint32_t* group_count, uint64_t* V_out) {
    __shared__ uint32_t ws[8];
    __shared__ uint32_t s_b;
    __shared__ unsigned long long s_excl;
    if (threadIdx.x == 0) s_b = atomicAdd(ticket, 1u);
    __syncthreads();
    const uint32_t b = s_b;
    const uint64_t base = (uint64_t)b * SCAN_CHUNK + threadIdx.x * 16;
    uint32_t v[16], s = 0;
    if (base + 16 <= nd) {
        const uint4* q = (const uint4*)(cnt + base);
        const uint4 a0 = q[0], a1 = q[1], a2 = q[2], a3 = q[3];
        v[0] = a0.x; v[1] = a0.y; v[2] = a0.z; v[3] = a0.w; v[4] = a1.x; v[5] = a1.y; v[6] = a1.z; v[7] = a1.w;
        v[8] = a2.x; v[9] = a2.y; v[10] = a2.z; v[11] = a2.w; v[12] = a3.x; v[13] = a3.y; v[14] = a3.z; v[15] = a3.w;
    } else {
        for (int k = 0; k < 16; ++k) v[k] = (base + k < nd) ? cnt[base + k] : 0;
    }
    for (int k = 0; k < 16; ++k) s += v[k];
    uint32_t inc = s;
    for (int o = 1; o < 32; o <<= 1) { uint32_t t = __shfl_up_sync(0xFFFFFFFFu, inc, o); if ((threadIdx.x & 31) >= o) inc += t; }
    if ((threadIdx.x & 31) == 31) ws[threadIdx.x >> 5] = inc;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long total = 0;
        for (int k = 0; k < 8; ++k) total += ws[k];
        volatile unsigned long long* vs = state;
        if (b == 0) { vs[0] = (2ull << 62) | total; s_excl = 0; }
        else {
            vs[b] = (1ull << 62) | total;
            __threadfence();
            unsigned long long excl = 0;
            for (uint32_t j = b; j-- > 0;) {
                unsigned long long e;
                do { e = vs[j]; } while ((e >> 62) == 0);
                excl += e & ((1ull << 62) - 1);
                if ((e >> 62) == 2) break;
            }
            vs[b] = (2ull << 62) | (excl + total);
            s_excl = excl;
        }
        __threadfence();
        if (b + 1 == gridDim.x) { *V_out = s_excl + total; *ticket = 0; }
    }
    __syncthreads();
    uint32_t off = (uint32_t)s_excl;
    for (uint32_t k = 0; k < (threadIdx.x >> 5); ++k) off += ws[k];
    off += inc - s;
    uint32_t mine = 0;
    for (int k = 0; k < 16; ++k) mine += v[k] != 0;
    uint32_t incl = mine;
    for (int o = 1; o < 32; o <<= 1) { uint32_t t = __shfl_up_sync(0xFFFFFFFFu, incl, o); if ((threadIdx.x & 31) >= o) incl += t; }
    const uint32_t totalg = __shfl_sync(0xFFFFFFFFu, incl, 31);
    uint32_t gbase = 0;
    if ((threadIdx.x & 31) == 0 && totalg) gbase = atomicAdd(group_count, totalg);
    gbase = __shfl_sync(0xFFFFFFFFu, gbase, 0) + incl - mine;
    for (int k = 0; k < 16; ++k) {
        if (base + k < nd) dir[base + k] = off;
        off += v[k];
        if (v[k]) groups[gbase++] = (uint32_t)(base + k);
    }
}

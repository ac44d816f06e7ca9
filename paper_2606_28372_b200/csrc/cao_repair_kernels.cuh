// cao_repair_kernels.cuh -- S5: repair to the nearest valid configuration (O9).
//
// repair(c) = c if valid, else argmin over the valid table of (Hamming, sum |didx|, L).  Two exact routes:
//   probe : the Hamming-1 neighbours of c are tested in the bitmap by increasing |delta|; the first level
//           with a valid neighbour gives the minimum (1, |delta|, L') directly.
//   scan  : candidates without a valid Hamming-1 neighbour are compacted into a worklist; each CTA takes a
//           tile of 128 candidates (one per thread, row in registers) and a chunk of the valid table, staged
//           through shared memory in 512-row tiles and read back as broadcast LDS.128; per (candidate,row):
//           one VABSDIFF4.ACC per word for sum|didx|, a carry trick + one POPC per row for the Hamming count.
//           Chunks of the same candidate are merged with a 64-bit atomicMin on the packed key (order-free).
#pragma once
#include "cao_host.h"

// Hamming-1 probe of an INVALID, in-domain row with linear index L.  Returns the key or CAO_KEY_NONE.
template <int ROWW>
__device__ __forceinline__ uint64_t probe_h1(const SpaceMeta& sm, const uint32_t (&w)[ROWW], uint64_t L) {
    for (int delta = 1; delta < sm.M; ++delta) {
        // all bit tests of one |delta| level are independent loads (no short-circuit), so they overlap in flight
        uint64_t cand[ROWW * 8];
        bool hit[ROWW * 8];
#pragma unroll
        for (int d = 0; d < ROWW * 4; ++d) {
            const int c = (int)((w[d >> 2] >> ((d & 3) * 8)) & 0xFFu);
            const uint64_t step = d < sm.n ? (uint64_t)delta * sm.stride[d] : 0;
            const bool okm = d < sm.n && c >= delta, okp = d < sm.n && c + delta < (int)sm.m[d];
            cand[2 * d] = okm ? L - step : L;  cand[2 * d + 1] = okp ? L + step : L;
            hit[2 * d] = okm;                  hit[2 * d + 1] = okp;
        }
#pragma unroll
        for (int e = 0; e < ROWW * 8; ++e) hit[e] = hit[e] && bit_test(sm.bitmap, cand[e]);
        uint64_t bestL = ~0ull;
#pragma unroll
        for (int e = 0; e < ROWW * 8; ++e) if (hit[e] && cand[e] < bestL) bestL = cand[e];
        if (bestL != ~0ull) return make_key(1u, (uint32_t)delta, rank_of(sm, bestL));
    }
    return CAO_KEY_NONE;
}

// Validity + probe of one row; in_domain = every index byte is < m_d.
template <int ROWW>
__device__ __forceinline__ uint64_t validate_probe(const SpaceMeta& sm, const uint32_t (&w)[ROWW], bool use_probe, bool& valid) {
    bool in_dom = true;
#pragma unroll
    for (int d = 0; d < ROWW * 4; ++d)
        if (d < sm.n && ((w[d >> 2] >> ((d & 3) * 8)) & 0xFFu) >= sm.m[d]) in_dom = false;
    valid = false;
    if (!in_dom) return CAO_KEY_NONE;
    uint64_t L = row_lin<ROWW>(sm, w);
    if (bit_test(sm.bitmap, L)) { valid = true; return make_key(0, 0, rank_of(sm, L)); }
    return use_probe ? probe_h1<ROWW>(sm, w, L) : CAO_KEY_NONE;
}

// Appends `slot` to the worklist (warp-aggregated by the compiler's REDUX path or plain atomics; order-free).
__device__ __forceinline__ void worklist_push(uint32_t* wl, uint32_t* wl_count, uint32_t slot) {
    uint32_t pos = atomicAdd(wl_count, 1u);
    wl[pos] = slot;
}

// ---------------------------------------------------------------------------------------------
// Thread groups: G threads (a multiple of 32) that synchronise among themselves -- __syncwarp() for one warp, a named
// barrier otherwise.  The fused generation kernel runs several groups per CTA; the standalone probe kernel one.
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
__device__ __forceinline__ uint64_t warp_min_u64(uint64_t v) {
#pragma unroll
    for (int o = 16; o; o >>= 1) { uint64_t t = __shfl_xor_sync(0xFFFFFFFFu, v, o); v = t < v ? t : v; }
    return v;
}
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

// Appends the threads with `pred` to a list: returns this thread's position (one shared-memory atomic per warp).
__device__ __forceinline__ uint32_t grp_push(bool pred, uint32_t* counter, bool one_warp = false) {
    const uint32_t bal = __ballot_sync(0xFFFFFFFFu, pred), lane = threadIdx.x & 31;
    uint32_t base = 0;
    if (lane == 0 && bal) {
        if (one_warp) { base = *counter; *counter = base + (uint32_t)__popc(bal); }     // a single warp owns the counter
        else base = atomicAdd(counter, (uint32_t)__popc(bal));
    }
    base = __shfl_sync(0xFFFFFFFFu, base, 0);
    return base + __popc(bal & ((1u << lane) - 1u));
}

// Group-cooperative probe of ONE candidate c (n index bytes, in-domain, linear index L) at Hamming levels
// 2 .. pm.levels, in turn.  A row at Hamming distance exactly h is h neighbours (d, v != c_d) of strictly increasing
// dimension.  Every neighbour t contributes ptab[t] = (|v - c_d| << 40) + (v - c_d) * stride_d, so the packed key
// (sum |delta| << 40 | L') of a row is L + the sum of its neighbours' contributions (the fields cannot interfere:
// 0 <= L' < 2^40, sum |delta| < 2^13).  The first two neighbours come from the flattened pair list (spread over the
// threads, four independent bit tests in flight), levels >= 4 add a depth-first walk over the middle ones, the last one
// is a serial loop with eight loads in flight.  The level minimum is exact because Hamming is the primary key.  ptab:
// pm.NB words of shared memory owned by the group.  *slot must be ~0 and visible to the group on entry.  Returns the
// level that found a valid neighbour (0 = none), group-uniform, and leaves (sad << 40 | L') in *slot.
static __device__ __noinline__ int probe_levels_grp(const Grp g, const uint64_t* __restrict__ bitmap, const uint64_t* stride,
                                                    const ProbeMeta& pm, const uint16_t* nb, const uint32_t* pairs,
                                                    const uint8_t* c, uint64_t L, uint64_t* ptab, unsigned long long* slot) {
    const uint32_t NB = pm.NB, C2 = pm.C2;
    const uint64_t M40 = (1ull << 40) - 1;
    for (uint32_t t = g.t; t < NB; t += g.G) {
        const uint32_t e = nb[t], d = e >> 8, kq = e & 255u, cd = c[d];
        const int dv = (int)(kq + (kq >= cd)) - (int)cd;
        ptab[t] = ((uint64_t)(uint32_t)abs(dv) << 40) + (uint64_t)((int64_t)dv * (int64_t)stride[d]);
    }
    g.sync();
    for (int level = 2; level <= pm.levels; ++level) {
        uint64_t best = ~0ull;
        if (level == 2) {
            for (uint32_t q0 = 0; q0 < C2; q0 += 4 * g.G) {             // four independent bit tests per thread and pass
                uint64_t k2[4]; bool bit[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const uint32_t q = q0 + u * g.G + g.t;
                    const uint32_t pr = pairs[q < C2 ? q : 0];
                    k2[u] = L + ptab[pr & 0xFFFFu] + ptab[pr >> 16];
                    bit[u] = bit_test(bitmap, k2[u] & M40) && q < C2;
                }
#pragma unroll
                for (int u = 0; u < 4; ++u) if (bit[u]) best = k2[u] < best ? k2[u] : best;
            }
        } else if (level == 3 && pm.C3) {
            const uint32_t C3 = pm.C3;                                  // flat triple list: eight independent bit tests per thread and pass
            const uint32_t* __restrict__ tri = pm.triples;
            for (uint32_t q0 = 0; q0 < C3; q0 += 8 * g.G) {
                uint64_t k3[8]; bool bit[8];
#pragma unroll
                for (int u = 0; u < 8; ++u) {
                    const uint32_t q = q0 + u * g.G + g.t;
                    const uint32_t tr = __ldg(&tri[q < C3 ? q : 0]);
                    k3[u] = L + ptab[tr & 1023u] + ptab[(tr >> 10) & 1023u] + ptab[tr >> 20];
                    bit[u] = bit_test(bitmap, k3[u] & M40) && q < C3;
                }
#pragma unroll
                for (int u = 0; u < 8; ++u) if (bit[u]) best = k3[u] < best ? k3[u] : best;
            }
        } else {
            const int extra = level - 3;                                // middle neighbours walked depth-first (0 .. 3)
            for (uint32_t q = g.t; q < C2; q += g.G) {
                const uint32_t pr = pairs[q];
                uint64_t Kst[CAO_MAX_PROBE_LEVEL - 2]; uint32_t tcur[CAO_MAX_PROBE_LEVEL - 2];
                Kst[0] = L + ptab[pr & 0xFFFFu] + ptab[pr >> 16];
                tcur[0] = pm.nb_first[(nb[pr >> 16] >> 8) + 1];
                int depth = 0;
                for (;;) {
                    if (depth == extra) {                               // innermost neighbour: serial loop, 8 loads in flight
                        const uint64_t Kb = Kst[depth];
                        for (uint32_t t0 = tcur[depth]; t0 < NB; t0 += 8) {
                            uint64_t k3[8]; bool bit[8];
#pragma unroll
                            for (int u = 0; u < 8; ++u) {
                                k3[u] = Kb + ptab[t0 + u < NB ? t0 + u : t0];
                                bit[u] = bit_test(bitmap, k3[u] & M40) && t0 + u < NB;
                            }
#pragma unroll
                            for (int u = 0; u < 8; ++u) if (bit[u]) best = k3[u] < best ? k3[u] : best;
                        }
                        if (depth == 0) break;
                        --depth; ++tcur[depth];
                        continue;
                    }
                    if (tcur[depth] >= NB) {                            // this middle position is exhausted
                        if (depth == 0) break;
                        --depth; ++tcur[depth];
                        continue;
                    }
                    const uint32_t tm = tcur[depth];
                    Kst[depth + 1] = Kst[depth] + ptab[tm];
                    tcur[depth + 1] = pm.nb_first[(nb[tm] >> 8) + 1];
                    ++depth;
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

// Hamming >= 2 probe of the worklist: one CTA per candidate.  Candidates without a valid neighbour up to `pm.levels`
// go on to the table scan (wl_out).
template <int ROWW>
__global__ void __launch_bounds__(256) k_probe23(const __grid_constant__ SpaceMeta sm, const __grid_constant__ ProbeMeta pm,
                                                 const uint8_t* __restrict__ cand_rows, const uint32_t* __restrict__ wl,
                                                 const uint32_t* __restrict__ wl_count, unsigned long long* key,
                                                 uint32_t* wl_out, uint32_t* wl_out_count, unsigned long long* n_scanned) {
    __shared__ __align__(16) uint32_t s_cw[ROWW];
    __shared__ unsigned long long s_best;
    __shared__ uint64_t s_stride[CAO_MAX_DIMS];
    __shared__ uint64_t s_ptab[CAO_MAX_NB_PROBE];
    const uint32_t count = *wl_count, tid = threadIdx.x;
    if (tid < (uint32_t)sm.n) s_stride[tid] = sm.stride[tid];
    const Grp g{tid, blockDim.x, 0};
    for (uint32_t ci = blockIdx.x; ci < count; ci += gridDim.x) {
        const uint32_t slot = wl[ci];
        __syncthreads();
        if (tid < ROWW) s_cw[tid] = ((const uint32_t*)(cand_rows + (uint64_t)slot * (ROWW * 4)))[tid];
        if (tid == 0) s_best = ~0ull;
        __syncthreads();
        uint64_t Lc = 0;
        for (int d = 0; d < sm.n; ++d) Lc += (uint64_t)((const uint8_t*)s_cw)[d] * s_stride[d];
        const int found = probe_levels_grp(g, sm.bitmap, s_stride, pm, pm.nb, pm.pairs, (const uint8_t*)s_cw, Lc, s_ptab, &s_best);
        if (tid == 0) {
            const uint64_t best = s_best;
            if (found) key[slot] = make_key((uint32_t)found, (uint32_t)(best >> 40), rank_of(sm, best & ((1ull << 40) - 1)));
            else { wl_out[atomicAdd(wl_out_count, 1u)] = slot; if (n_scanned) atomicAdd(n_scanned, 1ull); }
        }
    }
}

#define SCAN_TC 128          // candidates per tile = threads per CTA
#define SCAN_TR 512          // valid rows per shared-memory tile

// WU = words of a row that carry indices (ceil(n/4)); row stride in HBM = 4 or 8 words.
// SMALL: every index < 128, so a byte of c^v is non-zero iff adding 0x7f carries into its bit 7.
// KM: key layout.  0 = north_star's (Hamming << 13 + sum|didx|) << 32 | rank; 1 = NEXT-1 index distance (L215, L270):
// sum|didx| << 32 | rank (the Hamming count is not computed).
// 16-byte asynchronous global -> shared copy (LDGSTS; bypasses registers and L1) and its group fences.
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(smem_dst)), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

template <int WU, bool SMALL, int KM = 0>
__global__ void __launch_bounds__(SCAN_TC) k_scan(const __grid_constant__ SpaceMeta sm, const uint8_t* __restrict__ cand_rows,
                                                  const uint32_t* __restrict__ wl, const uint32_t* __restrict__ wl_count,
                                                  unsigned long long* key) {
    constexpr int ROWW = WU <= 4 ? 4 : 8;
    constexpr int TQ = SCAN_TR * (ROWW / 4);                             // 16-byte quads per tile
    __shared__ uint4 tile[2][TQ];                                        // double buffer: tile rt+1 streams in (cp.async) while rt is scanned
    const uint32_t count = *wl_count;
    if (count == 0 || sm.V == 0) return;
    const uint32_t tid = threadIdx.x;
    const uint32_t ntiles = (count + SCAN_TC - 1) / SCAN_TC;
    const uint32_t nrt = (sm.V + SCAN_TR - 1) / SCAN_TR;                 // row tiles in the table
    uint32_t nchunks = gridDim.x / ntiles; if (nchunks < 1) nchunks = 1; if (nchunks > nrt) nchunks = nrt;
    const uint32_t tpc = (nrt + nchunks - 1) / nchunks;                  // row tiles per chunk
    nchunks = (nrt + tpc - 1) / tpc;
    const uint64_t items = (uint64_t)ntiles * nchunks;
    const uint4* table = (const uint4*)sm.rows;
    auto stage = [&](uint32_t rt, int buf) {                             // issue the copies of row tile rt into buffer buf
        const uint32_t r0 = rt * SCAN_TR, nr = min((uint32_t)SCAN_TR, sm.V - r0);
        const uint4* src = table + (uint64_t)r0 * (ROWW / 4);
        for (uint32_t q = tid; q < nr * (ROWW / 4); q += SCAN_TC) cp_async16(&tile[buf][q], &src[q]);
        cp_async_commit();
    };
    for (uint64_t item = blockIdx.x; item < items; item += gridDim.x) {
        const uint32_t ct = (uint32_t)(item / nchunks), rc = (uint32_t)(item - (uint64_t)ct * nchunks);
        const uint32_t ci = ct * SCAN_TC + tid;
        const bool has = ci < count;
        const uint32_t slot = has ? wl[ci] : 0;
        uint32_t c[ROWW];
        if (has) load_row_rw<ROWW>(cand_rows + (uint64_t)slot * (ROWW * 4), c);
        else { for (int k = 0; k < ROWW; ++k) c[k] = 0; }
        uint32_t bestk = 0xFFFFFFFFu, bestr = 0xFFFFFFFFu;
        uint32_t rt1 = (rc + 1) * tpc; if (rt1 > nrt) rt1 = nrt;
        const uint32_t rt0 = rc * tpc;
        __syncthreads();                                                 // the previous item's last tile is no longer read
        if (rt0 < rt1) stage(rt0, 0);
        for (uint32_t rt = rt0; rt < rt1; ++rt) {
            const int buf = (int)((rt - rt0) & 1u);
            if (rt + 1 < rt1) { stage(rt + 1, buf ^ 1); cp_async_wait<1>(); }   // (buf ^ 1 was released by the barrier below)
            else cp_async_wait<0>();
            __syncthreads();                                             // tile rt has landed for every thread
            const uint32_t r0 = rt * SCAN_TR;
            const uint32_t nr = min((uint32_t)SCAN_TR, sm.V - r0);
            const uint4* tl = tile[buf];
#pragma unroll 4
            for (uint32_t r = 0; r < nr; ++r) {
                uint32_t v[ROWW];
                { uint4 a = tl[r * (ROWW / 4)]; v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w; }
                if (ROWW == 8) { uint4 b = tl[r * 2 + 1]; v[4] = b.x; v[5] = b.y; v[6] = b.z; v[7] = b.w; }
                // Per index word: ad = per-byte |c - v| (one VABSDIFF4), then both sums come from IDP.4A (dot product with
                // 0x01010101), which issues on the fma pipe -- no POPC (quarter rate), no XOR, no flag merging:
                //   sum |delta idx| = sum of the bytes of ad;
                //   SMALL (every index < 128): t = ad + 0x7f7f7f7f has byte 127 where ad_b = 0 and 128 + (ad_b - 1) otherwise, i.e.
                //   as SIGNED bytes t_b = ad_b + 127 - 256 [ad_b != 0], so 256 * Hamming = sum ad_b + 508 per word - sum s8(t_b).
                //   general: flags f = 0x80 per differing byte from the carry trick on c ^ v, 128 * Hamming = sum f_b.
                uint32_t sad = 0, fs = 0; int ts = 0;
#pragma unroll
                for (int k = 0; k < WU; ++k) {
                    if (KM == 0 && SMALL) {
                        const uint32_t ad = __vabsdiffu4(c[k], v[k]);
                        sad = __dp4a(ad, 0x01010101u, sad);
                        ts = __dp4a((int)(ad + 0x7f7f7f7fu), 0x01010101, ts);
                    } else {
                        sad = sad4_acc(c[k], v[k], sad);
                        if (KM == 0) {
                            const uint32_t x = c[k] ^ v[k];
                            const uint32_t t = ((x & 0x7f7f7f7fu) + 0x7f7f7f7fu) | x;
                            fs = __dp4a(t & 0x80808080u, 0x01010101u, fs);
                        }
                    }
                }
                const uint32_t hamk = SMALL ? ((sad + 508u * WU - (uint32_t)ts) << 5) : (fs << 6);      // Hamming << 13
                uint32_t k32 = KM == 1 ? sad : hamk + sad;
                if (k32 < bestk) { bestk = k32; bestr = r0 + r; }         // ascending rank: ties keep the smallest L
            }
            __syncthreads();                                             // everyone is done with tile rt: its buffer may be refilled
        }
        if (has && bestr != 0xFFFFFFFFu) atomicMin(&key[slot], ((unsigned long long)bestk << 32) | bestr);
    }
}

// ---------------------------------------------------------------------------------------------
// Standalone batched repair (cao_space_repair): probe kernel, k_probe23, k_scan, finish kernel.  The caller's rows are
// copied to `clean` with the padding bytes (positions >= n) zeroed, so that padding never adds to Hamming or sum |d|;
// rows with an index outside its domain are invalid and skip the neighbour probes (A27): they go straight to the scan.
template <int ROWW>
__global__ void __launch_bounds__(256) k_repair_probe(const __grid_constant__ SpaceMeta sm, const uint8_t* __restrict__ rows_in,
                                                      uint8_t* clean, uint64_t count, int use_probe, unsigned long long* key,
                                                      uint32_t* wl, uint32_t* wl_count, uint32_t* wl2, uint32_t* wl2_count) {
    uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= count) return;
    uint32_t w[ROWW];
    load_row<ROWW>(rows_in + i * (ROWW * 4), w);
#pragma unroll
    for (int z = 0; z < ROWW; ++z) {
        const int first = z * 4;
        if (first >= sm.n) w[z] = 0;
        else if (first + 4 > sm.n) w[z] &= 0xFFFFFFFFu >> (8 * (first + 4 - sm.n));
    }
    store_row<ROWW>(clean + i * (ROWW * 4), w);
    bool valid;
    bool in_dom = true;
#pragma unroll
    for (int d = 0; d < ROWW * 4; ++d)
        if (d < sm.n && ((w[d >> 2] >> ((d & 3) * 8)) & 0xFFu) >= sm.m[d]) in_dom = false;
    uint64_t k = validate_probe<ROWW>(sm, w, use_probe != 0, valid);
    key[i] = k;
    if (k == CAO_KEY_NONE) { if (in_dom && wl2 != wl) worklist_push(wl, wl_count, (uint32_t)i); else worklist_push(wl2, wl2_count, (uint32_t)i); }
}

static __global__ void __launch_bounds__(256) k_repair_finish(const unsigned long long* __restrict__ key, uint64_t count,
                                                       uint32_t* rank_out, uint64_t* key_out) {
    uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= count) return;
    unsigned long long k = key[i];
    if (rank_out) rank_out[i] = (uint32_t)k;
    if (key_out) key_out[i] = k;
}

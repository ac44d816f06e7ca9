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
// Hamming-2 / Hamming-3 probe of the worklist: one CTA per candidate.  All index rows at Hamming distance
// exactly h are enumerated as h targets (dimension, value) of strictly increasing dimension; the outer
// targets are walked by the whole warp, the innermost one is spread over the lanes.  Each probe is one bit
// test at L + sum (v - c) * stride; the level minimum of (sum |v - c|, L') is exact because Hamming is the
// primary key.  Candidates without a valid neighbour up to `levels` go on to the table scan (wl_out).
__device__ __forceinline__ uint64_t warp_min_u64(uint64_t v) {
#pragma unroll
    for (int o = 16; o; o >>= 1) { uint64_t t = __shfl_xor_sync(0xFFFFFFFFu, v, o); v = t < v ? t : v; }
    return v;
}

// Block-cooperative probe of ONE candidate whose row sits in shared memory (s_cw, ROWW words).  *s_best must be
// ~0 and visible to the block on entry.  Threads walk the flattened list of target pairs (t1 < t2, different
// dimensions); level 3 adds a serial walk over the targets of the dimensions after t2's.  Returns the level
// that found a valid neighbour (0 = none) -- block-uniform -- and leaves (sad << 40 | L') in *s_best.
template <int ROWW>
__device__ __forceinline__ int probe23_cta(const SpaceMeta& sm, const ProbeMeta& pm, const uint32_t* s_cw,
                                           unsigned long long* s_best) {
    const uint8_t* c = (const uint8_t*)s_cw;
    const uint32_t tid = threadIdx.x, T = pm.T, C2 = pm.C2;
    uint64_t L = 0;
    for (int d = 0; d < sm.n; ++d) L += (uint64_t)c[d] * sm.stride[d];
    int found = 0;
    for (int level = 2; level <= pm.levels && !found; ++level) {
        uint64_t best = ~0ull;
        for (uint32_t q = tid; q < C2; q += blockDim.x) {
            const uint32_t pr = __ldg(&pm.pairs[q]);
            const uint32_t e1 = __ldg(&pm.tgt[pr & 0xFFFFu]), e2 = __ldg(&pm.tgt[pr >> 16]);
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
                    const uint32_t e3 = __ldg(&pm.tgt[t3]), d3 = e3 >> 8;
                    const int dv3 = (int)(e3 & 255) - (int)c[d3];
                    const uint64_t L3 = L2 + (int64_t)dv3 * (int64_t)sm.stride[d3];
                    const bool bit3 = bit_test(sm.bitmap, L3);              // unconditional: dv3 == 0 re-reads L2 (a legal index)
                    if (dv3 != 0 && bit3) { uint64_t k = ((uint64_t)(s2 + (uint32_t)abs(dv3)) << 40) | L3; best = k < best ? k : best; }
                }
            }
        }
        best = warp_min_u64(best);
        if ((tid & 31) == 0 && best != ~0ull) atomicMin(s_best, best);
        __syncthreads();
        const bool hit = *s_best != ~0ull;
        __syncthreads();                                                // everyone has read the slot before the next level writes it
        if (hit) found = level;
    }
    return found;
}

template <int ROWW>
__global__ void __launch_bounds__(256) k_probe23(const __grid_constant__ SpaceMeta sm, const __grid_constant__ ProbeMeta pm,
                                                 const uint8_t* __restrict__ cand_rows, const uint32_t* __restrict__ wl,
                                                 const uint32_t* __restrict__ wl_count, unsigned long long* key,
                                                 uint32_t* wl_out, uint32_t* wl_out_count, unsigned long long* n_scanned) {
    // One CTA per worklist candidate.
    __shared__ uint32_t s_cw[ROWW];
    __shared__ unsigned long long s_best;
    const uint32_t count = *wl_count, tid = threadIdx.x;
    for (uint32_t ci = blockIdx.x; ci < count; ci += gridDim.x) {
        const uint32_t slot = wl[ci];
        __syncthreads();
        if (tid < ROWW) s_cw[tid] = ((const uint32_t*)(cand_rows + (uint64_t)slot * (ROWW * 4)))[tid];
        if (tid == 0) s_best = ~0ull;
        __syncthreads();
        const int found = probe23_cta<ROWW>(sm, pm, s_cw, &s_best);
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
template <int WU, bool SMALL>
__global__ void __launch_bounds__(SCAN_TC) k_scan(const __grid_constant__ SpaceMeta sm, const uint8_t* __restrict__ cand_rows,
                                                  const uint32_t* __restrict__ wl, const uint32_t* __restrict__ wl_count,
                                                  unsigned long long* key) {
    constexpr int ROWW = WU <= 4 ? 4 : 8;
    __shared__ uint4 tile[SCAN_TR * (ROWW / 4)];
    const uint32_t count = *wl_count;
    if (count == 0 || sm.V == 0) return;
    const uint32_t tid = threadIdx.x;
    const uint32_t ntiles = (count + SCAN_TC - 1) / SCAN_TC;
    const uint32_t nrt = (sm.V + SCAN_TR - 1) / SCAN_TR;                 // row tiles in the table
    uint32_t nchunks = gridDim.x / ntiles; if (nchunks < 1) nchunks = 1; if (nchunks > nrt) nchunks = nrt;
    const uint32_t tpc = (nrt + nchunks - 1) / nchunks;                  // row tiles per chunk
    nchunks = (nrt + tpc - 1) / tpc;
    const uint64_t items = (uint64_t)ntiles * nchunks;
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
        for (uint32_t rt = rc * tpc; rt < rt1; ++rt) {
            const uint32_t r0 = rt * SCAN_TR;
            const uint32_t nr = min((uint32_t)SCAN_TR, sm.V - r0);
            __syncthreads();
            const uint4* src = (const uint4*)(sm.rows + (uint64_t)r0 * (ROWW * 4));
            for (uint32_t q = tid; q < nr * (ROWW / 4); q += SCAN_TC) tile[q] = __ldg(&src[q]);
            __syncthreads();
#pragma unroll 4
            for (uint32_t r = 0; r < nr; ++r) {
                uint32_t v[ROWW];
                { uint4 a = tile[r * (ROWW / 4)]; v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w; }
                if (ROWW == 8) { uint4 b = tile[r * 2 + 1]; v[4] = b.x; v[5] = b.y; v[6] = b.z; v[7] = b.w; }
                uint32_t sad = 0, hb = 0, ham = 0;
#pragma unroll
                for (int k = 0; k < WU; ++k) {
                    sad = sad4_acc(c[k], v[k], sad);
                    uint32_t x = c[k] ^ v[k];
                    uint32_t t = SMALL ? (x + 0x7f7f7f7fu) : (((x & 0x7f7f7f7fu) + 0x7f7f7f7fu) | x);
                    if ((k & 3) == 0 && k) { ham += __popc(hb); hb = 0; }
                    hb |= (t & 0x80808080u) >> (k & 3);
                }
                ham += __popc(hb);
                uint32_t k32 = (ham << 13) + sad;
                if (k32 < bestk) { bestk = k32; bestr = r0 + r; }         // ascending rank: ties keep the smallest L
            }
        }
        if (has && bestr != 0xFFFFFFFFu) atomicMin(&key[slot], ((unsigned long long)bestk << 32) | bestr);
    }
}

// ---------------------------------------------------------------------------------------------
// Standalone batched repair (cao_space_repair): probe kernel, k_scan, finish kernel.
template <int ROWW>
__global__ void __launch_bounds__(256) k_repair_probe(const __grid_constant__ SpaceMeta sm, const uint8_t* __restrict__ rows_in,
                                                      uint64_t count, int use_probe, unsigned long long* key,
                                                      uint32_t* wl, uint32_t* wl_count, uint32_t* wl2, uint32_t* wl2_count) {
    uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= count) return;
    uint32_t w[ROWW];
    load_row<ROWW>(rows_in + i * (ROWW * 4), w);
    bool valid;
    bool in_dom = true;
#pragma unroll
    for (int d = 0; d < ROWW * 4; ++d)
        if (d < sm.n && ((w[d >> 2] >> ((d & 3) * 8)) & 0xFFu) >= sm.m[d]) in_dom = false;
    uint64_t k = validate_probe<ROWW>(sm, w, use_probe != 0, valid);
    key[i] = k;
    // rows with an index outside its domain skip the neighbour probes and go straight to the scan (wl2)
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

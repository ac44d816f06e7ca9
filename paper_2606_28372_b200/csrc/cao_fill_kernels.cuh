// cao_fill_kernels.cuh -- S1 pass 2 (valid table from the bitmap) and the batched is-valid query.
#pragma once
#include "cao_host.h"

// Decode L into index bytes packed in ROWW uint32 words (4 bytes per word, padding zero).
template <int ROWW>
__device__ __forceinline__ void decode_row(const SpaceMeta& sm, uint64_t L, uint32_t (&w)[ROWW]) {
#pragma unroll
    for (int k = 0; k < ROWW; ++k) w[k] = 0;
#pragma unroll
    for (int d = ROWW * 4 - 1; d >= 0; --d) {
        if (d < sm.n) {
            uint32_t m = sm.m[d];
            if (m > 1) {
                uint64_t q = div_magic(L, sm.magic[d]);
                uint32_t idx = (uint32_t)(L - q * m);
                L = q;
                w[d >> 2] |= idx << ((d & 3) * 8);
            }
        }
    }
}

// A warp owns 32 consecutive 512-config groups per pass (grid-stride): lane l reads the directory count of
// group g0 + l, so sparse regions cost one directory word per 512 configs and nothing else.  Groups are then
// processed in pairs (32 half words of the bitmap = 1024 configs): a shuffle scan gives each half word its
// first rank; the pair's W rows are contiguous in the table and are produced one row per lane -- output j
// belongs to the last lane t with offset o_t <= j (binary search over the 32 offsets in shared memory), its
// config is the (j - o_t)-th set bit of that lane's half word.  Row and Ltab stores are fully coalesced.
template <int ROWW>
__global__ void __launch_bounds__(256) k_fill(const __grid_constant__ SpaceMeta sm, uint64_t n_words,
                                              uint8_t* rows, uint64_t* Ltab, uint32_t* dir_out,
                                              const uint32_t* __restrict__ dir, uint64_t nd, uint32_t gpw) {
    // gpw = groups per warp pass: 2 for dense spaces (one pair per warp, maximum parallelism), 32 for sparse ones
    __shared__ uint32_t s_off[8][33];
    __shared__ uint32_t s_bits[8][32];
    const uint32_t lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const uint64_t nwarps = (uint64_t)gridDim.x * 8, wid = (uint64_t)blockIdx.x * 8 + wib;
    for (uint64_t g0 = wid * gpw; g0 < nd; g0 += nwarps * gpw) {
        const uint64_t gl = g0 + lane;
        uint32_t gbase = 0, gcnt = 0;
        if (lane < gpw && gl < nd) {
            gbase = dir[gl]; gcnt = dir[gl + 1] - gbase;
            dir_out[gl] = gbase;
            if (gl + 1 == nd) dir_out[nd] = gbase + gcnt;
        }
        const uint32_t nonempty = __ballot_sync(0xFFFFFFFFu, gcnt != 0);
        for (uint32_t pp = 0; pp < gpw / 2; ++pp) {
            if (!((nonempty >> (2 * pp)) & 3u)) continue;               // both groups of the pair are empty
            const uint64_t g = g0 + 2 * pp + (lane >> 4);                // this lane's group
            const uint32_t base = __shfl_sync(0xFFFFFFFFu, gbase, 2 * pp + (lane >> 4));
            const uint32_t cnt = __shfl_sync(0xFFFFFFFFu, gcnt, 2 * pp + (lane >> 4));
            const uint64_t hw = g * 16 + (lane & 15);
            uint32_t bits = 0;
            if (cnt && g < nd && hw < 2 * n_words) bits = ((const uint32_t*)sm.bitmap)[hw];
            const uint32_t pc = __popc(bits);
            uint32_t inc = pc;
#pragma unroll
            for (int o = 1; o < 16; o <<= 1) { uint32_t t = __shfl_up_sync(0xFFFFFFFFu, inc, o, 16); if ((lane & 15) >= o) inc += t; }
            const uint32_t r = base + inc - pc;                          // rank of this half word's first valid config
            const uint32_t r0 = __shfl_sync(0xFFFFFFFFu, r, 0);
            const uint32_t off = g < nd ? r - r0 : 0xFFFFFFFFu;          // lanes past the directory own no rows
            __syncwarp();
            s_off[wib][lane] = off; s_bits[wib][lane] = bits;
            uint32_t tot = pc;
#pragma unroll
            for (int o = 16; o; o >>= 1) tot += __shfl_xor_sync(0xFFFFFFFFu, tot, o);
            __syncwarp();
            const uint64_t hw0 = (g0 + 2 * pp) * 16;
            for (uint32_t j = lane; j < tot; j += 32) {
                uint32_t t = 0;                                          // last lane with off <= j
#pragma unroll
                for (int step = 16; step; step >>= 1) { const uint32_t c = t + step; if (c < 32 && s_off[wib][c] <= j) t = c; }
                const uint32_t b = (uint32_t)kth_set_bit32(s_bits[wib][t], j - s_off[wib][t]);
                const uint64_t L = (hw0 + t) * 32 + b;
                uint32_t w[ROWW];
                decode_row<ROWW>(sm, L, w);
                const uint64_t rr = (uint64_t)r0 + j;
                uint4* dst = (uint4*)(rows + rr * (ROWW * 4));
                dst[0] = make_uint4(w[0], w[1], w[2], w[3]);
                if (ROWW == 8) dst[1] = make_uint4(w[4], w[5], w[6], w[7]);
                Ltab[rr] = L;
            }
        }
    }
}

// Batched Search Space query "is valid" (L139): out[i] = bitmap[L(row_i)]; rows with an index out of its
// domain are invalid.
template <int ROWW>
__global__ void __launch_bounds__(256) k_is_valid(const __grid_constant__ SpaceMeta sm, const uint8_t* __restrict__ rows_in,
                                                  uint64_t count, uint8_t* out) {
    uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= count) return;
    const uint4* src = (const uint4*)(rows_in + i * (ROWW * 4));
    uint32_t w[ROWW];
    uint4 a = __ldg(&src[0]); w[0] = a.x; w[1] = a.y; w[2] = a.z; w[3] = a.w;
    if (ROWW == 8) { uint4 b = __ldg(&src[1]); w[4] = b.x; w[5] = b.y; w[6] = b.z; w[7] = b.w; }
    bool ok = true;
#pragma unroll
    for (int d = 0; d < ROWW * 4; ++d)
        if (d < sm.n && ((w[d >> 2] >> ((d & 3) * 8)) & 0xFFu) >= sm.m[d]) ok = false;
    out[i] = ok ? (uint8_t)bit_test(sm.bitmap, row_lin<ROWW>(sm, w)) : (uint8_t)0;
}

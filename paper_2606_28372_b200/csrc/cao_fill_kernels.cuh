// cao_fill_kernels.cuh -- S1 pass 2 (valid table from the bitmap) and the batched is-valid query.
#pragma once
#include "cao_host.h"

// Decode L into index bytes packed in ROWW uint32 words (4 bytes per word, padding zero); digits [d_lo, d_hi).
template <int ROWW>
__device__ __forceinline__ void decode_digits(const SpaceMeta& sm, uint64_t q, int d_lo, int d_hi, uint32_t (&w)[ROWW]) {
#pragma unroll
    for (int k = 0; k < ROWW; ++k) w[k] = 0;
    for (int d = d_hi - 1; d >= d_lo; --d) {
        const uint32_t m = sm.m[d];
        if (m > 1) {
            const uint64_t q2 = div_magic(q, sm.magic[d]);
            const uint32_t idx = (uint32_t)(q - q2 * m);
            q = q2;
#pragma unroll
            for (int k = 0; k < ROWW; ++k) if (k == (d >> 2)) w[k] |= idx << ((d & 3) * 8);
        }
    }
}

// One warp per NON-EMPTY 512-config group (list from k_cnt_apply, any order; grid-stride).  Lane l < 16 holds half word
// l of the group's bitmap; a shuffle scan gives each half word its first rank; the group's rows -- contiguous in the
// table from dir[g] -- are produced one per lane: output j belongs to the last half word with offset <= j (binary
// search in shared memory), its config is the (j - offset)-th set bit.  A group spans at most three blocks of B configs
// (B >= 256): lanes 0..2 decode their outer digits once, the inner index bytes come from the lookup table of k_inner_lut
// (lut == nullptr: decode them too).  Row (uint4) and Ltab stores are coalesced.
template <int ROWW, bool L32>
__global__ void __launch_bounds__(256) k_fill(const __grid_constant__ SpaceMeta sm, uint64_t n_words, uint8_t* rows, void* Ltab,
                                              const uint32_t* __restrict__ dir, const uint32_t* __restrict__ groups,
                                              const uint32_t* __restrict__ group_count, const uint32_t* __restrict__ lut,
                                              uint64_t B, uint64_t magicB, int32_t t) {
    __shared__ uint32_t s_off[8][17];
    __shared__ uint32_t s_bits[8][16];
    __shared__ __align__(16) uint32_t s_outer[8][3][ROWW];
    const uint32_t lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const uint32_t ngroups = *group_count;
    const uint64_t nwarps = (uint64_t)gridDim.x * 8, wid = (uint64_t)blockIdx.x * 8 + wib;
    for (uint64_t li = wid; li < ngroups; li += nwarps) {
        const uint64_t g = groups[li];
        const uint32_t r0 = dir[g];
        const uint64_t hw = g * 16 + (lane & 15);
        uint32_t bits = 0;
        if (lane < 16 && hw < 2 * n_words) bits = ((const uint32_t*)sm.bitmap)[hw];
        const uint32_t pc = __popc(bits);
        uint32_t inc = pc;
#pragma unroll
        for (int o = 1; o < 16; o <<= 1) { uint32_t v = __shfl_up_sync(0xFFFFFFFFu, inc, o, 16); if ((lane & 15) >= o) inc += v; }
        const uint32_t tot = __shfl_sync(0xFFFFFFFFu, inc, 15);
        const uint64_t L0 = g << CAO_DIR_SHIFT;
        const uint64_t o_first = B > 1 ? div_magic(L0, magicB) : L0;
        __syncwarp();
        if (lane < 16) { s_off[wib][lane] = inc - pc; s_bits[wib][lane] = bits; }
        if (lane == 16) s_off[wib][16] = 0xFFFFFFFFu;
        if (lane < 3) {
            uint32_t w[ROWW];
            decode_digits<ROWW>(sm, o_first + lane, 0, t, w);           // blocks past the end decode to garbage nobody reads
#pragma unroll
            for (int k = 0; k < ROWW; ++k) s_outer[wib][lane][k] = w[k];
        }
        __syncwarp();
        for (uint32_t j = lane; j < tot; j += 32) {
            uint32_t tt = 0;                                             // last half word with off <= j
#pragma unroll
            for (int step = 8; step; step >>= 1) { const uint32_t c = tt + step; if (s_off[wib][c] <= j) tt = c; }
            const uint32_t b = (uint32_t)kth_set_bit32(s_bits[wib][tt], j - s_off[wib][tt]);
            const uint64_t L = L0 + tt * 32 + b;
            const uint64_t o = B > 1 ? div_magic(L, magicB) : L;
            const uint64_t p = L - o * B;
            uint32_t w[ROWW];
            if (lut) {
                const uint4* q = (const uint4*)(lut + p * ROWW);
                const uint4 a = __ldg(&q[0]); w[0] = a.x; w[1] = a.y; w[2] = a.z; w[3] = a.w;
                if (ROWW == 8) { const uint4 c = __ldg(&q[1]); w[4] = c.x; w[5] = c.y; w[6] = c.z; w[7] = c.w; }
            } else {
                decode_digits<ROWW>(sm, p, t, sm.n, w);
            }
            const uint32_t* ob = s_outer[wib][(uint32_t)(o - o_first)];
#pragma unroll
            for (int k = 0; k < ROWW; ++k) w[k] |= ob[k];
            const uint64_t rr = (uint64_t)r0 + j;
            uint4* dst = (uint4*)(rows + rr * (ROWW * 4));
            dst[0] = make_uint4(w[0], w[1], w[2], w[3]);
            if (ROWW == 8) dst[1] = make_uint4(w[4], w[5], w[6], w[7]);
            if (L32) ((uint32_t*)Ltab)[rr] = (uint32_t)L; else ((uint64_t*)Ltab)[rr] = L;
        }
    }
}

// Batched Search Space query "is valid" (L139): out[i] = bitmap[L(row_i)]; rows with an index out of its
// domain are invalid (A27).
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

// cao_device.cuh -- device-side primitives shared by the libcao kernels (sm_100a).
// Citations: "Lnnn" = PAPER.md line, "Ox"/"Ax" = readings in DESIGN.md.  Nothing here is shared
// with oracle/ (the CPU oracle has its own copies of every formula).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#define CAO_MAX_DIMS 32
#define CAO_MAX_STACK 32
#define CAO_DIR_SHIFT 9          // rank directory granularity: one u32 per 512 configs (8 bitmap words)

// ---------------------------------------------------------------------------------------------
// Space description handed to every kernel BY VALUE (__grid_constant__), so several spaces can be
// in flight on different streams without sharing a __constant__ symbol.
struct SpaceMeta {
    uint64_t N;                         // Cartesian size
    uint64_t stride[CAO_MAX_DIMS];      // stride[n-1] = 1 (A1: first param most significant)
    uint64_t magic[CAO_MAX_DIMS];       // ceil(2^64 / m_d) for m_d >= 2 (exact division of any L < 2^56)
    const uint64_t* bitmap;             // ceil(N/64) words
    const uint8_t* rows;                // V x rowB, ascending L, padding bytes zero
    const void* Ltab;                   // V linear indices: u32 when N <= 2^32 (ltab32), else u64
    const uint32_t* dir;                // ceil(N/512)+1 exclusive counts
    const float* obj;                   // V
    uint32_t V;
    int32_t n, rowB, M;                 // M = max_d m_d (O6)
    int32_t ltab32;
    uint16_t m[CAO_MAX_DIMS];
};

// Neighbour lists of the Hamming-level probes (S5).  A point has NB = sum (m_d - 1) Hamming-1 neighbours; neighbour
// t = (dimension d, k) with k = 0 .. m_d - 2 stands for the value index v = k + (k >= c_d) != c_d of a candidate c, so
// no probe is ever wasted on the candidate's own value.  Entries are sorted by (d, k).
#define CAO_MAX_PROBE_LEVEL 6
#define CAO_MAX_NB_PROBE 368            // NB above this never probes beyond level 1 (the pair list would exceed 2^16 entries)
struct ProbeMeta {
    const uint16_t* nb;                 // NB entries: d << 8 | k
    const uint32_t* pairs;              // C2 entries: t1 | t2 << 16, dimension(t1) < dimension(t2)
    const uint32_t* triples;            // C3 entries: t1 | t2 << 10 | t3 << 20, strictly increasing dimensions (0 entries: level 3 walks)
    uint32_t NB, C2, C3;
    int32_t levels;                     // highest Hamming level probed in the bitmap before the table scan (0..6)
    uint16_t nb_first[CAO_MAX_DIMS + 1];    // first neighbour of dimension d; nb_first[n..] = NB
};

// ---------------------------------------------------------------------------------------------
// O3: Philox4x32-10 (Salmon et al., SC'11).
static __device__ __noinline__ uint4 philox4x32_10(uint4 c, uint32_t k0, uint32_t k1) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        uint32_t h0 = __umulhi(0xD2511F53u, c.x), l0 = 0xD2511F53u * c.x;
        uint32_t h1 = __umulhi(0xCD9E8D57u, c.z), l1 = 0xCD9E8D57u * c.z;
        c = make_uint4(h1 ^ c.y ^ k0, l1, h0 ^ c.w ^ k1, l0);
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    return c;
}

// K consecutive counter blocks (c.w, c.w + 1, ...) at once: K independent chains interleaved round by round, so a lone
// warp is not bound by the multiply latency, and the round keys are advanced once per round for all K.
template <int K>
static __device__ __forceinline__ void philox4x32_10_multi(uint4 c, uint32_t k0, uint32_t k1, uint4 (&out)[K]) {
    uint4 s[K];
#pragma unroll
    for (int q = 0; q < K; ++q) s[q] = make_uint4(c.x, c.y, c.z, c.w + q);
#pragma unroll
    for (int r = 0; r < 10; ++r) {
#pragma unroll
        for (int q = 0; q < K; ++q) {
            const uint32_t h0 = __umulhi(0xD2511F53u, s[q].x), l0 = 0xD2511F53u * s[q].x;
            const uint32_t h1 = __umulhi(0xCD9E8D57u, s[q].z), l1 = 0xCD9E8D57u * s[q].z;
            s[q] = make_uint4(h1 ^ s[q].y ^ k0, l1, h0 ^ s[q].w ^ k1, l0);
        }
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
#pragma unroll
    for (int q = 0; q < K; ++q) out[q] = s[q];
}

struct PhiloxPair { uint4 a, b; };
static __device__ __noinline__ PhiloxPair philox4x32_10_x2(uint4 c, uint32_t k0, uint32_t k1) {
    uint4 o[2];
    philox4x32_10_multi<2>(c, k0, k1, o);
    PhiloxPair r; r.a = o[0]; r.b = o[1];
    return r;
}

enum : uint32_t { S_INIT = 0, S_OP = 1, S_MUT = 2, S_REINIT = 3 };

// Slot-addressed draws for one (seed, run, generation, individual, stream): counter =
// (run, gen, ind, stream<<24 | slot>>2), word slot&3.  The last block is cached, so walking
// the slots in ascending order costs one Philox call per four draws.
struct Draws {
    uint32_t k0, k1, run, gen, ind, stream, cur;
    uint4 blk;
    __device__ __forceinline__ Draws(uint64_t seed, uint32_t run_, uint32_t gen_, uint32_t ind_, uint32_t stream_)
        : k0((uint32_t)seed), k1((uint32_t)(seed >> 32)), run(run_), gen(gen_), ind(ind_), stream(stream_),
          cur(0xFFFFFFFFu) {}
    __device__ __forceinline__ uint32_t operator()(uint32_t slot) {
        uint32_t b = slot >> 2;
        if (b != cur) { blk = philox4x32_10(make_uint4(run, gen, ind, (stream << 24) | b), k0, k1); cur = b; }
        uint32_t s = slot & 3;
        return s == 0 ? blk.x : s == 1 ? blk.y : s == 2 ? blk.z : blk.w;
    }
};

// The same addressing with TWO blocks per Philox call (slots 8b .. 8b+7): for the operators that walk many slots.
struct Draws2 {
    uint32_t k0, k1, run, gen, ind, stream, cur;
    uint4 blk[2];
    __device__ __forceinline__ Draws2(uint64_t seed, uint32_t run_, uint32_t gen_, uint32_t ind_, uint32_t stream_)
        : k0((uint32_t)seed), k1((uint32_t)(seed >> 32)), run(run_), gen(gen_), ind(ind_), stream(stream_),
          cur(0xFFFFFFFFu) {}
    __device__ __forceinline__ uint32_t operator()(uint32_t slot) {
        const uint32_t b = slot >> 3;
        if (b != cur) {
            const PhiloxPair r = philox4x32_10_x2(make_uint4(run, gen, ind, (stream << 24) | (b << 1)), k0, k1);
            blk[0] = r.a; blk[1] = r.b; cur = b;
        }
        const uint4 v = (slot & 4) ? blk[1] : blk[0];
        const uint32_t s = slot & 3;
        return s == 0 ? v.x : s == 1 ? v.y : s == 2 ? v.z : v.w;
    }
};

__device__ __forceinline__ float u01(uint32_t w) { return __fmul_rn((float)(w >> 8), 5.9604644775390625e-08f); }
__device__ __forceinline__ uint32_t below(uint32_t w, uint32_t k) { return __umulhi(w, k); }

// ---------------------------------------------------------------------------------------------
// fp32 helpers: every operation is one IEEE rounding (__f*_rn never contracts into an FMA).
// O7: exp(-z) for z >= 0, add/mul only.
__device__ __forceinline__ float exp_neg_spec(float z) {
    const float LOG2E = 0x1.715476p+0f, RSQRT2 = 0x1.6a09e6p-1f;
    const float c0 = 1.0f, c1 = -0x1.62e430p-1f, c2 = 0x1.ebfbe0p-3f, c3 = -0x1.c6b08ep-5f,
                c4 = 0x1.3b2ab6p-7f, c5 = -0x1.5d87fep-10f, c6 = 0x1.430912p-13f, c7 = -0x1.ffcbfcp-17f;
    float t = __fmul_rn(z, LOG2E);
    float kf = floorf(t);
    const bool tiny = !(kf < 126.0f);                               // result 0 (also for NaN); decided by a select at the end, so
    float fr = __fsub_rn(t, kf);                                        // the dependent chain below can overlap independent work
    float u = __fsub_rn(fr, 0.5f);
    float p = c7;
    p = __fadd_rn(__fmul_rn(p, u), c6);
    p = __fadd_rn(__fmul_rn(p, u), c5);
    p = __fadd_rn(__fmul_rn(p, u), c4);
    p = __fadd_rn(__fmul_rn(p, u), c3);
    p = __fadd_rn(__fmul_rn(p, u), c2);
    p = __fadd_rn(__fmul_rn(p, u), c1);
    p = __fadd_rn(__fmul_rn(p, u), c0);
    p = __fmul_rn(p, RSQRT2);
    float scale = __uint_as_float((uint32_t)(127 - (int)(tiny ? 0.0f : kf)) << 23);
    return tiny ? 0.0f : __fmul_rn(p, scale);
}

__device__ __forceinline__ float clamp_pos(float x, float hi) {   // NaN -> 0, -0 -> +0
    x = (x > 0.0f) ? x : 0.0f;
    x = (x < hi) ? x : hi;
    return x;
}
// O6: coord(k) = k / (M-1) (IEEE division), snap = rint(x*(M-1)) half-to-even, clamped (A10, A11).
__device__ __forceinline__ float coord_M(int M, int k) { return M > 1 ? __fdiv_rn((float)k, (float)(M - 1)) : 0.0f; }
__device__ __forceinline__ int snap_M(int M, int m_d, float x) {
    float g = __fmul_rn(x, (float)(M - 1));
    int k = __float2int_rn(g);
    k = max(k, 0);
    k = min(k, m_d - 1);
    return k;
}
// O5: round_and_clip(i_best + F*(i_a - i_b)), two fp32 roundings, half-to-even (Alg.1, A8).
__device__ __forceinline__ int de_mutate_index(float F, int ibest, int ia, int ib, int top) {
    float t = __fmul_rn(F, (float)(ia - ib));
    float mf = __fadd_rn((float)ibest, t);
    int v = __float2int_rn(mf);
    v = max(v, 0);
    v = min(v, top);
    return v;
}

// ---------------------------------------------------------------------------------------------
// Bitmap / rank directory.
__device__ __forceinline__ bool bit_test(const uint64_t* __restrict__ bitmap, uint64_t L) {
    return (__ldg(&bitmap[L >> 6]) >> (L & 63)) & 1ull;
}
// rank of a VALID L: directory entry of its 512-block + popcount of the bits below it in the block.  The eight
// words of the block (one 64-byte line; the bitmap buffer is padded to 256 bytes) are loaded unconditionally
// as four 128-bit loads, so the rank costs one round trip instead of a dependent chain.
__device__ __forceinline__ uint32_t rank_of(const SpaceMeta& sm, uint64_t L) {
    const uint32_t wi = (uint32_t)(L >> 6) & 7u;
    const ulonglong2* blk = (const ulonglong2*)(sm.bitmap + ((L >> 6) & ~7ull));
    uint32_t r = __ldg(&sm.dir[L >> CAO_DIR_SHIFT]);
    const uint64_t below_mask = (1ull << (L & 63)) - 1ull;
#pragma unroll
    for (int h = 0; h < 4; ++h) {
        const ulonglong2 v = __ldg(&blk[h]);
        const uint32_t q0 = 2 * h, q1 = 2 * h + 1;
        r += q0 < wi ? __popcll(v.x) : q0 == wi ? __popcll(v.x & below_mask) : 0;
        r += q1 < wi ? __popcll(v.y) : q1 == wi ? __popcll(v.y & below_mask) : 0;
    }
    return r;
}

__device__ __forceinline__ uint64_t ltab_at(const SpaceMeta& sm, uint32_t r) {
    return sm.ltab32 ? (uint64_t)__ldg(&((const uint32_t*)sm.Ltab)[r]) : __ldg(&((const uint64_t*)sm.Ltab)[r]);
}

// Exact L / m and L % m through the precomputed reciprocal (m >= 2, L < 2^56).
__device__ __forceinline__ uint64_t div_magic(uint64_t L, uint64_t magic) { return __umul64hi(L, magic); }

// Row bytes live in uint32 words (4 index bytes per word, byte d&3 of word d>>2).
__device__ __forceinline__ uint32_t row_byte(const uint32_t* w, int d) { return (w[d >> 2] >> ((d & 3) * 8)) & 0xFFu; }

// Saturating int64 arithmetic of the constraint programs (A3): clamp to +-2^62.
#define CAO_SAT (1ll << 62)
__device__ __forceinline__ int64_t sat64(int64_t v) { return v > CAO_SAT ? CAO_SAT : (v < -CAO_SAT ? -CAO_SAT : v); }
__device__ __forceinline__ int64_t sat_add(int64_t a, int64_t b) {      // |a|,|b| <= 2^62
    if (b > 0 && a > CAO_SAT - b) return CAO_SAT;
    if (b < 0 && a < -CAO_SAT - b) return -CAO_SAT;
    return a + b;
}
__device__ __forceinline__ int64_t sat_mul(int64_t a, int64_t b) {
    int64_t hi = __mul64hi(a, b);
    int64_t lo = (int64_t)((uint64_t)a * (uint64_t)b);
    if (hi != (lo >> 63)) return ((a < 0) != (b < 0)) ? -CAO_SAT : CAO_SAT;
    return sat64(lo);
}

// O1: postfix interpreter over the VALUES x[d].  Runs from token pc with the stack st[0..sp).  Returns 1/0 at
// the end of the program (a zero divisor makes the constraint false: 0).  If stop_t >= 0 it stops BEFORE the
// first PUSH_PARAM d with d >= stop_t and returns 2 with the resume point in *pc_out / *sp_out: the prefix of
// a program that reads only outer digits is executed once per block of configs, not once per config.
static __device__ __noinline__ int eval_core(const int32_t* __restrict__ w, int nw, const int64_t* __restrict__ x, int pc,
                                             int64_t* st, int sp, int stop_t, int* pc_out, int* sp_out) {
    for (; pc < nw; ++pc) {
        int op = w[pc];
        if (op == 1) {
            if (stop_t >= 0 && w[pc + 1] >= stop_t) { *pc_out = pc; *sp_out = sp; return 2; }
            st[sp++] = sat64(x[w[++pc]]); continue;
        }
        if (op == 2) {
            uint64_t lo = (uint32_t)w[pc + 1], hi = (uint32_t)w[pc + 2]; pc += 2;
            st[sp++] = sat64((int64_t)(lo | (hi << 32))); continue;
        }
        if (op == 8) { st[sp - 1] = -st[sp - 1]; continue; }
        if (op == 19) { st[sp - 1] = (st[sp - 1] == 0); continue; }
        int64_t b = st[--sp], a = st[sp - 1], r = 0;
        switch (op) {
            case 3: r = sat_add(a, b); break;
            case 4: r = sat_add(a, -b); break;
            case 5: r = sat_mul(a, b); break;
            case 6: if (b == 0) return 0; r = a / b; break;
            case 7: if (b == 0) return 0; r = a % b; break;
            case 9: r = a < b ? a : b; break;
            case 10: r = a > b ? a : b; break;
            case 11: r = a < b; break;  case 12: r = a <= b; break;
            case 13: r = a > b; break;  case 14: r = a >= b; break;
            case 15: r = a == b; break; case 16: r = a != b; break;
            case 17: r = (a != 0) && (b != 0); break;
            case 18: r = (a != 0) || (b != 0); break;
        }
        st[sp - 1] = r;
    }
    return st[0] != 0;
}
static __device__ __forceinline__ int eval_program(const int32_t* __restrict__ w, int nw, const int64_t* __restrict__ x) {
    int64_t st[CAO_MAX_STACK];
    int a, b;
    return eval_core(w, nw, x, 0, st, 0, -1, &a, &b);
}
// k-th (0-based) set bit of a word that has more than k bits set: binary search on popcounts of the low part.
__device__ __forceinline__ int kth_set_bit32(uint32_t w, uint32_t k) {
    int pos = 0; uint32_t c;
    c = __popc(w & 0xFFFFu); if (k >= c) { pos += 16; k -= c; w >>= 16; }
    c = __popc(w & 0xFFu);   if (k >= c) { pos += 8;  k -= c; w >>= 8; }
    c = __popc(w & 0xFu);    if (k >= c) { pos += 4;  k -= c; w >>= 4; }
    c = __popc(w & 0x3u);    if (k >= c) { pos += 2;  k -= c; w >>= 2; }
    c = w & 1u;              if (k >= c) { pos += 1; }
    return pos;
}
__device__ __forceinline__ int kth_set_bit64(uint64_t word, uint32_t k) {
    const uint32_t lo = (uint32_t)word, hi = (uint32_t)(word >> 32), cl = __popc(lo);
    return k < cl ? kth_set_bit32(lo, k) : 32 + kth_set_bit32(hi, k - cl);
}
// ---------------------------------------------------------------------------------------------
// Packed index rows: ROWW uint32 words (ROWW = 4 for n <= 16, 8 for n <= 32), 16-byte aligned.
template <int ROWW>
__device__ __forceinline__ void load_row(const uint8_t* __restrict__ p, uint32_t (&w)[ROWW]) {
    const uint4* q = (const uint4*)p;
    uint4 a = __ldg(&q[0]); w[0] = a.x; w[1] = a.y; w[2] = a.z; w[3] = a.w;
    if (ROWW == 8) { uint4 b = __ldg(&q[1]); w[4] = b.x; w[5] = b.y; w[6] = b.z; w[7] = b.w; }
}
template <int ROWW>
__device__ __forceinline__ void load_row_rw(const uint8_t* p, uint32_t (&w)[ROWW]) {     // state written by earlier kernels
    const uint4* q = (const uint4*)p;
    uint4 a = q[0]; w[0] = a.x; w[1] = a.y; w[2] = a.z; w[3] = a.w;
    if (ROWW == 8) { uint4 b = q[1]; w[4] = b.x; w[5] = b.y; w[6] = b.z; w[7] = b.w; }
}
template <int ROWW>
__device__ __forceinline__ void store_row(uint8_t* p, const uint32_t (&w)[ROWW]) {
    uint4* q = (uint4*)p;
    q[0] = make_uint4(w[0], w[1], w[2], w[3]);
    if (ROWW == 8) q[1] = make_uint4(w[4], w[5], w[6], w[7]);
}
template <int ROWW>
__device__ __forceinline__ uint64_t row_lin(const SpaceMeta& sm, const uint32_t (&w)[ROWW]) {
    uint64_t L = 0;
#pragma unroll
    for (int d = 0; d < ROWW * 4; ++d)
        if (d < sm.n) L += (uint64_t)((w[d >> 2] >> ((d & 3) * 8)) & 0xFFu) * sm.stride[d];
    return L;
}

// Sum of absolute byte differences with accumulate: one VABSDIFF4.U8.ACC.
__device__ __forceinline__ uint32_t sad4_acc(uint32_t a, uint32_t b, uint32_t c) {
    uint32_t r;
    asm("vabsdiff4.u32.u32.u32.add %0, %1, %2, %3;" : "=r"(r) : "r"(a), "r"(b), "r"(c));
    return r;
}

// Repair key (O9): ham << 45 | sad << 32 | rank; rank is monotone in L, so the order equals (ham, sad, L).
#define CAO_KEY_NONE 0xFFFFFFFFFFFFFFFFull
__device__ __forceinline__ uint64_t make_key(uint32_t ham, uint32_t sad, uint32_t rank) {
    return ((uint64_t)ham << 45) | ((uint64_t)sad << 32) | rank;
}
__device__ __forceinline__ uint32_t fbits(float f) { return __float_as_uint(f); }

// cao_runs.cu -- host side of the repair query and of the runs half of include/cao.h (S2-S7).
#include <algorithm>
#include <cmath>
#include <cstring>
#include <mutex>
#include <curand_kernel.h>
#include "cao_runs_kernels.cuh"
#include "cao_var_kernels.cuh"

// Fused generation kernel, one object per algorithm (cao_gen_algo.cu).
struct GenLayout;
#define CAO_GEN_DECL(A)                                                                                                   \
    int cao_gen_setup_##A(int roww, unsigned threads, size_t smem, int wide, int* occ);                                             \
    int cao_gen_launch_##A(int roww, unsigned grid, unsigned threads, size_t smem, cudaStream_t st, const SpaceMeta& sm,  \
                           const ProbeMeta& pm, const RunsMeta& rm, const GenLayout& lay, uint32_t g_first, uint32_t n_gens);
CAO_GEN_DECL(0) CAO_GEN_DECL(1) CAO_GEN_DECL(2) CAO_GEN_DECL(3)
#include "cao_gen_layout.h"

#define SCAN_GRID (cao_sm_count() * 8)

struct cao_runs {
    const cao_space* s = nullptr;
    SpaceMeta sm{};
    RunsMeta rm{};
    uint32_t gen = 0;
    unsigned block = 32;
    int mode = 1;                      // 1 = fused persistent k_gen, 0 = phased (k_op / k_probe23 / k_scan / k_finish)
    bool var_on = false;               // a non-default cao_variant: phased pipeline only
    GenLayout lay{};                   // shared-memory slice of one group of the fused kernel
    unsigned gen_threads = 256, gen_grid = 0;
    size_t gen_smem = 0;
    size_t smem_init = 0, smem_op = 0, smem_fin = 0;
    // raw state views for cao_runs_debug_state
    uint64_t bytes_idx = 0, bytes_pi = 0, bytes_pn = 0;
};

// ---------------------------------------------------------------------------------------------
// in_domain: every candidate byte is a legal index (< m_d <= 128 when M <= 128), which the SMALL byte trick needs.
// index_distance: the NEXT-1 key (sum|didx|, L) of L215 / L270 instead of north_star's (Hamming, sum|didx|, L).
template <int WU>
static void launch_scan_wu(const SpaceMeta& sm, const uint8_t* cand, const uint32_t* wl, const uint32_t* wl_count,
                           unsigned long long* key, bool in_domain, bool index_distance, cudaStream_t st) {
    if (index_distance) k_scan<WU, false, 1><<<SCAN_GRID, SCAN_TC, 0, st>>>(sm, cand, wl, wl_count, key);
    else if (sm.M <= 128 && in_domain) k_scan<WU, true><<<SCAN_GRID, SCAN_TC, 0, st>>>(sm, cand, wl, wl_count, key);
    else k_scan<WU, false><<<SCAN_GRID, SCAN_TC, 0, st>>>(sm, cand, wl, wl_count, key);
}
#define DISPATCH_WU(n_dims, CALL)                                                   \
    switch (((n_dims) + 3) / 4) {                                                   \
        case 1: { CALL(1); } break; case 2: { CALL(2); } break; case 3: { CALL(3); } break; case 4: { CALL(4); } break; \
        case 5: { CALL(5); } break; case 6: { CALL(6); } break; case 7: { CALL(7); } break; default: { CALL(8); } break; \
    }
static int launch_scan(const SpaceMeta& sm, const uint8_t* cand, const uint32_t* wl, const uint32_t* wl_count,
                       unsigned long long* key, bool in_domain, cudaStream_t st, bool index_distance = false) {
    ProfScope ps(PK_SCAN, st);
#define CALL_SCAN(W) launch_scan_wu<W>(sm, cand, wl, wl_count, key, in_domain, index_distance, st)
    DISPATCH_WU(sm.n, CALL_SCAN);
    CAO_LAUNCHED("k_scan");
    return CAO_OK;
}
// NEXT-1 neighbour-rule scan (Alg.2: kind 0, per-rule nearest member; Alg.3: kind 1, per-rule member counts).
static int launch_scan_nb(const SpaceMeta& sm, int kind, const uint8_t* cand, const uint32_t* wl, const uint32_t* wl_count,
                          const uint8_t* present, const XAddr& xa, unsigned long long* key3, uint32_t* cnt3, cudaStream_t st) {
    ProfScope ps(PK_SCAN, st);
#define CALL_NB(W) if (kind == 0) k_scan_nb<W, 0><<<SCAN_GRID, SCAN_TC, 0, st>>>(sm, cand, wl, wl_count, present, xa, key3, cnt3); \
                   else k_scan_nb<W, 1><<<SCAN_GRID, SCAN_TC, 0, st>>>(sm, cand, wl, wl_count, present, xa, key3, cnt3)
    DISPATCH_WU(sm.n, CALL_NB);
    CAO_LAUNCHED("k_scan_nb");
    return CAO_OK;
}
static int launch_pick_nb(const SpaceMeta& sm, const uint8_t* cand, const uint32_t* wl, const uint32_t* wl_count, const uint8_t* present,
                          const uint32_t* cnt3, const uint32_t* w_arr, uint64_t seed, uint32_t first_run, uint32_t P, uint32_t gen,
                          unsigned long long* key, uint8_t* rule, cudaStream_t st) {
    ProfScope ps(PK_SCAN, st);
#define CALL_PICK(W) k_pick_nb<W><<<cao_sm_count() * 4, 256, 0, st>>>(sm, cand, wl, wl_count, present, cnt3, w_arr, seed, first_run, P, gen, key, rule)
    DISPATCH_WU(sm.n, CALL_PICK);
    CAO_LAUNCHED("k_pick_nb");
    return CAO_OK;
}
static int launch_present(const SpaceMeta& sm, uint8_t* present, cudaStream_t st) {
    CAO_CUDA(cudaMemsetAsync(present, 0, (size_t)CAO_MAX_DIMS * 256 + 256, st));
    const unsigned grid = (unsigned)((sm.V + 255) / 256);
    if (sm.rowB == 16) k_present<4><<<grid, 256, 0, st>>>(sm, present);
    else k_present<8><<<grid, 256, 0, st>>>(sm, present);
    CAO_LAUNCHED("k_present");
    k_all_present<<<1, 256, 0, st>>>(sm, present, (uint32_t*)(present + CAO_MAX_DIMS * 256));
    CAO_LAUNCHED("k_all_present");
    return CAO_OK;
}

// Hamming-2/3 probe of worklist wl; survivors go to wl2 (the scan's input).
static int launch_probe23(const cao_space* s, const SpaceMeta& sm, const uint8_t* cand, const uint32_t* wl, const uint32_t* wl_count,
                          unsigned long long* key, uint32_t* wl2, uint32_t* wl2_count, unsigned long long* n_scanned,
                          int levels, cudaStream_t st) {
    ProbeMeta pm = s->probe;
    pm.levels = levels;
    ProfScope ps(PK_PROBE, st);
    if (sm.rowB == 16) k_probe23<4><<<cao_sm_count() * 8, 256, 0, st>>>(sm, pm, cand, wl, wl_count, key, wl2, wl2_count, n_scanned);
    else k_probe23<8><<<cao_sm_count() * 8, 256, 0, st>>>(sm, pm, cand, wl, wl_count, key, wl2, wl2_count, n_scanned);
    CAO_LAUNCHED("k_probe23");
    return CAO_OK;
}

// Dispatch over (algorithm, row words).
#define DISPATCH_ALGO_ROWW(algo, roww, CALL)                                         \
    do {                                                                             \
        if ((roww) == 4) {                                                           \
            switch (algo) {                                                          \
                case CAO_DE: { CALL(CAO_DE, 4); } break;                             \
                case CAO_PSO: { CALL(CAO_PSO, 4); } break;                           \
                case CAO_FIREFLY: { CALL(CAO_FIREFLY, 4); } break;                   \
                default: { CALL(CAO_GA, 4); } break;                                 \
            }                                                                        \
        } else {                                                                     \
            switch (algo) {                                                          \
                case CAO_DE: { CALL(CAO_DE, 8); } break;                             \
                case CAO_PSO: { CALL(CAO_PSO, 8); } break;                           \
                case CAO_FIREFLY: { CALL(CAO_FIREFLY, 8); } break;                   \
                default: { CALL(CAO_GA, 8); } break;                                 \
            }                                                                        \
        }                                                                            \
    } while (0)

// Integer-issue peak (bench.py): 8 independent chains per thread of ONE instruction kind, nothing else in the loop.
template <int KIND>
__global__ void __launch_bounds__(256) k_int_peak(uint32_t* out, uint32_t iters) {
    uint32_t a[8];
    const uint32_t b = threadIdx.x * 2654435761u + 12345u, c = blockIdx.x * 40503u + 7u;
#pragma unroll
    for (int j = 0; j < 8; ++j) a[j] = b ^ (c + j * 0x9E3779B9u);
    for (uint32_t it = 0; it < iters; ++it) {
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            if (KIND == 0) asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a[j]) : "r"(b), "r"(c));
            if (KIND == 1) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a[j]) : "r"(b), "r"(c));
            if (KIND == 2) asm volatile("vabsdiff4.u32.u32.u32.add %0, %0, %1, %2;" : "+r"(a[j]) : "r"(b), "r"(c));
            if (KIND == 3) asm volatile("popc.b32 %0, %0;" : "+r"(a[j]));
            if (KIND == 4) asm volatile("add.u32 %0, %0, %1;" : "+r"(a[j]) : "r"(b));
            if (KIND == 5) asm volatile("dp4a.u32.u32 %0, %1, %2, %0;" : "+r"(a[j]) : "r"(b), "r"(c));
        }
    }
    uint32_t x = 0;
#pragma unroll
    for (int j = 0; j < 8; ++j) x ^= a[j];
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = x;
}

// ---------------------------------------------------------------------------------------------
// Scratch of cao_space_repair_noalloc: one fixed array in the library's own device image, so the entry point never has to
// ask the CUDA allocator for anything.  Sized for CAO_REPAIR_NOALLOC_MAX_ROWS rows of the wider row format (32 bytes):
// packed keys + two worklists + their counters + the padding-cleaned copy of the rows -- the same regions, in the same
// order, as cao_space_repair_scratch_bytes.  Every GPU on which the library's kernels get loaded keeps its own copy of
// these 3 MiB until the process ends.
#define CAO_NOALLOC_SCRATCH_BYTES ((size_t)CAO_REPAIR_NOALLOC_MAX_ROWS * (8 + 4 + 4 + 32) + 256)
static_assert(CAO_NOALLOC_SCRATCH_BYTES % 256 == 0, "regions of the static scratch stay 256-byte aligned");
static __device__ __align__(256) unsigned char g_noalloc_scratch[CAO_NOALLOC_SCRATCH_BYTES];
// In host code `g_noalloc_scratch` is only a handle for the runtime, not something a kernel can dereference: the real
// device address differs per GPU and is looked up once per device with cudaGetSymbolAddress (noalloc_scratch_ptr).
#define CAO_NOALLOC_MAX_DEVICES 64
static std::mutex g_noalloc_mu;
static void* g_noalloc_ptr[CAO_NOALLOC_MAX_DEVICES] = {};

// Device address of the static scratch on the CURRENT device; resolved on the first call per device, cached afterwards.
static int noalloc_scratch_ptr(void** out) {
    int dev = -1;
    CAO_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= CAO_NOALLOC_MAX_DEVICES)
        return cao_fail(CAO_E_CUDA, "cao_space_repair_noalloc: device ordinal " + std::to_string(dev) + " is outside 0.." +
                                        std::to_string(CAO_NOALLOC_MAX_DEVICES - 1));
    std::lock_guard<std::mutex> lk(g_noalloc_mu);
    if (!g_noalloc_ptr[dev]) {
        void* p = nullptr;
        CAO_CUDA(cudaGetSymbolAddress(&p, g_noalloc_scratch));
        if (!p || ((uintptr_t)p & 255)) return cao_fail(CAO_E_CUDA, "cao_space_repair_noalloc: the static scratch has no usable device address");
        g_noalloc_ptr[dev] = p;
    }
    *out = g_noalloc_ptr[dev];
    return CAO_OK;
}

extern "C" {

// ---------------------------------------------------------------------------------------------
int cao_space_repair_scratch_bytes(const cao_space* s, uint64_t count, uint64_t* bytes) {
    if (!s || !bytes) return cao_fail(CAO_E_INVALID_ARG, "cao_space_repair_scratch_bytes: NULL argument");
    *bytes = align256(std::max<uint64_t>(1, count) * 8) + 2 * align256(std::max<uint64_t>(1, count) * 4) + 256 +
             align256(std::max<uint64_t>(1, count) * (uint64_t)s->meta.rowB);
    return CAO_OK;
}

int cao_space_repair(const cao_space* s, const uint8_t* d_idx_rows, uint64_t count, uint32_t* d_rank_out,
                     uint64_t* d_key_out, int32_t use_probe, void* d_scratch, void* stream) {
    if (!s) return cao_fail(CAO_E_INVALID_ARG, "cao_space_repair: NULL space");
    if (!s->filled) return cao_fail(CAO_E_STATE, "cao_space_repair: space not built");
    if (count == 0) return CAO_OK;
    if (!d_idx_rows || (!d_rank_out && !d_key_out)) return cao_fail(CAO_E_INVALID_ARG, "cao_space_repair: NULL argument");
    if (count >= (1ull << 32)) return cao_fail(CAO_E_TOO_LARGE, "cao_space_repair: count >= 2^32");
    if (s->meta.V == 0) return cao_fail(CAO_E_EMPTY_SPACE, "cao_space_repair: the space has no valid configuration");
    if (!d_scratch || ((uintptr_t)d_scratch & 255) || ((uintptr_t)d_idx_rows & 15))
        return cao_fail(CAO_E_WORKSPACE, "cao_space_repair: scratch must be 256-byte aligned, rows 16-byte aligned");
    cudaStream_t st = (cudaStream_t)stream;
    uint8_t* sc = (uint8_t*)d_scratch;
    unsigned long long* key = (unsigned long long*)sc;
    uint32_t* wl = (uint32_t*)(sc + align256(count * 8));
    uint32_t* wl2 = (uint32_t*)(sc + align256(count * 8) + align256(count * 4));
    uint32_t* wl_count = (uint32_t*)(sc + align256(count * 8) + 2 * align256(count * 4));
    uint32_t* wl2_count = wl_count + 1;
    uint8_t* clean = sc + align256(count * 8) + 2 * align256(count * 4) + 256;      // rows with zeroed padding
    CAO_CUDA(cudaMemsetAsync(wl_count, 0, 8, st));
    const int levels = use_probe < 0 || use_probe > CAO_MAX_PROBE_LEVEL ? s->probe.levels : (s->probe.C2 == 0 ? std::min(use_probe, 1) : use_probe);
    const bool two = levels >= 2;
    unsigned grid = (unsigned)((count + 255) / 256);
    {   // without Hamming-2/3 probes everything unresolved goes to the scan list directly
        ProfScope ps(PK_QUERY, st);
        uint32_t* a = two ? wl : wl2; uint32_t* ac = two ? wl_count : wl2_count;
        if (s->meta.rowB == 16) k_repair_probe<4><<<grid, 256, 0, st>>>(s->meta, d_idx_rows, clean, count, levels >= 1, key, a, ac, wl2, wl2_count);
        else k_repair_probe<8><<<grid, 256, 0, st>>>(s->meta, d_idx_rows, clean, count, levels >= 1, key, a, ac, wl2, wl2_count);
    }
    CAO_LAUNCHED("k_repair_probe");
    int rc = CAO_OK;
    if (two) { rc = launch_probe23(s, s->meta, clean, wl, wl_count, key, wl2, wl2_count, nullptr, levels, st); if (rc) return rc; }
    rc = launch_scan(s->meta, clean, wl2, wl2_count, key, false, st);
    if (rc) return rc;
    k_repair_finish<<<grid, 256, 0, st>>>(key, count, d_rank_out, d_key_out);
    CAO_LAUNCHED("k_repair_finish");
    return CAO_OK;
}

// cao_space_repair for callers that cannot bring scratch memory because they cannot allocate (who they are: include/cao.h).
// Inputs and outputs stay the caller's; the scratch is g_noalloc_scratch.  Nothing on this path allocates:
// cudaGetDevice / cudaGetSymbolAddress (first call per device only), one cudaMemsetAsync of the two worklist counters,
// then the launches of cao_space_repair.  The per-kernel timing option creates CUDA events, so it has to be off.
int cao_space_repair_noalloc(const cao_space* s, const uint8_t* d_idx_rows, uint64_t count, uint32_t* d_rank_out,
                             uint64_t* d_key_out, int32_t use_probe, void* stream) {
    if (!s) return cao_fail(CAO_E_INVALID_ARG, "cao_space_repair_noalloc: NULL space");
    if (!s->filled) return cao_fail(CAO_E_STATE, "cao_space_repair_noalloc: space not built");
    if (count > CAO_REPAIR_NOALLOC_MAX_ROWS)
        return cao_fail(CAO_E_TOO_LARGE, "cao_space_repair_noalloc: " + std::to_string(count) + " rows, the static scratch holds at most " +
                                             std::to_string(CAO_REPAIR_NOALLOC_MAX_ROWS) + " per call (split the batch, or use cao_space_repair)");
    if (count == 0) return CAO_OK;
    if (!d_idx_rows || (!d_rank_out && !d_key_out)) return cao_fail(CAO_E_INVALID_ARG, "cao_space_repair_noalloc: NULL argument");
    if (s->meta.V == 0) return cao_fail(CAO_E_EMPTY_SPACE, "cao_space_repair_noalloc: the space has no valid configuration");
    if ((uintptr_t)d_idx_rows & 15) return cao_fail(CAO_E_WORKSPACE, "cao_space_repair_noalloc: rows must be 16-byte aligned");
    if (g_cao_prof_on.load(std::memory_order_relaxed) != 0)
        return cao_fail(CAO_E_STATE, "cao_space_repair_noalloc: cao_profile_enable is on, and its timing events are allocations; switch it off");
    void* scratch = nullptr;
    int rc = noalloc_scratch_ptr(&scratch);
    if (rc) return rc;
    // The worklist counters are cleared by cao_space_repair's cudaMemsetAsync and every key of rows 0..count-1 is written by
    // k_repair_probe before anything reads it, so whatever the previous call left in the array cannot leak into this one.
    return cao_space_repair(s, d_idx_rows, count, d_rank_out, d_key_out, use_probe, scratch, stream);
}

// Shared-memory slice of one group of the fused kernel (cao_gen_kernels.cuh): word offsets.
// width: 0 = automatic, 1 / 2 / 4 = threads per group as a multiple of roundup32(P).  Automatic: while the runs of this
// launch fill only part of the GPU's resident thread slots (148 SMs x 3 CTAs x 256 threads), a run gets more lanes --
// Firefly four per firefly (its operator is a dependent chain per attractor), the others two (their cooperative phases:
// neighbour probes, scans, GA mutation, stride over the group).  Results do not depend on the width.
static GenLayout gen_layout(const cao_space* s, int algo, uint32_t P, uint32_t R, int width) {
    GenLayout L{};
    const uint32_t n = (uint32_t)s->meta.n, roww = (uint32_t)s->meta.rowB / 4;
    uint32_t off = GRP_SHARED_WORDS;
    auto take = [&](uint32_t words) { uint32_t o = off; off = (off + std::max(1u, words) + 3u) & ~3u; return o; };
    L.rank = take(P); L.f = take(P);
    const bool cont = algo == CAO_PSO || algo == CAO_FIREFLY;
    L.idx = take(cont ? 0 : P * roww);
    L.x = take(cont ? n * P : 0);
    L.v = take(algo == CAO_PSO ? n * P : 0); L.pb = take(algo == CAO_PSO ? n * P : 0); L.pbf = take(algo == CAO_PSO ? P : 0);
    L.cand = take(P * roww); L.key = take(2 * P);
    L.scr = take(algo == CAO_GA ? 3 * P : P);
    L.wl = take(P); L.cw = take(GEN_NB * roww); L.skey = take(2 * GEN_NB); L.bestrow = take(roww);
    L.Lc = take(2 * P); L.aux4 = take(4 * P);
    L.ptab = take(s->probe.levels >= 2 ? 2 * s->probe.NB : 0);
    L.words = off;
    const uint32_t G0 = (P + 31) / 32 * 32;
    const double slots = (double)cao_sm_count() * 3 * 256;
    uint32_t f = 1;
    if (width == 0) {
        if (algo == CAO_FIREFLY) { if (roww == 4 && G0 * 4 <= 256 && (double)R * G0 * 4 <= 1.25 * slots) f = 4; }
        else if (G0 * 2 <= 256 && (double)R * G0 * 2 <= 0.6 * slots) f = 2;
    } else if ((uint32_t)width * G0 <= 256 && !(algo == CAO_FIREFLY && width == 4 && roww != 4)) f = (uint32_t)width;
    L.wide = algo == CAO_FIREFLY && f == 4 ? 1 : 0;
    if (algo == CAO_FIREFLY && f == 2) f = 1;                           // Firefly is either one warp-lane or four lanes per firefly
    L.G = G0 * f;
    L.NG = L.G <= 256 ? 256 / L.G : 1;
    L.NB = 0;
    for (uint32_t d = 0; d < n; ++d) L.NB += (uint32_t)s->meta.m[d] - 1u;
    L.nb_words = (L.NB / 2 + 4) & ~3u;
    const uint64_t tab_bytes = (uint64_t)s->probe.C2 * 4;
    L.probe_in_smem = s->probe.levels >= 2 && tab_bytes <= 16384;
    L.cta_words = 3 * CAO_MAX_DIMS + L.nb_words + (L.probe_in_smem ? (uint32_t)((tab_bytes + 15) / 16 * 4) : 0);
    // keep one CTA below the 227 KB opt-in limit: fewer groups per CTA for large populations / many dimensions
    while (L.NG > 1 && ((uint64_t)L.cta_words + (uint64_t)L.NG * L.words) * 4 > 200 * 1024) --L.NG;
    return L;
}

// ---------------------------------------------------------------------------------------------
struct RunsLayout {
    uint64_t cand, key, valid, rep_rank, eval_rank, tap_f, accept, active, idx, rank, f, x, v, pb, pbf, dedup,
        uniq, gens_done, stagn, best_rank, best_f, traj, wl, wl2, wl_count, counters, rcache, ticket, total;
    uint64_t rule, key3, cnt3, present;   // SURVEY 8(f) variants only
    uint64_t zero_from, zero_bytes;       // region that must start as zero: dedup .. stagn
    uint32_t dedup_words;
};

static const cao_variant CAO_VARIANT_DEFAULT = {1, 0, 0, 0, 0, 0, 1e20f, 0};
static bool variant_is_default(const cao_variant& v) {
    return v.constraint_aware == 1 && v.repair_mode == 0 && v.de_mutation == 0 && v.de_crossover == 0 && v.ga_crossover == 0 &&
           v.init_lhs == 0;
}
static RunsLayout runs_layout(const SpaceMeta& sm, int algo, uint64_t P, uint64_t R, uint64_t max_gens,
                              const cao_variant& var = CAO_VARIANT_DEFAULT) {
    RunsLayout L{};
    const uint64_t RP = R * P, rowB = sm.rowB, n = sm.n;
    uint64_t off = 0;
    auto take = [&](uint64_t bytes) { uint64_t o = off; off = align256(off + std::max<uint64_t>(1, bytes)); return o; };
    L.cand = take(RP * rowB); L.key = take(RP * 8); L.valid = take(RP); L.rep_rank = take(RP * 4);
    L.eval_rank = take(RP * 4); L.tap_f = take(RP * 4); L.accept = take(RP); L.active = take(R);
    const bool cont = algo == CAO_PSO || algo == CAO_FIREFLY;
    L.idx = take(cont ? 0 : RP * rowB); L.rank = take(RP * 4); L.f = take(RP * 4);
    L.x = take(cont ? RP * n * 4 : 0);
    L.v = take(algo == CAO_PSO ? RP * n * 4 : 0); L.pb = take(algo == CAO_PSO ? RP * n * 4 : 0);
    L.pbf = take(algo == CAO_PSO ? RP * 4 : 0);
    L.dedup_words = (uint32_t)(((uint64_t)sm.V + 31) / 32);
    L.zero_from = off;
    L.dedup = take(R * L.dedup_words * 4);
    L.uniq = take(R * 4); L.gens_done = take(R * 4); L.stagn = take(R * 4);
    L.wl_count = take(8); L.counters = take(32 * 8); L.ticket = take(8);
    L.zero_bytes = off - L.zero_from;
    L.best_rank = take(R * 4); L.best_f = take(R * 4);
    L.traj = take((max_gens + 1) * R * 12);
    L.wl = take(RP * 4);
    L.wl2 = take(RP * 4);
    L.rcache = take(R * CAO_RCACHE * 16);
    if (!variant_is_default(var)) {
        const bool paper = var.constraint_aware && var.repair_mode == 1;
        L.rule = take(RP);
        L.key3 = take(paper && cont ? RP * 24 : 0);
        L.cnt3 = take(paper && algo == CAO_GA ? RP * 12 : 0);
        L.present = take(paper ? (uint64_t)CAO_MAX_DIMS * 256 + 256 : 0);
    }
    L.total = off;
    return L;
}

static int check_runs_args(const cao_space* s, int32_t algo, int32_t pop, uint32_t n_runs, uint32_t max_gens) {
    if (!s) return cao_fail(CAO_E_INVALID_ARG, "runs: NULL space");
    if (!s->filled) return cao_fail(CAO_E_STATE, "runs: space not built");
    if (algo < 0 || algo > 3) return cao_fail(CAO_E_INVALID_ARG, "runs: unknown algorithm");
    if (pop < 1 || n_runs < 1) return cao_fail(CAO_E_INVALID_ARG, "runs: pop and n_runs must be >= 1");
    if (pop > 1024) return cao_fail(CAO_E_TOO_LARGE, "runs: pop > 1024");
    if (s->meta.V == 0) return cao_fail(CAO_E_EMPTY_SPACE, "runs: the space has no valid configuration");
    if ((uint64_t)pop > s->meta.V) return cao_fail(CAO_E_POP_GT_VALID, "runs: population larger than the number of valid configurations");
    if (algo == CAO_DE && pop < 3) return cao_fail(CAO_E_INVALID_ARG, "runs: DE needs pop >= 3");
    if (algo == CAO_GA && pop < 2) return cao_fail(CAO_E_INVALID_ARG, "runs: GA needs pop >= 2");
    if ((uint64_t)pop * n_runs >= (1ull << 32)) return cao_fail(CAO_E_TOO_LARGE, "runs: pop * n_runs >= 2^32");
    if (max_gens >= (1u << 24)) return cao_fail(CAO_E_TOO_LARGE, "runs: max_gens >= 2^24");
    return CAO_OK;
}

static int check_variant(int32_t algo, int32_t pop, const cao_variant& v) {
    if (v.constraint_aware < 0 || v.constraint_aware > 1 || v.repair_mode < 0 || v.repair_mode > 1 || v.de_mutation < 0 ||
        v.de_mutation > 5 || v.de_crossover < 0 || v.de_crossover > 1 || v.ga_crossover < 0 || v.ga_crossover > 3 ||
        v.init_lhs < 0 || v.init_lhs > 1)
        return cao_fail(CAO_E_INVALID_ARG, "runs: unknown cao_variant switch value");
    static const int donors[6] = {2, 3, 2, 3, 4, 5};
    if (algo == CAO_DE && pop < donors[v.de_mutation] + 1) return cao_fail(CAO_E_INVALID_ARG, "runs: DE population smaller than donors + 1");
    if (v.init_lhs && (algo != CAO_DE || !v.constraint_aware))
        return cao_fail(CAO_E_INVALID_ARG, "runs: init_lhs is DE's constraint-aware initial sample (L223)");
    if (!(v.penalty > 0.0f) || !(v.penalty < 3.0e38f)) return cao_fail(CAO_E_INVALID_ARG, "runs: penalty must be > 0 and finite");
    return CAO_OK;
}

int cao_runs_workspace_bytes_ex(const cao_space* s, int32_t algo, const cao_variant* var, int32_t pop, uint32_t n_runs,
                                uint32_t max_gens, uint64_t* bytes) {
    if (!bytes) return cao_fail(CAO_E_INVALID_ARG, "cao_runs_workspace_bytes: NULL argument");
    int rc = check_runs_args(s, algo, pop, n_runs, max_gens);
    if (rc) return rc;
    const cao_variant v = var ? *var : CAO_VARIANT_DEFAULT;
    if ((rc = check_variant(algo, pop, v))) return rc;
    *bytes = runs_layout(s->meta, algo, (uint64_t)pop, n_runs, max_gens, v).total;
    return CAO_OK;
}
int cao_runs_workspace_bytes(const cao_space* s, int32_t algo, int32_t pop, uint32_t n_runs, uint32_t max_gens, uint64_t* bytes) {
    return cao_runs_workspace_bytes_ex(s, algo, nullptr, pop, n_runs, max_gens, bytes);
}

int cao_runs_create(const cao_space* s, int32_t algo, const cao_hparams* hp, uint32_t n_runs, uint32_t first_run, int32_t pop,
                    uint32_t budget_unique, uint32_t max_gens, uint64_t seed, void* d_workspace, void* stream, cao_runs** out) {
    return cao_runs_create_ex(s, algo, hp, nullptr, n_runs, first_run, pop, budget_unique, max_gens, seed, d_workspace, stream, out);
}

int cao_runs_create_ex(const cao_space* s, int32_t algo, const cao_hparams* hp, const cao_variant* var, uint32_t n_runs,
                       uint32_t first_run, int32_t pop, uint32_t budget_unique, uint32_t max_gens, uint64_t seed, void* d_workspace,
                       void* stream, cao_runs** out) {
    if (!out || !hp) return cao_fail(CAO_E_INVALID_ARG, "cao_runs_create: NULL argument");
    int rc = check_runs_args(s, algo, pop, n_runs, max_gens);
    if (rc) return rc;
    const cao_variant vr = var ? *var : CAO_VARIANT_DEFAULT;
    if ((rc = check_variant(algo, pop, vr))) return rc;
    if (!s->meta.obj) return cao_fail(CAO_E_STATE, "cao_runs_create: call cao_space_set_objective first");
    if (algo == CAO_GA && (hp->ga_beta_b < 1 || hp->ga_beta_b > 16 || hp->ga_mutation_chance < 1))
        return cao_fail(CAO_E_INVALID_ARG, "cao_runs_create: ga_beta_b must be 1..16 and ga_mutation_chance >= 1");
    if (!d_workspace || ((uintptr_t)d_workspace & 255)) return cao_fail(CAO_E_WORKSPACE, "cao_runs_create: workspace must be non-NULL and 256-byte aligned");
    cudaStream_t st = (cudaStream_t)stream;
    const RunsLayout L = runs_layout(s->meta, algo, (uint64_t)pop, n_runs, max_gens, vr);
    uint8_t* w = (uint8_t*)d_workspace;
    cao_runs* r = new cao_runs();
    r->s = s; r->sm = s->meta;
    RunsMeta& m = r->rm;
    m.var = vr; r->var_on = !variant_is_default(vr); m.var_on = r->var_on ? 1 : 0;
    m.rule = nullptr; m.key3 = nullptr; m.cnt3 = nullptr; m.present = nullptr;
    if (r->var_on) {
        m.rule = w + L.rule; m.key3 = (unsigned long long*)(w + L.key3); m.cnt3 = (uint32_t*)(w + L.cnt3); m.present = w + L.present;
    }
    m.R = n_runs; m.first_run = first_run; m.P = (uint32_t)pop; m.budget = budget_unique; m.max_gens = max_gens;
    m.dedup_words = L.dedup_words; m.algo = algo; m.probe_levels = s->probe.levels; m.seed = seed; m.hp = *hp;
    m.cand = w + L.cand; m.key = (unsigned long long*)(w + L.key); m.valid = w + L.valid;
    m.rep_rank = (uint32_t*)(w + L.rep_rank); m.eval_rank = (uint32_t*)(w + L.eval_rank); m.tap_f = (float*)(w + L.tap_f);
    m.accept = w + L.accept; m.active = w + L.active;
    m.idx = w + L.idx; m.rank = (uint32_t*)(w + L.rank); m.f = (float*)(w + L.f);
    m.x = (float*)(w + L.x); m.v = (float*)(w + L.v); m.pb = (float*)(w + L.pb); m.pbf = (float*)(w + L.pbf);
    m.dedup = (uint32_t*)(w + L.dedup); m.uniq = (uint32_t*)(w + L.uniq); m.gens_done = (uint32_t*)(w + L.gens_done);
    m.stagn = (uint32_t*)(w + L.stagn); m.best_rank = (uint32_t*)(w + L.best_rank); m.best_f = (float*)(w + L.best_f);
    m.traj = (uint32_t*)(w + L.traj); m.wl = (uint32_t*)(w + L.wl); m.wl_count = (uint32_t*)(w + L.wl_count);
    m.wl2 = (uint32_t*)(w + L.wl2); m.wl2_count = m.wl_count + 1;
    m.counters = (unsigned long long*)(w + L.counters);
    m.rcache = (ulonglong2*)(w + L.rcache);
    m.ticket = (uint32_t*)(w + L.ticket);
    const uint64_t RP = (uint64_t)n_runs * pop;
    r->bytes_idx = RP * s->meta.rowB; r->bytes_pi = RP * 4; r->bytes_pn = RP * s->meta.n * 4;
    r->block = (unsigned)((pop + 31) / 32 * 32);
    r->lay = gen_layout(s, algo, (uint32_t)pop, n_runs, 0);
    r->gen_threads = r->lay.G * r->lay.NG;
    r->gen_smem = ((size_t)r->lay.cta_words + (size_t)r->lay.NG * r->lay.words) * 4;
    {   // default execution mode: how many invalid candidates will fall through the bitmap probes to the table scan?
        // For a uniformly random invalid point, P(no valid row within Hamming distance L) ~ exp(-density * E_L), E_L =
        // number of rows within distance L (levels probed).  Scans by a single group are slow, so above 1 % the phased
        // pipeline (whole-GPU k_scan per generation) is the default; cao_runs_set_mode overrides.
        double e[CAO_MAX_PROBE_LEVEL + 1] = {1, 0, 0, 0, 0, 0, 0}, E = 0;
        for (int d = 0; d < s->meta.n; ++d) for (int h = CAO_MAX_PROBE_LEVEL; h >= 1; --h) e[h] += e[h - 1] * (double)(s->meta.m[d] - 1);
        for (int h = 1; h <= s->probe.levels; ++h) E += e[h];
        const double p_scan = std::exp(-(double)s->meta.V / (double)s->meta.N * E);
        r->mode = p_scan > 0.01 ? 0 : 1;
    }
    if (r->gen_smem > 227 * 1024) r->mode = 0;                         // the population does not fit one SM: phased only
    if (r->var_on) r->mode = 0;                                         // SURVEY 8(f) variants run through the phased pipeline
    const size_t P = (size_t)pop, n = (size_t)s->meta.n;
    r->smem_init = P * 4;
    r->smem_op = algo == CAO_GA ? P * 16 : algo == CAO_FIREFLY ? (P * n + 2 * P) * 4 : 0;
    r->smem_fin = algo == CAO_DE ? P * 16 : 0;
    int rc2 = CAO_OK;
    do {
        if ((rc2 = cao_cuda_check(cudaMemsetAsync(w + L.zero_from, 0, L.zero_bytes, st), "memset state"))) break;
        if ((rc2 = cao_cuda_check(cudaMemsetAsync(w + L.best_rank, 0xFF, (uint64_t)n_runs * 4, st), "memset best_rank"))) break;
        if ((rc2 = cao_cuda_check(cudaMemsetAsync(w + L.cand, 0, L.idx - L.cand, st), "memset taps"))) break;
        if ((rc2 = cao_cuda_check(cudaMemsetAsync(w + L.key, 0xFF, RP * 8, st), "memset keys"))) break;   // no key yet
        if ((rc2 = cao_cuda_check(cudaMemsetAsync(w + L.rcache, 0xFF, (uint64_t)n_runs * CAO_RCACHE * 16, st), "memset repair cache"))) break;
        if (r->var_on) {
            if ((rc2 = cao_cuda_check(cudaMemsetAsync(w + L.rule, 0xFF, RP, st), "memset rule tap"))) break;
            if (vr.constraint_aware && vr.repair_mode == 1 && (rc2 = launch_present(r->sm, w + L.present, st))) break;
        }
        if (vr.init_lhs) {                                              // A35: LHS points -> ordinary repair pipeline -> k_init reads the ranks
            { ProfScope ps(PK_INIT, st);
              if (s->meta.rowB == 16) k_lhs_points<4><<<n_runs, r->block, r->smem_init, st>>>(r->sm, r->rm);
              else k_lhs_points<8><<<n_runs, r->block, r->smem_init, st>>>(r->sm, r->rm); }
            ++g_cao_launches;
            if ((rc2 = cao_cuda_check(cudaGetLastError(), "k_lhs_points"))) break;
            const int levels = s->probe.levels;
            if (levels >= 2 && (rc2 = launch_probe23(s, r->sm, m.cand, m.wl, m.wl_count, m.key, m.wl2, m.wl2_count, nullptr, levels, st))) break;
            if ((rc2 = launch_scan(r->sm, m.cand, levels >= 2 ? m.wl2 : m.wl, levels >= 2 ? m.wl2_count : m.wl_count, m.key, true, st))) break;
        }
#define CALL_INIT(A, W) \
        if (r->smem_op > 48 * 1024) { rc2 = cao_smem_optin_max(k_op<A, W, 256>, "shared-memory opt-in of k_op");               \
                                      if (!rc2) rc2 = cao_smem_optin_max(k_op<A, W, 1024>, "shared-memory opt-in of k_op"); } \
        if (!rc2) k_init<A, W><<<n_runs, r->block, r->smem_init, st>>>(r->sm, r->rm)
        { ProfScope ps(PK_INIT, st); DISPATCH_ALGO_ROWW(algo, s->meta.rowB / 4, CALL_INIT); }
        if (rc2) break;
        ++g_cao_launches;
        rc2 = cao_cuda_check(cudaGetLastError(), "k_init");
    } while (0);
    if (rc2) { delete r; return rc2; }
    *out = r;
    return CAO_OK;
}

void cao_runs_destroy(cao_runs* r) { delete r; }

int cao_runs_step(cao_runs* r, uint32_t n_generations, void* stream) {
    if (!r) return cao_fail(CAO_E_INVALID_ARG, "cao_runs_step: NULL runs");
    cudaStream_t st = (cudaStream_t)stream;
    const int algo = r->rm.algo, roww = r->sm.rowB / 4;
    if (r->mode == 1) {                                                 // fused: one launch for all the generations
        const uint32_t left = r->rm.max_gens - r->gen, ng = std::min(n_generations, left);   // g <= max_gens (O10)
        if (ng == 0) return CAO_OK;
        if (r->gen_grid == 0) {                                         // first launch: opt-in shared memory, persistent grid size
            int occ = 0, dev = 0, sms = 0;
            CAO_CUDA(cudaGetDevice(&dev));
            CAO_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
            int rc = CAO_OK;
            switch (algo) {
                case CAO_DE: rc = cao_gen_setup_0(roww, r->gen_threads, r->gen_smem, (int)r->lay.wide, &occ); break;
                case CAO_PSO: rc = cao_gen_setup_1(roww, r->gen_threads, r->gen_smem, (int)r->lay.wide, &occ); break;
                case CAO_FIREFLY: rc = cao_gen_setup_2(roww, r->gen_threads, r->gen_smem, (int)r->lay.wide, &occ); break;
                default: rc = cao_gen_setup_3(roww, r->gen_threads, r->gen_smem, (int)r->lay.wide, &occ); break;
            }
            if (rc) return rc;
            if (occ < 1) return cao_fail(CAO_E_TOO_LARGE, "cao_runs_step: the population state does not fit the shared memory of one SM");
            const uint64_t need = ((uint64_t)r->rm.R + r->lay.NG - 1) / r->lay.NG;
            r->gen_grid = (unsigned)std::min<uint64_t>(need, (uint64_t)sms * (uint64_t)occ);
        }
        int rc = CAO_OK;
        {
            ProfScope ps(PK_GEN, st);
            switch (algo) {
#define CALL_GEN(A) rc = cao_gen_launch_##A(roww, r->gen_grid, r->gen_threads, r->gen_smem, st, r->sm, r->s->probe, r->rm, r->lay, r->gen, ng)
                case CAO_DE: CALL_GEN(0); break;
                case CAO_PSO: CALL_GEN(1); break;
                case CAO_FIREFLY: CALL_GEN(2); break;
                default: CALL_GEN(3); break;
            }
        }
        if (rc) return rc;
        r->gen += ng;
        return CAO_OK;
    }
    for (uint32_t it = 0; it < n_generations; ++it) {
        if (r->gen >= r->rm.max_gens) break;                            // g <= max_gens (O10)
        const uint32_t g = r->gen + 1;
#define CALL_OP(A, W) if (r->block <= 256) k_op<A, W, 256><<<r->rm.R, r->block, r->smem_op, st>>>(r->sm, r->rm, g); \
                      else k_op<A, W, 1024><<<r->rm.R, r->block, r->smem_op, st>>>(r->sm, r->rm, g)
        { ProfScope ps(PK_OP, st); DISPATCH_ALGO_ROWW(algo, roww, CALL_OP); }
        CAO_LAUNCHED("k_op");
        int rc = CAO_OK;
        const int levels = r->s->probe.levels;
        const cao_variant& vr = r->rm.var;
        if (!vr.constraint_aware) {
            // NEXT-2: nothing is repaired (L272, L284)
        } else if (vr.repair_mode == 1) {                               // NEXT-1: the paper's own repairs, all by table scan (wl2)
            const RunsMeta& m = r->rm;
            if (algo == CAO_DE) rc = launch_scan(r->sm, m.cand, m.wl2, m.wl2_count, m.key, true, st, true);
            else if (algo == CAO_GA) {
                rc = launch_scan_nb(r->sm, 1, m.cand, m.wl2, m.wl2_count, m.present, XAddr{nullptr, 1, 0, 0, 0}, m.key3, m.cnt3, st);
                if (!rc) rc = launch_pick_nb(r->sm, m.cand, m.wl2, m.wl2_count, m.present, m.cnt3, nullptr, m.seed, m.first_run, m.P, g, m.key, m.rule, st);
            } else {
                const XAddr xa{m.x, m.P, (uint64_t)r->sm.n * m.P, m.P, 1};
                rc = launch_scan_nb(r->sm, 0, m.cand, m.wl2, m.wl2_count, m.present, xa, m.key3, m.cnt3, st);
            }
            if (rc) return rc;
        } else {
            if (levels >= 2) {
                rc = launch_probe23(r->s, r->sm, r->rm.cand, r->rm.wl, r->rm.wl_count, r->rm.key, r->rm.wl2, r->rm.wl2_count,
                                    &r->rm.counters[1], levels, st);
                if (rc) return rc;
            }
            rc = launch_scan(r->sm, r->rm.cand, levels >= 2 ? r->rm.wl2 : r->rm.wl, levels >= 2 ? r->rm.wl2_count : r->rm.wl_count, r->rm.key, true, st);
            if (rc) return rc;
        }
#define CALL_FIN(A, W) k_finish<A, W><<<r->rm.R, r->block, r->smem_fin, st>>>(r->sm, r->rm, g)
        { ProfScope ps(PK_FINISH, st); DISPATCH_ALGO_ROWW(algo, roww, CALL_FIN); }
        CAO_LAUNCHED("k_finish");
        r->gen = g;
    }
    return CAO_OK;
}

int cao_runs_set_fused_width(cao_runs* r, int32_t width) {
    if (!r || (width != 0 && width != 1 && width != 2 && width != 4))
        return cao_fail(CAO_E_INVALID_ARG, "cao_runs_set_fused_width: width must be 0 (automatic), 1, 2 or 4");
    if (r->gen_grid != 0) return cao_fail(CAO_E_STATE, "cao_runs_set_fused_width: call before the first fused cao_runs_step");
    const GenLayout L = gen_layout(r->s, r->rm.algo, r->rm.P, r->rm.R, width);
    const size_t smem = ((size_t)L.cta_words + (size_t)L.NG * L.words) * 4;
    if (smem > 227 * 1024) return cao_fail(CAO_E_TOO_LARGE, "cao_runs_set_fused_width: the groups do not fit the shared memory of one SM");
    r->lay = L; r->gen_threads = L.G * L.NG; r->gen_smem = smem;
    return CAO_OK;
}
int cao_runs_fused_width(const cao_runs* r, int32_t* width) {
    if (!r || !width) return cao_fail(CAO_E_INVALID_ARG, "cao_runs_fused_width: NULL argument");
    *width = (int32_t)(r->lay.G / ((r->rm.P + 31) / 32 * 32));
    return CAO_OK;
}

int cao_runs_mode(const cao_runs* r, int32_t* mode) {
    if (!r || !mode) return cao_fail(CAO_E_INVALID_ARG, "cao_runs_mode: NULL argument");
    *mode = r->mode;
    return CAO_OK;
}

int cao_runs_set_mode(cao_runs* r, int32_t mode) {
    if (!r || (mode != 0 && mode != 1)) return cao_fail(CAO_E_INVALID_ARG, "cao_runs_set_mode: mode must be 0 (phased) or 1 (fused)");
    if (mode == 1 && r->var_on)
        return cao_fail(CAO_E_INVALID_ARG, "cao_runs_set_mode: runs with a non-default cao_variant use the phased pipeline only");
    if (mode == 1 && r->gen_smem > 227 * 1024)
        return cao_fail(CAO_E_TOO_LARGE, "cao_runs_set_mode: the population state does not fit the shared memory of one SM (fused mode)");
    r->mode = mode;
    return CAO_OK;
}

int cao_runs_best(const cao_runs* r, float* d_best_f, uint32_t* d_best_rank, uint32_t* d_uniq, uint32_t* d_gens_done, void* stream) {
    if (!r) return cao_fail(CAO_E_INVALID_ARG, "cao_runs_best: NULL runs");
    cudaStream_t st = (cudaStream_t)stream;
    const uint64_t b = (uint64_t)r->rm.R * 4;
    if (d_best_f) CAO_CUDA(cudaMemcpyAsync(d_best_f, r->rm.best_f, b, cudaMemcpyDeviceToDevice, st));
    if (d_best_rank) CAO_CUDA(cudaMemcpyAsync(d_best_rank, r->rm.best_rank, b, cudaMemcpyDeviceToDevice, st));
    if (d_uniq) CAO_CUDA(cudaMemcpyAsync(d_uniq, r->rm.uniq, b, cudaMemcpyDeviceToDevice, st));
    if (d_gens_done) CAO_CUDA(cudaMemcpyAsync(d_gens_done, r->rm.gens_done, b, cudaMemcpyDeviceToDevice, st));
    return CAO_OK;
}

int cao_runs_trajectory(const cao_runs* r, const void** d_traj, uint32_t* gens_recorded) {
    if (!r) return cao_fail(CAO_E_INVALID_ARG, "cao_runs_trajectory: NULL runs");
    if (d_traj) *d_traj = r->rm.traj;
    if (gens_recorded) *gens_recorded = r->gen;
    return CAO_OK;
}

int cao_runs_debug_last(const cao_runs* r, const uint8_t** d_postsnap_rows, const uint8_t** d_valid, const uint32_t** d_repaired_rank,
                        const uint32_t** d_eval_rank, const float** d_f, const uint8_t** d_accept, const uint8_t** d_active) {
    if (!r) return cao_fail(CAO_E_INVALID_ARG, "cao_runs_debug_last: NULL runs");
    if (d_postsnap_rows) *d_postsnap_rows = r->rm.cand;
    if (d_valid) *d_valid = r->rm.valid;
    if (d_repaired_rank) *d_repaired_rank = r->rm.rep_rank;
    if (d_eval_rank) *d_eval_rank = r->rm.eval_rank;
    if (d_f) *d_f = r->rm.tap_f;
    if (d_accept) *d_accept = r->rm.accept;
    if (d_active) *d_active = r->rm.active;
    return CAO_OK;
}

int cao_runs_debug_rule(const cao_runs* r, const uint8_t** d_rule) {
    if (!r || !d_rule) return cao_fail(CAO_E_INVALID_ARG, "cao_runs_debug_rule: NULL argument");
    if (!r->var_on) return cao_fail(CAO_E_STATE, "cao_runs_debug_rule: only runs with a non-default cao_variant record the rule");
    *d_rule = r->rm.rule;
    return CAO_OK;
}

int cao_runs_debug_state(const cao_runs* r, int32_t which, const void** d_ptr, uint64_t* bytes) {
    if (!r || !d_ptr || !bytes) return cao_fail(CAO_E_INVALID_ARG, "cao_runs_debug_state: NULL argument");
    const int a = r->rm.algo;
    const bool cont = a == CAO_PSO || a == CAO_FIREFLY;
    switch (which) {
        case 0: if (cont) break; *d_ptr = r->rm.idx; *bytes = r->bytes_idx; return CAO_OK;
        case 1: *d_ptr = r->rm.rank; *bytes = r->bytes_pi; return CAO_OK;
        case 2: *d_ptr = r->rm.f; *bytes = r->bytes_pi; return CAO_OK;
        case 3: if (!cont) break; *d_ptr = r->rm.x; *bytes = r->bytes_pn; return CAO_OK;
        case 4: if (a != CAO_PSO) break; *d_ptr = r->rm.v; *bytes = r->bytes_pn; return CAO_OK;
        case 5: if (a != CAO_PSO) break; *d_ptr = r->rm.pb; *bytes = r->bytes_pn; return CAO_OK;
        case 6: if (a != CAO_PSO) break; *d_ptr = r->rm.pbf; *bytes = r->bytes_pi; return CAO_OK;
        default: break;
    }
    return cao_fail(CAO_E_INVALID_ARG, "cao_runs_debug_state: this algorithm has no such state array");
}

int cao_runs_counters(const cao_runs* r, void* stream, uint64_t* n_repaired, uint64_t* n_scanned, uint64_t* n_evaluated) {
    if (!r) return cao_fail(CAO_E_INVALID_ARG, "cao_runs_counters: NULL runs");
    unsigned long long h[3] = {0, 0, 0};
    CAO_CUDA(cudaMemcpyAsync(h, r->rm.counters, 24, cudaMemcpyDeviceToHost, (cudaStream_t)stream));
    CAO_CUDA(cudaStreamSynchronize((cudaStream_t)stream));
    if (n_repaired) *n_repaired = h[0];
    if (n_scanned) *n_scanned = h[1];
    if (n_evaluated) *n_evaluated = h[2];
    return CAO_OK;
}

int cao_runs_stats(const cao_runs* r, void* stream, uint64_t* h_out32) {
    if (!r || !h_out32) return cao_fail(CAO_E_INVALID_ARG, "cao_runs_stats: NULL argument");
    CAO_CUDA(cudaMemcpyAsync(h_out32, r->rm.counters, 32 * 8, cudaMemcpyDeviceToHost, (cudaStream_t)stream));
    CAO_CUDA(cudaStreamSynchronize((cudaStream_t)stream));
    return CAO_OK;
}

// ---------------------------------------------------------------------------------------------
// NEXT-1 standalone.  Scratch: key | key3 | cnt3 | wl | wl_count | rule | present | clean rows.
struct ModeScratch { uint64_t key, key3, cnt3, wl, wl_count, rule, present, clean, total; };
static ModeScratch mode_scratch(const cao_space* s, uint64_t count) {
    ModeScratch L{};
    const uint64_t c = std::max<uint64_t>(1, count);
    uint64_t off = 0;
    auto take = [&](uint64_t bytes) { uint64_t o = off; off = align256(off + bytes); return o; };
    L.key = take(c * 8); L.key3 = take(c * 24); L.cnt3 = take(c * 12); L.wl = take(c * 4); L.wl_count = take(256);
    L.rule = take(c); L.present = take((uint64_t)CAO_MAX_DIMS * 256 + 256); L.clean = take(c * (uint64_t)s->meta.rowB);
    L.total = off;
    return L;
}
int cao_space_repair_mode_scratch_bytes(const cao_space* s, uint64_t count, uint64_t* bytes) {
    if (!s || !bytes) return cao_fail(CAO_E_INVALID_ARG, "cao_space_repair_mode_scratch_bytes: NULL argument");
    *bytes = mode_scratch(s, count).total;
    return CAO_OK;
}
int cao_space_repair_mode(const cao_space* s, int32_t mode, const uint8_t* d_idx_rows, const float* d_x, const uint32_t* d_w,
                          uint64_t count, uint32_t* d_rank_out, uint8_t* d_rule_out, void* d_scratch, void* stream) {
    if (!s) return cao_fail(CAO_E_INVALID_ARG, "cao_space_repair_mode: NULL space");
    if (!s->filled) return cao_fail(CAO_E_STATE, "cao_space_repair_mode: space not built");
    if (mode < 1 || mode > 3) return cao_fail(CAO_E_INVALID_ARG, "cao_space_repair_mode: mode must be 1 (index distance), 2 (Alg.2) or 3 (Alg.3)");
    if (count == 0) return CAO_OK;
    if (!d_idx_rows || !d_rank_out || (mode == 2 && !d_x) || (mode == 3 && !d_w))
        return cao_fail(CAO_E_INVALID_ARG, "cao_space_repair_mode: NULL argument");
    if (count >= (1ull << 32)) return cao_fail(CAO_E_TOO_LARGE, "cao_space_repair_mode: count >= 2^32");
    if (s->meta.V == 0) return cao_fail(CAO_E_EMPTY_SPACE, "cao_space_repair_mode: the space has no valid configuration");
    if (!d_scratch || ((uintptr_t)d_scratch & 255) || ((uintptr_t)d_idx_rows & 15))
        return cao_fail(CAO_E_WORKSPACE, "cao_space_repair_mode: scratch must be 256-byte aligned, rows 16-byte aligned");
    cudaStream_t st = (cudaStream_t)stream;
    const ModeScratch L = mode_scratch(s, count);
    uint8_t* sc = (uint8_t*)d_scratch;
    unsigned long long* key = (unsigned long long*)(sc + L.key); unsigned long long* key3 = (unsigned long long*)(sc + L.key3);
    uint32_t* cnt3 = (uint32_t*)(sc + L.cnt3); uint32_t* wl = (uint32_t*)(sc + L.wl); uint32_t* wl_count = (uint32_t*)(sc + L.wl_count);
    uint8_t* rule = sc + L.rule; uint8_t* present = sc + L.present; uint8_t* clean = sc + L.clean;
    CAO_CUDA(cudaMemsetAsync(wl_count, 0, 8, st));
    int rc = launch_present(s->meta, present, st);
    if (rc) return rc;
    const unsigned grid = (unsigned)((count + 255) / 256);
    {
        ProfScope ps(PK_QUERY, st);
        if (s->meta.rowB == 16) k_mode_probe<4><<<grid, 256, 0, st>>>(s->meta, d_idx_rows, clean, count, key, key3, cnt3, wl, wl_count, rule);
        else k_mode_probe<8><<<grid, 256, 0, st>>>(s->meta, d_idx_rows, clean, count, key, key3, cnt3, wl, wl_count, rule);
    }
    CAO_LAUNCHED("k_mode_probe");
    if (mode == 1) rc = launch_scan(s->meta, clean, wl, wl_count, key, true, st, true);
    else if (mode == 2) rc = launch_scan_nb(s->meta, 0, clean, wl, wl_count, present, XAddr{d_x, 1, (uint64_t)s->meta.n, 1, 0}, key3, cnt3, st);
    else {
        rc = launch_scan_nb(s->meta, 1, clean, wl, wl_count, present, XAddr{nullptr, 1, 0, 0, 0}, key3, cnt3, st);
        if (!rc) rc = launch_pick_nb(s->meta, clean, wl, wl_count, present, cnt3, d_w, 0, 0, 1, 0, key, rule, st);
    }
    if (rc) return rc;
    k_mode_finish<<<grid, 256, 0, st>>>(mode, key, key3, count, d_rank_out, rule, d_rule_out);
    CAO_LAUNCHED("k_mode_finish");
    return CAO_OK;
}

// ---------------------------------------------------------------------------------------------
// NEXT-4
static uint64_t next_pow2(uint64_t v) { uint64_t p = 1; while (p < v) p <<= 1; return p; }
int cao_space_sort_objective(const cao_space* s, float* d_sorted, void* d_scratch, void* stream) {
    if (!s || !d_sorted || !d_scratch) return cao_fail(CAO_E_INVALID_ARG, "cao_space_sort_objective: NULL argument");
    if (!s->filled || !s->meta.obj) return cao_fail(CAO_E_STATE, "cao_space_sort_objective: build the space and set the objective first");
    if (s->meta.V == 0) return cao_fail(CAO_E_EMPTY_SPACE, "cao_space_sort_objective: the space has no valid configuration");
    cudaStream_t st = (cudaStream_t)stream;
    if (s->meta.V > (1ull << 31)) return cao_fail(CAO_E_TOO_LARGE, "cao_space_sort_objective: more than 2^31 valid configurations");
    const uint32_t V = s->meta.V, n2 = (uint32_t)next_pow2(V);
    uint32_t* buf = (uint32_t*)d_scratch;
    const unsigned grid = (n2 + 255) / 256;
    k_sort_load<<<grid, 256, 0, st>>>(s->meta.obj, V, buf, n2);
    CAO_LAUNCHED("k_sort_load");
    for (uint32_t k = 2; k <= n2; k <<= 1)
        for (uint32_t j = k >> 1; j > 0; j >>= 1) { k_bitonic_step<<<grid, 256, 0, st>>>(buf, n2, j, k); ++g_cao_launches; }
    CAO_CUDA(cudaGetLastError());
    k_sort_store<<<(V + 255) / 256, 256, 0, st>>>(buf, V, d_sorted);
    CAO_LAUNCHED("k_sort_store");
    return CAO_OK;
}
int cao_space_baseline(const cao_space* s, const float* d_sorted, const uint64_t* d_t, uint32_t S, double* d_B, void* stream) {
    if (!s || !d_sorted || !d_t || !d_B) return cao_fail(CAO_E_INVALID_ARG, "cao_space_baseline: NULL argument");
    if (!s->filled || s->meta.V == 0) return cao_fail(CAO_E_STATE, "cao_space_baseline: space not built or empty");
    if (S == 0) return CAO_OK;
    k_baseline<<<(S + 31) / 32, 32, 0, (cudaStream_t)stream>>>(d_sorted, s->meta.V, d_t, S, d_B);
    CAO_LAUNCHED("k_baseline");
    return CAO_OK;
}
int cao_runs_score(const cao_runs* r, const float* d_sorted, const uint64_t* d_t, const double* d_B, uint32_t S, double* d_per_t,
                   double* d_score, void* d_scratch, void* stream) {
    if (!r || !d_sorted || !d_t || !d_B || !d_per_t || !d_score || !d_scratch) return cao_fail(CAO_E_INVALID_ARG, "cao_runs_score: NULL argument");
    if (S == 0) return cao_fail(CAO_E_INVALID_ARG, "cao_runs_score: no sampling point");
    cudaStream_t st = (cudaStream_t)stream;
    const uint64_t items = (uint64_t)S * r->rm.R;
    k_score_runs<<<(unsigned)((items + 255) / 256), 256, 0, st>>>(r->rm.traj, r->rm.R, r->gen, d_sorted, r->sm.V, d_t, d_B, S, (double*)d_scratch);
    CAO_LAUNCHED("k_score_runs");
    k_score_reduce<<<(S + 31) / 32, 32, 0, st>>>((const double*)d_scratch, r->rm.R, S, d_per_t, d_score);
    CAO_LAUNCHED("k_score_reduce");
    k_score_final<<<1, 1, 0, st>>>(d_per_t, S, d_score);
    CAO_LAUNCHED("k_score_final");
    return CAO_OK;
}

// ---------------------------------------------------------------------------------------------
__global__ void k_test_philox(const uint32_t* __restrict__ in, uint32_t* out, uint64_t count) {
    uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= count) return;
    const uint32_t* p = in + i * 6;
    uint4 r = philox4x32_10(make_uint4(p[0], p[1], p[2], p[3]), p[4], p[5]);
    ((uint4*)out)[i] = r;
}
__global__ void k_test_exp_neg(const float* __restrict__ z, float* out, uint64_t count) {
    uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < count) out[i] = exp_neg_spec(z[i]);
}
int cao_test_philox(const uint32_t* d_ctr_key, uint32_t* d_out, uint64_t count, void* stream) {
    if (count == 0) return CAO_OK;
    if (!d_ctr_key || !d_out) return cao_fail(CAO_E_INVALID_ARG, "cao_test_philox: NULL argument");
    k_test_philox<<<(unsigned)((count + 255) / 256), 256, 0, (cudaStream_t)stream>>>(d_ctr_key, d_out, count);
    CAO_LAUNCHED("k_test_philox");
    return CAO_OK;
}
// The same counters and keys through cuRAND's own device function curand_Philox4x32_10 (an independent implementation).
__global__ void k_test_curand_philox(const uint32_t* __restrict__ in, uint32_t* out, uint64_t count) {
    uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= count) return;
    const uint32_t* p = in + i * 6;
    uint4 r = curand_Philox4x32_10(make_uint4(p[0], p[1], p[2], p[3]), make_uint2(p[4], p[5]));
    ((uint4*)out)[i] = r;
}
int cao_test_curand_philox(const uint32_t* d_ctr_key, uint32_t* d_out, uint64_t count, void* stream) {
    if (count == 0) return CAO_OK;
    if (!d_ctr_key || !d_out) return cao_fail(CAO_E_INVALID_ARG, "cao_test_curand_philox: NULL argument");
    k_test_curand_philox<<<(unsigned)((count + 255) / 256), 256, 0, (cudaStream_t)stream>>>(d_ctr_key, d_out, count);
    CAO_LAUNCHED("k_test_curand_philox");
    return CAO_OK;
}
int cao_test_int_peak(int32_t kind, uint32_t iters, uint32_t n_ctas, uint32_t* d_out, void* stream) {
    if (!d_out || n_ctas == 0) return cao_fail(CAO_E_INVALID_ARG, "cao_test_int_peak: NULL / empty argument");
    cudaStream_t st = (cudaStream_t)stream;
    switch (kind) {
        case 0: k_int_peak<0><<<n_ctas, 256, 0, st>>>(d_out, iters); break;
        case 1: k_int_peak<1><<<n_ctas, 256, 0, st>>>(d_out, iters); break;
        case 2: k_int_peak<2><<<n_ctas, 256, 0, st>>>(d_out, iters); break;
        case 3: k_int_peak<3><<<n_ctas, 256, 0, st>>>(d_out, iters); break;
        case 4: k_int_peak<4><<<n_ctas, 256, 0, st>>>(d_out, iters); break;
        case 5: k_int_peak<5><<<n_ctas, 256, 0, st>>>(d_out, iters); break;
        default: return cao_fail(CAO_E_INVALID_ARG, "cao_test_int_peak: kind must be 0..5");
    }
    CAO_LAUNCHED("k_int_peak");
    return CAO_OK;
}
int cao_test_exp_neg(const float* d_z, float* d_out, uint64_t count, void* stream) {
    if (count == 0) return CAO_OK;
    if (!d_z || !d_out) return cao_fail(CAO_E_INVALID_ARG, "cao_test_exp_neg: NULL argument");
    k_test_exp_neg<<<(unsigned)((count + 255) / 256), 256, 0, (cudaStream_t)stream>>>(d_z, d_out, count);
    CAO_LAUNCHED("k_test_exp_neg");
    return CAO_OK;
}

}  // extern "C"

// cao_host.h -- host-side objects behind the opaque handles of include/cao.h.
#pragma once
#include <cstdint>
#include <string>
#include <vector>
#include <atomic>
#include <cuda_runtime.h>
#include "../../include/cao.h"
#include "cao_device.cuh"

extern thread_local std::string g_cao_err;
extern std::atomic<uint64_t> g_cao_launches;
int cao_fail(int code, const std::string& msg);
int cao_cuda_check(cudaError_t e, const char* what);
#define CAO_CUDA(x) do { int rc_ = cao_cuda_check((x), #x); if (rc_) return rc_; } while (0)
#define CAO_LAUNCHED(what) do { ++g_cao_launches; int rc_ = cao_cuda_check(cudaGetLastError(), what); if (rc_) return rc_; } while (0)

// Optional per-kernel-class device timing (cao_profile_*): CUDA events on the launching stream around each launch.
enum { PK_TABLE = 0, PK_ENUM, PK_CSCAN, PK_FILL, PK_INIT, PK_OP, PK_SCAN, PK_FINISH, PK_QUERY, PK_PROBE, PK_GEN, PK_RESID, PK_MASKS, PK_RESPRE, PK_N };
extern std::atomic<int> g_cao_prof_on;
void cao_prof_mark(int cls, bool end, cudaStream_t st);
struct ProfScope {
    int cls; cudaStream_t st; bool on;
    ProfScope(int c, cudaStream_t s) : cls(c), st(s), on(g_cao_prof_on.load(std::memory_order_relaxed) != 0) { if (on) cao_prof_mark(cls, false, st); }
    ~ProfScope() { if (on) cao_prof_mark(cls, true, st); }
};

static inline uint64_t align256(uint64_t x) { return (x + 255) & ~255ull; }

// Multiprocessors of the current device (cached per device ordinal): every persistent / grid-stride grid is sized as a
// multiple of it.  Without a usable device (host-side planning on a CPU-only box) it answers 148, the B200's count; the
// value only shapes grids and chunking, never results.
unsigned cao_sm_count();

// Opt-in to more than 48 KB of dynamic shared memory.  cudaFuncAttributeMaxDynamicSharedMemorySize REPLACES the kernel's
// limit, it does not raise it: two live objects (two cao_runs, two cao_space) that share a kernel instantiation and each
// set "their" size would lower the limit under one another, and the larger one's next launch would fail with
// cudaErrorInvalidValue.  So every site sets the same value, the most the device grants this kernel (opt-in limit per
// block minus the kernel's static shared memory).  The limit is only a permission: what a launch occupies, and hence the
// residency, still follows the size given at launch.
template <class K>
static inline int cao_smem_optin_max(K* kernel, const char* what) {
    int dev = 0, optin = 0;
    cudaFuncAttributes fa{};
    int rc = cao_cuda_check(cudaGetDevice(&dev), what);
    if (!rc) rc = cao_cuda_check(cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev), what);
    if (!rc) rc = cao_cuda_check(cudaFuncGetAttributes(&fa, kernel), what);
    if (!rc) rc = cao_cuda_check(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, optin - (int)fa.sharedSizeBytes), what);
    return rc;
}
#define CAO_SMEM_OPTIN(kernel) do { int rc_ = cao_smem_optin_max(kernel, "shared-memory opt-in of " #kernel); if (rc_) return rc_; } while (0)

// Value classes of a residual constraint (cao_enum_kernels.cuh, pass 1c).
#define CAO_MAX_RC 4
struct ResClassArgs {
    long long* keys;                   // CAO_HS prefix values (CAO_CLS_EMPTY = free)
    uint64_t* table;                   // CAO_HS x Wb inner masks
    int32_t* overflow;                 // more distinct values than slots: the constraint falls back to the per-config path
    int32_t pc0, r;                    // first token of the suffix; residual constraint number
};

// One constraint in the enumeration plan.
struct ConsPlan {
    bool tabled = false;
    std::vector<int> scope;            // parameters the program reads, descending
    std::vector<int> outer;            // scope digits < t (outer part)
    std::vector<uint32_t> cstride;     // mixed-radix strides of the outer scope digits (row index of the table)
    uint64_t rows = 1;                 // product of m_d over the outer scope digits
    uint64_t table_off = 0;            // u64-word offset of the table inside the tables region
    uint64_t flag_off = 0;             // byte offset of its row flags inside the flags region
};

struct cao_space {
    std::vector<std::vector<int64_t>> dom;
    std::vector<std::vector<int32_t>> cons;
    int mode = 0;
    bool planned = false, counted = false, filled = false;
    SpaceMeta meta{};
    // enumeration plan
    int t = 0;                         // first inner digit: digits t..n-1 form one bitmap block of B configs
    uint64_t B = 0, n_blocks = 0, nd = 0, n_words = 0;
    uint32_t Wb = 0, CH = 1;           // u64 words per block mask; blocks per thread of k_enum (product of the last outer digits)
    int n_inv = 0, chunk_digits = 0;   // tabled constraints that do not read those digits; how many digits
    uint64_t off_keys = 0; bool use_keys = false;
    cudaStream_t side2 = nullptr; cudaEvent_t ev_fork2 = nullptr, ev_join2 = nullptr;   // residual prefix || masks
    std::vector<ConsPlan> plan;
    std::vector<int32_t> desc;         // descriptor words uploaded to the device
    int n_tab = 0, n_res = 0, n_rc = 0;
    int rc_pc0[CAO_MAX_RC] = {0, 0, 0, 0}, rc_r[CAO_MAX_RC] = {0, 0, 0, 0};
    uint64_t off_rc[CAO_MAX_RC] = {0, 0, 0, 0}, rc_bytes = 0;
    bool use_lut = false;
    // scratch layout (byte offsets)
    uint64_t off_dom = 0, off_desc = 0, off_tables = 0, off_flags = 0, off_lut = 0, off_cnt = 0, off_part = 0, off_V = 0,
             off_live = 0, off_groups = 0, off_pre = 0, scratch_bytes = 0;
    uint64_t tables_words = 0, flags_bytes = 0, n_part = 0, max_table_threads = 0, max_table_ci = 1;
    uint64_t bitmap_bytes = 0;
    void* d_scratch = nullptr;
    void* d_table = nullptr;
    // table layout
    uint64_t off_rows = 0, off_Ltab = 0, off_dir = 0, off_tgt = 0, table_bytes = 0;
    // Hamming-level probes (S5)
    ProbeMeta probe{};
    std::vector<uint16_t> h_nb;
    std::vector<uint32_t> h_pairs, h_triples;
    uint64_t off_pairs = 0, off_triples = 0;
    int probe_levels_req = -1;         // -1 = cost model
    // the zero fill of the bitmap runs on a side stream, overlapped with the table build
    cudaStream_t side = nullptr;
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
    // cao_space_rebuild replays a captured CUDA graph of the whole of S1 (launch-bound on small spaces)
    cudaGraphExec_t rebuild_exec = nullptr;
    uint64_t rebuild_launches = 0;
};

// Arguments of the pass-1 kernels, passed by value.
struct EnumArgs {
    uint64_t B, n_blocks;
    const int64_t* dom;                // [n][256]
    const int32_t* desc;
    const uint64_t* tables;
    const uint8_t* flags;              // one byte per table row: the row has a bit set
    uint64_t* bitmap;                  // zero-filled
    uint32_t* cnt;                     // per-512 counts (zeroed)
    uint32_t* live;                    // blocks that survive the tabled constraints
    uint32_t* live_count;
    uint32_t* keys;                    // [live][n_tab] table row index of every survivor (NULL: k_masks recomputes them)
    int32_t n_inv;                     // the first n_inv tabled constraints do not read the last outer digits (chunk-invariant)
    uint32_t Wb, CH;
    int32_t t, n_tab, n_res;
    uint32_t desc_words, desc_in_smem; // the descriptor words are staged in shared memory by every CTA (when they fit)
    int32_t n_rc;                      // residual constraints with value classes
    int8_t rc_of[32];                  // residual r -> class table (or -1); at most 32 residual constraints are looked at
    ResClassArgs rc[CAO_MAX_RC];
};

struct cao_runs;

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
enum { PK_TABLE = 0, PK_ENUM, PK_CSCAN, PK_FILL, PK_INIT, PK_OP, PK_SCAN, PK_FINISH, PK_QUERY, PK_PROBE, PK_GEN, PK_N };
extern std::atomic<int> g_cao_prof_on;
void cao_prof_mark(int cls, bool end, cudaStream_t st);
struct ProfScope {
    int cls; cudaStream_t st; bool on;
    ProfScope(int c, cudaStream_t s) : cls(c), st(s), on(g_cao_prof_on.load(std::memory_order_relaxed) != 0) { if (on) cao_prof_mark(cls, false, st); }
    ~ProfScope() { if (on) cao_prof_mark(cls, true, st); }
};

static inline uint64_t align256(uint64_t x) { return (x + 255) & ~255ull; }

// One constraint in the enumeration plan.
struct ConsPlan {
    bool tabled = false;
    std::vector<int> scope;            // parameters the program reads, ascending
    std::vector<int> outer;            // scope digits < t (outer part)
    std::vector<uint32_t> cstride;     // mixed-radix strides of the outer scope digits (row index of the table)
    uint64_t rows = 1;                 // product of m_d over the outer scope digits
    uint64_t table_off = 0;            // u64-word offset of the table inside the tables region
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
    uint32_t Wb = 0, nb = 0, nb_tabled = 0;           // u64 words per block mask; blocks per CTA
    std::vector<ConsPlan> plan;
    std::vector<int32_t> desc;         // descriptor words uploaded to the device
    int n_tab = 0, n_res = 0, n_rc = 0;
    int rc_pc0[4] = {0, 0, 0, 0};
    uint64_t off_rc[4] = {0, 0, 0, 0}, rc_bytes = 0;
    // scratch layout (byte offsets)
    uint64_t off_dom = 0, off_desc = 0, off_tables = 0, off_cnt = 0, off_part = 0, off_V = 0, scratch_bytes = 0;
    uint64_t tables_words = 0, n_part = 0, max_table_threads = 0, max_table_ci = 1;
    uint64_t bitmap_bytes = 0;
    void* d_scratch = nullptr;
    void* d_table = nullptr;
    // table layout
    uint64_t off_rows = 0, off_Ltab = 0, off_dir = 0, off_tgt = 0, table_bytes = 0;
    // Hamming-level probes (S5)
    ProbeMeta probe{};
    std::vector<uint16_t> h_nb;
    std::vector<uint32_t> h_pairs;
    uint64_t off_pairs = 0;
    int probe_levels_req = -1;         // -1 = cost model
};

// Arguments of the pass-1 kernel, passed by value.
// Residual constraint handled through value classes: blocks whose program prefix leaves the
// same single stack value share one inner mask.
#define CAO_HS 4096                         // hash slots = maximum number of distinct prefix values
#define CAO_MAX_RC 4
#define CAO_CLS_EMPTY ((long long)0x8080808080808080ll)   // below -2^62: never a saturated value
#define CAO_CLS_FALSE 0xFFFFFFFFu
#define CAO_CLS_OVERFLOW 0xFFFFFFFEu
struct ResClassArgs {
    long long* keys;                   // CAO_HS prefix values (CAO_CLS_EMPTY = free)
    uint64_t* table;                   // CAO_HS x Wb inner masks
    uint32_t* blk_class;               // n_blocks: hash slot of the block's prefix value
    int32_t* overflow;                 // set if more than the table holds: the constraint falls back to phase 1b
    int32_t pc0;                       // first token of the suffix
};

struct EnumArgs {
    uint64_t B, magicB, n_blocks, n_words;
    const int64_t* dom;                // [n][256]
    const int32_t* desc;
    const uint64_t* tables;
    uint64_t* bitmap;
    uint32_t* cnt;                     // per-512 counts (zeroed)
    uint32_t Wb, nb;
    int32_t t, n_tab, n_res, n_rc;     // the first n_rc residual constraints use value classes
    ResClassArgs rc[CAO_MAX_RC];
};

struct cao_runs;

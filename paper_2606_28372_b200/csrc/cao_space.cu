// cao_space.cu -- host side of the search-space half of include/cao.h (S1, is-valid; L129-143).
#include <algorithm>
#include <cstring>
#include "cao_enum_kernels.cuh"
#include "cao_fill_kernels.cuh"

thread_local std::string g_cao_err;
std::atomic<uint64_t> g_cao_launches{0};
int cao_fail(int code, const std::string& msg) { g_cao_err = msg; return code; }
int cao_cuda_check(cudaError_t e, const char* what) {
    if (e == cudaSuccess) return 0;
    return cao_fail(CAO_E_CUDA, std::string(what) + ": " + cudaGetErrorString(e));
}

// ---------------------------------------------------------------------------------------------
// Profiling: event pairs per launch, summed per kernel class when read.
#include <mutex>
std::atomic<int> g_cao_prof_on{0};
namespace {
struct ProfRec { int cls; cudaEvent_t e0, e1; };
std::mutex g_prof_mu;
std::vector<ProfRec> g_prof_pending;
std::vector<cudaEvent_t> g_prof_pool;
double g_prof_ms[PK_N];
uint64_t g_prof_n[PK_N];
cudaEvent_t prof_event() {
    if (!g_prof_pool.empty()) { cudaEvent_t e = g_prof_pool.back(); g_prof_pool.pop_back(); return e; }
    cudaEvent_t e = nullptr; cudaEventCreate(&e); return e;
}
void prof_drain() {
    for (auto& r : g_prof_pending) {
        if (!r.e0 || !r.e1) continue;
        float ms = 0.0f;
        if (cudaEventSynchronize(r.e1) == cudaSuccess && cudaEventElapsedTime(&ms, r.e0, r.e1) == cudaSuccess) {
            g_prof_ms[r.cls] += ms; g_prof_n[r.cls] += 1;
        }
        g_prof_pool.push_back(r.e0); g_prof_pool.push_back(r.e1);
    }
    g_prof_pending.clear();
}
}  // namespace
unsigned cao_sm_count() {
    static std::atomic<int> cache[64];                                   // zero-initialised: 0 = not asked yet
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) { cudaGetLastError(); return 148u; }
    sms = cache[dev].load(std::memory_order_relaxed);
    if (sms > 0) return (unsigned)sms;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1) { cudaGetLastError(); return 148u; }
    cache[dev].store(sms, std::memory_order_relaxed);
    return (unsigned)sms;
}

void cao_prof_mark(int cls, bool end, cudaStream_t st) {
    std::lock_guard<std::mutex> lk(g_prof_mu);
    if (!end) {
        ProfRec r{cls, prof_event(), nullptr};
        if (r.e0) cudaEventRecord(r.e0, st);
        g_prof_pending.push_back(r);
    } else {
        for (size_t k = g_prof_pending.size(); k-- > 0;) {
            ProfRec& r = g_prof_pending[k];
            if (r.cls == cls && !r.e1) { r.e1 = prof_event(); if (r.e1) cudaEventRecord(r.e1, st); break; }
        }
    }
}

static bool program_ok(const int32_t* w, int nw, int n_params) {
    int sp = 0;
    for (int pc = 0; pc < nw; ++pc) {
        int32_t op = w[pc];
        if (op == CAO_OP_PUSH_PARAM) { if (pc + 1 >= nw || w[pc + 1] < 0 || w[pc + 1] >= n_params) return false; ++pc; ++sp; }
        else if (op == CAO_OP_PUSH_CONST) { if (pc + 2 >= nw) return false; pc += 2; ++sp; }
        else if (op == CAO_OP_NEG || op == CAO_OP_NOT) { if (sp < 1) return false; }
        else if (op >= CAO_OP_ADD && op <= CAO_OP_OR) { if (sp < 2) return false; --sp; }
        else return false;
        if (sp > CAO_MAX_STACK) return false;
    }
    return sp == 1;
}

extern "C" {

const char* cao_last_error(void) { return g_cao_err.c_str(); }
uint64_t cao_launch_count(void) { return g_cao_launches.load(); }

int cao_profile_enable(int32_t on) {
    std::lock_guard<std::mutex> lk(g_prof_mu);
    if (on) { prof_drain(); for (int c = 0; c < PK_N; ++c) { g_prof_ms[c] = 0.0; g_prof_n[c] = 0; } }
    g_cao_prof_on.store(on ? 1 : 0);
    return CAO_OK;
}
int cao_profile_read(int32_t cls, double* ms_total, uint64_t* launches) {
    if (cls < 0 || cls >= PK_N) return cao_fail(CAO_E_INVALID_ARG, "cao_profile_read: unknown kernel class");
    std::lock_guard<std::mutex> lk(g_prof_mu);
    prof_drain();
    if (ms_total) *ms_total = g_prof_ms[cls];
    if (launches) *launches = g_prof_n[cls];
    return CAO_OK;
}
const char* cao_profile_name(int32_t cls) {
    static const char* names[PK_N] = {"k_build_tables+k_inner_lut", "k_enum", "k_cnt_reduce+k_cnt_apply", "k_fill", "k_init",
                                      "k_op", "k_scan", "k_finish", "k_is_valid/k_repair_probe/k_repair_finish", "k_probe23", "k_gen",
                                      "k_residual", "k_keys+k_masks", "k_res_prefix+k_res_class_table"};
    return cls >= 0 && cls < PK_N ? names[cls] : "";
}

int cao_space_create(cao_space** out) {
    if (!out) return cao_fail(CAO_E_INVALID_ARG, "cao_space_create: out is NULL");
    *out = new cao_space();
    return CAO_OK;
}
void cao_space_destroy(cao_space* s) {
    if (!s) return;
    if (s->rebuild_exec) cudaGraphExecDestroy(s->rebuild_exec);
    if (s->ev_fork) cudaEventDestroy(s->ev_fork);
    if (s->ev_join) cudaEventDestroy(s->ev_join);
    if (s->side) cudaStreamDestroy(s->side);
    if (s->ev_fork2) cudaEventDestroy(s->ev_fork2);
    if (s->ev_join2) cudaEventDestroy(s->ev_join2);
    if (s->side2) cudaStreamDestroy(s->side2);
    delete s;
}

int cao_space_add_param(cao_space* s, const char*, const int64_t* h_values, int32_t n_values) {
    if (!s || !h_values) return cao_fail(CAO_E_INVALID_ARG, "cao_space_add_param: NULL argument");
    if (s->planned) return cao_fail(CAO_E_STATE, "cao_space_add_param: space already planned/built");
    if (n_values < 1) return cao_fail(CAO_E_INVALID_ARG, "cao_space_add_param: n_values < 1");
    if (n_values > 256 || s->dom.size() >= CAO_MAX_DIMS) return cao_fail(CAO_E_TOO_LARGE, "cao_space_add_param: more than 32 params or 256 values");
    s->dom.emplace_back(h_values, h_values + n_values);
    return CAO_OK;
}

int cao_space_add_constraint(cao_space* s, const int32_t* h_rpn, int32_t n_words) {
    if (!s || !h_rpn || n_words < 1) return cao_fail(CAO_E_INVALID_ARG, "cao_space_add_constraint: NULL/empty program");
    if (s->planned) return cao_fail(CAO_E_STATE, "cao_space_add_constraint: space already planned/built");
    if (!program_ok(h_rpn, n_words, (int)s->dom.size())) return cao_fail(CAO_E_INVALID_ARG, "cao_space_add_constraint: malformed program");
    s->cons.emplace_back(h_rpn, h_rpn + n_words);
    return CAO_OK;
}

int cao_space_set_build_mode(cao_space* s, int32_t mode) {
    if (!s || (mode != 0 && mode != 1)) return cao_fail(CAO_E_INVALID_ARG, "cao_space_set_build_mode: mode must be 0 or 1");
    if (s->planned) return cao_fail(CAO_E_STATE, "cao_space_set_build_mode: after build_workspace_bytes");
    s->mode = mode;
    return CAO_OK;
}

int cao_space_set_probe_levels(cao_space* s, int32_t levels) {
    if (!s || levels < -1 || levels > CAO_MAX_PROBE_LEVEL) return cao_fail(CAO_E_INVALID_ARG, "cao_space_set_probe_levels: levels must be -1 (auto) or 0..6");
    if (s->counted) return cao_fail(CAO_E_STATE, "cao_space_set_probe_levels: call before cao_space_build_count");
    s->probe_levels_req = levels;
    return CAO_OK;
}
int cao_space_probe_levels(const cao_space* s, int32_t* levels) {
    if (!s || !levels) return cao_fail(CAO_E_INVALID_ARG, "cao_space_probe_levels: NULL argument");
    if (!s->counted) return cao_fail(CAO_E_STATE, "cao_space_probe_levels: space not built");
    *levels = s->probe.levels;
    return CAO_OK;
}

static int plan_space(cao_space* s) {
    const int n = (int)s->dom.size();
    if (n < 1) return cao_fail(CAO_E_INVALID_ARG, "space has no parameters");
    SpaceMeta& M = s->meta;
    std::memset(&M, 0, sizeof(M));
    M.n = n; M.rowB = n <= 16 ? 16 : 32; M.M = 1;
    unsigned __int128 N = 1;
    for (int d = n - 1; d >= 0; --d) {
        M.stride[d] = (uint64_t)N;
        uint32_t m = (uint32_t)s->dom[d].size();
        M.m[d] = (uint16_t)m;
        M.M = std::max<int>(M.M, (int)m);
        M.magic[d] = m > 1 ? (uint64_t)((((unsigned __int128)1 << 64) + m - 1) / m) : 0;
        N *= m;
        if (N >= ((unsigned __int128)1 << 40)) return cao_fail(CAO_E_TOO_LARGE, "Cartesian size N >= 2^40");
    }
    M.N = (uint64_t)N;
    M.ltab32 = M.N <= (1ull << 32) ? 1 : 0;                       // Ltab holds u32 when every L fits (SURVEY 8(a) layout)
    // inner block: smallest trailing product >= 256 (or the whole space)
    uint64_t B = 1; int t = n;
    while (t > 0 && B < 256) { --t; B *= M.m[t]; }
    s->t = t; s->B = B; s->Wb = (uint32_t)((B + 63) / 64); s->n_blocks = M.N / B;
    s->n_words = (M.N + 63) / 64; s->nd = (M.N + 511) / 512;
    // chunk of k_enum = all combinations of the last k outer digits (product CH <= 32, and enough threads left)
    s->CH = 1; s->chunk_digits = 0;
    for (int d = t - 1; d >= 0; --d) {
        const uint64_t c2 = (uint64_t)s->CH * M.m[d];
        if (c2 > 32 || s->n_blocks / c2 < (uint64_t)cao_sm_count() * 256) break;
        s->CH = (uint32_t)c2; s->chunk_digits += 1;
    }
    // per-constraint plan
    s->plan.assign(s->cons.size(), ConsPlan());
    uint64_t total_words = 0, total_flags = 0;
    for (size_t c = 0; c < s->cons.size(); ++c) {
        ConsPlan& p = s->plan[c];
        const auto& w = s->cons[c];
        bool used[CAO_MAX_DIMS] = {false};
        for (size_t pc = 0; pc < w.size(); ++pc) {
            if (w[pc] == CAO_OP_PUSH_PARAM) { used[w[pc + 1]] = true; ++pc; }
            else if (w[pc] == CAO_OP_PUSH_CONST) pc += 2;
        }
        uint64_t rows = 1; bool ok = true;
        for (int d = n - 1; d >= 0; --d) if (used[d]) {
            p.scope.push_back(d);
            if (d < t) {
                p.outer.push_back(d); p.cstride.push_back((uint32_t)rows);
                rows *= M.m[d];
                if (rows > (1ull << 24)) { ok = false; rows = 1ull << 24; }
            }
        }
        p.rows = rows;
        uint64_t words = rows * s->Wb;
        p.tabled = s->mode == 0 && ok && words * 8 <= (8ull << 20) && (total_words + words) * 8 <= (128ull << 20);
        if (p.tabled) { p.table_off = total_words; total_words += words; p.flag_off = total_flags; total_flags += rows; }
    }
    s->tables_words = total_words; s->flags_bytes = total_flags;
    // descriptors: small tables first (the cheapest, usually most selective tests come first), then residual programs
    std::vector<int> tab, res;
    for (size_t c = 0; c < s->cons.size(); ++c) (s->plan[c].tabled ? tab : res).push_back((int)c);
    std::stable_sort(tab.begin(), tab.end(), [&](int a, int b) { return s->plan[a].rows < s->plan[b].rows; });
    // chunk-invariant constraints (no outer scope digit among the last chunk_digits) come first
    auto invariant = [&](int c) { for (int d : s->plan[c].outer) if (d >= t - s->chunk_digits) return false; return true; };
    std::stable_sort(tab.begin(), tab.end(), [&](int a, int b) { return invariant(a) > invariant(b); });
    s->n_inv = 0;
    for (int c : tab) if (invariant(c)) s->n_inv += 1;
    s->n_tab = (int)tab.size(); s->n_res = (int)res.size();
    std::vector<int32_t>& D = s->desc;
    D.assign(tab.size() + res.size() + s->cons.size(), 0);       // [tab offs][res offs][program offs of every constraint]
    std::vector<int32_t> prog_off(s->cons.size());
    for (size_t c = 0; c < s->cons.size(); ++c) {
        prog_off[c] = (int32_t)D.size();
        D[tab.size() + res.size() + c] = (int32_t)D.size();
        D.insert(D.end(), s->cons[c].begin(), s->cons[c].end());
    }
    s->max_table_threads = 0; s->max_table_ci = 1;
    for (size_t k = 0; k < tab.size(); ++k) {
        const ConsPlan& p = s->plan[tab[k]];
        D[k] = (int32_t)D.size();
        D.push_back((int32_t)(uint32_t)p.table_off); D.push_back((int32_t)(uint32_t)(p.table_off >> 32));
        D.push_back((int32_t)(uint32_t)p.flag_off);
        D.push_back((int32_t)p.outer.size());
        for (size_t e = 0; e < p.outer.size(); ++e) { D.push_back(p.outer[e]); D.push_back((int32_t)p.cstride[e]); }
        D.push_back(prog_off[tab[k]]); D.push_back((int32_t)s->cons[tab[k]].size()); D.push_back((int32_t)p.rows);
        // inner scope: the digits >= t the program reads; the inner pattern of a row depends on them only, so the
        // program runs once per (row, inner-scope combination) and the result is replicated over the block
        std::vector<int> inner; uint64_t Ci = 1;
        for (int d : p.scope) if (d >= t) inner.push_back(d);           // scope is descending in d
        std::vector<uint32_t> istride(inner.size());
        for (size_t e = 0; e < inner.size(); ++e) { istride[e] = (uint32_t)Ci; Ci *= M.m[inner[e]]; }
        D.push_back((int32_t)inner.size()); D.push_back((int32_t)Ci);
        for (size_t e = 0; e < inner.size(); ++e) { D.push_back(inner[e]); D.push_back((int32_t)istride[e]); }
        s->max_table_threads = std::max<uint64_t>(s->max_table_threads, p.rows * s->Wb * 64);
        s->max_table_ci = std::max<uint64_t>(s->max_table_ci, Ci);
    }
    for (size_t k = 0; k < res.size(); ++k) {
        D[tab.size() + k] = (int32_t)D.size();
        D.push_back((int32_t)s->cons[res[k]].size());
        D.insert(D.end(), s->cons[res[k]].begin(), s->cons[res[k]].end());
    }
    // Value classes: a residual program whose tokens before the first inner parameter leave exactly one stack value,
    // and whose remaining tokens read inner parameters only, depends on the outer digits through that one value.
    s->n_rc = 0;
    if (s->mode == 0 && (uint64_t)CAO_HS * s->Wb * 8 <= (32ull << 20)) {
        for (size_t k = 0; k < res.size() && k < 32 && s->n_rc < CAO_MAX_RC; ++k) {
            const auto& w = s->cons[res[k]];
            int sp = 0, pc0 = -1; bool ok = true;
            for (size_t pc = 0; pc < w.size(); ++pc) {
                const int op = w[pc];
                if (op == CAO_OP_PUSH_PARAM) {
                    const int d = w[pc + 1];
                    if (pc0 < 0 && d >= t) { pc0 = (int)pc; if (sp != 1) ok = false; }
                    else if (pc0 >= 0 && d < t) ok = false;               // the suffix reads an outer parameter
                    ++pc; ++sp;
                } else if (op == CAO_OP_PUSH_CONST) { pc += 2; ++sp; }
                else if (op == CAO_OP_NEG || op == CAO_OP_NOT) {}
                else --sp;
            }
            if (ok && pc0 > 0) { s->rc_pc0[s->n_rc] = pc0; s->rc_r[s->n_rc] = (int)k; ++s->n_rc; }
        }
    }
    s->use_lut = B * (uint64_t)M.rowB <= (1ull << 20);            // inner index bytes of every pattern (pass 2)
    // scratch layout
    uint64_t off = 0;
    s->off_dom = off; off = align256(off + (uint64_t)n * 256 * 8);
    s->off_desc = off; off = align256(off + D.size() * 4);
    s->off_tables = off; off = align256(off + std::max<uint64_t>(1, total_words) * 8);
    s->off_flags = off; off = align256(off + std::max<uint64_t>(1, total_flags));
    s->off_lut = off; off = align256(off + (s->use_lut ? B * (uint64_t)M.rowB : 1));
    s->n_part = (s->nd + 1 + SCAN_CHUNK - 1) / SCAN_CHUNK;
    s->off_part = off; off = align256(off + s->n_part * 8);      // chunk sums (u32) / look-back states (u64)
    s->off_V = off; off = align256(off + 32);                     // V (u64), scan ticket, live count, group count
    s->off_cnt = off; off = align256(off + (s->nd + 1) * 4);
    s->off_live = off; off = align256(off + s->n_blocks * 4);
    s->use_keys = s->n_tab > 0 && s->n_blocks * (uint64_t)s->n_tab * 4 <= (64ull << 20);
    s->off_keys = off; off = align256(off + (s->use_keys ? s->n_blocks * (uint64_t)s->n_tab * 4 : 1));
    s->off_pre = off; off = align256(off + (s->n_res ? s->n_blocks * (uint64_t)s->n_res * sizeof(ResPrefix) : 1));
    s->off_groups = off; off = align256(off + (s->nd + 1) * 4);
    s->rc_bytes = align256((uint64_t)CAO_HS * 8) + align256((uint64_t)CAO_HS * s->Wb * 8) + 256;
    for (int k = 0; k < s->n_rc; ++k) { s->off_rc[k] = off; off += s->rc_bytes; }
    s->scratch_bytes = off;
    s->bitmap_bytes = align256(s->n_words * 8);
    s->planned = true;
    return CAO_OK;
}

int cao_space_build_workspace_bytes(cao_space* s, uint64_t* bitmap_bytes, uint64_t* scratch_bytes) {
    if (!s || !bitmap_bytes || !scratch_bytes) return cao_fail(CAO_E_INVALID_ARG, "cao_space_build_workspace_bytes: NULL argument");
    if (!s->planned) { int rc = plan_space(s); if (rc) return rc; }
    *bitmap_bytes = s->bitmap_bytes; *scratch_bytes = s->scratch_bytes;
    return CAO_OK;
}

// S1 pass 1 on `st`: zero fill (side stream) || constraint tables, then block masks -> bitmap + per-512 counts,
// residual constraints on the survivors, and the first half of the count scan (V).
static int launch_pass1(cao_space* s, void* d_bitmap, uint8_t* sc, cudaStream_t st, bool with_reduce = true) {
    if (!s->side) {
        CAO_CUDA(cudaStreamCreateWithFlags(&s->side, cudaStreamNonBlocking));
        CAO_CUDA(cudaEventCreateWithFlags(&s->ev_fork, cudaEventDisableTiming));
        CAO_CUDA(cudaEventCreateWithFlags(&s->ev_join, cudaEventDisableTiming));
        CAO_CUDA(cudaStreamCreateWithFlags(&s->side2, cudaStreamNonBlocking));
        CAO_CUDA(cudaEventCreateWithFlags(&s->ev_fork2, cudaEventDisableTiming));
        CAO_CUDA(cudaEventCreateWithFlags(&s->ev_join2, cudaEventDisableTiming));
    }
    s->meta.bitmap = (const uint64_t*)d_bitmap;
    // fork: the zero fill of the bitmap (N/8 bytes, HBM-bound) overlaps the table build (latency-bound)
    CAO_CUDA(cudaEventRecord(s->ev_fork, st));
    CAO_CUDA(cudaStreamWaitEvent(s->side, s->ev_fork, 0));
    if (s->use_lut) {                                                   // the inner-digit LUT (needed by k_fill only) is off the critical path too
        ProfScope ps(PK_TABLE, s->side);
        k_inner_lut<<<(unsigned)((s->B + 255) / 256), 256, 0, s->side>>>(s->meta, (uint32_t*)(sc + s->off_lut), s->B, s->t, s->meta.rowB / 4);
        CAO_LAUNCHED("k_inner_lut");
    }
    CAO_CUDA(cudaMemsetAsync(d_bitmap, 0, s->bitmap_bytes, s->side));
    CAO_CUDA(cudaMemsetAsync(sc + s->off_part, 0, (s->off_cnt - s->off_part) + (s->nd + 1) * 4, s->side));   // scan states, V, tickets, counts
    for (int k = 0; k < s->n_rc; ++k) {                                 // class tables start empty
        uint8_t* b = sc + s->off_rc[k];
        CAO_CUDA(cudaMemsetAsync(b, 0x80, (uint64_t)CAO_HS * 8, s->side));
        CAO_CUDA(cudaMemsetAsync(b + align256((uint64_t)CAO_HS * 8) + align256((uint64_t)CAO_HS * s->Wb * 8), 0, 4, s->side));
    }
    CAO_CUDA(cudaEventRecord(s->ev_join, s->side));
    const int64_t* d_dom = (const int64_t*)(sc + s->off_dom);
    const int32_t* d_desc = (const int32_t*)(sc + s->off_desc);
    uint64_t* d_tables = (uint64_t*)(sc + s->off_tables);
    uint8_t* d_flags = sc + s->off_flags;
    if (s->n_tab) {
        ProfScope ps(PK_TABLE, st);
        dim3 grid((unsigned)std::min<uint64_t>((s->max_table_threads + 8191) / 8192, (uint64_t)cao_sm_count() * 8), (unsigned)s->n_tab);
        const uint32_t ci_cap = s->B <= 8192 ? (uint32_t)((s->B + 7) & ~7ull) : 0;
        const size_t tsm = 2 * (size_t)ci_cap + (size_t)std::max<uint64_t>(256, s->max_table_ci);
        if (tsm > 48 * 1024) CAO_SMEM_OPTIN(k_build_tables);
        k_build_tables<<<grid, 256, tsm, st>>>(s->meta, d_dom, d_desc, d_tables, d_flags, s->B, s->Wb, s->t, ci_cap);
        CAO_LAUNCHED("k_build_tables");
    }
    CAO_CUDA(cudaStreamWaitEvent(st, s->ev_join, 0));                   // join
    uint32_t* ctl = (uint32_t*)(sc + s->off_V);                         // [0..1] V, [2] scan ticket, [3] live count, [4] group count
    EnumArgs ea{};
    ea.B = s->B; ea.n_blocks = s->n_blocks; ea.dom = d_dom; ea.desc = d_desc; ea.tables = d_tables; ea.flags = d_flags;
    ea.bitmap = (uint64_t*)d_bitmap; ea.cnt = (uint32_t*)(sc + s->off_cnt);
    ea.live = (uint32_t*)(sc + s->off_live); ea.live_count = ctl + 3;
    ea.keys = s->use_keys ? (uint32_t*)(sc + s->off_keys) : nullptr; ea.n_inv = s->n_inv;
    ea.Wb = s->Wb; ea.CH = s->CH; ea.t = s->t; ea.n_tab = s->n_tab; ea.n_res = s->n_res;
    ea.desc_words = (uint32_t)s->desc.size(); ea.desc_in_smem = s->desc.size() <= 8192;
    ea.n_rc = s->n_rc;
    for (int r = 0; r < 32; ++r) ea.rc_of[r] = -1;
    for (int k = 0; k < s->n_rc; ++k) {
        uint8_t* b = sc + s->off_rc[k];
        ResClassArgs& rc = ea.rc[k];
        rc.keys = (long long*)b; b += align256((uint64_t)CAO_HS * 8);
        rc.table = (uint64_t*)b; b += align256((uint64_t)CAO_HS * s->Wb * 8);
        rc.overflow = (int32_t*)b;
        rc.pc0 = s->rc_pc0[k]; rc.r = s->rc_r[k];
        ea.rc_of[s->rc_r[k]] = (int8_t)k;
    }
    const unsigned bd = 256;
    const size_t smem_desc = ea.desc_in_smem ? (size_t)ea.desc_words * 4 : 0;
    const size_t smem_dig = smem_desc + (((size_t)bd * (size_t)std::max(1, s->t) + 3) & ~(size_t)3);
    const size_t smem_enum = smem_dig + (size_t)bd * s->CH * 4;
    {
        const uint64_t threads = (s->n_blocks + s->CH - 1) / s->CH;
        if (smem_enum > 48 * 1024) {
            CAO_SMEM_OPTIN(k_enum);
            CAO_SMEM_OPTIN(k_masks);
        }
        {
            ProfScope ps(PK_ENUM, st);
            k_enum<<<(unsigned)((threads + bd - 1) / bd), bd, smem_enum, st>>>(s->meta, ea);
        }
        CAO_LAUNCHED("k_enum");
        if (s->n_res) {                                                 // fork: the residual prefixes need the live list only
            CAO_CUDA(cudaEventRecord(s->ev_fork2, st));
            CAO_CUDA(cudaStreamWaitEvent(s->side2, s->ev_fork2, 0));
        }
        if (s->use_keys) {
            ProfScope ps(PK_MASKS, st);
            k_keys<<<(unsigned)std::min<uint64_t>((s->n_blocks + bd - 1) / bd, (uint64_t)cao_sm_count() * 4), bd, smem_dig, st>>>(s->meta, ea);
            CAO_LAUNCHED("k_keys");
        }
        ProfScope ps(PK_MASKS, st);
        const uint64_t items = s->n_blocks * (uint64_t)s->Wb;
        k_masks<<<(unsigned)std::min<uint64_t>((items + bd - 1) / bd, (uint64_t)cao_sm_count() * 16), bd, smem_dig, st>>>(s->meta, ea);
        CAO_LAUNCHED("k_masks");
    }
    if (s->n_res) {
        ResPrefix* pre = (ResPrefix*)(sc + s->off_pre);
        const uint64_t items = s->n_blocks * (uint64_t)s->n_res;
        {
            ProfScope ps(PK_RESPRE, s->side2);
            k_res_prefix<<<(unsigned)std::min<uint64_t>((items + bd - 1) / bd, (uint64_t)cao_sm_count() * 8), bd, smem_desc, s->side2>>>(s->meta, ea, pre);
        }
        CAO_LAUNCHED("k_res_prefix");
        if (s->n_rc) {
            ProfScope ps(PK_RESPRE, s->side2);
            k_res_class_table<<<dim3(cao_sm_count() * 4, (unsigned)s->n_rc), 256, 0, s->side2>>>(s->meta, ea);
            CAO_LAUNCHED("k_res_class_table");
        }
        CAO_CUDA(cudaEventRecord(s->ev_join2, s->side2));
        CAO_CUDA(cudaStreamWaitEvent(st, s->ev_join2, 0));              // join: k_residual needs the masks and the prefixes
        ProfScope ps(PK_RESID, st);
        const uint64_t warps = std::min<uint64_t>(s->n_blocks, (uint64_t)cao_sm_count() * 64);
        k_residual<<<(unsigned)((warps + 7) / 8), bd, smem_desc, st>>>(s->meta, ea, pre);
        CAO_LAUNCHED("k_residual");
    }
    if (with_reduce) {
        ProfScope ps(PK_CSCAN, st);
        k_cnt_reduce<<<(unsigned)s->n_part, 256, 0, st>>>(ea.cnt, s->nd + 1, (uint32_t*)(sc + s->off_part), s->n_part, ctl + 2, (uint64_t*)ctl);
        CAO_LAUNCHED("k_cnt_reduce");
    }
    return CAO_OK;
}

// S1 pass 2 on `st`: rank directory + list of non-empty groups, then rows and Ltab.
static int launch_fill(cao_space* s, uint8_t* tb, cudaStream_t st, bool single_pass = false) {
    uint8_t* sc = (uint8_t*)s->d_scratch;
    uint8_t* rows = tb + s->off_rows; void* Ltab = tb + s->off_Ltab; uint32_t* dir = (uint32_t*)(tb + s->off_dir);
    const uint32_t* cnt = (const uint32_t*)(sc + s->off_cnt);
    uint32_t* ctl = (uint32_t*)(sc + s->off_V);
    uint32_t* groups = (uint32_t*)(sc + s->off_groups);
    CAO_CUDA(cudaMemsetAsync(ctl + 4, 0, 4, st));
    if (single_pass) {                                                  // rebuild: reduce + apply in one decoupled-look-back pass
        ProfScope ps(PK_CSCAN, st);
        k_cnt_scan1<<<(unsigned)s->n_part, 256, 0, st>>>(cnt, s->nd + 1, (unsigned long long*)(sc + s->off_part), ctl + 2, dir, groups, ctl + 4, (uint64_t*)ctl);
        CAO_LAUNCHED("k_cnt_scan1");
    } else {
        ProfScope ps(PK_CSCAN, st);
        k_cnt_apply<<<(unsigned)s->n_part, 256, 0, st>>>(cnt, s->nd + 1, (const uint32_t*)(sc + s->off_part), dir, groups, ctl + 4);
        CAO_LAUNCHED("k_cnt_apply");
    }
    const uint32_t* lut = s->use_lut ? (const uint32_t*)(sc + s->off_lut) : nullptr;
    const uint64_t magicB = s->B > 1 ? (uint64_t)((((unsigned __int128)1 << 64) + s->B - 1) / s->B) : 0;
    const unsigned grid = (unsigned)std::min<uint64_t>((s->nd + 7) / 8, (uint64_t)cao_sm_count() * 8);   // a warp per group, grid-stride over the list
    {
        ProfScope ps(PK_FILL, st);
#define CALL_FILL(W, L32) k_fill<W, L32><<<grid, 256, 0, st>>>(s->meta, s->n_words, rows, Ltab, dir, groups, ctl + 4, lut, s->B, magicB, s->t)
        if (s->meta.rowB == 16) { if (s->meta.ltab32) CALL_FILL(4, true); else CALL_FILL(4, false); }
        else { if (s->meta.ltab32) CALL_FILL(8, true); else CALL_FILL(8, false); }
    }
    CAO_LAUNCHED("k_fill");
    return CAO_OK;
}

int cao_space_build_count(cao_space* s, void* d_bitmap, void* d_scratch, void* stream, uint64_t* h_V) {
    if (!s || !h_V) return cao_fail(CAO_E_INVALID_ARG, "cao_space_build_count: NULL argument");
    if (!s->planned) return cao_fail(CAO_E_STATE, "cao_space_build_count: call cao_space_build_workspace_bytes first");
    if (!d_bitmap || !d_scratch || ((uintptr_t)d_bitmap & 255) || ((uintptr_t)d_scratch & 255))
        return cao_fail(CAO_E_WORKSPACE, "cao_space_build_count: bitmap/scratch must be non-NULL and 256-byte aligned");
    cudaStream_t st = (cudaStream_t)stream;
    const int n = s->meta.n;
    uint8_t* sc = (uint8_t*)d_scratch;
    std::vector<int64_t> hdom((size_t)n * 256, 0);
    for (int d = 0; d < n; ++d) std::copy(s->dom[d].begin(), s->dom[d].end(), hdom.begin() + (size_t)d * 256);
    CAO_CUDA(cudaMemcpyAsync(sc + s->off_dom, hdom.data(), hdom.size() * 8, cudaMemcpyHostToDevice, st));
    CAO_CUDA(cudaMemcpyAsync(sc + s->off_desc, s->desc.data(), s->desc.size() * 4, cudaMemcpyHostToDevice, st));
    { int rc = launch_pass1(s, d_bitmap, sc, st); if (rc) return rc; }
    uint64_t* d_V = (uint64_t*)(sc + s->off_V);
    uint64_t V = 0;
    CAO_CUDA(cudaMemcpyAsync(&V, d_V, 8, cudaMemcpyDeviceToHost, st));
    CAO_CUDA(cudaStreamSynchronize(st));
    if (V >= (1ull << 32)) return cao_fail(CAO_E_TOO_LARGE, "V >= 2^32");
    s->meta.V = (uint32_t)V; s->d_scratch = d_scratch; s->counted = true; s->filled = false;
    if (s->rebuild_exec) { cudaGraphExecDestroy(s->rebuild_exec); s->rebuild_exec = nullptr; }     // new buffers
    *h_V = V;
    const uint64_t rowB = s->meta.rowB;
    uint64_t off = 0;
    s->off_rows = off; off = align256(off + std::max<uint64_t>(1, V) * rowB);
    s->off_Ltab = off; off = align256(off + std::max<uint64_t>(1, V) * (s->meta.ltab32 ? 4 : 8));
    s->off_dir = off; off = align256(off + (s->nd + 1) * 4);
    // neighbour lists and the cost model that decides how many Hamming levels are probed before the scan:
    // e_h = number of index rows at Hamming distance exactly h from a point (elementary symmetric polynomial of m_d - 1)
    {
        const int n = s->meta.n;
        s->h_nb.clear();
        for (int d = 0; d < n; ++d) {
            s->probe.nb_first[d] = (uint16_t)s->h_nb.size();
            for (int k = 0; k + 1 < (int)s->meta.m[d]; ++k) s->h_nb.push_back((uint16_t)(d << 8 | k));
        }
        for (int d = n; d <= CAO_MAX_DIMS; ++d) s->probe.nb_first[d] = (uint16_t)s->h_nb.size();
        s->probe.NB = (uint32_t)s->h_nb.size();
        double e[CAO_MAX_PROBE_LEVEL + 1] = {1, 0, 0, 0, 0, 0, 0};
        for (int d = 0; d < n; ++d) for (int h = CAO_MAX_PROBE_LEVEL; h >= 1; --h) e[h] += e[h - 1] * (double)(s->meta.m[d] - 1);
        const double scan_cost = (double)V * (5.0 * ((n + 3) / 4) + 6.0);
        int lv = 1;
        while (lv < CAO_MAX_PROBE_LEVEL && e[lv + 1] * 60.0 <= scan_cost) ++lv;
        if (s->probe_levels_req >= 0) lv = std::min(CAO_MAX_PROBE_LEVEL, std::max(0, s->probe_levels_req));
        if (e[2] > 65536.0 || s->probe.NB > CAO_MAX_NB_PROBE) lv = std::min(lv, 1);   // the pair list would not fit its budget
        s->h_pairs.clear();
        if (lv >= 2)
            for (uint32_t t1 = 0; t1 < s->probe.NB; ++t1)
                for (uint32_t t2 = s->probe.nb_first[(s->h_nb[t1] >> 8) + 1]; t2 < s->probe.NB; ++t2)
                    s->h_pairs.push_back(t1 | (t2 << 16));
        s->probe.C2 = (uint32_t)s->h_pairs.size();
        // flat list of the Hamming-3 neighbour triples (the level that dominates the slow runs): every lane takes
        // triples with eight independent bit tests in flight instead of walking the third neighbour serially per pair
        s->h_triples.clear();
        if (lv >= 3 && e[3] <= 131072.0)
            for (uint32_t t1 = 0; t1 < s->probe.NB; ++t1)
                for (uint32_t t2 = s->probe.nb_first[(s->h_nb[t1] >> 8) + 1]; t2 < s->probe.NB; ++t2)
                    for (uint32_t t3 = s->probe.nb_first[(s->h_nb[t2] >> 8) + 1]; t3 < s->probe.NB; ++t3)
                        s->h_triples.push_back(t1 | (t2 << 10) | (t3 << 20));
        s->probe.C3 = (uint32_t)s->h_triples.size();
        s->probe.levels = lv;
    }
    s->off_tgt = off; off = align256(off + std::max<uint64_t>(1, s->h_nb.size()) * 2);
    s->off_pairs = off; off = align256(off + std::max<uint64_t>(1, s->h_pairs.size()) * 4);
    s->off_triples = off; off = align256(off + std::max<uint64_t>(1, s->h_triples.size()) * 4);
    s->table_bytes = off;
    return CAO_OK;
}

int cao_space_table_bytes(const cao_space* s, uint64_t* bytes) {
    if (!s || !bytes) return cao_fail(CAO_E_INVALID_ARG, "cao_space_table_bytes: NULL argument");
    if (!s->counted) return cao_fail(CAO_E_STATE, "cao_space_table_bytes: call cao_space_build_count first");
    *bytes = s->table_bytes;
    return CAO_OK;
}

int cao_space_build_fill(cao_space* s, void* d_table, void* stream) {
    if (!s) return cao_fail(CAO_E_INVALID_ARG, "cao_space_build_fill: NULL space");
    if (!s->counted) return cao_fail(CAO_E_STATE, "cao_space_build_fill: call cao_space_build_count first");
    if (!d_table || ((uintptr_t)d_table & 255)) return cao_fail(CAO_E_WORKSPACE, "cao_space_build_fill: table must be non-NULL and 256-byte aligned");
    cudaStream_t st = (cudaStream_t)stream;
    uint8_t* tb = (uint8_t*)d_table;
    uint8_t* rows = tb + s->off_rows; void* Ltab = tb + s->off_Ltab; uint32_t* dir = (uint32_t*)(tb + s->off_dir);
    s->d_table = d_table;
    { int rc = launch_fill(s, tb, st); if (rc) return rc; }
    if (!s->h_nb.empty())
        CAO_CUDA(cudaMemcpyAsync(tb + s->off_tgt, s->h_nb.data(), s->h_nb.size() * 2, cudaMemcpyHostToDevice, st));
    s->probe.nb = (const uint16_t*)(tb + s->off_tgt);
    if (!s->h_pairs.empty())
        CAO_CUDA(cudaMemcpyAsync(tb + s->off_pairs, s->h_pairs.data(), s->h_pairs.size() * 4, cudaMemcpyHostToDevice, st));
    s->probe.pairs = (const uint32_t*)(tb + s->off_pairs);
    if (!s->h_triples.empty())
        CAO_CUDA(cudaMemcpyAsync(tb + s->off_triples, s->h_triples.data(), s->h_triples.size() * 4, cudaMemcpyHostToDevice, st));
    s->probe.triples = (const uint32_t*)(tb + s->off_triples);
    s->meta.rows = rows; s->meta.Ltab = Ltab; s->meta.dir = dir;
    s->d_table = d_table;
    s->filled = true;
    return CAO_OK;
}

int cao_space_rebuild(cao_space* s, void* stream) {
    if (!s) return cao_fail(CAO_E_INVALID_ARG, "cao_space_rebuild: NULL space");
    if (!s->filled) return cao_fail(CAO_E_STATE, "cao_space_rebuild: the space must have been built once");
    cudaStream_t st = (cudaStream_t)stream;
    // The sequence (two zero fills on the side stream, ~10 short kernels) is launch-bound on small spaces: it is captured
    // once into a CUDA graph and replayed.  Not on the legacy default stream (capture is illegal there) and not while
    // per-kernel profiling is on (its events must be real).
    const bool can_graph = st != nullptr && st != cudaStreamLegacy && st != cudaStreamPerThread && !g_cao_prof_on.load();
    // count scan: one look-back pass while the chain of chunks is short (measured: 2 us faster on configs[1] / [2], 4 us
    // slower on configs[3]'s 274 chunks than reduce + apply)
    const bool single = s->n_part <= 32;
    if (can_graph && !s->rebuild_exec) {
        const uint64_t l0 = g_cao_launches.load();
        if (cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
            int rc = launch_pass1(s, (void*)s->meta.bitmap, (uint8_t*)s->d_scratch, st, !single);
            if (!rc) rc = launch_fill(s, (uint8_t*)s->d_table, st, single);
            cudaGraph_t graph = nullptr;
            const cudaError_t e = cudaStreamEndCapture(st, &graph);
            if (!rc && e == cudaSuccess && graph && cudaGraphInstantiate(&s->rebuild_exec, graph, 0) == cudaSuccess)
                s->rebuild_launches = g_cao_launches.load() - l0;
            else s->rebuild_exec = nullptr;
            if (graph) cudaGraphDestroy(graph);
            g_cao_launches.store(l0);                                   // nothing ran yet
            cudaGetLastError();
        }
    }
    if (can_graph && s->rebuild_exec) {
        CAO_CUDA(cudaGraphLaunch(s->rebuild_exec, st));
        g_cao_launches += s->rebuild_launches;
        return CAO_OK;
    }
    int rc = launch_pass1(s, (void*)s->meta.bitmap, (uint8_t*)s->d_scratch, st, !single);
    if (rc) return rc;
    return launch_fill(s, (uint8_t*)s->d_table, st, single);
}

int cao_space_build_stats(const cao_space* s, void* stream, uint64_t* h_out4) {
    if (!s || !h_out4) return cao_fail(CAO_E_INVALID_ARG, "cao_space_build_stats: NULL argument");
    if (!s->filled) return cao_fail(CAO_E_STATE, "cao_space_build_stats: space not built");
    uint32_t ctl[8] = {0};
    CAO_CUDA(cudaMemcpyAsync(ctl, (uint8_t*)s->d_scratch + s->off_V, 32, cudaMemcpyDeviceToHost, (cudaStream_t)stream));
    CAO_CUDA(cudaStreamSynchronize((cudaStream_t)stream));
    h_out4[0] = s->n_blocks; h_out4[1] = ctl[3]; h_out4[2] = ctl[4]; h_out4[3] = s->B;
    return CAO_OK;
}

int cao_space_ltab_bytes(const cao_space* s, int32_t* bytes) {
    if (!s || !bytes) return cao_fail(CAO_E_INVALID_ARG, "cao_space_ltab_bytes: NULL argument");
    if (!s->planned) return cao_fail(CAO_E_STATE, "cao_space_ltab_bytes: space not planned yet");
    *bytes = s->meta.ltab32 ? 4 : 8;
    return CAO_OK;
}

int cao_space_sizes(const cao_space* s, uint64_t* N, uint64_t* V, int32_t* n, int32_t* row_bytes) {
    if (!s) return cao_fail(CAO_E_INVALID_ARG, "cao_space_sizes: NULL space");
    if (!s->planned) return cao_fail(CAO_E_STATE, "cao_space_sizes: space not planned yet");
    if (N) *N = s->meta.N;
    if (V) *V = s->counted ? s->meta.V : 0;
    if (n) *n = s->meta.n;
    if (row_bytes) *row_bytes = s->meta.rowB;
    return CAO_OK;
}

int cao_space_views(const cao_space* s, const uint64_t** d_bitmap, const uint8_t** d_rows, const void** d_Ltab,
                    const uint32_t** d_rank_dir) {
    if (!s) return cao_fail(CAO_E_INVALID_ARG, "cao_space_views: NULL space");
    if (!s->filled) return cao_fail(CAO_E_STATE, "cao_space_views: space not built");
    if (d_bitmap) *d_bitmap = s->meta.bitmap;
    if (d_rows) *d_rows = s->meta.rows;
    if (d_Ltab) *d_Ltab = s->meta.Ltab;
    if (d_rank_dir) *d_rank_dir = s->meta.dir;
    return CAO_OK;
}

int cao_space_is_valid(const cao_space* s, const uint8_t* d_idx_rows, uint64_t count, uint8_t* d_out, void* stream) {
    if (!s || (count && (!d_idx_rows || !d_out))) return cao_fail(CAO_E_INVALID_ARG, "cao_space_is_valid: NULL argument");
    if (!s->counted) return cao_fail(CAO_E_STATE, "cao_space_is_valid: space not built");
    if (count == 0) return CAO_OK;
    if ((uintptr_t)d_idx_rows & 15) return cao_fail(CAO_E_WORKSPACE, "cao_space_is_valid: rows must be 16-byte aligned");
    unsigned grid = (unsigned)((count + 255) / 256);
    if (s->meta.rowB == 16) k_is_valid<4><<<grid, 256, 0, (cudaStream_t)stream>>>(s->meta, d_idx_rows, count, d_out);
    else k_is_valid<8><<<grid, 256, 0, (cudaStream_t)stream>>>(s->meta, d_idx_rows, count, d_out);
    CAO_LAUNCHED("k_is_valid");
    return CAO_OK;
}

int cao_space_set_objective(cao_space* s, const float* d_obj) {
    if (!s || !d_obj) return cao_fail(CAO_E_INVALID_ARG, "cao_space_set_objective: NULL argument");
    if (!s->filled) return cao_fail(CAO_E_STATE, "cao_space_set_objective: space not built");
    s->meta.obj = d_obj;
    return CAO_OK;
}

}  // extern "C"

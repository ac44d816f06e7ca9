// cao_oracle.cc -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, single-threaded CPU oracle for the hot path of "Constraint-aware Optimization in
// Auto-Tuning" (arxiv/paper_2606_28372; citations "Lnnn" are line numbers of PAPER.md, "Ox"/"Ax"
// are the readings listed in DESIGN.md).  Only tests/, __graft_entry__.smoke() and bench.py's
// cpu_baseline / --impl reference legs may load this library.  It shares no code with the CUDA
// path (paper_2606_28372_b200/csrc): no headers, no tables, no helpers.
//
// What is the plain definition (result reached exactly by the CUDA path):
//   enumerate (O1, L129-137), validity (L139), repair = argmin (Hamming, sum|didx|, L) over ALL
//   valid rows (O9; L143, L215, L270), objective lookup + per-run memoisation (O10; L268, L125).
// What is an algorithm followed step by step (randomised heuristics; every random number is
// addressed by (seed, run, generation, individual, stream, slot), never consumed sequentially):
//   init (O4; L139, L282(i)), DE best1bin (O5; Alg.1), PSO (O6; L276-282),
//   Firefly (O7; L284 -- update rule not in the paper, Yang's form, reading A14),
//   GA (O8; L286-292, Alg.3).
// Pins (tests/test_oracle_*.py): Philox known-answer vectors, itertools brute force on tiny
// spaces, hand-counted cfg0, exact V of cfg1-3, worked repair examples, exp against libm,
// invariants of the paper (only valid configs evaluated, repair identity on valid, DE population
// duplicate-free, PSO/FF positions untouched by repair, GA mutation = valid Hamming-1 neighbour).
// The four operator loops have no closed form: their parity with the *paper* is unpinned
// (DESIGN.md "Parity unpinned"); they are pinned by those invariants and by the independent
// prototype values recorded in SURVEY.md section 8(c).
//
// SURVEY 8(f) rows (readings A28-A36 in DESIGN.md), selected per Runs by `Variant` (all-default = the path above):
//   NEXT-1 paper-verbatim repair: DE index-distance key (L215, L270); neighbour rules strictly-adjacent / adjacent /
//          Hamming (L139-143) and the NEIGHBORS cascade (Alg.2); Euclidean-nearest choice for PSO / Firefly
//          (Alg.2); random choice for GA (Alg.3).  Plain definitions: every rule is a loop over ALL
//          valid rows.
//   NEXT-2 non-constraint-aware variants: random Cartesian initial population, no repair, static penalty (L107, L272, L284).
//   NEXT-3 operator variants: DE rand1 / currenttobest1 / randtobest1 / best2 / rand2, binomial / exponential crossover
//          (L219, L272); GA two-point / uniform / disruptive-uniform crossover (L288); Latin Hypercube initial sample (L223).
//   NEXT-4 performance score P (Eq.2) over trajectories against a calculated random-search baseline -- PARITY WITH
//          THE PAPER UNPINNED: the baseline formula of [29] is not in the paper (reading A36).
//
// Build: g++ -std=c++17 -O2 -ffp-contract=off -fno-fast-math -shared -fPIC (oracle/build.py).
// fp32 arithmetic is IEEE single (x86-64 SSE2), one rounding per written operation.

#include <cstdint>
#include <cstring>
#include <cmath>
#include <vector>
#include <algorithm>

namespace {

// ------------------------------------------------------------------ O3: Philox4x32-10
// Salmon et al., SC'11.  One round: (c0,c1,c2,c3) <- (hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1, lo(M0*c0)),
// then the key is bumped by the Weyl constants.
void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    const uint64_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = M0 * (uint64_t)c0;
        uint64_t p1 = M1 * (uint64_t)c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

enum Stream : uint32_t { S_INIT = 0, S_OP = 1, S_MUT = 2, S_REINIT = 3, S_REPAIR = 5 };   // 4 is reserved

// draw(stream, slot) for (seed, run, generation, individual):
// counter = (run, generation, individual, stream<<24 | slot>>2), key = (seed_lo, seed_hi), word slot&3.
uint32_t draw(uint64_t seed, uint32_t run, uint32_t gen, uint32_t ind, uint32_t stream, uint32_t slot) {
    uint32_t ctr[4] = { run, gen, ind, (stream << 24) | (slot >> 2) };
    uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    uint32_t out[4];
    philox4x32_10(ctr, key, out);
    return out[slot & 3];
}

float u01(uint32_t w) { return (float)(w >> 8) * 5.9604644775390625e-08f; }          // (w>>8) * 2^-24, exact
uint32_t below(uint32_t w, uint32_t k) { return (uint32_t)(((uint64_t)w * (uint64_t)k) >> 32); }

// ------------------------------------------------------------------ O7: exp(-z), add/mul only
// 2^-t with t = z*log2(e):  2^-floor(t) * 2^-1/2 * exp(-ln2 * (frac(t) - 1/2)), degree-7 Taylor
// polynomial in u = frac - 1/2 (|u| <= 1/2), Horner, every operation rounded to fp32.
float exp_neg_spec(float z) {
    const float LOG2E = 0x1.715476p+0f, RSQRT2 = 0x1.6a09e6p-1f;
    const float c[8] = { 1.0f, -0x1.62e430p-1f, 0x1.ebfbe0p-3f, -0x1.c6b08ep-5f,
                         0x1.3b2ab6p-7f, -0x1.5d87fep-10f, 0x1.430912p-13f, -0x1.ffcbfcp-17f };
    float t = z * LOG2E;
    float kf = floorf(t);
    if (!(kf < 126.0f)) return 0.0f;
    float fr = t - kf;
    float u = fr - 0.5f;
    float p = c[7];
    for (int i = 6; i >= 0; --i) { p = p * u; p = p + c[i]; }
    p = p * RSQRT2;
    uint32_t bits = (uint32_t)(127 - (int)kf) << 23;
    float scale; std::memcpy(&scale, &bits, 4);
    return p * scale;
}

float clamp_pos(float x, float hi) {        // NaN -> 0, -0 -> +0 (explicit selects, O6)
    x = (x > 0.0f) ? x : 0.0f;
    x = (x < hi) ? x : hi;
    return x;
}

uint32_t fbits(float f) { uint32_t b; std::memcpy(&b, &f, 4); return b; }

// ------------------------------------------------------------------ O1: constraint programs
enum Op : int32_t { PUSH_PARAM = 1, PUSH_CONST = 2, ADD = 3, SUB = 4, MUL = 5, DIV = 6, MOD = 7, NEG = 8,
                    MIN_ = 9, MAX_ = 10, LT = 11, LE = 12, GT = 13, GE = 14, EQ = 15, NE = 16,
                    AND_ = 17, OR_ = 18, NOT_ = 19 };

const __int128 SAT = (__int128)1 << 62;
int64_t sat(__int128 v) { if (v > SAT) v = SAT; if (v < -SAT) v = -SAT; return (int64_t)v; }

// Returns 1 / 0; a division or modulo by zero anywhere makes the whole constraint false (A3).
// Malformed programs are rejected at add time, so the stack cannot under/overflow here.
int eval_program(const std::vector<int32_t>& w, const int64_t* x) {
    int64_t st[64]; int sp = 0;
    for (size_t pc = 0; pc < w.size(); ++pc) {
        int32_t op = w[pc];
        if (op == PUSH_PARAM) { st[sp++] = sat(x[w[++pc]]); continue; }
        if (op == PUSH_CONST) {
            uint64_t lo = (uint32_t)w[pc + 1], hi = (uint32_t)w[pc + 2]; pc += 2;
            st[sp++] = sat((int64_t)(lo | (hi << 32))); continue;
        }
        if (op == NEG) { st[sp - 1] = sat(-(__int128)st[sp - 1]); continue; }
        if (op == NOT_) { st[sp - 1] = (st[sp - 1] == 0); continue; }
        int64_t b = st[--sp], a = st[sp - 1], r = 0;
        switch (op) {
            case ADD: r = sat((__int128)a + b); break;
            case SUB: r = sat((__int128)a - b); break;
            case MUL: r = sat((__int128)a * b); break;
            case DIV: if (b == 0) return 0; r = a / b; break;       // C: truncates toward zero
            case MOD: if (b == 0) return 0; r = a % b; break;
            case MIN_: r = a < b ? a : b; break;
            case MAX_: r = a > b ? a : b; break;
            case LT: r = a < b; break;  case LE: r = a <= b; break;
            case GT: r = a > b; break;  case GE: r = a >= b; break;
            case EQ: r = a == b; break; case NE: r = a != b; break;
            case AND_: r = (a != 0) && (b != 0); break;
            case OR_: r = (a != 0) || (b != 0); break;
        }
        st[sp - 1] = r;
    }
    return st[0] != 0;
}

// Validates a program: known opcodes, param index in range, stack depth 1 at the end, depth <= 64.
bool program_ok(const int32_t* w, int nw, int n_params) {
    int sp = 0;
    for (int pc = 0; pc < nw; ++pc) {
        int32_t op = w[pc];
        if (op == PUSH_PARAM) { if (pc + 1 >= nw || w[pc + 1] < 0 || w[pc + 1] >= n_params) return false; ++pc; ++sp; }
        else if (op == PUSH_CONST) { if (pc + 2 >= nw) return false; pc += 2; ++sp; }
        else if (op == NEG || op == NOT_) { if (sp < 1) return false; }
        else if (op >= ADD && op <= OR_) { if (sp < 2) return false; --sp; }
        else return false;
        if (sp > 64) return false;
    }
    return sp == 1;
}

struct Space {
    std::vector<std::vector<int64_t>> dom;        // dom[d][idx]; first param = most significant digit (A1)
    std::vector<std::vector<int32_t>> cons;
    int n = 0;
    uint64_t N = 0, V = 0;
    std::vector<uint64_t> stride;
    std::vector<uint64_t> bitmap;                 // bit (L&63) of word (L>>6)
    std::vector<uint8_t> rows;                    // V x n index rows, ascending L; position = rank
    std::vector<uint64_t> Ltab;                   // V linear indices
    std::vector<float> obj;                       // V objective values by rank
    bool built = false;
    int M = 1;                                    // max_d m_d
    std::vector<std::vector<uint8_t>> present;    // present[d][k] = 1 iff some valid configuration has idx_d = k (A28)

    bool valid_idx(const uint8_t* idx) const {    // all constraints true for this index row
        int64_t x[32];
        for (int d = 0; d < n; ++d) x[d] = dom[d][idx[d]];
        for (const auto& c : cons) if (!eval_program(c, x)) return false;
        return true;
    }
    uint64_t lin(const uint8_t* idx) const { uint64_t L = 0; for (int d = 0; d < n; ++d) L += idx[d] * stride[d]; return L; }
    bool bit(uint64_t L) const { return (bitmap[L >> 6] >> (L & 63)) & 1; }
    // rank of a valid L = its position in the sorted table (binary search; the table is the definition)
    uint32_t rank_of(uint64_t L) const {
        return (uint32_t)(std::lower_bound(Ltab.begin(), Ltab.end(), L) - Ltab.begin());
    }
};

// O1: for L = 0..N-1 decode, evaluate, set bit, append.
void enumerate(Space& s) {
    s.n = (int)s.dom.size();
    s.stride.assign(s.n, 1);
    for (int d = s.n - 2; d >= 0; --d) s.stride[d] = s.stride[d + 1] * s.dom[d + 1].size();
    s.N = s.n ? s.stride[0] * s.dom[0].size() : 0;
    s.M = 1; for (auto& d : s.dom) s.M = std::max<int>(s.M, (int)d.size());
    s.bitmap.assign((s.N + 63) / 64, 0);
    s.rows.clear(); s.Ltab.clear();
    // idx holds the mixed-radix digits of L, idx_d = (L / stride_d) mod m_d; it is advanced like an odometer
    // (last digit fastest) instead of re-dividing every L.  orc_space_count_range() below does the literal
    // division decode and the tests check the two against each other.
    // The odometer counts in unsigned (a 256-value digit must reach 256 to carry); idx is its byte copy.
    unsigned odo[32] = { 0 };
    uint8_t idx[32] = { 0 };
    for (uint64_t L = 0; L < s.N; ++L) {
        if (s.valid_idx(idx)) {
            s.bitmap[L >> 6] |= (uint64_t)1 << (L & 63);
            s.rows.insert(s.rows.end(), idx, idx + s.n);
            s.Ltab.push_back(L);
        }
        for (int d = s.n - 1; d >= 0; --d) {
            if (++odo[d] < s.dom[d].size()) { idx[d] = (uint8_t)odo[d]; break; }
            odo[d] = 0; idx[d] = 0;
        }
    }
    s.V = s.Ltab.size();
    s.present.assign(s.n, {});
    for (int d = 0; d < s.n; ++d) s.present[d].assign(s.dom[d].size(), 0);
    for (uint64_t r = 0; r < s.V; ++r) for (int d = 0; d < s.n; ++d) s.present[d][s.rows[r * s.n + d]] = 1;
    s.built = true;
}

// O9: repair(c) = c if valid else argmin over ALL valid rows of (Hamming, sum |didx|, L).
struct RepairKey { uint32_t ham, sad; uint64_t L; uint32_t rank; };
// A27: a row with an index outside its domain (idx_d >= m_d) is not a point of X: it is invalid, and its repair is
// the same argmin taken over its byte values.
bool in_domain(const Space& s, const uint8_t* c) {
    for (int d = 0; d < s.n; ++d) if (c[d] >= s.dom[d].size()) return false;
    return true;
}
RepairKey repair(const Space& s, const uint8_t* c) {
    if (in_domain(s, c)) {
        uint64_t Lc = s.lin(c);
        if (s.bit(Lc)) return RepairKey{ 0, 0, Lc, s.rank_of(Lc) };
    }
    RepairKey best{ 0xFFFFFFFFu, 0xFFFFFFFFu, ~0ull, 0xFFFFFFFFu };
    for (uint64_t r = 0; r < s.V; ++r) {
        const uint8_t* v = &s.rows[r * s.n];
        uint32_t ham = 0, sad = 0;
        for (int d = 0; d < s.n; ++d) {
            ham += (v[d] != c[d]);
            sad += (uint32_t)std::abs((int)v[d] - (int)c[d]);
        }
        uint64_t L = s.Ltab[r];
        bool less = ham < best.ham || (ham == best.ham && (sad < best.sad || (sad == best.sad && L < best.L)));
        if (less) best = RepairKey{ ham, sad, L, (uint32_t)r };
    }
    return best;
}

// ------------------------------------------------------------------ NEXT-1: paper-verbatim neighbour rules and repairs
const uint32_t RANK_NONE = 0xFFFFFFFFu;

// L215 "Index-distance" / L270: nearest valid by the sum of absolute index differences alone; ties -> smallest L (A5).
RepairKey repair_index_distance(const Space& s, const uint8_t* c) {
    if (in_domain(s, c)) {
        uint64_t Lc = s.lin(c);
        if (s.bit(Lc)) return RepairKey{ 0, 0, Lc, s.rank_of(Lc) };
    }
    RepairKey best{ 0xFFFFFFFFu, 0xFFFFFFFFu, ~0ull, RANK_NONE };
    for (uint64_t r = 0; r < s.V; ++r) {
        const uint8_t* v = &s.rows[r * s.n];
        uint32_t ham = 0, sad = 0;
        for (int d = 0; d < s.n; ++d) { ham += (v[d] != c[d]); sad += (uint32_t)std::abs((int)v[d] - (int)c[d]); }
        uint64_t L = s.Ltab[r];
        if (sad < best.sad || (sad == best.sad && L < best.L)) best = RepairKey{ ham, sad, L, (uint32_t)r };
    }
    return best;
}

// present(d, k): some valid configuration has idx_d = k ("the ... value that gives a valid configuration", L141; A28).
bool value_present(const Space& s, int d, int k) { return s.present[d][k] != 0; }     // filled by enumerate() from the valid table
// The three neighbour rules of L139-143 between an index row c and a VALID row v != c:
//   0 strictly-adjacent: every parameter identical or the previous/next value (|v_d - c_d| <= 1);
//   1 adjacent: every parameter identical or the nearest previous/next value that occurs in a valid configuration (A28);
//   2 Hamming: all parameters identical except one.
// near_lo[d] / near_hi[d]: nearest present index below / above c_d, or -1.
bool is_neighbor(const Space& s, int rule, const uint8_t* c, const uint8_t* v, const int* near_lo, const int* near_hi) {
    int differ = 0;
    for (int d = 0; d < s.n; ++d) {
        if (v[d] == c[d]) continue;
        ++differ;
        if (rule == 0 && std::abs((int)v[d] - (int)c[d]) > 1) return false;
        if (rule == 1 && (int)v[d] != near_lo[d] && (int)v[d] != near_hi[d]) return false;
    }
    if (differ == 0) return false;
    if (rule == 2 && differ != 1) return false;
    return true;
}
// list_neighbors(p, rule) (Alg.2 L3): ranks of the valid neighbours of c under `rule`, ascending L.
std::vector<uint32_t> list_neighbors(const Space& s, const uint8_t* c, int rule) {
    int near_lo[32], near_hi[32];
    for (int d = 0; d < s.n; ++d) {
        near_lo[d] = near_hi[d] = -1;
        for (int k = (int)c[d] - 1; k >= 0; --k) if (value_present(s, d, k)) { near_lo[d] = k; break; }
        for (int k = (int)c[d] + 1; k < (int)s.dom[d].size(); ++k) if (value_present(s, d, k)) { near_hi[d] = k; break; }
    }
    std::vector<uint32_t> out;
    for (uint64_t r = 0; r < s.V; ++r)
        if (is_neighbor(s, rule, c, &s.rows[r * s.n], near_lo, near_hi)) out.push_back((uint32_t)r);
    return out;
}
// NEIGHBORS (Alg.2): the first non-empty of strictly-adjacent, adjacent, Hamming; *rule_out = which (3 = none).
std::vector<uint32_t> neighbors_cascade(const Space& s, const uint8_t* c, int* rule_out) {
    for (int rule = 0; rule < 3; ++rule) {
        std::vector<uint32_t> nb = list_neighbors(s, c, rule);
        if (!nb.empty()) { *rule_out = rule; return nb; }
    }
    *rule_out = 3;
    return {};
}
float coord_M(int M, int k);
// Alg.2: the neighbour nearest to the continuous position x by Euclidean distance in continuous space
// (compared on the squared distance, A30; fp32, one rounding per operation; ties -> smallest L, A5).
uint32_t repair_alg2(const Space& s, const uint8_t* c, const float* x, int* rule_out) {
    std::vector<uint32_t> nb = neighbors_cascade(s, c, rule_out);
    uint32_t best = RANK_NONE; float bestd = 0.0f;
    for (uint32_t r : nb) {
        const uint8_t* v = &s.rows[(uint64_t)r * s.n];
        float acc = 0.0f;
        for (int d = 0; d < s.n; ++d) { float df = coord_M(s.M, v[d]) - x[d]; float q = df * df; acc = acc + q; }
        if (best == RANK_NONE || acc < bestd) { best = r; bestd = acc; }     // ascending L: ties keep the first
    }
    return best;
}
// Alg.3: a random member of the first non-empty neighbour set (w = the 32-bit draw).
uint32_t repair_alg3(const Space& s, const uint8_t* c, uint32_t w, int* rule_out) {
    std::vector<uint32_t> nb = neighbors_cascade(s, c, rule_out);
    if (nb.empty()) return RANK_NONE;
    return nb[below(w, (uint32_t)nb.size())];
}

// ------------------------------------------------------------------ runs
enum Algo : int { A_DE = 0, A_PSO = 1, A_FF = 2, A_GA = 3 };
struct HParams { float de_F, de_CR, pso_w, pso_c1, pso_c2, ff_B0, ff_gamma, ff_alpha; int32_t ga_mutation_chance, ga_beta_b; };

// SURVEY 8(f) switches; the all-default value is the north_star path.
struct Variant {
    int32_t aware;          // 1 constraint-aware (default); 0 = NEXT-2: random Cartesian init, no repair, static penalty
    int32_t repair_mode;    // 0 unified key (A4); 1 = NEXT-1: DE index-distance / PSO,FF Alg.2 / GA Alg.3
    int32_t de_mutation;    // 0 best1 (default), 1 rand1, 2 currenttobest1, 3 randtobest1, 4 best2, 5 rand2   (NEXT-3)
    int32_t de_crossover;   // 0 binomial (default), 1 exponential
    int32_t ga_crossover;   // 0 single_point (default), 1 two_point, 2 uniform, 3 disruptive_uniform
    int32_t init_lhs;       // 1 = Latin Hypercube initial population (DE, L223)
    float penalty;          // objective of an unevaluated invalid configuration (L107: 1e20 under minimisation)
    int32_t reserved;
};
const Variant VARIANT_DEFAULT = { 1, 0, 0, 0, 0, 0, 1e20f, 0 };
const int DE_DONORS[6] = { 2, 3, 2, 3, 4, 5 };

struct Run {
    uint32_t id = 0;                     // global run index (RNG key)
    std::vector<uint8_t> idx;            // P x n   DE/GA individuals (valid rows)
    std::vector<uint32_t> rank;          // P       rank of each individual (DE/GA) / last evaluated rank (PSO/FF)
    std::vector<float> f;                // P       objective of each individual / last evaluation
    std::vector<float> x, v, pb;         // P x n   PSO/FF position, PSO velocity, PSO personal best
    std::vector<float> pbf;              // P       PSO personal-best objective
    std::vector<uint8_t> seen;           // V       memoisation: 1 if this run ever evaluated the rank
    uint32_t uniq = 0, gens_done = 0, stagnation = 0;
    float best_f = 0; uint32_t best_rank = 0xFFFFFFFFu;
};

struct Runs {
    const Space* s; Algo algo; HParams hp; uint32_t R, first_run; int P; uint32_t budget, max_gens; uint64_t seed;
    Variant var = VARIANT_DEFAULT;
    uint32_t gen = 0;                    // generations stepped so far (trajectory rows 0..gen)
    std::vector<Run> run;
    std::vector<uint8_t> traj;           // (gen+1) x R x 12 bytes {f32 best_f, u32 best_rank, u32 uniq}
    // taps of the last stepped generation, [run][ind]:
    std::vector<uint8_t> tap_cand;       // R x P x n   post-snap, pre-repair rows
    std::vector<uint8_t> tap_valid;      // R x P       1 if the post-snap row was valid
    std::vector<uint32_t> tap_rep;       // R x P       rank after repair (before GA mutation)
    std::vector<uint32_t> tap_eval;      // R x P       rank evaluated
    std::vector<float> tap_f;            // R x P       f of the evaluated rank
    std::vector<uint8_t> tap_accept;     // R x P       DE accept flag / PSO pbest-improved flag
    std::vector<uint8_t> tap_active;     // R           run was active this generation
    uint64_t n_repaired = 0;             // candidates whose post-snap row was invalid (all generations)
    uint64_t n_evaluated = 0;            // candidates evaluated (all generations, incl. gen 0 and re-inits)
    uint64_t n_penalised = 0;            // candidates that stayed invalid and received the static penalty (NEXT-1 / NEXT-2)
    std::vector<uint8_t> tap_rule;       // R x P       NEXT-1: neighbour rule that repaired the candidate (0/1/2), 3 = none, 255 = n/a
};

// O6 continuous embedding (L278-280): the dimension with most values (M of them) spans [0,1] with grid step
// eps = 1/(M-1); dimension d spans [0, (m_d-1)*eps] (A10).  snap = nearest grid point, half-to-even (A11).
float coord_M(int M, int k) { return M > 1 ? (float)k / (float)(M - 1) : 0.0f; }
int snap_M(int M, int m_d, float x) {
    float g = x * (float)(M - 1);
    int k = (int)rintf(g);
    if (k < 0) k = 0;
    if (k > m_d - 1) k = m_d - 1;
    return k;
}
float coord(const Space& s, int k) { return coord_M(s.M, k); }
int snap(const Space& s, int d, float x) { return snap_M(s.M, (int)s.dom[d].size(), x); }

// O5 mutation of one dimension on indices: round_and_clip(i_best + F*(i_a - i_b)), two fp32 roundings,
// rint = round-half-to-even (A8), clip to [0, top].
int de_mutate_index(float F, int ibest, int ia, int ib, int top) {
    int diff = ia - ib;
    float t = F * (float)diff;
    float mf = (float)ibest + t;
    int vd = (int)rintf(mf);
    if (vd < 0) vd = 0;
    if (vd > top) vd = top;
    return vd;
}

// O10: evaluate a rank for a run: memoise, count unique, track best-so-far = min (f bits, rank).
// rank == RANK_NONE (NEXT-1 / NEXT-2: the configuration stayed invalid): it cannot be compiled or measured (L135), so
// nothing is memoised or counted and the strategy sees the static penalty (L107, L284; A33).
float evaluate(Runs& rs, Run& r, uint32_t rank) {
    if (rank == RANK_NONE) { rs.n_penalised += 1; return rs.var.penalty; }
    float f = rs.s->obj[rank];
    if (!r.seen[rank]) { r.seen[rank] = 1; r.uniq += 1; }
    if (r.best_rank == 0xFFFFFFFFu || fbits(f) < fbits(r.best_f) || (fbits(f) == fbits(r.best_f) && rank < r.best_rank)) {
        r.best_f = f; r.best_rank = rank;
    }
    rs.n_evaluated += 1;
    return f;
}

// NEXT-3, L223 (A35): Latin Hypercube sample of P index rows.  Per dimension d the P strata [j/P, (j+1)/P) of the unit
// interval are assigned to the individuals by the permutation perm_d(i) = number of individuals whose draw(slot 1+d) is
// smaller (ties by individual); individual i takes the point (perm_d(i) + u) / P, u = u01(draw(slot 1+n+d)), scaled to m_d values.
void lhs_rows(const Runs& rs, const Run& r, uint32_t stream, uint32_t gen, std::vector<uint8_t>& out) {
    const Space& s = *rs.s; const int P = rs.P, n = s.n;
    out.assign((size_t)P * n, 0);
    for (int d = 0; d < n; ++d) {
        std::vector<uint32_t> w(P);
        for (int j = 0; j < P; ++j) w[j] = draw(rs.seed, r.id, gen, j, stream, 1 + d);
        for (int i = 0; i < P; ++i) {
            int perm = 0;
            for (int j = 0; j < P; ++j) perm += (w[j] < w[i]) || (w[j] == w[i] && j < i);
            float u = u01(draw(rs.seed, r.id, gen, i, stream, 1 + n + d));
            float t = (float)perm + u;
            t = t * (float)s.dom[d].size();
            t = t / (float)P;
            int k = (int)floorf(t);
            if (k > (int)s.dom[d].size() - 1) k = (int)s.dom[d].size() - 1;
            out[(size_t)i * n + d] = (uint8_t)k;
        }
    }
}

// O4: P distinct valid ranks, uniform with linear probing; fills DE/GA rows or PSO/FF positions.
// Variants: init_lhs (A35): the rank of individual i is the unified-key repair (O9) of its LHS point instead of a uniform
// draw, with the same linear probing; aware = 0 (NEXT-2, L272 / L284; A34): the initial population is random in the
// Cartesian space (DE/GA: idx_d = below(draw(slot 1+n+d), m_d); PSO/FF: x_d = u01(draw(slot 1+n+d)) * hi_d), not repaired.
void init_population(Runs& rs, Run& r, uint32_t stream, uint32_t gen) {
    const Space& s = *rs.s; const int P = rs.P, n = s.n;
    if (!rs.var.aware) {
        for (int i = 0; i < P; ++i) {
            uint8_t row[32];
            for (int d = 0; d < n; ++d) {
                uint32_t w = draw(rs.seed, r.id, gen, i, stream, 1 + n + d);
                float hi = coord_M(s.M, (int)s.dom[d].size() - 1);
                if (rs.algo == A_DE || rs.algo == A_GA) {
                    row[d] = (uint8_t)below(w, (uint32_t)s.dom[d].size());
                    r.idx[(size_t)i * n + d] = row[d];
                } else {
                    float xd = u01(w) * hi;
                    r.x[(size_t)i * n + d] = xd;
                    row[d] = (uint8_t)snap_M(s.M, (int)s.dom[d].size(), xd);
                    if (rs.algo == A_PSO) {
                        float u = u01(draw(rs.seed, r.id, gen, i, stream, 1 + d));
                        float c = u - 0.5f;
                        r.v[(size_t)i * n + d] = c * hi;
                        r.pb[(size_t)i * n + d] = xd;
                    }
                }
            }
            uint64_t L = s.lin(row);
            uint32_t rk = s.bit(L) ? s.rank_of(L) : RANK_NONE;
            r.rank[i] = rk;
            r.f[i] = evaluate(rs, r, rk);
            if (rs.algo == A_PSO) r.pbf[i] = r.f[i];
        }
        return;
    }
    std::vector<uint8_t> lhs;
    const bool use_lhs = rs.var.init_lhs && stream == S_INIT;          // L266: the stagnation re-init is "random"
    if (use_lhs) lhs_rows(rs, r, stream, gen, lhs);
    std::vector<uint32_t> taken;
    for (int i = 0; i < P; ++i) {
        uint32_t rk = use_lhs ? repair(s, &lhs[(size_t)i * n]).rank
                              : below(draw(rs.seed, r.id, gen, i, stream, 0), (uint32_t)s.V);
        while (std::find(taken.begin(), taken.end(), rk) != taken.end()) rk = (uint32_t)((rk + 1) % s.V);
        taken.push_back(rk);
        const uint8_t* row = &s.rows[(uint64_t)rk * n];
        r.rank[i] = rk;
        r.f[i] = evaluate(rs, r, rk);
        if (rs.algo == A_DE || rs.algo == A_GA) {
            std::copy(row, row + n, &r.idx[(size_t)i * n]);
        } else {
            for (int d = 0; d < n; ++d) {
                float xd = coord(s, row[d]);
                r.x[(size_t)i * n + d] = xd;
                if (rs.algo == A_PSO) {
                    float hi = coord(s, (int)s.dom[d].size() - 1);
                    float u = u01(draw(rs.seed, r.id, gen, i, stream, 1 + d));
                    float c = u - 0.5f;
                    r.v[(size_t)i * n + d] = c * hi;
                    r.pb[(size_t)i * n + d] = xd;
                }
            }
            if (rs.algo == A_PSO) r.pbf[i] = r.f[i];
        }
    }
}

void write_traj(Runs& rs, uint32_t g) {
    rs.traj.resize((size_t)(g + 1) * rs.R * 12);
    for (uint32_t k = 0; k < rs.R; ++k) {
        uint8_t* p = &rs.traj[((size_t)g * rs.R + k) * 12];
        const Run& r = rs.run[k];
        std::memcpy(p, &r.best_f, 4); std::memcpy(p + 4, &r.best_rank, 4); std::memcpy(p + 8, &r.uniq, 4);
    }
}

// S4-S6 for one candidate row: validity, repair, (tap), returns the rank after repair, or RANK_NONE when the
// candidate stays invalid (aware = 0: no repair, L272 / L284; repair_mode = 1: every neighbour set empty, Alg.2 L18 / Alg.3 L7).
// xcont: the continuous position the row was snapped from (PSO / Firefly), used by Alg.2 only.
uint32_t validate_and_repair(Runs& rs, size_t k, int i, const uint8_t* cand, const float* xcont = nullptr, uint32_t g = 0) {
    const Space& s = *rs.s; const int n = s.n, P = rs.P;
    size_t t = k * P + i;
    std::copy(cand, cand + n, &rs.tap_cand[t * n]);
    rs.tap_rule[t] = 255;
    uint64_t Lc = s.lin(cand);
    if (s.bit(Lc)) {                                            // operator outputs are in-domain by construction
        rs.tap_valid[t] = 1;
        rs.tap_rep[t] = s.rank_of(Lc);
        return rs.tap_rep[t];
    }
    rs.tap_valid[t] = 0;
    rs.n_repaired += 1;                                         // counts the invalid post-snap rows
    uint32_t rk = RANK_NONE;
    if (rs.var.aware) {
        if (rs.var.repair_mode == 0) rk = repair(s, cand).rank;
        else {
            int rule = 255;
            if (rs.algo == A_DE) rk = repair_index_distance(s, cand).rank;
            else if (rs.algo == A_GA) rk = repair_alg3(s, cand, draw(rs.seed, rs.run[k].id, g, i, S_REPAIR, 0), &rule);
            else rk = repair_alg2(s, cand, xcont, &rule);
            rs.tap_rule[t] = (uint8_t)rule;
        }
    }
    rs.tap_rep[t] = rk;
    return rk;
}

// The row an individual holds after S5: the valid table row of its rank, or its own (still invalid) candidate row.
const uint8_t* row_after_repair(const Space& s, uint32_t rk, const uint8_t* cand) {
    return rk == RANK_NONE ? cand : &s.rows[(uint64_t)rk * s.n];
}

// NEXT-3 (L219, L272): k distinct donors from X \ {x_i}: donor z = below(draw(OP, z), P-1-z) mapped past i and the
// earlier donors in ascending order (for two donors this is exactly O5's a, b).
void de_donors(const Runs& rs, const Run& r, uint32_t g, int i, int nd, uint32_t* donor) {
    std::vector<uint32_t> taken{ (uint32_t)i };
    for (int z = 0; z < nd; ++z) {
        uint32_t a = below(draw(rs.seed, r.id, g, i, S_OP, z), (uint32_t)(rs.P - 1 - z));
        std::sort(taken.begin(), taken.end());
        for (uint32_t t : taken) if (a >= t) a += 1;
        taken.push_back(a);
        donor[z] = a;
    }
}
// Mutation of one dimension on indices (Alg.1 L183-188 generalised to the operators of L272), fp32, one rounding per
// operation, round half-to-even, clip (A8).  base / diff pairs by operator:
//   best1 best + F(r0-r1) | rand1 r0 + F(r1-r2) | currenttobest1 x + F(best-x) + F(r0-r1) | randtobest1 r0 + F(best-r0) + F(r1-r2)
//   best2 best + F(r0-r1) + F(r2-r3) | rand2 r0 + F(r1-r2) + F(r3-r4)
int de_mutate_variant(int op, float F, int xi, int best, const int* r, int top) {
    int base, p1, q1, p2 = 0, q2 = 0; bool two = true;
    switch (op) {
        case 1: base = r[0]; p1 = r[1]; q1 = r[2]; two = false; break;
        case 2: base = xi; p1 = best; q1 = xi; p2 = r[0]; q2 = r[1]; break;
        case 3: base = r[0]; p1 = best; q1 = r[0]; p2 = r[1]; q2 = r[2]; break;
        case 4: base = best; p1 = r[0]; q1 = r[1]; p2 = r[2]; q2 = r[3]; break;
        case 5: base = r[0]; p1 = r[1]; q1 = r[2]; p2 = r[3]; q2 = r[4]; break;
        default: base = best; p1 = r[0]; q1 = r[1]; two = false; break;
    }
    float t1 = F * (float)(p1 - q1);
    float mf = (float)base + t1;
    if (two) { float t2 = F * (float)(p2 - q2); mf = mf + t2; }
    int vd = (int)rintf(mf);
    if (vd < 0) vd = 0;
    if (vd > top) vd = top;
    return vd;
}

// O5: one synchronous DE generation (best1bin by default; NEXT-3 operators through rs.var).
void step_de(Runs& rs, size_t k, uint32_t g) {
    const Space& s = *rs.s; Run& r = rs.run[k]; const int n = s.n, P = rs.P;
    const std::vector<uint8_t> old = r.idx;                     // population at generation start (A6)
    const std::vector<float> oldf = r.f;
    // best-so-far at generation start; while nothing valid has been evaluated (NEXT-2 only): individual 0 (A34)
    const uint8_t* best = r.best_rank == RANK_NONE ? &old[0] : &s.rows[(uint64_t)r.best_rank * n];
    std::vector<uint64_t> oldL(P), uL(P);
    for (int j = 0; j < P; ++j) oldL[j] = s.lin(&old[(size_t)j * n]);
    std::vector<uint32_t> urank(P); std::vector<float> uf(P);
    std::vector<uint8_t> urow((size_t)P * n);
    const int mut = rs.var.de_mutation, nd = DE_DONORS[mut];
    for (int i = 0; i < P; ++i) {
        // donors distinct, all != i (A9: any may coincide with best)
        uint32_t don[5];
        de_donors(rs, r, g, i, nd, don);
        uint32_t jrand = below(draw(rs.seed, r.id, g, i, S_OP, nd), n);
        uint8_t v[32], u[32];
        for (int d = 0; d < n; ++d) {
            // Alg.1: m = i_r1 + F*(i_r2 - i_r3) on indices, r1 = best; round half-to-even, clip (A8)
            int rr[5];
            for (int z = 0; z < nd; ++z) rr[z] = old[(size_t)don[z] * n + d];
            v[d] = (uint8_t)(mut == 0 ? de_mutate_index(rs.hp.de_F, best[d], rr[0], rr[1], (int)s.dom[d].size() - 1)
                                      : de_mutate_variant(mut, rs.hp.de_F, old[(size_t)i * n + d], best[d], rr, (int)s.dom[d].size() - 1));
        }
        if (rs.var.de_crossover == 0) {
            // Alg.1: binomial crossover
            for (int d = 0; d < n; ++d) {
                float rr = u01(draw(rs.seed, r.id, g, i, S_OP, nd + 1 + d));
                u[d] = (rr < rs.hp.de_CR || (uint32_t)d == jrand) ? v[d] : old[(size_t)i * n + d];
            }
        } else {
            // exponential crossover (L272): a run of consecutive dimensions (cyclic) from j_rand, continued while r < CR
            for (int d = 0; d < n; ++d) u[d] = old[(size_t)i * n + d];
            int d = (int)jrand, c = 0;
            do { u[d] = v[d]; d = (d + 1) % n; ++c; }
            while (c < n && u01(draw(rs.seed, r.id, g, i, S_OP, nd + 1 + c)) < rs.hp.de_CR);
        }
        urank[i] = validate_and_repair(rs, k, i, u);
        const uint8_t* ur = row_after_repair(s, urank[i], u);
        std::copy(ur, ur + n, &urow[(size_t)i * n]);
        rs.tap_eval[k * P + i] = urank[i];
        uf[i] = evaluate(rs, r, urank[i]);                      // all P trials are evaluated
        rs.tap_f[k * P + i] = uf[i];
        uL[i] = s.lin(ur);
    }
    // selection (Alg.1): f(u) <= f(x) and u not in X (old members) and not an earlier trial (A7)
    bool any = false;
    for (int i = 0; i < P; ++i) {
        bool acc = uf[i] <= oldf[i];
        for (int j = 0; j < P && acc; ++j) if (oldL[j] == uL[i]) acc = false;
        for (int j = 0; j < i && acc; ++j) if (uL[j] == uL[i]) acc = false;
        rs.tap_accept[k * P + i] = acc;
        if (acc) {
            any = true;
            std::copy(&urow[(size_t)i * n], &urow[(size_t)i * n] + n, &r.idx[(size_t)i * n]);
            r.f[i] = uf[i]; r.rank[i] = urank[i];
        }
    }
    // L266: population unchanged over two consecutive generations -> re-initialise (evaluated in this step)
    r.stagnation = any ? 0 : r.stagnation + 1;
    if (r.stagnation == 2) { init_population(rs, r, S_REINIT, g); r.stagnation = 0; }
}

// O6: one synchronous PSO generation.
void step_pso(Runs& rs, size_t k, uint32_t g) {
    const Space& s = *rs.s; Run& r = rs.run[k]; const int n = s.n, P = rs.P;
    int gb = 0;                                                // gbest = argmin (pbest_f bits, i) at generation start
    for (int i = 1; i < P; ++i) if (fbits(r.pbf[i]) < fbits(r.pbf[gb])) gb = i;
    const std::vector<float> gbest(r.pb.begin() + (size_t)gb * n, r.pb.begin() + (size_t)(gb + 1) * n);
    for (int i = 0; i < P; ++i) {
        uint8_t cand[32];
        for (int d = 0; d < n; ++d) {
            size_t q = (size_t)i * n + d;
            float hi = coord(s, (int)s.dom[d].size() - 1);
            float r1 = u01(draw(rs.seed, r.id, g, i, S_OP, 2 * d));
            float r2 = u01(draw(rs.seed, r.id, g, i, S_OP, 2 * d + 1));
            float a = rs.hp.pso_c1 * r1;
            float b = r.pb[q] - r.x[q];
            float t1 = a * b;
            float c = rs.hp.pso_c2 * r2;
            float e = gbest[d] - r.x[q];
            float t2 = c * e;
            float vv = rs.hp.pso_w * r.v[q];
            vv = vv + t1;
            vv = vv + t2;
            float xx = r.x[q] + vv;
            xx = clamp_pos(xx, hi);
            r.v[q] = vv; r.x[q] = xx;
            cand[d] = (uint8_t)snap(s, d, xx);
        }
        uint32_t rk = validate_and_repair(rs, k, i, cand, &r.x[(size_t)i * n], g);   // repair affects evaluation only (L282)
        rs.tap_eval[k * P + i] = rk;
        float f = evaluate(rs, r, rk);
        rs.tap_f[k * P + i] = f; r.f[i] = f; r.rank[i] = rk;
        bool improved = f < r.pbf[i];                           // strict (A13)
        rs.tap_accept[k * P + i] = improved;
        if (improved) { r.pbf[i] = f; for (int d = 0; d < n; ++d) r.pb[(size_t)i * n + d] = r.x[(size_t)i * n + d]; }
    }
}

// O7: one synchronous Firefly generation (Yang's rule; A14-A16).
void step_ff(Runs& rs, size_t k, uint32_t g) {
    const Space& s = *rs.s; Run& r = rs.run[k]; const int n = s.n, P = rs.P;
    const std::vector<float> xo = r.x, fo = r.f;                // start-of-generation positions / intensities
    for (int i = 0; i < P; ++i) {
        float xi[32];
        for (int d = 0; d < n; ++d) xi[d] = xo[(size_t)i * n + d];
        for (int j = 0; j < P; ++j) {
            if (!(fo[j] < fo[i])) continue;                     // only brighter (lower cost) fireflies attract
            float r2 = 0.0f;
            for (int d = 0; d < n; ++d) { float df = xo[(size_t)j * n + d] - xi[d]; float q = df * df; r2 = r2 + q; }
            float z = rs.hp.ff_gamma * r2;
            float beta = rs.hp.ff_B0 * exp_neg_spec(z);
            for (int d = 0; d < n; ++d) {
                float df = xo[(size_t)j * n + d] - xi[d];
                float sft = beta * df;
                xi[d] = xi[d] + sft;
                float e = u01(draw(rs.seed, r.id, g, i, S_OP, (uint32_t)(j * n + d))) - 0.5f;
                e = rs.hp.ff_alpha * e;
                xi[d] = xi[d] + e;
            }
        }
        uint8_t cand[32];
        for (int d = 0; d < n; ++d) {
            float hi = coord(s, (int)s.dom[d].size() - 1);
            xi[d] = clamp_pos(xi[d], hi);
            r.x[(size_t)i * n + d] = xi[d];
            cand[d] = (uint8_t)snap(s, d, xi[d]);
        }
        uint32_t rk = validate_and_repair(rs, k, i, cand, &r.x[(size_t)i * n], g);
        rs.tap_eval[k * P + i] = rk;
        float f = evaluate(rs, r, rk);
        rs.tap_f[k * P + i] = f; r.f[i] = f; r.rank[i] = rk;
        rs.tap_accept[k * P + i] = 0;
    }
}

// O8: one GA generation (single-point crossover by default, repair, then 1-in-X mutation; population replaced).
void step_ga(Runs& rs, size_t k, uint32_t g) {
    const Space& s = *rs.s; Run& r = rs.run[k]; const int n = s.n, P = rs.P;
    const int B = rs.hp.ga_beta_b;
    std::vector<int> order(P);
    for (int i = 0; i < P; ++i) order[i] = i;
    std::vector<uint64_t> L(P);
    for (int i = 0; i < P; ++i) L[i] = s.lin(&r.idx[(size_t)i * n]);
    std::sort(order.begin(), order.end(), [&](int a, int b) {   // L288: sorted by cost; ties by (L, i)
        if (fbits(r.f[a]) != fbits(r.f[b])) return fbits(r.f[a]) < fbits(r.f[b]);
        if (L[a] != L[b]) return L[a] < L[b];
        return a < b;
    });
    const std::vector<uint8_t> old = r.idx;
    for (int i = 0; i < P; ++i) {
        // Beta(1,B) selection over sorted positions = min of B uniform positions (A18)
        uint32_t sa = P, sb = P;
        for (int q = 0; q < B; ++q) sa = std::min(sa, below(draw(rs.seed, r.id, g, i, S_OP, q), P));
        for (int q = 0; q < B; ++q) sb = std::min(sb, below(draw(rs.seed, r.id, g, i, S_OP, B + q), P));
        if (sb == sa) sb = (sa + 1) % P;                        // A17
        const uint8_t* pa = &old[(size_t)order[sa] * n];
        const uint8_t* pbb = &old[(size_t)order[sb] * n];
        uint8_t child[32];
        if (rs.var.ga_crossover == 0) {                         // single point (Table IV)
            int cut = (n > 1) ? 1 + (int)below(draw(rs.seed, r.id, g, i, S_OP, 2 * B), n - 1) : 1;
            for (int d = 0; d < n; ++d) child[d] = d < cut ? pa[d] : pbb[d];
        } else if (rs.var.ga_crossover == 1) {                  // two point (L288; A31): B's genes between the two cuts
            uint32_t c1 = below(draw(rs.seed, r.id, g, i, S_OP, 2 * B), n + 1);
            uint32_t c2 = below(draw(rs.seed, r.id, g, i, S_OP, 2 * B + 1), n + 1);
            uint32_t lo = std::min(c1, c2), hi = std::max(c1, c2);
            for (int d = 0; d < n; ++d) child[d] = ((uint32_t)d >= lo && (uint32_t)d < hi) ? pbb[d] : pa[d];
        } else if (rs.var.ga_crossover == 2) {                  // uniform (L288): every gene from A or B with probability 1/2
            for (int d = 0; d < n; ++d) child[d] = below(draw(rs.seed, r.id, g, i, S_OP, 2 * B + d), 2) == 0 ? pa[d] : pbb[d];
        } else {                                                // disruptive uniform (L288; A31): uniform, but at least
            int D = 0;                                          // half of the DIFFERING genes come from B
            for (int d = 0; d < n; ++d) D += (pa[d] != pbb[d]);
            int need = (D + 1) / 2, rem = D;
            for (int d = 0; d < n; ++d) {
                child[d] = pa[d];
                if (pa[d] == pbb[d]) continue;
                bool coin = below(draw(rs.seed, r.id, g, i, S_OP, 2 * B + d), 2) == 1;
                bool take = coin || need >= rem;
                if (take) { child[d] = pbb[d]; if (need > 0) --need; }
                --rem;
            }
        }
        uint32_t rk = validate_and_repair(rs, k, i, child, nullptr, g);   // A4 unified key, or Alg.3 (repair_mode 1)
        uint8_t cur[32];
        { const uint8_t* rr = row_after_repair(s, rk, child); std::copy(rr, rr + n, cur); }
        // L290, L311, L393: mutate with probability 1/X
        if (below(draw(rs.seed, r.id, g, i, S_MUT, 0), (uint32_t)rs.hp.ga_mutation_chance) == 0) {
            if (rs.var.aware) {                                 // ... into a random valid Hamming-1 neighbour (L311)
                std::vector<uint64_t> nb;                       // valid Hamming-1 neighbours, (d asc, value index asc)
                for (int d = 0; d < n; ++d)
                    for (int val = 0; val < (int)s.dom[d].size(); ++val) {
                        if (val == cur[d]) continue;
                        uint8_t t[32]; std::copy(cur, cur + n, t); t[d] = (uint8_t)val;
                        if (s.valid_idx(t)) nb.push_back(s.lin(t));
                    }
                if (!nb.empty()) {
                    uint32_t pick = below(draw(rs.seed, r.id, g, i, S_MUT, 1), (uint32_t)nb.size());
                    rk = s.rank_of(nb[pick]);
                    std::copy(&s.rows[(uint64_t)rk * n], &s.rows[(uint64_t)rk * n] + n, cur);
                }
            } else {                                            // NEXT-2 (L309): one parameter gets a different value, if any
                int d = (int)below(draw(rs.seed, r.id, g, i, S_MUT, 1), n);
                int md = (int)s.dom[d].size();
                if (md > 1) {
                    int val = (int)below(draw(rs.seed, r.id, g, i, S_MUT, 2), md - 1);
                    if (val >= cur[d]) val += 1;
                    cur[d] = (uint8_t)val;
                    uint64_t Lm = s.lin(cur);
                    rk = s.bit(Lm) ? s.rank_of(Lm) : RANK_NONE;
                }
            }
        }
        rs.tap_eval[k * P + i] = rk;
        float f = evaluate(rs, r, rk);
        rs.tap_f[k * P + i] = f;
        rs.tap_accept[k * P + i] = 0;
        std::copy(cur, cur + n, &r.idx[(size_t)i * n]);         // L288: fully refreshed
        r.f[i] = f; r.rank[i] = rk;
    }
}

// ------------------------------------------------------------------ NEXT-4: performance score (Eq.2; A36)
// Calculated baseline B(t): the expected best (minimum) objective of t draws without replacement from the V feasible
// configurations ("a statistical approximation of random search over the feasible solutions", L357):
//   B(t) = sum_{i=1..V-t+1} f_(i) * C(V-i, t-1) / C(V, t),  f_(1) <= f_(2) <= ... the sorted objective values;
// the weights follow w_1 = t/V, w_{i+1} = w_i * (V-t-i+1) / (V-i).  fp64.
double baseline_at(const std::vector<float>& sorted, uint64_t t) {
    const uint64_t V = sorted.size();
    if (t < 1) t = 1;
    if (t > V) t = V;
    double w = (double)t / (double)V, acc = 0.0;
    for (uint64_t i = 1; i + t <= V + 1; ++i) {
        acc += w * (double)sorted[i - 1];
        w = w * (double)(V - t - i + 1) / (double)(V - i);
    }
    return acc;
}
// Budget of [29] as quoted in L361: the time (here: unique evaluations) the baseline needs to reach `frac` (0.95) of the
// distance between the search-space median and the optimum.  median = lower median of the sorted objective values.
uint64_t baseline_budget(const std::vector<float>& sorted, double frac) {
    const uint64_t V = sorted.size();
    const double opt = sorted[0], med = sorted[(V - 1) / 2];
    const double target = med - frac * (med - opt);
    for (uint64_t t = 1; t <= V; ++t) if (baseline_at(sorted, t) <= target) return t;
    return V;
}
// P_t of one run (L359-361; A36): (B(t) - best_r(t)) / (B(t) - f_opt), best_r(t) = best-so-far objective at the last
// recorded generation whose unique-evaluation count is <= t (generation 0 if none); a run that has not evaluated any
// valid configuration by then counts as the worst feasible objective.  0 = baseline, 1 = optimum found at once.
// Where the baseline has itself reached the optimum the quotient is undefined; see the guard below.
double score_run_at(const Runs& rs, const std::vector<float>& sorted, uint32_t k, uint64_t t) {
    const uint32_t G = rs.gen;
    uint32_t gsel = 0;
    for (uint32_t g = 0; g <= G; ++g) {
        uint32_t uq; std::memcpy(&uq, &rs.traj[((size_t)g * rs.R + k) * 12 + 8], 4);
        if (uq <= t) gsel = g;
    }
    float bf; uint32_t br;
    std::memcpy(&bf, &rs.traj[((size_t)gsel * rs.R + k) * 12], 4);
    std::memcpy(&br, &rs.traj[((size_t)gsel * rs.R + k) * 12 + 4], 4);
    const double best = br == RANK_NONE ? (double)sorted.back() : (double)bf;
    const double B = baseline_at(sorted, t), opt = sorted[0];
    // B(t) = f_opt (t >= V, or every objective value equal): random search has reached the optimum itself and the ratio is
    // 0/0 or x/0.  A36: the term is then 1 for a run that holds the optimum and 0 otherwise.
    if (B - opt == 0.0) return best == opt ? 1.0 : 0.0;
    return (B - best) / (B - opt);
}

}  // namespace

// ============================================================================ C entry points
extern "C" {

void orc_philox4x32_10(const uint32_t* ctr, const uint32_t* key, uint32_t* out) { philox4x32_10(ctr, key, out); }
uint32_t orc_draw(uint64_t seed, uint32_t run, uint32_t gen, uint32_t ind, uint32_t stream, uint32_t slot) {
    return draw(seed, run, gen, ind, stream, slot);
}
float orc_u01(uint32_t w) { return u01(w); }
uint32_t orc_below(uint32_t w, uint32_t k) { return below(w, k); }
float orc_exp_neg_spec(float z) { return exp_neg_spec(z); }
void orc_exp_neg_spec_many(const float* z, float* out, uint64_t count) { for (uint64_t i = 0; i < count; ++i) out[i] = exp_neg_spec(z[i]); }

int orc_de_mutate_index(float F, int ibest, int ia, int ib, int top) { return de_mutate_index(F, ibest, ia, ib, top); }
float orc_clamp_pos(float x, float hi) { return clamp_pos(x, hi); }
float orc_coord(int M, int k) { return coord_M(M, k); }
int orc_snap(int M, int m_d, float x) { return snap_M(M, m_d, x); }

void* orc_space_create() { return new Space(); }
void orc_space_destroy(void* p) { delete (Space*)p; }
int orc_space_add_param(void* p, const int64_t* values, int32_t nv) {
    Space* s = (Space*)p;
    if (nv < 1 || nv > 256 || s->dom.size() >= 32 || s->built) return -1;
    s->dom.emplace_back(values, values + nv);
    return 0;
}
int orc_space_add_constraint(void* p, const int32_t* w, int32_t nw) {
    Space* s = (Space*)p;
    if (s->built || !program_ok(w, nw, (int)s->dom.size())) return -1;
    s->cons.emplace_back(w, w + nw);
    return 0;
}
int orc_space_build(void* p) { Space* s = (Space*)p; if (s->dom.empty()) return -1; enumerate(*s); return 0; }
// Single-constraint / single-config evaluation on VALUES (used by the bytecode pins).
int orc_eval_program(const int32_t* w, int32_t nw, const int64_t* x, int32_t n_params) {
    if (!program_ok(w, nw, n_params)) return -1;
    std::vector<int32_t> prog(w, w + nw);
    return eval_program(prog, x);
}
uint64_t orc_space_N(const void* p) { return ((const Space*)p)->N; }
uint64_t orc_space_V(const void* p) { return ((const Space*)p)->V; }
int32_t orc_space_n(const void* p) { return ((const Space*)p)->n; }
const uint64_t* orc_space_bitmap(const void* p) { return ((const Space*)p)->bitmap.data(); }
const uint8_t* orc_space_rows(const void* p) { return ((const Space*)p)->rows.data(); }
const uint64_t* orc_space_Ltab(const void* p) { return ((const Space*)p)->Ltab.data(); }
int orc_space_is_valid(const void* p, const uint8_t* idx) { const Space* s = (const Space*)p; return in_domain(*s, idx) && s->bit(s->lin(idx)); }
// Count of valid configs among L in [L0, L1) evaluated directly (no table): for sampled-range checks.
uint64_t orc_space_count_range(const void* p, uint64_t L0, uint64_t L1) {
    const Space* s = (const Space*)p;
    int n = (int)s->dom.size();
    std::vector<uint64_t> stride(n, 1);
    for (int d = n - 2; d >= 0; --d) stride[d] = stride[d + 1] * s->dom[d + 1].size();
    uint64_t cnt = 0; uint8_t idx[32];
    Space tmp; tmp.dom = s->dom; tmp.cons = s->cons; tmp.n = n;
    for (uint64_t L = L0; L < L1; ++L) {
        for (int d = 0; d < n; ++d) idx[d] = (uint8_t)((L / stride[d]) % s->dom[d].size());
        cnt += tmp.valid_idx(idx);
    }
    return cnt;
}
// Brute-force repair of `count` rows (n bytes each): rank + key parts.
void orc_space_repair(const void* p, const uint8_t* rows, uint64_t count, uint32_t* rank, uint32_t* ham, uint32_t* sad, uint64_t* L) {
    const Space* s = (const Space*)p;
    for (uint64_t i = 0; i < count; ++i) {
        RepairKey k = repair(*s, rows + i * s->n);
        if (rank) rank[i] = k.rank;
        if (ham) ham[i] = k.ham;
        if (sad) sad[i] = k.sad;
        if (L) L[i] = k.L;
    }
}
int orc_space_set_objective(void* p, const float* obj) { Space* s = (Space*)p; if (!s->built) return -1; s->obj.assign(obj, obj + s->V); return 0; }

void* orc_runs_create_ex(const void* sp, int algo, const HParams* hp, const Variant* var, uint32_t n_runs, uint32_t first_run,
                         int32_t pop, uint32_t budget, uint32_t max_gens, uint64_t seed) {
    const Space* s = (const Space*)sp;
    const Variant v = var ? *var : VARIANT_DEFAULT;
    if (!s->built || s->obj.size() != s->V || pop < 1 || (uint64_t)pop > s->V || pop > 1024) return nullptr;
    if (algo == A_DE && pop < 3) return nullptr;
    if (algo == A_GA && (pop < 2 || hp->ga_beta_b < 1 || hp->ga_mutation_chance < 1)) return nullptr;
    if (v.aware < 0 || v.aware > 1 || v.repair_mode < 0 || v.repair_mode > 1 || v.de_mutation < 0 || v.de_mutation > 5 ||
        v.de_crossover < 0 || v.de_crossover > 1 || v.ga_crossover < 0 || v.ga_crossover > 3 || v.init_lhs < 0 || v.init_lhs > 1)
        return nullptr;
    if (algo == A_DE && pop < DE_DONORS[v.de_mutation] + 1) return nullptr;
    if (v.init_lhs && (algo != A_DE || !v.aware)) return nullptr;       // L223: LHS is DE's initial sample of valid candidates
    if (!(v.penalty > 0.0f) || !(v.penalty < 3.0e38f)) return nullptr;
    Runs* rs = new Runs();
    rs->s = s; rs->algo = (Algo)algo; rs->hp = *hp; rs->var = v; rs->R = n_runs; rs->first_run = first_run; rs->P = pop;
    rs->budget = budget; rs->max_gens = max_gens; rs->seed = seed;
    const size_t P = pop, n = s->n;
    rs->run.resize(n_runs);
    for (uint32_t k = 0; k < n_runs; ++k) {
        Run& r = rs->run[k];
        r.id = first_run + k;
        r.idx.assign(P * n, 0); r.rank.assign(P, 0); r.f.assign(P, 0.0f);
        if (algo == A_PSO || algo == A_FF) r.x.assign(P * n, 0.0f);
        if (algo == A_PSO) { r.v.assign(P * n, 0.0f); r.pb.assign(P * n, 0.0f); r.pbf.assign(P, 0.0f); }
        r.seen.assign(s->V, 0);
        r.best_f = v.penalty;                                   // until a valid configuration has been evaluated (A33)
        init_population(*rs, r, S_INIT, 0);                     // generation 0 (S2)
    }
    rs->tap_rule.assign((size_t)n_runs * P, 255);
    rs->tap_cand.assign((size_t)n_runs * P * n, 0); rs->tap_valid.assign((size_t)n_runs * P, 0);
    rs->tap_rep.assign((size_t)n_runs * P, 0); rs->tap_eval.assign((size_t)n_runs * P, 0);
    rs->tap_f.assign((size_t)n_runs * P, 0.0f); rs->tap_accept.assign((size_t)n_runs * P, 0);
    rs->tap_active.assign(n_runs, 0);
    write_traj(*rs, 0);
    return rs;
}
void* orc_runs_create(const void* sp, int algo, const HParams* hp, uint32_t n_runs, uint32_t first_run, int32_t pop,
                      uint32_t budget, uint32_t max_gens, uint64_t seed) {
    return orc_runs_create_ex(sp, algo, hp, nullptr, n_runs, first_run, pop, budget, max_gens, seed);
}
void orc_runs_destroy(void* p) { delete (Runs*)p; }

// O10: a run is active for generation g iff (budget == 0 or uniq < budget) and g <= max_gens; an active
// run evaluates all P candidates of that generation (A20); inactive runs are frozen, their row repeats.
void orc_runs_step(void* p, uint32_t n_generations) {
    Runs* rs = (Runs*)p;
    for (uint32_t it = 0; it < n_generations; ++it) {
        uint32_t g = rs->gen + 1;
        for (size_t k = 0; k < rs->R; ++k) {
            Run& r = rs->run[k];
            bool active = (rs->budget == 0 || r.uniq < rs->budget) && g <= rs->max_gens;
            rs->tap_active[k] = active;
            if (!active) continue;
            switch (rs->algo) {
                case A_DE: step_de(*rs, k, g); break;
                case A_PSO: step_pso(*rs, k, g); break;
                case A_FF: step_ff(*rs, k, g); break;
                case A_GA: step_ga(*rs, k, g); break;
            }
            r.gens_done += 1;
        }
        rs->gen = g;
        write_traj(*rs, g);
    }
}
uint32_t orc_runs_gen(const void* p) { return ((const Runs*)p)->gen; }
void orc_runs_best(const void* p, float* best_f, uint32_t* best_rank, uint32_t* uniq, uint32_t* gens_done) {
    const Runs* rs = (const Runs*)p;
    for (uint32_t k = 0; k < rs->R; ++k) {
        best_f[k] = rs->run[k].best_f; best_rank[k] = rs->run[k].best_rank;
        uniq[k] = rs->run[k].uniq; gens_done[k] = rs->run[k].gens_done;
    }
}
const uint8_t* orc_runs_trajectory(const void* p) { return ((const Runs*)p)->traj.data(); }
const uint8_t* orc_runs_tap_cand(const void* p) { return ((const Runs*)p)->tap_cand.data(); }
const uint8_t* orc_runs_tap_valid(const void* p) { return ((const Runs*)p)->tap_valid.data(); }
const uint32_t* orc_runs_tap_rep(const void* p) { return ((const Runs*)p)->tap_rep.data(); }
const uint32_t* orc_runs_tap_eval(const void* p) { return ((const Runs*)p)->tap_eval.data(); }
const float* orc_runs_tap_f(const void* p) { return ((const Runs*)p)->tap_f.data(); }
const uint8_t* orc_runs_tap_accept(const void* p) { return ((const Runs*)p)->tap_accept.data(); }
const uint8_t* orc_runs_tap_active(const void* p) { return ((const Runs*)p)->tap_active.data(); }
uint64_t orc_runs_n_repaired(const void* p) { return ((const Runs*)p)->n_repaired; }
uint64_t orc_runs_n_evaluated(const void* p) { return ((const Runs*)p)->n_evaluated; }
uint64_t orc_runs_n_penalised(const void* p) { return ((const Runs*)p)->n_penalised; }
const uint8_t* orc_runs_tap_rule(const void* p) { return ((const Runs*)p)->tap_rule.data(); }

// ---- NEXT-1 queries on single rows (for the pins and the GPU parity of the standalone repair modes)
// Ranks of the valid neighbours of `row` under rule 0 strictly-adjacent / 1 adjacent / 2 Hamming (ascending L); returns
// the count, writes at most cap ranks.
uint64_t orc_space_neighbors(const void* p, const uint8_t* row, int rule, uint32_t* out, uint64_t cap) {
    const Space* s = (const Space*)p;
    std::vector<uint32_t> nb = list_neighbors(*s, row, rule);
    for (uint64_t i = 0; i < nb.size() && i < cap; ++i) out[i] = nb[i];
    return nb.size();
}
// mode 1: index-distance (L270); 2: Alg.2 with positions x (count x n floats); 3: Alg.3 with draws w (count words).
// rank = 0xFFFFFFFF when every neighbour set is empty; rule = set used (0/1/2, 3 none, 255 n/a); valid rows map to themselves.
void orc_space_repair_mode(const void* p, int mode, const uint8_t* rows, const float* x, const uint32_t* w, uint64_t count,
                           uint32_t* rank, uint8_t* rule) {
    const Space* s = (const Space*)p;
    for (uint64_t i = 0; i < count; ++i) {
        const uint8_t* c = rows + i * s->n;
        int ru = 255; uint32_t rk;
        if (in_domain(*s, c) && s->bit(s->lin(c))) rk = s->rank_of(s->lin(c));
        else if (mode == 1) rk = repair_index_distance(*s, c).rank;
        else if (mode == 2) rk = repair_alg2(*s, c, x + i * s->n, &ru);
        else rk = repair_alg3(*s, c, w[i], &ru);
        rank[i] = rk; if (rule) rule[i] = (uint8_t)ru;
    }
}
int orc_de_mutate_variant(int op, float F, int xi, int best, const int* r, int top) { return de_mutate_variant(op, F, xi, best, r, top); }
// LHS rows (P x n) of run `run_id` for (seed, stream INIT, generation 0) on this space (pins of A35).
void orc_lhs_rows(const void* sp, uint64_t seed, uint32_t run_id, int32_t pop, uint8_t* out) {
    Runs rs; rs.s = (const Space*)sp; rs.P = pop; rs.seed = seed; rs.algo = A_DE;
    Run r; r.id = run_id;
    std::vector<uint8_t> rows;
    lhs_rows(rs, r, S_INIT, 0, rows);
    std::copy(rows.begin(), rows.end(), out);
}
// ---- NEXT-4
double orc_baseline(const void* p, uint64_t t) {
    const Space* s = (const Space*)p;
    std::vector<float> sorted = s->obj; std::sort(sorted.begin(), sorted.end());
    return baseline_at(sorted, t);
}
uint64_t orc_baseline_budget(const void* p, double frac) {
    const Space* s = (const Space*)p;
    std::vector<float> sorted = s->obj; std::sort(sorted.begin(), sorted.end());
    return baseline_budget(sorted, frac);
}
// per_t[s] = mean over the runs of P_t at t[s]; returns their mean over s (Eq.2 for one search space).
double orc_runs_score(const void* p, const uint64_t* t, uint32_t S, double* per_t) {
    const Runs* rs = (const Runs*)p;
    std::vector<float> sorted = rs->s->obj; std::sort(sorted.begin(), sorted.end());
    double total = 0.0;
    for (uint32_t q = 0; q < S; ++q) {
        double acc = 0.0;
        for (uint32_t k = 0; k < rs->R; ++k) acc += score_run_at(*rs, sorted, k, t[q]);
        acc /= (double)rs->R;
        if (per_t) per_t[q] = acc;
        total += acc;
    }
    return S ? total / (double)S : 0.0;
}
// State copies, [run][ind][dim] / [run][ind]; which = 0 idx(u8) 1 rank(u32) 2 f(f32) 3 x 4 v 5 pbest 6 pbest_f
void orc_runs_state(const void* p, int which, void* out) {
    const Runs* rs = (const Runs*)p;
    uint8_t* o = (uint8_t*)out;
    for (uint32_t k = 0; k < rs->R; ++k) {
        const Run& r = rs->run[k];
        const void* src = nullptr; size_t bytes = 0;
        switch (which) {
            case 0: src = r.idx.data(); bytes = r.idx.size(); break;
            case 1: src = r.rank.data(); bytes = r.rank.size() * 4; break;
            case 2: src = r.f.data(); bytes = r.f.size() * 4; break;
            case 3: src = r.x.data(); bytes = r.x.size() * 4; break;
            case 4: src = r.v.data(); bytes = r.v.size() * 4; break;
            case 5: src = r.pb.data(); bytes = r.pb.size() * 4; break;
            case 6: src = r.pbf.data(); bytes = r.pbf.size() * 4; break;
        }
        if (bytes) std::memcpy(o, src, bytes);
        o += bytes;
    }
}

}  // extern "C"

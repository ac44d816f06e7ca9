"""Pins of the SURVEY 8(f) rows in the oracle (NEXT-1 paper-verbatim repairs, NEXT-2 non-constraint-aware variants,
NEXT-3 operator variants and LHS, NEXT-4 performance score): hand-worked values on cfg0 (tests/golden/neighbors_cfg0.txt),
itertools / numpy brute force on tiny spaces, closed forms and special cases, invariants of the paper."""
import itertools
import os
from fractions import Fraction
from math import comb
import numpy as np
import pytest

import oracle as O
import workloads as W
from conftest import oracle_space

GOLD = os.path.join(os.path.dirname(__file__), "golden", "neighbors_cfg0.txt")
NONE = 0xFFFFFFFF


def _gold():
    nb, idx, alg2, alg3 = [], [], [], []
    for ln in open(GOLD):
        if ln.startswith("#") or not ln.strip():
            continue
        kind, rest = ln.split(None, 1)
        if kind == "nb":
            left, right = rest.split(":")
            i, j, t, rule = (int(x) for x in left.split())
            nb.append(((i, j, t), rule, [int(x) for x in right.split()]))
        elif kind == "idx":
            left, right = rest.split("->")
            idx.append((tuple(int(x) for x in left.split()), int(right)))
        elif kind == "alg2":
            left, right = rest.split("->")
            r = right.split()
            alg2.append(([float(x) for x in left.split()], tuple(int(x) for x in r[:3]), int(r[3]), int(r[4])))
        elif kind == "alg3":
            left, right = rest.split("->")
            l = left.split()
            alg3.append((tuple(int(x) for x in l[:3]), int(l[3], 16), int(right)))
    return nb, idx, alg2, alg3


# ------------------------------------------------------------------------------------------------ NEXT-1
def test_worked_neighbour_sets_and_repairs_cfg0():
    sp, s = oracle_space(0)
    Lt = s.Ltab()
    nb, idx, alg2, alg3 = _gold()
    assert len(nb) == 7 and len(idx) == 3 and len(alg2) == 3 and len(alg3) == 4
    for c, rule, want in nb:
        assert list(Lt[s.neighbors(c, rule)]) == want, (c, rule)
    for c, want in idx:
        assert int(Lt[s.repair_mode("index", [c])[0][0]]) == want
    for x, snapped, rule, want in alg2:
        c = [O.snap(max(sp.m), m, v) for v, m in zip(x, sp.m)]
        assert tuple(c) == snapped
        rk, ru = s.repair_mode("alg2", [c], x=[x])
        assert (int(Lt[rk[0]]), int(ru[0])) == (want, rule)
    for c, w, want in alg3:
        rk, _ = s.repair_mode("alg3", [c], w=[w])
        assert int(Lt[rk[0]]) == want


def _gapped_space():
    """x in {1..5} but only x in {1,5} is feasible; y in {1,2,3}; (x, y) = (1, 1) and (5, 3) infeasible."""
    from workloads.rpn import P, OR, AND, NOT
    doms = [[1, 2, 3, 4, 5], [1, 2, 3]]
    rpn = [OR(P(0).eq(1), P(0).eq(5)).program(),
           NOT(OR(AND(P(0).eq(1), P(1).eq(1)), AND(P(0).eq(5), P(1).eq(3)))).program()]
    return O.OracleSpace(doms, rpn).build()


def test_adjacent_skips_values_that_never_occur_in_a_valid_configuration():
    # L141: "the nearest previous/next value that gives a valid configuration" (A28).  x = 3 (index 2), y = 2 (index 1):
    # indices 1, 2, 3 of x occur in no valid configuration, so the strictly-adjacent set is empty, while the adjacent
    # rule reaches x index 0 and 4 and y index 0, 1, 2: valid rows (0,1) (0,2) (4,0) (4,1)  [(0,0) and (4,2) are infeasible].
    s = _gapped_space()
    assert s.V == 4
    rows = s.rows()
    assert s.neighbors([2, 1], 0).size == 0
    assert sorted(map(tuple, rows[s.neighbors([2, 1], 1)])) == [(0, 1), (0, 2), (4, 0), (4, 1)]
    assert sorted(map(tuple, rows[s.neighbors([2, 1], 2)])) == [(0, 1), (4, 1)]        # Hamming: only x changes
    # cascade: Alg.3 picks from the adjacent set (rule 1), Alg.2 the Euclidean-nearest of it
    rk, ru = s.repair_mode("alg3", [[2, 1]] * 4, w=[0, 1 << 30, 1 << 31, 3 << 30])
    assert list(ru) == [1] * 4 and sorted(map(tuple, rows[rk])) == [(0, 1), (0, 2), (4, 0), (4, 1)]
    x = np.array([[0.55, 0.30]], np.float32)                   # coord = k/4: nearest of the four is (4,1) = (1.0, .25)
    rk, ru = s.repair_mode("alg2", [[2, 1]], x=x)
    assert tuple(rows[rk[0]]) == (4, 1) and ru[0] == 1
    # a row whose three sets are all empty stays unrepaired (Alg.2 L18, Alg.3 L7): single-row space
    from workloads.rpn import P
    s1 = O.OracleSpace([[1, 2, 3, 4, 5, 6, 7]], [(P(0).eq(1)).program()]).build()
    # value 7 (index 6): strictly-adjacent {5} invalid; adjacent: nearest present below = index 0 -> valid row (0,)
    assert list(s1.repair_mode("alg3", [[6]], w=[5])[0]) == [0]
    s2 = O.OracleSpace([[1, 2], [1, 2]], [(P(0) + P(1)).eq(2).program()]).build()     # only (1,1) valid
    # (2,2) = idx (1,1): strictly adjacent to (0,0) -> repaired by rule 0
    assert list(s2.repair_mode("alg3", [[1, 1]], w=[0])[1]) == [0]


@pytest.mark.parametrize("seed", range(24))
def test_neighbour_rules_and_repairs_against_itertools(seed):
    sp = W.random_tiny_space(seed, max_N=1500)
    s = O.OracleSpace.from_space(sp).build()
    doms, m, n = sp.domains, sp.m, sp.n
    stride = [int(np.prod(m[d + 1:])) for d in range(n)]
    lin = lambda r: sum(int(a) * b for a, b in zip(r, stride))
    allrows = list(itertools.product(*[range(k) for k in m]))
    valid = [r for r in allrows if all(p([doms[d][r[d]] for d in range(n)]) for p in sp.preds)]
    assert len(valid) == s.V
    if not valid:
        return
    present = [{r[d] for r in valid} for d in range(n)]
    rng = np.random.default_rng(seed)
    invalid = [r for r in allrows if r not in set(valid)]
    if not invalid:
        return
    Lt = s.Ltab()
    M = max(m)
    for c in [invalid[i] for i in rng.choice(len(invalid), size=min(12, len(invalid)), replace=False)]:
        lo = [max([k for k in present[d] if k < c[d]], default=None) for d in range(n)]
        hi = [min([k for k in present[d] if k > c[d]], default=None) for d in range(n)]
        sets = [
            [v for v in valid if all(abs(v[d] - c[d]) <= 1 for d in range(n))],
            [v for v in valid if all(v[d] in (c[d], lo[d], hi[d]) for d in range(n))],
            [v for v in valid if sum(v[d] != c[d] for d in range(n)) == 1],
        ]
        for rule in range(3):
            assert list(Lt[s.neighbors(c, rule)]) == sorted(lin(v) for v in sets[rule]), (c, rule)
        # index distance
        want = min(valid, key=lambda v: (sum(abs(v[d] - c[d]) for d in range(n)), lin(v)))
        assert int(Lt[s.repair_mode("index", [c])[0][0]]) == lin(want)
        # cascade
        first = next((q for q in range(3) if sets[q]), 3)
        w = int(rng.integers(0, 2 ** 32))
        rk, ru = s.repair_mode("alg3", [c], w=[w])
        if first == 3:
            assert rk[0] == NONE and ru[0] == 3
        else:
            members = sorted(sets[first], key=lin)
            assert int(Lt[rk[0]]) == lin(members[(w * len(members)) >> 32]) and ru[0] == first
            x = (np.array(c, np.float32) / np.float32(max(M - 1, 1)) + rng.uniform(-0.08, 0.08, n).astype(np.float32)).astype(np.float32)
            def dist(v):
                acc = np.float32(0)
                for d in range(n):
                    cv = np.float32(v[d]) / np.float32(M - 1) if M > 1 else np.float32(0)
                    df = np.float32(cv - x[d]); acc = np.float32(acc + np.float32(df * df))
                return acc
            best = min(members, key=lambda v: (dist(v), lin(v)))
            rk, ru = s.repair_mode("alg2", [c], x=[x])
            assert int(Lt[rk[0]]) == lin(best) and ru[0] == first


def test_paper_repairs_are_the_identity_on_valid_rows():
    sp, s = oracle_space(0)
    rows = s.rows()
    for mode, kw in (("index", {}), ("alg2", dict(x=np.zeros((len(rows), 3)))), ("alg3", dict(w=np.arange(len(rows))))):
        rk, _ = s.repair_mode(mode, rows, **kw)
        assert np.array_equal(rk, np.arange(len(rows)))          # Alg.1 L205 / Alg.3: valid configurations are kept


# ------------------------------------------------------------------------------------------------ NEXT-3
def test_de_mutation_variants_closed_forms():
    F = np.float32(0.7)
    rng = np.random.default_rng(1)
    f32 = np.float32
    for _ in range(400):
        xi, best = int(rng.integers(0, 16)), int(rng.integers(0, 16))
        r = [int(v) for v in rng.integers(0, 16, 5)]
        top = int(rng.integers(1, 16))
        forms = {
            "best1": f32(f32(best) + f32(F * f32(r[0] - r[1]))),
            "rand1": f32(f32(r[0]) + f32(F * f32(r[1] - r[2]))),
            "currenttobest1": f32(f32(f32(xi) + f32(F * f32(best - xi))) + f32(F * f32(r[0] - r[1]))),
            "randtobest1": f32(f32(f32(r[0]) + f32(F * f32(best - r[0]))) + f32(F * f32(r[1] - r[2]))),
            "best2": f32(f32(f32(best) + f32(F * f32(r[0] - r[1]))) + f32(F * f32(r[2] - r[3]))),
            "rand2": f32(f32(f32(r[0]) + f32(F * f32(r[1] - r[2]))) + f32(F * f32(r[3] - r[4]))),
        }
        for op, mf in forms.items():
            want = int(min(max(int(np.rint(mf)), 0), top))        # numpy rint = half-to-even (A8)
            assert O.de_mutate_variant(op, 0.7, xi, best, r, top) == want, (op, xi, best, r)
    # best1 through the variant routine equals O5's pinned de_mutate_index
    for a in range(8):
        for b in range(8):
            assert O.de_mutate_variant("best1", 0.7, 0, 3, [a, b], 7) == O.de_mutate_index(0.7, 3, a, b, 7)


def _de_runs(s, **kw):
    var = O.Variant.make(**{k: v for k, v in kw.items() if k in ("de_mutation", "de_crossover", "aware", "repair_mode", "init_lhs")})
    hp = O.HParams.default()
    if "CR" in kw:
        hp.de_CR = kw["CR"]
    return O.OracleRuns(s, "de", n_runs=kw.get("R", 6), pop=kw.get("P", 12), max_gens=8, seed=kw.get("seed", 3), hparams=hp, variant=var)


@pytest.mark.parametrize("mut", ["best1", "rand1", "currenttobest1", "randtobest1", "best2", "rand2"])
def test_de_exponential_crossover_special_cases(mut):
    sp, s = oracle_space(1)
    n = sp.n
    # CR = 0: exactly the j_rand gene comes from the mutant -> the trial differs from x_i in at most one parameter
    r = _de_runs(s, de_mutation=mut, de_crossover="exp", CR=0.0)
    before = r.state()["idx"].copy()
    r.step(1)
    cand = r.taps()["cand"]
    assert ((cand != before).sum(axis=2) <= 1).all()
    # CR = 1 (u01 < 1 always): the whole mutant is taken, for binomial and exponential alike -> identical trials
    ra = _de_runs(s, de_mutation=mut, de_crossover="exp", CR=1.0); ra.step(1)
    rb = _de_runs(s, de_mutation=mut, de_crossover="bin", CR=1.0); rb.step(1)
    assert np.array_equal(ra.taps()["cand"], rb.taps()["cand"])
    # in between: the genes taken from the mutant form one cyclic run (exponential) -- checked where mutant != x_i
    rc = _de_runs(s, de_mutation=mut, de_crossover="exp", CR=0.6)
    before = rc.state()["idx"].copy()
    rc.step(1)
    cand, mutant = rc.taps()["cand"], ra.taps()["cand"]           # same seed: ra's trials are the full mutants
    for k in range(cand.shape[0]):
        for i in range(cand.shape[1]):
            took = [d for d in range(n) if cand[k, i, d] != before[k, i, d]]
            assert all(cand[k, i, d] == mutant[k, i, d] for d in took)
            if took:                                              # contained in a cyclic window no longer than the run
                span = min(max((d - s0) % n for d in took) for s0 in took)
                assert span < n


def test_de_donors_are_distinct_and_not_the_target():
    # with F = 0 the mutant is the base vector itself: rand1 -> x_r0, currenttobest1 -> x_i, best1 -> best
    sp, s = oracle_space(1)
    hp = O.HParams.default(); hp.de_F = 0.0; hp.de_CR = 1.0
    for mut, base in (("rand1", "donor"), ("rand2", "donor"), ("currenttobest1", "self"), ("best2", "best")):
        r = O.OracleRuns(s, "de", n_runs=8, pop=10, max_gens=4, seed=5, hparams=hp, variant=O.Variant.make(de_mutation=mut))
        before = r.state()["idx"].copy()
        best_rank = r.best()["best_rank"].copy()
        r.step(1)
        cand = r.taps()["cand"]
        for k in range(8):
            for i in range(10):
                if base == "self":
                    assert np.array_equal(cand[k, i], before[k, i])
                elif base == "best":
                    assert np.array_equal(cand[k, i], s.rows()[best_rank[k]])
                else:
                    others = [j for j in range(10) if j != i and np.array_equal(before[k, j], cand[k, i])]
                    assert others, "the rand base vector must be another member of the population"


@pytest.mark.parametrize("xo", ["two_point", "uniform", "disruptive_uniform"])
def test_ga_crossover_variants(xo):
    sp, s = oracle_space(1)
    n, P, B = sp.n, 16, 3
    hp = O.HParams.default(); hp.ga_mutation_chance = 1 << 30          # (almost) never mutate
    r = O.OracleRuns(s, "ga", n_runs=12, pop=P, max_gens=3, seed=11, hparams=hp, variant=O.Variant.make(ga_crossover=xo))
    st = r.state()
    idx, f = st["idx"].copy(), st["f"].copy()
    r.step(1)
    cand = r.taps()["cand"]
    stride = [int(np.prod(sp.m[d + 1:])) for d in range(n)]
    frac_b = []
    for k in range(12):
        L = (idx[k].astype(np.int64) * np.array(stride)).sum(axis=1)
        order = sorted(range(P), key=lambda a: (f[k, a].view(np.uint32), L[a], a))
        for i in range(P):
            dr = lambda slot: O.draw(11, k, 1, i, "op", slot)
            sa = min(O.below(dr(q), P) for q in range(B)); sb = min(O.below(dr(B + q), P) for q in range(B))
            if sb == sa:
                sb = (sa + 1) % P
            A, Bp = idx[k, order[sa]], idx[k, order[sb]]
            child = cand[k, i]
            assert all(child[d] in (A[d], Bp[d]) for d in range(n))
            differ = [d for d in range(n) if A[d] != Bp[d]]
            fromB = [d for d in differ if child[d] == Bp[d]]
            if xo == "two_point":                                       # B's genes form one contiguous window
                c1, c2 = O.below(dr(2 * B), n + 1), O.below(dr(2 * B + 1), n + 1)
                lo, hi = min(c1, c2), max(c1, c2)
                assert all((lo <= d < hi) == (child[d] == Bp[d]) for d in differ)
            if xo == "disruptive_uniform":                              # at least half of the differing genes are swapped
                assert len(fromB) >= (len(differ) + 1) // 2
            if differ:
                frac_b.append(len(fromB) / len(differ))
    if xo == "uniform":
        assert 0.4 < np.mean(frac_b) < 0.6
    if xo == "disruptive_uniform":
        assert np.mean(frac_b) > 0.55


def test_lhs_strata_are_each_hit_once():
    # P a multiple of every m_d: value k of dimension d owns P/m_d strata, so it is drawn exactly P/m_d times (L223, A35)
    sp, s = oracle_space(0)                                             # m = (5, 6, 4)
    for run in range(5):
        rows = s.lhs_rows(seed=7, run_id=run, pop=60)
        for d, md in enumerate(sp.m):
            assert np.array_equal(np.bincount(rows[:, d], minlength=md), np.full(md, 60 // md))
    # general P: individual with stratum j lands in [floor(j m / P), floor((j+1) m / P)], every stratum used once
    rows = s.lhs_rows(seed=7, run_id=0, pop=7)
    for d, md in enumerate(sp.m):
        srt = np.sort(rows[:, d])
        for j in range(7):
            assert (j * md) // 7 <= srt[j] <= min(((j + 1) * md) // 7, md - 1)


def test_lhs_population_is_valid_and_distinct():
    sp, s = oracle_space(1)
    r = O.OracleRuns(s, "de", n_runs=10, pop=24, max_gens=2, seed=2, variant=O.Variant.make(init_lhs=True))
    st = r.state()
    for k in range(10):
        assert len(set(st["rank"][k])) == 24                            # L223 "valid candidates", O4 distinct
        assert all(s.is_valid(row) for row in st["idx"][k])
    # the LHS points themselves, where valid, are kept as they are (repair is the identity on valid rows)
    pts = s.lhs_rows(seed=2, run_id=0, pop=24)
    kept = sum(1 for i in range(24) if s.is_valid(pts[i]) and np.array_equal(pts[i], st["idx"][0, i]))
    assert kept >= sum(1 for i in range(24) if s.is_valid(pts[i])) - 2  # minus collisions moved by linear probing


# ------------------------------------------------------------------------------------------------ NEXT-2
@pytest.mark.parametrize("algo", ["de", "pso", "firefly", "ga"])
def test_unaware_variant_never_repairs_and_penalises_invalid(algo):
    sp, s = oracle_space(1)
    r = O.OracleRuns(s, algo, n_runs=6, pop=16, max_gens=12, seed=4, variant=O.Variant.make(aware=False, penalty=1e20))
    st = r.state()
    # L272 / L284: random initial population -- not restricted to valid configurations (density 18 %)
    n_valid0 = int((st["rank"] != NONE).sum())
    assert 0 < n_valid0 < 6 * 16
    assert np.all(st["f"][st["rank"] == NONE] == np.float32(1e20))
    tot_pen = 6 * 16 - n_valid0
    for g in range(1, 13):
        r.step(1)
        t = r.taps()
        act = t["active"].astype(bool)
        valid = t["valid"].astype(bool)[act]
        if algo != "ga":                                                # (GA may still mutate after the validity test)
            assert np.all(t["eval_rank"][act][~valid] == NONE)
            assert np.all(t["f"][act][~valid] == np.float32(1e20))
            for k in np.nonzero(act)[0]:                                # no repair: a valid candidate is evaluated as it is
                for i in range(16):
                    if t["valid"][k, i]:
                        assert np.array_equal(s.rows()[t["eval_rank"][k, i]], t["cand"][k, i])
        assert np.all(t["rep_rank"][act][~valid] == NONE)
    b = r.best()
    traj = r.trajectory()
    assert np.all(np.diff(traj["uniq"].astype(np.int64), axis=0) >= 0)
    # only valid configurations are ever evaluated (L135): every evaluated rank indexes the valid table; penalised ones do not count
    assert r.n_evaluated + r.n_penalised >= 6 * 16 * 13 and r.n_penalised > tot_pen
    assert np.all(b["uniq"] <= r.n_evaluated)
    # best-so-far only ever holds a valid configuration, or nothing
    ok = b["best_rank"] != NONE
    assert np.all(b["best_f"][ok] == s._obj[b["best_rank"][ok]]) and np.all(b["best_f"][~ok] == np.float32(1e20))


def test_aware_beats_unaware_on_a_sparse_space():
    # the paper's headline (L405-411): constraint-awareness helps, most on sparse spaces.  Same budget of generations.
    sp, s = oracle_space(1)
    gain = []
    for algo in ("pso", "ga"):
        fa = O.OracleRuns(s, algo, n_runs=20, pop=16, max_gens=15, seed=1)
        fu = O.OracleRuns(s, algo, n_runs=20, pop=16, max_gens=15, seed=1, variant=O.Variant.make(aware=False))
        fa.step(15); fu.step(15)
        gain.append(np.median(fu.best()["best_f"]) - np.median(fa.best()["best_f"]))
    assert all(g > 0 for g in gain)


@pytest.mark.parametrize("algo", ["de", "pso", "firefly", "ga"])
def test_paper_repair_mode_invariants(algo):
    sp, s = oracle_space(1)
    r = O.OracleRuns(s, algo, n_runs=4, pop=16, max_gens=6, seed=9, variant=O.Variant.make(repair_mode=1))
    rows = s.rows()
    for g in range(6):
        before = r.state()
        r.step(1)
        t = r.taps()
        for k in range(4):
            for i in range(16):
                c, rk = t["cand"][k, i], t["rep_rank"][k, i]
                if t["valid"][k, i]:
                    assert np.array_equal(rows[rk], c) and t["rule"][k, i] == 255
                    continue
                if algo == "de":                                        # L270: nearest by the sum of index differences
                    want, _ = s.repair_mode("index", [c])
                    assert rk == want[0]
                    continue
                rule = t["rule"][k, i]
                if rk == NONE:
                    assert rule == 3 and all(s.neighbors(c, q).size == 0 for q in range(3))
                    assert t["f"][k, i] == np.float32(1e20) or algo == "ga"
                    continue
                assert all(s.neighbors(c, q).size == 0 for q in range(rule)) and rk in s.neighbors(c, rule)
        if algo in ("pso", "firefly"):                                  # L282: the repair does not move the particle
            x = r.state()["x"]
            M = max(sp.m)
            snapped = np.array([[[O.snap(M, sp.m[d], float(x[k, i, d])) for d in range(sp.n)] for i in range(16)] for k in range(4)])
            assert np.array_equal(snapped, t["cand"])


# ------------------------------------------------------------------------------------------------ NEXT-4
def test_baseline_closed_forms_and_brute_force():
    from workloads.rpn import P
    s = O.OracleSpace([[1, 2, 3, 4, 5, 6, 7, 8, 9]], []).build()
    obj = np.array([5.0, 3.0, 9.0, 1.5, 7.25, 2.0, 8.0, 4.0, 6.0], np.float32)
    s.set_objective(obj)
    V = 9
    assert s.baseline(1) == pytest.approx(float(obj.astype(np.float64).mean()), rel=1e-14)   # one draw: the mean
    assert s.baseline(V) == pytest.approx(1.5, rel=1e-14)                                   # all drawn: the optimum
    srt = sorted(float(v) for v in obj)
    for t in range(1, V + 1):                                       # expected minimum over all C(V,t) subsets, exact rationals
        want = sum(Fraction(min(c)) for c in itertools.combinations(srt, t)) / comb(V, t)
        assert s.baseline(t) == pytest.approx(float(want), rel=1e-13)
    # budget (L361): first t whose baseline is within 5 % of the median-optimum distance from the optimum
    med, opt = srt[(V - 1) // 2], srt[0]
    want_t = next(t for t in range(1, V + 1)
                  if float(sum(Fraction(min(c)) for c in itertools.combinations(srt, t)) / comb(V, t)) <= med - 0.95 * (med - opt))
    assert s.baseline_budget(0.95) == want_t


def test_score_special_cases_and_direct_evaluation():
    sp, s = oracle_space(0)
    obj = s._obj
    r = O.OracleRuns(s, "ga", n_runs=12, pop=8, max_gens=10, seed=0)
    r.step(10)
    traj = r.trajectory()
    ts = [8, 10, 14, 20, 30]
    score, per = r.score(ts)
    fopt = float(obj.min())
    want = []
    for t in ts:
        B = s.baseline(t)
        acc = 0.0
        for k in range(12):
            g = max([gg for gg in range(11) if traj["uniq"][gg, k] <= t], default=0)
            acc += (B - float(traj["best_f"][g, k])) / (B - fopt)
        want.append(acc / 12)
    assert per == pytest.approx(want, rel=1e-12) and score == pytest.approx(np.mean(want), rel=1e-12)
    # a run that holds the optimum from generation 0 scores exactly 1 at every sampling point (L361)
    best_rank = int(np.argmin(obj))
    for seed in range(200):
        r1 = O.OracleRuns(s, "ga", n_runs=1, pop=8, max_gens=1, seed=seed)
        if r1.best()["best_rank"][0] == best_rank:
            r1.step(1)
            assert r1.score([8, 9, 12])[0] == pytest.approx(1.0, abs=1e-12)
            break
    else:
        pytest.skip("no seed starts at the optimum")
    # t = V: B(V) is the optimum itself (every draw taken), the quotient would be x/0; A36: 1 for runs that hold the optimum, else 0
    V = s.V
    assert s.baseline(V) == fopt
    scV, perV = r.score([V])
    g_last = [max(gg for gg in range(11) if traj["uniq"][gg, k] <= V) for k in range(12)]
    wantV = np.mean([1.0 if float(traj["best_f"][g_last[k], k]) == fopt else 0.0 for k in range(12)])
    assert np.isfinite(perV).all() and perV[0] == wantV and scV == wantV
    assert np.isfinite(r.score([8, V, 10 * V])[0])
    # a run stuck at the baseline value scores 0: uniform-random search itself averages to ~0 over many runs
    ru = O.OracleRuns(s, "ga", n_runs=400, pop=8, max_gens=0, seed=5)     # generation 0 = 8 uniform valid draws
    sc, _ = ru.score([8])
    assert abs(sc) < 0.08

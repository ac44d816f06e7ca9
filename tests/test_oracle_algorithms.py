"""Pins of the four generation steps (O4-O8, O10): the independent-prototype values of SURVEY.md 8(c)
and the invariants the paper fixes.  Parity of these heuristics with the *paper* is unpinned."""
import os
import zlib
import numpy as np
import pytest

import oracle as O
import workloads as W
from conftest import oracle_space

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _gold():
    out = {}
    with open(os.path.join(GOLD, "prototype_cfg0.txt")) as fh:
        for ln in fh:
            if ln.startswith("#") or not ln.strip():
                continue
            k, *rest = ln.split()
            out[k] = rest
    return out


def _cfg0_space_with_test_objective():
    sp = W.space_cfg0()
    s = O.OracleSpace.from_space(sp).build()
    s.set_objective(W.test_objective_37(s.V))
    return sp, s


@pytest.mark.parametrize("algo", ["de", "ga", "pso", "firefly"])
def test_prototype_values_cfg0(algo):
    g = _gold()
    sp, s = _cfg0_space_with_test_objective()
    r = O.OracleRuns(s, algo, n_runs=100, pop=20, budget=0, max_gens=50, seed=0)
    if algo == "de":
        assert [int(x) for x in r.state()["rank"][0]] == [int(x) for x in g["gen0_ranks_run0"]]
    r.step(50)
    t = r.trajectory()
    crc = 0
    for k in range(100):
        crc = zlib.crc32(np.ascontiguousarray(t[:, k]).tobytes(), crc)
    b = r.best()
    rep, uniq, nf1, sbr, want_crc = g[algo]
    assert r.n_repaired == int(rep)
    assert int(b["uniq"].sum()) == int(uniq)
    assert int((b["best_f"] == 1.0).sum()) == int(nf1)
    assert int(b["best_rank"].sum()) == int(sbr)
    assert "%08x" % crc == want_crc
    if algo == "de":
        for item in g["traj_de_run0"]:
            gg, vals = item.split(":")
            f, rk, uq = (int(x) for x in vals.split(","))
            row = t[int(gg), 0]
            assert (float(row["best_f"]), int(row["best_rank"]), int(row["uniq"])) == (float(f), rk, uq)


def _hamming(a, b):
    return int((np.asarray(a) != np.asarray(b)).sum())


@pytest.mark.parametrize("algo", ["de", "ga", "pso", "firefly"])
@pytest.mark.parametrize("cfg", [0, 1])
def test_invariants(cfg, algo):
    sp, s = oracle_space(cfg)
    R, P, G = (12, 20, 25) if cfg == 0 else (2, 32, 3)
    rows, Ls = s.rows(), s.Ltab()
    obj = s._obj
    r = O.OracleRuns(s, algo, n_runs=R, pop=P, budget=0, max_gens=1000, seed=11)
    M = max(sp.m)
    prev_best = r.best()
    evaluated = np.full(R, P, np.int64)
    for g in range(1, G + 1):
        x_before = r.state().get("x")
        r.step(1)
        tp, st, b = r.taps(), r.state(), r.best()
        # only valid configurations are ever evaluated (L139, L270, L282): ranks index the valid table, f = obj[rank]
        assert (tp["eval_rank"] < s.V).all() and (tp["f"] == obj[tp["eval_rank"]]).all()
        for k in range(R):
            for i in range(P):
                c = tp["cand"][k, i]
                v = s.is_valid(c)
                assert bool(tp["valid"][k, i]) == v
                if v:                                        # repair is the identity on valid configs
                    assert (rows[tp["rep_rank"][k, i]] == c).all()
        evaluated += P
        # best-so-far never gets worse; uniq bounded by evaluations and V
        assert (b["best_f"] <= prev_best["best_f"]).all()
        assert (b["uniq"] <= np.minimum(evaluated + P * g, s.V)).all() and (b["uniq"] >= prev_best["uniq"]).all()
        assert (b["best_f"] == obj[b["best_rank"]]).all()
        prev_best = b
        if algo == "de":
            # L161/L223: the population never holds the same configuration twice
            for k in range(R):
                Lp = (st["idx"][k].astype(np.uint64) * np.array(_strides(sp.m), np.uint64)).sum(axis=1)
                assert len(set(Lp.tolist())) == P
                assert all(s.is_valid(row) for row in st["idx"][k])
        if algo in ("pso", "firefly"):
            # L282: the particle's own position is NOT replaced by the repaired configuration; the candidate is
            # the snap of the continuous position, whatever repair did for the evaluation
            for k in range(R):
                for i in range(P):
                    snapped = [O.snap(M, sp.m[d], float(st["x"][k, i, d])) for d in range(sp.n)]
                    assert snapped == [int(q) for q in tp["cand"][k, i]]
            hi = np.array([O.coord(M, mm - 1) for mm in sp.m], np.float32)
            assert (st["x"] >= 0).all() and (st["x"] <= hi[None, None, :]).all()
        if algo == "ga":
            # L288: population fully refreshed with valid children; L311: mutation = one valid Hamming-1 neighbour
            assert (st["rank"] == tp["eval_rank"]).all()
            for k in range(R):
                for i in range(P):
                    assert (st["idx"][k, i] == rows[tp["eval_rank"][k, i]]).all()
                    if tp["eval_rank"][k, i] != tp["rep_rank"][k, i]:
                        assert _hamming(rows[tp["eval_rank"][k, i]], rows[tp["rep_rank"][k, i]]) == 1


def _strides(m):
    st = [1] * len(m)
    for d in range(len(m) - 2, -1, -1):
        st[d] = st[d + 1] * m[d + 1]
    return st


def test_ga_parent_selection_is_beta_1_b():
    # min of b uniform positions has CDF 1 - (1 - x)^b over the sorted population (A18)
    b, Pn, trials = 3, 20, 30000
    counts = np.zeros(Pn)
    for t in range(trials):
        sa = min(O.below(O.draw(5, t, 1, 0, "op", q), Pn) for q in range(b))
        counts[sa] += 1
    edges = np.arange(Pn + 1) / Pn
    expect = trials * ((1 - edges[:-1]) ** b - (1 - edges[1:]) ** b)
    chi2 = ((counts - expect) ** 2 / expect).sum()
    assert chi2 < 60.0                                       # 19 dof, p ~ 1e-6 cut-off


def test_budget_freezes_runs_and_run_offset_is_a_pure_relabel():
    sp, s = oracle_space(0)
    a = O.OracleRuns(s, "de", n_runs=6, pop=20, budget=40, max_gens=30, seed=3)
    a.step(35)
    t = a.trajectory()
    b = a.best()
    assert (b["gens_done"] <= 30).all() and (b["uniq"] < 40 + 20).all()      # overshoot < P (A20)
    for k in range(6):
        gd = int(b["gens_done"][k])
        assert (t[gd:, k] == t[gd, k]).all()                 # frozen rows repeat
        if gd < 30:
            assert t[gd, k]["uniq"] >= 40 and (gd == 0 or t[gd - 1, k]["uniq"] < 40)
    # runs are keyed by global run index: a shard [2, 6) reproduces runs 2..5 exactly
    c = O.OracleRuns(s, "de", n_runs=4, pop=20, budget=40, max_gens=30, seed=3, first_run=2)
    c.step(35)
    assert (c.trajectory() == t[:, 2:6]).all()


def test_de_stagnation_reinit_happens_and_keeps_best():
    # a 4-config valid set with P=4 cannot accept anything (every trial is already in X): re-init every 2nd generation
    s = O.OracleSpace([[1, 2, 3, 4, 5, 6]], [(W.P(0) < 5).program()]).build()      # x0 < 5  -> V = 4
    assert s.V == 4
    s.set_objective(np.array([4, 3, 2, 1], np.float32))
    r = O.OracleRuns(s, "de", n_runs=3, pop=4, budget=0, max_gens=10, seed=1)
    before = r.n_evaluated
    r.step(4)
    assert r.n_evaluated - before == 3 * (4 * 4 + 2 * 4)      # 4 generations of trials + 2 re-inits of 4
    assert (r.best()["best_f"] == 1.0).all() and (r.best()["uniq"] == 4).all()
    assert not r.taps()["accept"].any()

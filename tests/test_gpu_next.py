"""GPU parity, through the C ABI, of the SURVEY 8(f) rows against the CPU oracle on the same seeded inputs:
NEXT-1 paper-verbatim repairs (standalone and inside the runs), NEXT-2 non-constraint-aware variants, NEXT-3 operator
variants and LHS, NEXT-4 performance score.  Bit-exact everywhere (integers, fp32 and fp64 bit patterns)."""
import numpy as np
import pytest

import oracle as O
import workloads as W
from conftest import oracle_space

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu
NONE = 0xFFFFFFFF

_GPU_SPACES = {}


def gpu_space(cfg, os_, sp):
    import paper_2606_28372_b200 as cao
    if cfg not in _GPU_SPACES:
        _GPU_SPACES[cfg] = cao.Space.from_space(sp).build()
    g = _GPU_SPACES[cfg]
    g.set_objective(os_._obj)
    return g


def _np(t):
    return t.cpu().numpy()


def compare(gr, orr, n, taps=True):
    gt = _np(gr.trajectory()).view(np.uint32)
    ot = orr.trajectory()
    assert gt.shape[0] == orr.gen + 1
    assert np.array_equal(gt[:, :, 0], ot["best_f"].view(np.uint32))
    assert np.array_equal(gt[:, :, 1], ot["best_rank"])
    assert np.array_equal(gt[:, :, 2], ot["uniq"])
    gb, ob = gr.best(), orr.best()
    for key in ("best_f", "best_rank", "uniq", "gens_done"):
        assert np.array_equal(_np(gb[key]).view(np.uint32), ob[key].view(np.uint32)), key
    gs, os_ = gr.state(), orr.state()
    for key in os_:
        assert np.array_equal(np.ascontiguousarray(_np(gs[key])).view(np.uint8).reshape(-1), np.ascontiguousarray(os_[key]).view(np.uint8).reshape(-1)), key
    if taps and orr.gen > 0:
        gtp, otp = gr.taps(), orr.taps()
        act = otp["active"].astype(bool)
        assert np.array_equal(_np(gtp["active"]), otp["active"])
        assert np.array_equal(_np(gtp["cand"])[act][:, :, :n], otp["cand"][act])
        assert np.array_equal(_np(gtp["valid"])[act], otp["valid"][act])
        assert np.array_equal(_np(gtp["rep_rank"]).view(np.uint32)[act], otp["rep_rank"][act])
        assert np.array_equal(_np(gtp["eval_rank"]).view(np.uint32)[act], otp["eval_rank"][act])
        assert np.array_equal(_np(gtp["f"]).view(np.uint32)[act], otp["f"].view(np.uint32)[act])
        assert np.array_equal(_np(gtp["accept"])[act], otp["accept"][act])
        assert np.array_equal(_np(gr.rule_tap())[act], otp["rule"][act])
    st = gr.stats()
    assert st["n_repaired"] == orr.n_repaired
    assert st["n_penalised"] == orr.n_penalised
    assert st["n_evaluated"] - st["n_penalised"] == orr.n_evaluated


def run_pair(cfg, algo, R, P, gens, budget=0, seed=0, first_run=0, hp=None, **var):
    import paper_2606_28372_b200 as cao
    sp, os_ = oracle_space(cfg)
    g = gpu_space(cfg, os_, sp)
    kw = dict(n_runs=R, pop=P, budget=budget, max_gens=gens, seed=seed, first_run=first_run)
    orr = O.OracleRuns(os_, algo, hparams=hp, variant=O.Variant.make(**var), **kw)
    ghp = None if hp is None else cao.HParams(*[getattr(hp, f[0]) for f in hp._fields_])
    gr = cao.Runs(g, algo, hparams=ghp, variant=cao.Variant.make(**var), **kw)
    assert gr.mode == "phased"
    compare(gr, orr, sp.n)
    for _ in range(gens):
        gr.step(1); orr.step(1)
        compare(gr, orr, sp.n)
    return gr, orr


ALGOS = ["de", "pso", "firefly", "ga"]


# ------------------------------------------------------------------------------------------------ NEXT-2
@pytest.mark.parametrize("algo", ALGOS)
def test_unaware_cfg0(algo):
    gr, orr = run_pair(0, algo, R=24, P=20, gens=20, seed=1, aware=False)
    assert orr.n_penalised > 0


@pytest.mark.parametrize("algo", ALGOS)
def test_unaware_cfg1_budget(algo):
    run_pair(1, algo, R=6, P=32, gens=14, budget=150, seed=2, aware=False)


def test_unaware_cfg3_firefly_rows_of_32_bytes():
    run_pair(3, "firefly", R=2, P=24, gens=4, seed=0, aware=False)
    run_pair(3, "ga", R=2, P=24, gens=4, seed=0, aware=False)


def test_unaware_custom_penalty():
    run_pair(0, "pso", R=8, P=12, gens=6, seed=5, aware=False, penalty=12345.0)


# ------------------------------------------------------------------------------------------------ NEXT-1
@pytest.mark.parametrize("algo", ALGOS)
def test_paper_repair_cfg0(algo):
    gr, orr = run_pair(0, algo, R=24, P=20, gens=20, seed=3, repair_mode=1)
    assert orr.n_repaired > 0


@pytest.mark.parametrize("algo", ALGOS)
def test_paper_repair_cfg1(algo):
    run_pair(1, algo, R=3, P=16, gens=6, seed=4, repair_mode=1)


@pytest.mark.parametrize("algo", ["firefly", "ga", "de"])
def test_paper_repair_cfg3_sparse(algo):
    # 20 dimensions, 32-byte rows (operator outputs stay close to valid rows; the all-sets-empty outcome of Alg.2 L18 /
    # Alg.3 L7 is covered by the uniformly random rows of test_standalone_repair_modes[3])
    run_pair(3, algo, R=2, P=16, gens=3, seed=0, repair_mode=1)


def _invalid_rows(sp, os_, count, seed):
    rng = np.random.default_rng(seed)
    rows = []
    while len(rows) < count:
        r = [int(rng.integers(0, m)) for m in sp.m]
        if not os_.is_valid(r):
            rows.append(r)
    return np.array(rows, np.uint8)


@pytest.mark.parametrize("cfg,count", [(0, 28), (1, 48), (2, 24), (3, 24)])
def test_standalone_repair_modes(cfg, count):
    sp, os_ = oracle_space(cfg)
    g = gpu_space(cfg, os_, sp)
    if cfg == 0:                                             # every invalid row of the space + some valid ones
        import itertools
        rows = np.array([r for r in itertools.product(*[range(m) for m in sp.m]) if not os_.is_valid(r)], np.uint8)
        rows = np.concatenate([rows, os_.rows()[:5]])
    else:
        rows = np.concatenate([_invalid_rows(sp, os_, count, cfg), os_.rows()[[0, os_.V // 2, os_.V - 1]]])
    rng = np.random.default_rng(100 + cfg)
    M = max(sp.m)
    x = (rows.astype(np.float32) / np.float32(M - 1) + rng.uniform(-0.4 / (M - 1), 0.4 / (M - 1), rows.shape).astype(np.float32)).astype(np.float32)
    w = rng.integers(0, 2 ** 32, rows.shape[0], dtype=np.uint64).astype(np.uint32)
    for mode, kw in (("index", {}), ("alg2", dict(x=x)), ("alg3", dict(w=w))):
        ork, oru = os_.repair_mode(mode, rows, **kw)
        grk, gru = g.repair_mode(mode, rows, **kw)
        assert np.array_equal(_np(grk).view(np.uint32), ork), mode
        assert np.array_equal(_np(gru), oru), mode
        if cfg == 3 and mode != "index":
            assert (ork == NONE).sum() > 0 and (oru == 3).sum() == (ork == NONE).sum()      # Alg.2 L18 / Alg.3 L7


# seeds of random_tiny_space(seed, max_N=1500) with 0 < V < N (something to repair, something to repair to)
@pytest.mark.parametrize("seed", [3, 6, 9, 10, 14, 18, 23, 25, 26, 30, 31, 39, 41, 44, 50, 58])
def test_standalone_repair_modes_tiny_spaces(seed):
    import paper_2606_28372_b200 as cao
    import itertools
    sp = W.random_tiny_space(seed, max_N=1500)
    os_ = O.OracleSpace.from_space(sp).build()
    assert 0 < os_.V < sp.N
    g = cao.Space.from_space(sp).build()
    rows = np.array([r for r in itertools.product(*[range(m) for m in sp.m]) if not os_.is_valid(r)][:200], np.uint8)
    rng = np.random.default_rng(seed)
    M = max(max(sp.m), 2)
    x = (rows.astype(np.float32) / np.float32(M - 1) + rng.uniform(-0.1, 0.1, rows.shape).astype(np.float32)).astype(np.float32)
    w = rng.integers(0, 2 ** 32, rows.shape[0], dtype=np.uint64).astype(np.uint32)
    for mode, kw in (("index", {}), ("alg2", dict(x=x)), ("alg3", dict(w=w))):
        ork, oru = os_.repair_mode(mode, rows, **kw)
        grk, gru = g.repair_mode(mode, rows, **kw)
        assert np.array_equal(_np(grk).view(np.uint32), ork), mode
        assert np.array_equal(_np(gru), oru), mode


# ------------------------------------------------------------------------------------------------ NEXT-3
@pytest.mark.parametrize("mut", ["rand1", "currenttobest1", "randtobest1", "best2", "rand2"])
@pytest.mark.parametrize("xo", ["bin", "exp"])
def test_de_operator_variants(mut, xo):
    run_pair(0, "de", R=16, P=20, gens=16, seed=6, de_mutation=mut, de_crossover=xo)
    run_pair(1, "de", R=3, P=16, gens=5, seed=6, de_mutation=mut, de_crossover=xo)


def test_de_best1_exp():
    run_pair(1, "de", R=4, P=16, gens=8, seed=7, de_crossover="exp")


@pytest.mark.parametrize("xo", ["two_point", "uniform", "disruptive_uniform"])
def test_ga_crossover_variants(xo):
    run_pair(0, "ga", R=16, P=20, gens=16, seed=8, ga_crossover=xo)
    run_pair(1, "ga", R=4, P=32, gens=8, seed=8, ga_crossover=xo)
    run_pair(3, "ga", R=2, P=16, gens=3, seed=8, ga_crossover=xo)


def test_de_lhs_initial_population():
    run_pair(0, "de", R=24, P=20, gens=10, seed=9, init_lhs=True)
    run_pair(1, "de", R=6, P=32, gens=6, seed=9, init_lhs=True)
    run_pair(3, "de", R=2, P=24, gens=2, seed=9, init_lhs=True)


def test_combined_switches():
    run_pair(1, "de", R=4, P=16, gens=6, seed=10, repair_mode=1, de_mutation="rand1", de_crossover="exp", init_lhs=True)
    run_pair(1, "ga", R=4, P=16, gens=6, seed=10, repair_mode=1, ga_crossover="uniform")
    run_pair(1, "ga", R=4, P=16, gens=6, seed=10, aware=False, ga_crossover="two_point")
    run_pair(1, "de", R=4, P=16, gens=6, seed=10, aware=False, de_mutation="rand2", de_crossover="exp")


def test_variant_errors_and_modes():
    import paper_2606_28372_b200 as cao
    sp, os_ = oracle_space(0)
    g = gpu_space(0, os_, sp)
    with pytest.raises(cao.CaoError) as e:
        cao.Runs(g, "de", n_runs=2, pop=8, variant=cao.Variant(1, 7, 0, 0, 0, 0, 1e20, 0))
    assert e.value.code == -1
    with pytest.raises(cao.CaoError):
        cao.Runs(g, "pso", n_runs=2, pop=8, variant=cao.Variant.make(init_lhs=True))
    with pytest.raises(cao.CaoError):
        cao.Runs(g, "de", n_runs=2, pop=5, variant=cao.Variant.make(de_mutation="rand2"))      # needs 5 donors + 1
    with pytest.raises(cao.CaoError):
        cao.Runs(g, "de", n_runs=2, pop=8, variant=cao.Variant.make(penalty=0.0))
    r = cao.Runs(g, "ga", n_runs=2, pop=8, variant=cao.Variant.make(ga_crossover="uniform"))
    with pytest.raises(cao.CaoError):
        r.set_mode("fused")
    # the all-default variant is the north_star path (fused allowed) and has no rule tap
    r0 = cao.Runs(g, "ga", n_runs=2, pop=8, variant=cao.Variant.make())
    assert r0.mode == "fused"
    with pytest.raises(cao.CaoError):
        r0.rule_tap()


# ------------------------------------------------------------------------------------------------ NEXT-4
@pytest.mark.parametrize("cfg", [0, 1])
def test_sorted_objective_baseline_and_score(cfg):
    import paper_2606_28372_b200 as cao
    sp, os_ = oracle_space(cfg)
    g = gpu_space(cfg, os_, sp)
    srt = g.sorted_objective()
    assert np.array_equal(_np(srt).view(np.uint32), np.sort(os_._obj).view(np.uint32))
    V = os_.V
    ts = [1, 2, 5, 20, 33, min(200, V), V] if cfg == 0 else [1, 8, 64, 500, 1000]
    B = g.baseline(srt, ts)
    want = np.array([os_.baseline(t) for t in ts], np.float64)
    assert np.array_equal(_np(B).view(np.uint64), want.view(np.uint64))           # same fp64 operation order
    for algo, var in (("ga", {}), ("pso", dict(aware=False))):
        kw = dict(n_runs=40, pop=16, max_gens=12, seed=3)
        orr = O.OracleRuns(os_, algo, variant=O.Variant.make(**var), **kw); orr.step(12)
        gr = cao.Runs(g, algo, variant=cao.Variant.make(**var), **kw); gr.step(12)
        t = [16, 20, 30, 50, 80, 120, 200] if cfg else [16, 20, 30, 50, 80, V, 3 * V]   # B(t >= V) = f_opt: guarded quotient (A36)
        sc, per = gr.score(srt, t)
        osc, oper = orr.score(t)
        assert np.array_equal(_np(per).view(np.uint64), oper.view(np.uint64)), algo
        assert _np(sc).view(np.uint64)[0] == np.float64(osc).view(np.uint64)


def test_unaware_penalty_below_objective_values():
    """A penalty smaller than some objective values: the first valid configuration a run evaluates becomes its best-so-far
    whatever its value (the oracle's rule, A33), it does not have to beat the penalty."""
    gr, orr = run_pair(0, "pso", R=16, P=12, gens=8, seed=9, aware=False, penalty=0.5)
    assert (orr.best()["best_f"][orr.best()["best_rank"] != 0xFFFFFFFF] > 0.5).any()
    run_pair(0, "de", R=16, P=12, gens=8, seed=9, aware=False, repair_mode=1, penalty=0.5)

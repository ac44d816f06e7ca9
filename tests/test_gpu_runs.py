"""GPU parity, through the C ABI, of the batched generation step (S2-S7) against the CPU oracle on the same
seeded inputs: post-snap rows, validity flags, repaired ranks, evaluated ranks, f, accept flags, population
state (fp32 bit patterns), uniq, best-so-far and whole trajectories -- all bit-exact (north_star)."""
import numpy as np
import pytest

import oracle as O
import workloads as W
from conftest import oracle_space

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

_GPU_SPACES = {}


def gpu_space(cfg, os_, sp, objective=None):
    import paper_2606_28372_b200 as cao
    if cfg not in _GPU_SPACES:
        _GPU_SPACES[cfg] = cao.Space.from_space(sp).build()
    g = _GPU_SPACES[cfg]
    g.set_objective(os_._obj if objective is None else objective)
    return g


def _np(t):
    return t.cpu().numpy()


def compare(gr, orr, n, gen_taps=True):
    """Everything observable after a step."""
    gt = _np(gr.trajectory()).view(np.uint32)
    ot = orr.trajectory()
    G = orr.gen + 1
    assert gt.shape[0] == G
    assert np.array_equal(gt[:, :, 0], ot["best_f"].view(np.uint32))
    assert np.array_equal(gt[:, :, 1], ot["best_rank"])
    assert np.array_equal(gt[:, :, 2], ot["uniq"])
    gb, ob = gr.best(), orr.best()
    assert np.array_equal(_np(gb["best_f"]).view(np.uint32), ob["best_f"].view(np.uint32))
    assert np.array_equal(_np(gb["best_rank"]).view(np.uint32), ob["best_rank"])
    assert np.array_equal(_np(gb["uniq"]).view(np.uint32), ob["uniq"])
    assert np.array_equal(_np(gb["gens_done"]).view(np.uint32), ob["gens_done"])
    gs, os_ = gr.state(), orr.state()
    for key in os_:
        a, b = _np(gs[key]), os_[key]
        if a.dtype == np.float32:
            assert np.array_equal(a.view(np.uint32), b.view(np.uint32)), key
        else:
            assert np.array_equal(a.view(b.dtype) if a.dtype.itemsize == b.dtype.itemsize else a, b), key
    if gen_taps and orr.gen > 0:
        gtp, otp = gr.taps(), orr.taps()
        act = otp["active"].astype(bool)
        assert np.array_equal(_np(gtp["active"]), otp["active"])
        assert np.array_equal(_np(gtp["cand"])[act][:, :, :n], otp["cand"][act])
        assert np.array_equal(_np(gtp["valid"])[act], otp["valid"][act])
        assert np.array_equal(_np(gtp["rep_rank"]).view(np.uint32)[act], otp["rep_rank"][act])
        assert np.array_equal(_np(gtp["eval_rank"]).view(np.uint32)[act], otp["eval_rank"][act])
        assert np.array_equal(_np(gtp["f"]).view(np.uint32)[act], otp["f"].view(np.uint32)[act])
        assert np.array_equal(_np(gtp["accept"])[act], otp["accept"][act])
    c = gr.counters()
    assert c["n_repaired"] == orr.n_repaired and c["n_evaluated"] == orr.n_evaluated


def run_pair(cfg, algo, R, P, gens, budget=0, seed=0, first_run=0, step_sizes=None, objective=None, hp=None):
    import paper_2606_28372_b200 as cao
    sp, os_ = oracle_space(cfg)
    if objective is not None:
        os_.set_objective(objective)
    g = gpu_space(cfg, os_, sp, objective)
    kw = dict(n_runs=R, pop=P, budget=budget, max_gens=gens, seed=seed, first_run=first_run)
    orr = O.OracleRuns(os_, algo, hparams=hp, **kw)
    ghp = None if hp is None else cao.HParams(*[getattr(hp, f[0]) for f in hp._fields_])
    # both execution modes; fused at the automatic group width (small run counts: widened groups, Firefly with four lanes
    # per firefly) and at width 1 (the shape of a filled GPU)
    grs = [cao.Runs(g, algo, hparams=ghp, mode="fused", **kw), cao.Runs(g, algo, hparams=ghp, mode="fused", fused_width=1, **kw),
           cao.Runs(g, algo, hparams=ghp, mode="phased", **kw)]
    assert grs[1].fused_width == 1 and grs[0].fused_width == (4 if algo == "firefly" and sp.n <= 16 and P <= 64 else 2 if P <= 128 and not (algo == "firefly") else 1)
    for gr in grs:
        compare(gr, orr, sp.n)
    done = 0
    for k in (step_sizes or [1] * gens):
        k = min(k, gens - done)
        if k <= 0:
            break
        orr.step(k); done += k
        for gr in grs:
            gr.step(k)
            compare(gr, orr, sp.n)
    gr = grs[0]
    return gr, orr


@pytest.mark.parametrize("algo", ["de", "pso", "firefly", "ga"])
def test_cfg0_every_generation(algo):
    """BASELINE configs[0] shape (P=20, 50 generations, 100 runs), all four algorithms, compared after every generation."""
    run_pair(0, algo, R=100, P=20, gens=50)


@pytest.mark.parametrize("algo", ["de", "pso", "firefly", "ga"])
def test_cfg0_prototype_objective_whole_run(algo):
    """The integer-valued objective of the secondary pins (many exact f ties), stepped in ragged chunks."""
    sp, os_ = oracle_space(0)
    obj = W.test_objective_37(os_.V)
    try:
        run_pair(0, algo, R=100, P=20, gens=50, step_sizes=[1, 2, 7, 40], objective=obj)
    finally:
        os_.set_objective(W.objective_table(os_.rows(), sp.m, 0))


@pytest.mark.parametrize("algo", ["de", "pso", "firefly", "ga"])
def test_cfg1_budget_and_generation_cap(algo):
    """configs[1]: GEMM-like space, P=32, budget of unique evaluations, frozen runs repeat their trajectory row."""
    gr, orr = run_pair(1, algo, R=6, P=32, gens=24, budget=400, step_sizes=[1, 1, 1, 5, 16])
    assert (orr.best()["uniq"] >= 1).all()


def test_cfg1_budget_freezes_runs():
    gr, orr = run_pair(1, "de", R=5, P=32, gens=12, budget=100, step_sizes=[3, 3, 3, 3])
    assert (orr.best()["gens_done"] < 12).any()                         # some run hit the budget and froze


def test_cfg2_ga():
    run_pair(2, "ga", R=3, P=64, gens=6, step_sizes=[1, 2, 3])


def test_cfg3_firefly_sparse():
    run_pair(3, "firefly", R=2, P=128, gens=4, step_sizes=[1, 3])


@pytest.mark.parametrize("algo", ["de", "pso", "firefly", "ga"])
def test_run_partition_invariance(algo):
    """RNG is keyed by the global run index: runs [3, 3+4) of a batch equal a batch created with first_run=3."""
    import paper_2606_28372_b200 as cao
    sp, os_ = oracle_space(0)
    g = gpu_space(0, os_, sp)
    a = cao.Runs(g, algo, n_runs=10, pop=20, max_gens=15, seed=5)
    b = cao.Runs(g, algo, n_runs=4, pop=20, max_gens=15, seed=5, first_run=3)
    a.step(15); b.step(15)
    assert torch.equal(a.trajectory()[:, 3:7], b.trajectory())
    orr = O.OracleRuns(os_, algo, n_runs=4, pop=20, max_gens=15, seed=5, first_run=3)
    orr.step(15)
    compare(b, orr, sp.n)


def test_step_beyond_cap_is_a_no_op_and_hparams():
    import paper_2606_28372_b200 as cao
    hp = O.HParams(0.5, 0.9, 0.7, 1.5, 1.5, 0.8, 2.0, 0.3, 2, 2)
    for algo in ["de", "pso", "firefly", "ga"]:
        gr, orr = run_pair(0, algo, R=7, P=9, gens=6, seed=1234567890123, step_sizes=[6], hp=hp)
        gr.step(5)
        assert gr.gen == 6


def test_small_populations_and_tiny_spaces():
    import paper_2606_28372_b200 as cao
    for seed in range(12):
        sp = W.random_tiny_space(seed)
        os_ = O.OracleSpace.from_space(sp).build()
        if os_.V < 4:
            continue
        obj = W.objective_table(os_.rows(), sp.m, seed)
        os_.set_objective(obj)
        g = cao.Space.from_space(sp).build()
        g.set_objective(obj)
        for algo in ["de", "pso", "firefly", "ga"]:
            P = int(min(os_.V, 3 + seed % 5))
            kw = dict(n_runs=5, pop=P, budget=0, max_gens=8, seed=seed)
            orr = O.OracleRuns(os_, algo, **kw); gr = cao.Runs(g, algo, **kw)
            for _ in range(8):
                gr.step(1); orr.step(1)
                compare(gr, orr, sp.n)


@pytest.mark.parametrize("levels", [0, 1, 2, 3, 4, 5, 6])
def test_forced_probe_levels_give_identical_runs(levels):
    """The Hamming-level probes are an exact shortcut of the scan: every setting reproduces the oracle."""
    import paper_2606_28372_b200 as cao
    sp, os_ = oracle_space(0)
    g = cao.Space.from_space(sp, probe_levels=levels).build()
    assert g.probe_levels == levels
    g.set_objective(os_._obj)
    for algo in ["de", "pso", "firefly", "ga"]:
        kw = dict(n_runs=30, pop=20, budget=0, max_gens=12, seed=3)
        orr = O.OracleRuns(os_, algo, **kw)
        grs = [cao.Runs(g, algo, mode=m, **kw) for m in ("fused", "phased")]
        for _ in range(4):
            orr.step(3)
            for gr in grs:
                gr.step(3)
                compare(gr, orr, sp.n)


def test_auto_probe_levels():
    import paper_2606_28372_b200 as cao
    sp, os_ = oracle_space(1)
    assert gpu_space(1, os_, sp).probe_levels == 6
    sp0, os0 = oracle_space(0)
    assert gpu_space(0, os0, sp0).probe_levels == 1


def test_default_execution_mode():
    """Fused unless the estimated share of candidates that reach the table scan is above 1 % (configs[3])."""
    import paper_2606_28372_b200 as cao
    for cfg, want in ((0, "fused"), (1, "fused"), (2, "fused"), (3, "phased")):
        sp, os_ = oracle_space(cfg)
        g = gpu_space(cfg, os_, sp)
        assert cao.Runs(g, "firefly", n_runs=2, pop=8, max_gens=1).mode == want, cfg


def test_fused_width_api():
    """cao_runs_set_fused_width: 0 / 1 / 2 / 4 only, before the first fused step; a width that does not apply falls back."""
    import paper_2606_28372_b200 as cao
    sp, os_ = oracle_space(0)
    g = gpu_space(0, os_, sp)
    r = cao.Runs(g, "ga", n_runs=4, pop=20, max_gens=4, mode="fused")
    with pytest.raises(cao.CaoError) as e:
        cao.lib().cao_runs_set_fused_width  # symbol exists
        cao.api._check(cao.lib().cao_runs_set_fused_width(r._h, 3))
    assert e.value.code == -1
    cao.api._check(cao.lib().cao_runs_set_fused_width(r._h, 4))
    assert r.fused_width == 4
    r.step(1)
    with pytest.raises(cao.CaoError) as e:
        cao.api._check(cao.lib().cao_runs_set_fused_width(r._h, 1))
    assert e.value.code == -2
    sp3, os3 = oracle_space(3)                               # 32-byte rows: Firefly's four-lane operator does not apply
    g3 = gpu_space(3, os3, sp3)
    r3 = cao.Runs(g3, "firefly", n_runs=2, pop=16, max_gens=2, mode="fused", fused_width=4)
    assert r3.fused_width == 1


def test_two_live_run_sets_share_a_kernel_instantiation():
    """Two run sets of one algorithm that need different amounts of opt-in shared memory, stepped in turn.  The opt-in
    limit belongs to the kernel instantiation, not to a run set: the set with the LARGER need is stepped first, then the
    smaller one, then the larger one again (the order in which a per-set limit would have been lowered under it)."""
    import paper_2606_28372_b200 as cao
    sp, os_ = oracle_space(1)
    g = gpu_space(1, os_, sp)
    # fused PSO, P=128: width 1 = two runs per CTA (~2x the shared memory of width 2 = one run per CTA), same k_gen<1,4,256>
    kw = dict(n_runs=6, pop=128, max_gens=6, seed=11)
    big = cao.Runs(g, "pso", mode="fused", fused_width=1, **kw)
    small = cao.Runs(g, "pso", mode="fused", fused_width=2, **kw)
    ref = cao.Runs(g, "pso", mode="phased", **kw)
    assert (big.fused_width, small.fused_width) == (1, 2)
    for k in (1, 2, 3):
        big.step(k); small.step(k); ref.step(k)
        torch.cuda.synchronize()
        assert torch.equal(big.trajectory(), ref.trajectory()) and torch.equal(small.trajectory(), ref.trajectory())
    # phased Firefly: k_op<2,4,1024> needs (P n + 2 P) 4 bytes: 64 KB at P=1024, 56 KB at P=896 -- both above the 48 KB default
    a = cao.Runs(g, "firefly", n_runs=2, pop=1024, max_gens=3, seed=3, mode="phased")
    b = cao.Runs(g, "firefly", n_runs=2, pop=896, max_gens=3, seed=3, mode="phased")
    orr = O.OracleRuns(os_, "firefly", n_runs=2, pop=1024, max_gens=3, seed=3)
    for _ in range(3):
        a.step(1); b.step(1); orr.step(1)
        torch.cuda.synchronize()
    compare(a, orr, sp.n)
    assert b.gen == 3


@pytest.mark.parametrize("algo", ["de", "ga"])
def test_objective_at_or_above_the_default_penalty(algo):
    """The objective contract is "> 0 and finite": a table whose every value exceeds the default penalty (1e20, L107) still
    has a best-so-far from generation 0 on, the same one in the fused kernel, the phased pipeline and the oracle."""
    sp, os_ = oracle_space(0)
    obj = (W.objective_table(os_.rows(), sp.m, 0).astype(np.float64) * 1e22).astype(np.float32)
    assert obj.min() >= 1e20 and np.isfinite(obj).all()
    try:
        gr, orr = run_pair(0, algo, R=20, P=20, gens=8, step_sizes=[1, 3, 4], objective=obj)
        assert (orr.best()["best_rank"] != 0xFFFFFFFF).all()
    finally:
        os_.set_objective(W.objective_table(os_.rows(), sp.m, 0))

"""GPU parity at the sizes and launch shapes bench.py times (through the C ABI, bit-exact against the CPU oracle).

The oracle is slow on purpose (every repair is a full table scan), so large batches are checked on WINDOWS of runs:
every random number is keyed by the global run index (O3), hence an OracleRuns created with first_run = k reproduces
runs [k, k + w) of any batch.  Windows are stepped on host threads in parallel (each oracle object stays
single-threaded; ctypes releases the GIL).  Covered here:
  * persistent fused kernel with more runs than resident groups (run tickets wrap), 1 / 2 / 4 warps per run,
    16- and 32-byte rows, both execution modes;
  * the BASELINE workloads at their full length: cfg1 budget 1000 to the 200-generation cap, cfg2 GA 150 generations,
    cfg3 Firefly 100 generations, cfg4 at 10^5 runs (3 GB of per-run dedup bitmaps);
  * exp_neg_spec on every fp32 in [0, 32); Philox against cuRAND's device function; rows outside the domain (A27).
"""
from concurrent.futures import ThreadPoolExecutor
import os
import numpy as np
import pytest

import oracle as O
import workloads as W
from conftest import oracle_space

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

_POOL = ThreadPoolExecutor(max_workers=max(2, min(16, os.cpu_count() or 2)))
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


def oracle_windows(os_, algo, windows, width, gens, **kw):
    """Steps one OracleRuns per window (first_run = k, `width` runs) for `gens` generations, in parallel."""
    def one(k0):
        r = O.OracleRuns(os_, algo, n_runs=width, first_run=k0, max_gens=gens, **kw)
        r.step(gens)
        return r
    return list(_POOL.map(one, windows))


def compare_window(gr, orr, n, k0, first_run=0, taps=True):
    """Runs [k0, k0 + orr.R) of the GPU batch against an oracle created with first_run = first_run + k0."""
    w = slice(k0, k0 + orr.R)
    gt = _np(gr.trajectory()[:, w]).view(np.uint32)
    ot = orr.trajectory()
    assert gt.shape[0] == orr.gen + 1
    assert np.array_equal(gt[:, :, 0], ot["best_f"].view(np.uint32)), ("best_f", k0)
    assert np.array_equal(gt[:, :, 1], ot["best_rank"]), ("best_rank", k0)
    assert np.array_equal(gt[:, :, 2], ot["uniq"]), ("uniq", k0)
    gb, ob = gr.best(), orr.best()
    for key in ("best_f", "best_rank", "uniq", "gens_done"):
        assert np.array_equal(_np(gb[key][w]).view(np.uint32), ob[key].view(np.uint32)), (key, k0)
    gs, os_ = gr.state(), orr.state()
    for key in os_:
        a, b = _np(gs[key][w]), os_[key]
        assert np.array_equal(a.view(np.uint32) if a.dtype.itemsize == 4 else a, b.view(np.uint32) if b.dtype.itemsize == 4 else b), (key, k0)
    if taps:
        gtp, otp = gr.taps(), orr.taps()
        act = otp["active"].astype(bool)
        assert np.array_equal(_np(gtp["active"][w]), otp["active"])
        assert np.array_equal(_np(gtp["cand"][w])[act][:, :, :n], otp["cand"][act])
        assert np.array_equal(_np(gtp["valid"][w])[act], otp["valid"][act])
        assert np.array_equal(_np(gtp["rep_rank"][w]).view(np.uint32)[act], otp["rep_rank"][act])
        assert np.array_equal(_np(gtp["eval_rank"][w]).view(np.uint32)[act], otp["eval_rank"][act])
        assert np.array_equal(_np(gtp["f"][w]).view(np.uint32)[act], otp["f"].view(np.uint32)[act])
        assert np.array_equal(_np(gtp["accept"][w])[act], otp["accept"][act])


def same_everywhere(a, b):
    """Two GPU batches (fused / phased) agree on every run: trajectories, results and population state."""
    assert torch.equal(a.trajectory(), b.trajectory())
    for key, v in a.best().items():
        assert torch.equal(v, b.best()[key]), key
    sb = b.state()
    for key, v in a.state().items():
        assert torch.equal(v.contiguous().view(torch.int32) if v.dtype == torch.float32 else v,
                           sb[key].contiguous().view(torch.int32) if v.dtype == torch.float32 else sb[key]), key


# ----------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("R", [1000, 1500, 20000])
@pytest.mark.parametrize("algo", ["de", "pso", "firefly", "ga"])
def test_cfg1_many_runs_sampled_windows(algo, R):
    """More runs than resident groups: the persistent kernel's tickets wrap around; windows at both ends and across
    the first wave boundary; fused against phased on ALL runs.  R = 1000 is the launch shape bench.py times: widened
    groups (two warps per run; Firefly four lanes per firefly, its own instantiation); 1500 and 20000 run one warp per run."""
    import paper_2606_28372_b200 as cao
    sp, os_ = oracle_space(1)
    g = gpu_space(1, os_, sp)
    gens, width = 30, 8
    windows = sorted({0, 1184, 1492, R - width} if R > 1492 + width else {0, 296, 500, R - width})
    kw = dict(pop=32, budget=0, seed=0)
    gf = cao.Runs(g, algo, n_runs=R, max_gens=gens, mode="fused", **kw)
    assert gf.fused_width == ((4 if algo == "firefly" else 2) if R == 1000 else 1)
    gf.step(7); gf.step(gens - 7)                                       # two launches: state leaves and re-enters shared memory
    ors = oracle_windows(os_, algo, windows, width, gens, **kw)
    for k0, orr in zip(windows, ors):
        compare_window(gf, orr, sp.n, k0)
    if R <= 2000:
        gp = cao.Runs(g, algo, n_runs=R, max_gens=gens, mode="phased", **kw)
        gp.step(gens)
        same_everywhere(gf, gp)


@pytest.mark.parametrize("algo", ["de", "pso", "firefly", "ga"])
def test_cfg2_two_warps_per_run(algo):
    """P = 64: groups of two warps (named barriers), 16-byte rows, 3.3 M valid rows."""
    import paper_2606_28372_b200 as cao
    sp, os_ = oracle_space(2)
    g = gpu_space(2, os_, sp)
    R, gens, width = 1300, 10, 3
    windows = [0, 640, R - width]
    kw = dict(pop=64, budget=0, seed=0)
    gf = cao.Runs(g, algo, n_runs=R, max_gens=gens, mode="fused", **kw)
    gf.step(gens)
    for k0, orr in zip(windows, oracle_windows(os_, algo, windows, width, gens, **kw)):
        compare_window(gf, orr, sp.n, k0)
    gp = cao.Runs(g, algo, n_runs=R, max_gens=gens, mode="phased", **kw)
    gp.step(gens)
    same_everywhere(gf, gp)


@pytest.mark.parametrize("P", [32, 128])
@pytest.mark.parametrize("algo", ["de", "pso", "firefly", "ga"])
def test_cfg3_wide_rows(algo, P):
    """n = 20: 32-byte rows (two 128-bit words per row); P = 128: four warps per run; most repairs need the scan."""
    import paper_2606_28372_b200 as cao
    sp, os_ = oracle_space(3)
    g = gpu_space(3, os_, sp)
    R, gens, width = (700, 8, 4) if P == 32 else (300, 6, 2)
    windows = [0, R // 2, R - width]
    kw = dict(pop=P, budget=0, seed=0)
    gf = cao.Runs(g, algo, n_runs=R, max_gens=gens, mode="fused", **kw)
    gf.step(gens)
    for k0, orr in zip(windows, oracle_windows(os_, algo, windows, width, gens, **kw)):
        compare_window(gf, orr, sp.n, k0)
    gp = cao.Runs(g, algo, n_runs=R, max_gens=gens, mode="phased", **kw)
    gp.step(gens)
    same_everywhere(gf, gp)


# ----------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("algo", ["de", "pso", "firefly", "ga"])
def test_cfg1_full_length_budget_1000(algo):
    """BASELINE configs[1] as bench.py runs it: budget 1000 unique evaluations, cap 200 generations; 16 runs."""
    import paper_2606_28372_b200 as cao
    sp, os_ = oracle_space(1)
    g = gpu_space(1, os_, sp)
    R, gens, width = 16, 200, 2
    kw = dict(pop=32, budget=1000, seed=0)
    windows = list(range(0, R, width))
    ors = oracle_windows(os_, algo, windows, width, gens, **kw)
    for mode in ("fused", "phased"):
        gr = cao.Runs(g, algo, n_runs=R, max_gens=gens, mode=mode, **kw)
        gr.step(gens)
        for k0, orr in zip(windows, ors):
            compare_window(gr, orr, sp.n, k0)
    if algo == "de":                                                    # the budget does bind: DE stops early
        assert max(int(o.best()["gens_done"].max()) for o in ors) < gens


def test_cfg2_ga_full_length():
    """BASELINE configs[2]: GA, P = 64, 150 generations (Table IV maxiter); 16 of the 10^4 runs."""
    import paper_2606_28372_b200 as cao
    sp, os_ = oracle_space(2)
    g = gpu_space(2, os_, sp)
    R, gens, width = 16, 150, 2
    kw = dict(pop=64, budget=0, seed=0)
    windows = list(range(0, R, width))
    ors = oracle_windows(os_, "ga", windows, width, gens, **kw)
    for mode in ("fused", "phased"):
        gr = cao.Runs(g, "ga", n_runs=R, max_gens=gens, mode=mode, **kw)
        gr.step(gens)
        for k0, orr in zip(windows, ors):
            compare_window(gr, orr, sp.n, k0)


def test_cfg3_firefly_full_length():
    """BASELINE configs[3]: Firefly, P = 128, 100 generations; 8 of the 1000 runs; most candidates need the scan."""
    import paper_2606_28372_b200 as cao
    sp, os_ = oracle_space(3)
    g = gpu_space(3, os_, sp)
    R, gens, width = 8, 100, 1
    kw = dict(pop=128, budget=0, seed=0)
    windows = list(range(0, R, width))
    ors = oracle_windows(os_, "firefly", windows, width, gens, **kw)
    for mode in ("fused", "phased"):
        gr = cao.Runs(g, "firefly", n_runs=R, max_gens=gens, mode=mode, **kw)
        gr.step(gens)
        for k0, orr in zip(windows, ors):
            compare_window(gr, orr, sp.n, k0)


# ---------------------------------------------------------------------------------------------------------- the shapes bench.py times
def test_cfg3_firefly_timed_shape():
    """bench.py's steps_cfg3: Firefly, P = 128, R = 1000, 100 generations, the library's default mode (phased).  The scan's
    (candidate tiles, table chunks) split is chosen on the device from the worklist length, so R = 1000 takes a split that
    the 8-run test above never takes; runs at the start, the middle and the end against the oracle."""
    import paper_2606_28372_b200 as cao
    sp, os_ = oracle_space(3)
    g = gpu_space(3, os_, sp)
    R, gens = 1000, 100
    windows = [0, 499, R - 1]
    kw = dict(pop=128, budget=0, seed=0)
    ors = oracle_windows(os_, "firefly", windows, 1, gens, **kw)
    gr = cao.Runs(g, "firefly", n_runs=R, max_gens=gens, **kw)
    assert gr.mode == "phased"
    gr.step(gens)
    for k0, orr in zip(windows, ors):
        compare_window(gr, orr, sp.n, k0)


def test_cfg2_ga_timed_shape():
    """bench.py's steps_cfg2: GA, P = 64, R = 10^4, 150 generations: 4 GB of per-run dedup bitmaps, byte offsets beyond 2^31."""
    import paper_2606_28372_b200 as cao
    sp, os_ = oracle_space(2)
    g = gpu_space(2, os_, sp)
    R, gens, width = 10_000, 150, 2
    windows = [0, 5_000, R - width]
    kw = dict(pop=64, budget=0, seed=0)
    ors = oracle_windows(os_, "ga", windows, width, gens, **kw)
    gr = cao.Runs(g, "ga", n_runs=R, max_gens=gens, **kw)
    assert gr.workspace_bytes > 4_000_000_000
    gr.step(gens)
    for k0, orr in zip(windows, ors):
        compare_window(gr, orr, sp.n, k0)
    del gr
    torch.cuda.empty_cache()


_NEXT_ROWS = [(a, v) for a in ("de", "pso", "firefly", "ga") for v in ("unaware", "paper_repair")] + \
             [("de", "rand1exp"), ("de", "lhs"), ("ga", "uniform")]


@pytest.mark.parametrize("algo,name", _NEXT_ROWS)
def test_cfg1_variant_rows_timed_shape(algo, name):
    """bench.py's next_rows_cfg1: every SURVEY 8(f) variant at R = 1000, budget 1000, cap 200 generations; first and last runs."""
    import paper_2606_28372_b200 as cao
    var = {"unaware": dict(aware=False), "paper_repair": dict(repair_mode=1), "rand1exp": dict(de_mutation="rand1", de_crossover="exp"),
           "lhs": dict(init_lhs=True), "uniform": dict(ga_crossover="uniform")}[name]
    sp, os_ = oracle_space(1)
    g = gpu_space(1, os_, sp)
    R, gens, width = 1000, 200, 2
    windows = [0, R - width]
    kw = dict(pop=32, budget=1000, seed=0)
    ors = oracle_windows(os_, algo, windows, width, gens, variant=O.Variant.make(**var), **kw)
    gr = cao.Runs(g, algo, n_runs=R, max_gens=gens, variant=cao.Variant.make(**var), **kw)
    gr.step(gens)
    for k0, orr in zip(windows, ors):
        compare_window(gr, orr, sp.n, k0)


@pytest.mark.parametrize("algo", ["de", "pso", "firefly", "ga"])
def test_cfg4_hundred_thousand_runs(algo):
    """BASELINE configs[4] at 10^5 runs, 200 generations, ONE launch: 3 GB of per-run dedup bitmaps (64-bit offsets),
    every SM slot re-used dozens of times; windows at the start, the middle and the very end."""
    import paper_2606_28372_b200 as cao
    sp, os_ = oracle_space(1)
    g = gpu_space(1, os_, sp)
    R, gens, width = 100_000, 200, 2
    windows = [0, 50_000, R - width]
    kw = dict(pop=32, budget=0, seed=0)
    gr = cao.Runs(g, algo, n_runs=R, max_gens=gens, **kw)
    gr.step(gens)
    for k0, orr in zip(windows, oracle_windows(os_, algo, windows, width, gens, **kw)):
        compare_window(gr, orr, sp.n, k0)
    c = gr.counters()
    assert c["n_evaluated"] >= R * 32 * (gens + 1)
    del gr
    torch.cuda.empty_cache()


# ----------------------------------------------------------------------------------------------------------
def test_exp_neg_spec_every_float_in_0_32():
    """exhaustive CPU-vs-GPU bit compare of exp_neg_spec over every fp32 in [0, 32) (1.1e9 inputs)."""
    import paper_2606_28372_b200 as cao
    lo, hi = int(np.float32(0.0).view(np.uint32)), int(np.float32(32.0).view(np.uint32))
    step = 1 << 24

    def chunk(b0):
        b1 = min(b0 + step, hi)
        z = np.arange(b0, b1, dtype=np.uint32).view(np.float32)
        return b0, O.exp_neg_spec_many(z)

    starts = list(range(lo, hi, step))
    for b0, want in _POOL.map(chunk, starts):
        b1 = min(b0 + step, hi)
        zt = torch.arange(b0, b1, dtype=torch.int64, device="cuda").to(torch.int32).view(torch.float32)
        got = cao.test_exp_neg(zt).view(torch.int32)
        assert torch.equal(got.cpu(), torch.from_numpy(want.view(np.int32))), hex(b0)


def test_philox_against_curand_device_function():
    """Second pin of O3 on the GPU box: cuRAND's curand_Philox4x32_10 agrees with the library and with the oracle."""
    import paper_2606_28372_b200 as cao
    rng = np.random.default_rng(11)
    ck = rng.integers(0, 2 ** 32, size=(20000, 6), dtype=np.uint64).astype(np.uint32)
    ck[0] = 0; ck[1] = 0xFFFFFFFF
    ck[2] = [0x243f6a88, 0x85a308d3, 0x13198a2e, 0x03707344, 0xa4093822, 0x299f31d0]
    t = torch.from_numpy(ck.view(np.int32)).cuda()
    ours = cao.test_philox(t).cpu().numpy().view(np.uint32)
    theirs = cao.test_curand_philox(t).cpu().numpy().view(np.uint32)
    assert np.array_equal(ours, theirs)
    assert tuple(int(x) for x in theirs[2]) == (0xd16cfe09, 0x94fdcceb, 0x5001e420, 0x24126ea1)
    for i in range(0, 20000, 97):
        assert np.array_equal(theirs[i], O.philox4x32_10(ck[i, :4], ck[i, 4:]))


@pytest.mark.parametrize("cfg", [0, 1, 3])
@pytest.mark.parametrize("levels", [0, 1, -1])
def test_repair_rows_outside_the_domain_and_dirty_padding(cfg, levels):
    """A27: a row with idx_d >= m_d is invalid; its repair is the same argmin over its byte values.  Bytes >= 128 on
    a space with M <= 128 (the scan's SMALL byte trick must not be used), and garbage in the padding bytes."""
    sp, os_ = oracle_space(cfg)
    g = gpu_space(cfg, os_, sp)
    rng = np.random.default_rng(5 + cfg)
    n, rb, cnt = sp.n, g.row_bytes, 96
    rows = np.stack([rng.integers(0, m, size=cnt) for m in sp.m], axis=1).astype(np.uint8)
    rows[::3, rng.integers(0, n)] = 200                                 # far outside, >= 128
    rows[1::3, rng.integers(0, n)] = max(sp.m)                          # just outside every domain
    rows[5::7] = rng.integers(128, 256, size=rows[5::7].shape).astype(np.uint8)
    padded = rng.integers(0, 256, size=(cnt, rb)).astype(np.uint8)      # dirty padding
    padded[:, :n] = rows
    want = os_.repair(rows)
    valid = np.array([os_.is_valid(r) for r in rows])
    assert not valid[::3].any() and not valid[1::3].any()
    rank, key = g.repair(torch.from_numpy(padded).cuda(), use_probe=levels if levels >= 0 else True)
    key = key.cpu().numpy().view(np.uint64)
    assert np.array_equal(rank.cpu().numpy().view(np.uint32), want["rank"])
    assert np.array_equal((key >> np.uint64(45)).astype(np.uint32), want["ham"])
    assert np.array_equal(((key >> np.uint64(32)) & np.uint64(0x1FFF)).astype(np.uint32), want["sad"])
    assert np.array_equal(g.is_valid(torch.from_numpy(padded).cuda()).cpu().numpy().astype(bool), valid)

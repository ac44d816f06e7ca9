"""GPU parity, through the C ABI, of S1 (enumerate/filter/compact), the is-valid query, S5 (repair) and the
arithmetic primitives (Philox, exp_neg_spec) against the CPU oracle: bit-exact."""
import numpy as np
import pytest

import oracle as O
import workloads as W
from conftest import oracle_space

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


def _gpu_space(sp, mode=0):
    import paper_2606_28372_b200 as cao
    return cao.Space.from_space(sp, build_mode=mode).build()


def _u64(t):
    a = t.cpu().numpy()
    return a.view(np.uint32).astype(np.uint64) if a.dtype.itemsize == 4 else a.view(np.uint64)


def _check_space(sp, os_, gs):
    N, V, n, rb = gs.sizes()
    assert (N, V, n) == (os_.N, os_.V, os_.n)
    assert np.array_equal(_u64(gs.bitmap()), os_.bitmap())
    if V:
        rows = gs.rows().cpu().numpy()
        assert np.array_equal(rows[:, :n], os_.rows())
        assert not rows[:, n:].any()                                   # padding bytes are zero
        assert np.array_equal(_u64(gs.Ltab()), os_.Ltab())
    # rank directory = exclusive count of valid L below each multiple of 512
    bits = np.unpackbits(os_.bitmap().view(np.uint8), bitorder="little")[:N]
    nd = (N + 511) // 512
    want = np.concatenate([[0], np.cumsum(np.add.reduceat(bits, np.arange(0, N, 512)))]) if N else np.zeros(1)
    assert np.array_equal(gs.rank_dir().cpu().numpy().astype(np.int64), want.astype(np.int64)[:nd + 1])


@pytest.mark.parametrize("mode", [0, 1])
@pytest.mark.parametrize("cfg", [0, 1, 2])
def test_enumerate_baseline_configs(cfg, mode):
    sp, os_ = oracle_space(cfg, with_objective=False)
    gs = _gpu_space(sp, mode)
    assert gs.V == sp.expect_V and gs.N == sp.expect_N
    _check_space(sp, os_, gs)


def test_enumerate_cfg3_full():
    """573 M Cartesian configs, 67,915 valid (1.2e-4): the whole bitmap and table against the oracle."""
    sp, os_ = oracle_space(3, with_objective=False)
    gs = _gpu_space(sp, 0)
    assert (gs.N, gs.V) == (573308928, 67915)
    _check_space(sp, os_, gs)


@pytest.mark.parametrize("mode", [0, 1])
def test_enumerate_random_tiny_spaces(mode):
    for seed in range(40):
        sp = W.random_tiny_space(seed)
        os_ = O.OracleSpace.from_space(sp).build()
        import paper_2606_28372_b200 as cao
        g = cao.Space.from_space(sp, build_mode=mode)
        g.alloc_build()
        V = g.build_count()
        assert V == os_.V, (seed, V, os_.V)
        g.alloc_table(); g.build_fill()
        _check_space(sp, os_, g)


def test_enumerate_edge_shapes():
    import paper_2606_28372_b200 as cao
    from workloads import P
    # single parameter, single value; no constraints
    for doms, progs in [([[5]], []), ([[1, 2, 3]], []), ([[1, 2, 3]], [(P(0) > 5).program()]),
                        ([list(range(200)), list(range(256))], [((P(0) + P(1)) % 7).eq(3).program()]),
                        ([[0, 1]] * 17, [(P(0) + P(16) >= 1).program()]),                      # 32-byte rows
                        ([[2 ** 40, 2 ** 41], [2 ** 30, -2 ** 31]], [(P(0) * P(1) > 0).program()]),   # saturation
                        ([[0, 1, 2], [0, 3]], [(P(1) // P(0) >= 0).program()])]:               # division by zero
        os_ = O.OracleSpace(doms, progs).build()
        for mode in (0, 1):
            g = cao.Space(doms, progs, build_mode=mode)
            g.alloc_build()
            assert g.build_count() == os_.V
            g.alloc_table(); g.build_fill()
            sp = type("S", (), {})()
            _check_space(sp, os_, g)


def test_is_valid_and_repair_cfg0_all_configs():
    sp, os_ = oracle_space(0, with_objective=False)
    gs = _gpu_space(sp)
    rows = np.array([[a, b, c] for a in range(5) for b in range(6) for c in range(4)], dtype=np.uint8)
    want_valid = np.array([os_.is_valid(r) for r in rows], dtype=np.uint8)
    assert np.array_equal(gs.is_valid(rows).cpu().numpy(), want_valid)
    want = os_.repair(rows)
    wkey = (want["ham"].astype(np.uint64) << np.uint64(45)) | (want["sad"].astype(np.uint64) << np.uint64(32)) | want["rank"].astype(np.uint64)
    for probe in (True, False, 1, 2, 3):
        rank, key = gs.repair(rows, use_probe=probe)
        assert np.array_equal(rank.cpu().numpy().view(np.uint32), want["rank"])
        assert np.array_equal(_u64(key), wkey)


@pytest.mark.parametrize("cfg,count", [(1, 300), (2, 40), (3, 200)])
def test_repair_random_rows(cfg, count):
    sp, os_ = oracle_space(cfg, with_objective=False)
    gs = _gpu_space(sp)
    rng = np.random.default_rng(100 + cfg)
    rows = np.stack([rng.integers(0, m, size=count) for m in sp.m], axis=1).astype(np.uint8)
    rows[:5] = os_.rows()[rng.integers(0, os_.V, size=5)]             # some valid rows: identity (Alg.1)
    want = os_.repair(rows)
    wkey = (want["ham"].astype(np.uint64) << np.uint64(45)) | (want["sad"].astype(np.uint64) << np.uint64(32)) | want["rank"].astype(np.uint64)
    assert (want["ham"][:5] == 0).all()
    for probe in (True, False, 1, 2, 3):
        rank, key = gs.repair(rows, use_probe=probe)
        assert np.array_equal(_u64(key), wkey)
        assert np.array_equal(rank.cpu().numpy().view(np.uint32), want["rank"])
    assert np.array_equal(gs.is_valid(rows).cpu().numpy(), (want["ham"] == 0).astype(np.uint8))


def test_repair_tiny_spaces_and_ragged_counts():
    import paper_2606_28372_b200 as cao
    for seed in range(25):
        sp = W.random_tiny_space(seed)
        os_ = O.OracleSpace.from_space(sp).build()
        if os_.V == 0:
            continue
        g = cao.Space.from_space(sp).build()
        rng = np.random.default_rng(seed)
        count = int(rng.integers(1, 700))
        rows = np.stack([rng.integers(0, m, size=count) for m in sp.m], axis=1).astype(np.uint8)
        want = os_.repair(rows)
        for probe in (True, False, 1, 2, 3):
            rank, key = g.repair(rows, use_probe=probe)
            assert np.array_equal(rank.cpu().numpy().view(np.uint32), want["rank"]), seed
            k = _u64(key)
            assert np.array_equal(k >> np.uint64(45), want["ham"].astype(np.uint64))
            assert np.array_equal((k >> np.uint64(32)) & np.uint64(0x1FFF), want["sad"].astype(np.uint64))


def test_empty_space_and_errors():
    import paper_2606_28372_b200 as cao
    from workloads import P
    g = cao.Space([[1, 2], [3, 4]], [(P(0) > 9).program()]).build()
    assert g.V == 0
    with pytest.raises(cao.CaoError) as e:
        g.repair(np.zeros((3, 2), np.uint8))
    assert e.value.code == -4
    g.set_objective if True else None
    sp, os_ = oracle_space(0)
    gs = _gpu_space(sp)
    gs.set_objective(os_._obj)
    with pytest.raises(cao.CaoError) as e:
        cao.Runs(gs, "de", n_runs=2, pop=93, max_gens=3)                # P > V
    assert e.value.code == -5
    assert gs.is_valid(np.zeros((0, 3), np.uint8)).numel() == 0


def test_philox_known_answers_and_random_parity():
    import paper_2606_28372_b200 as cao
    kat = [((0, 0, 0, 0), (0, 0), (0x6627e8d5, 0xe169c58d, 0xbc57ac4c, 0x9b00dbd8)),
           ((0xffffffff,) * 4, (0xffffffff,) * 2, (0x408f276d, 0x41c83b0e, 0xa20bc7c6, 0x6d5451fd)),
           ((0x243f6a88, 0x85a308d3, 0x13198a2e, 0x03707344), (0xa4093822, 0x299f31d0),
            (0xd16cfe09, 0x94fdcceb, 0x5001e420, 0x24126ea1))]              # Random123 known answers
    rng = np.random.default_rng(7)
    ck = rng.integers(0, 2 ** 32, size=(5000, 6), dtype=np.uint64).astype(np.uint32)
    for i, (c, k, _) in enumerate(kat):
        ck[i] = list(c) + list(k)
    out = cao.test_philox(torch.from_numpy(ck.view(np.int32)).cuda()).cpu().numpy().view(np.uint32)
    for i, (_, _, want) in enumerate(kat):
        assert tuple(int(x) for x in out[i]) == want
    for i in range(3, 5000, 7):
        assert np.array_equal(out[i], O.philox4x32_10(ck[i, :4], ck[i, 4:]))


def test_exp_neg_spec_bit_exact():
    import paper_2606_28372_b200 as cao
    rng = np.random.default_rng(3)
    z = np.concatenate([rng.uniform(0, 32, 2_000_000), rng.uniform(0, 1e-3, 100_000), rng.uniform(60, 200, 100_000),
                        [0.0, 1.0, 87.0, 87.5, 88.0, 126.0, 1e30, np.inf]]).astype(np.float32)
    got = cao.test_exp_neg(torch.from_numpy(z).cuda()).cpu().numpy()
    want = O.exp_neg_spec_many(z)
    assert np.array_equal(got.view(np.uint32), want.view(np.uint32))
    # every fp32 in a dense bit range [1.0, 1.0 + 2^22 ulps)
    zb = (np.arange(1 << 22, dtype=np.uint32) + np.float32(1.0).view(np.uint32)).view(np.float32)
    got = cao.test_exp_neg(torch.from_numpy(zb).cuda()).cpu().numpy()
    assert np.array_equal(got.view(np.uint32), O.exp_neg_spec_many(zb).view(np.uint32))


@pytest.mark.parametrize("cfg", [0, 1, 2, 3])
def test_rebuild_reproduces_the_space(cfg):
    """cao_space_rebuild: all of S1 again, asynchronously, into the same (wiped) buffers -- on the default stream (plain
    launches) and twice on a side stream (captured CUDA graph, then its replay); the count scan of the rebuild is the
    single-pass look-back variant (274 chunks on configs[3])."""
    sp, os_ = oracle_space(cfg, with_objective=False)
    gs = _gpu_space(sp)
    gs._bitmap.zero_(); gs.rows().zero_(); gs.Ltab().zero_(); gs.rank_dir().zero_()
    gs.rebuild()
    torch.cuda.synchronize()
    _check_space(sp, os_, gs)
    side = torch.cuda.Stream()
    for _ in range(2):
        gs._bitmap.zero_(); gs.rows().zero_(); gs.Ltab().zero_(); gs.rank_dir().zero_()
        torch.cuda.synchronize()
        with torch.cuda.stream(side):
            gs.rebuild()
        torch.cuda.synchronize()
        _check_space(sp, os_, gs)
    rows = np.stack([np.random.default_rng(1).integers(0, m, size=64) for m in sp.m], axis=1).astype(np.uint8)
    want = os_.repair(rows)
    rank, key = gs.repair(rows)                                         # probe tables survive the rebuild
    assert np.array_equal(rank.cpu().numpy().view(np.uint32), want["rank"])


def test_profile_classes_of_the_build():
    """Per-kernel timing of S1: the mask / key and residual-prefix kernels are booked under their own classes, not under the
    repair-probe and query classes that the generation step's analysis reads."""
    import paper_2606_28372_b200 as cao
    sp = W.space_cfg3()                                                 # has tabled and residual constraints
    cao.profile_enable(True)
    try:
        cao.Space.from_space(sp).build()
        torch.cuda.synchronize()
        prof = cao.profile_read()
    finally:
        cao.profile_enable(False)
    assert prof["k_keys+k_masks"][1] >= 1 and prof["k_enum"][1] == 1 and prof["k_fill"][1] == 1
    assert prof["k_probe23"][1] == 0 and prof["k_is_valid/k_repair_probe/k_repair_finish"][1] == 0
    assert len(prof) == 14

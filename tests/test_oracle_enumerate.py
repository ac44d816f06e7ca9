"""Pins of oracle enumeration (O1) and repair (O9) against independent brute force / closed counts (no GPU)."""
import itertools
import os
import numpy as np
import pytest

import oracle as O
import workloads as W
from conftest import oracle_space

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def brute_force(sp):
    """itertools.product over VALUES with the hand-written Python predicates (never the bytecode)."""
    valid_rows, Ls = [], []
    for L, idx in enumerate(itertools.product(*[range(len(d)) for d in sp.domains])):   # last digit fastest (A1)
        vals = [sp.domains[d][i] for d, i in enumerate(idx)]
        if all(p(vals) for p in sp.preds):
            valid_rows.append(idx); Ls.append(L)
    return np.array(valid_rows, np.uint8).reshape(-1, sp.n), np.array(Ls, np.uint64)


def check_space_against_bruteforce(sp):
    s = O.OracleSpace.from_space(sp).build()
    rows, Ls = brute_force(sp)
    assert s.N == sp.N and s.V == len(Ls)
    assert (s.rows() == rows).all() and (s.Ltab() == Ls).all()
    bm = s.bitmap()
    bits = np.zeros(len(bm) * 64, np.uint8)
    bits[Ls.astype(np.int64)] = 1
    want = np.packbits(bits.reshape(-1, 64), axis=1, bitorder="little").view("<u8").ravel()
    assert (bm == want).all()                               # bit (L & 63) of word (L >> 6); tail bits zero
    return s, rows, Ls


@pytest.mark.parametrize("seed", range(40))
def test_random_tiny_spaces_match_itertools(seed):
    check_space_against_bruteforce(W.random_tiny_space(seed))


def test_cfg0_hand_count():
    sp = W.space_cfg0()
    s, rows, Ls = check_space_against_bruteforce(sp)
    assert s.V == 92
    bad = {(16, 1), (64, 32), (128, 16), (128, 32), (256, 8), (256, 16), (256, 32)}
    got_bad = set()
    for ix in range(5):
        for iy in range(6):
            if not s.is_valid([ix, iy, 0]):
                got_bad.add((sp.domains[0][ix], sp.domains[1][iy]))
    assert got_bad == bad


def _numpy_valid_mask(sp):
    """Independent vectorised evaluation: one broadcast array per parameter, predicates on arrays."""
    grids = np.meshgrid(*[np.array(d, np.int64) for d in sp.domains], indexing="ij", sparse=True)
    mask = np.ones([len(d) for d in sp.domains], bool)
    for p in sp.preds:
        mask &= np.broadcast_to(p(grids), mask.shape)
    return mask.ravel()                                      # C order = last digit fastest


@pytest.mark.parametrize("cfg", [1, 2])
def test_cfg1_cfg2_counts_and_table(cfg):
    sp, s = oracle_space(cfg, with_objective=False)
    mask = _numpy_valid_mask(sp)
    assert s.N == sp.expect_N and int(mask.sum()) == sp.expect_V == s.V
    Ls = np.flatnonzero(mask).astype(np.uint64)
    assert (s.Ltab() == Ls).all()
    rows = s.rows()
    stride = np.cumprod([1] + sp.m[::-1][:-1])[::-1].astype(np.uint64)
    assert ((rows.astype(np.uint64) * stride).sum(axis=1) == Ls).all()     # rows decode L, most significant first
    bm = s.bitmap()
    assert int(np.unpackbits(bm.view(np.uint8)).sum()) == s.V               # popcount(bitmap) = V


def _cfg3_pruned_dfs():
    """Independent method for cfg3: depth-first search with early pruning on the product bound and on every
    divisibility pair as soon as both ends are assigned.  Returns the sorted valid linear indices."""
    t = W.CFG3_SEED0_TABLE
    doms = [[1 << e for e in es] for es in t["exps"]]
    m = [len(d) for d in doms]
    stride = [1] * 20
    for d in range(18, -1, -1):
        stride[d] = stride[d + 1] * m[d + 1]
    by_last = {d: [] for d in range(20)}
    for (a, b) in t["pairs"]:
        by_last[max(a, b)].append((a, b))
    out = []
    vals = [0] * 20

    def rec(d, prod, L):
        if d == 20:
            out.append(L); return
        for i, v in enumerate(doms[d]):
            p2 = prod * v
            if p2 > (1 << 20):
                break                                        # values ascend, all >= 1
            vals[d] = v
            if all(vals[b] % vals[a] == 0 for (a, b) in by_last[d]):
                rec(d + 1, p2, L + i * stride[d])
    rec(0, 1, 0)
    return np.array(out, np.uint64)


def test_cfg3_exact_table():
    Ls = _cfg3_pruned_dfs()
    assert len(Ls) == 67915 and (np.diff(Ls.astype(np.int64)) > 0).all()
    assert list(Ls[:5]) == [0, 2, 4, 6, 8] and int(Ls[-1]) == 382206080
    sp, s = oracle_space(3, with_objective=False)            # full oracle enumeration (~1 min)
    assert s.N == 573308928 and s.V == 67915
    assert (s.Ltab() == Ls).all()
    # literal division decode on sampled ranges agrees with the odometer table
    for L0 in (0, 382206080 - 1000, 123456789, 573308928 - 5000):
        L1 = min(L0 + 5000, s.N)
        want = int(((Ls >= L0) & (Ls < L1)).sum())
        assert s.count_range(L0, L1) == want


def test_count_range_decode_matches_table_on_tiny():
    for seed in range(10):
        sp = W.random_tiny_space(100 + seed)
        s = O.OracleSpace.from_space(sp).build()
        assert s.count_range(0, s.N) == s.V
        h = s.N // 2
        assert s.count_range(0, h) + s.count_range(h, s.N) == s.V


# ----------------------------------------------------------------------------- repair
def numpy_repair(rows, Ls, cand):
    """Independent brute force: all keys at once, lexicographic minimum via np.lexsort."""
    ham = (rows != cand[None, :]).sum(axis=1)
    sad = np.abs(rows.astype(np.int64) - cand[None, :].astype(np.int64)).sum(axis=1)
    order = np.lexsort((Ls, sad, ham))
    r = order[0]
    return int(r), int(ham[r]), int(sad[r]), int(Ls[r])


def nth_nonempty_tiny_space(base, k):
    """The k-th random tiny space, counting seeds from `base`, that has at least one valid configuration (an empty space
    has nothing to repair to: such seeds are passed over instead of skipping the test)."""
    seed, found = base, -1
    while True:
        sp = W.random_tiny_space(seed)
        s = O.OracleSpace.from_space(sp).build()
        found += s.V > 0
        if found == k:
            return sp, s
        seed += 1


@pytest.mark.parametrize("seed", range(25))
def test_repair_is_the_key_minimum_on_tiny_spaces(seed):
    sp, s = nth_nonempty_tiny_space(200, seed)
    rows, Ls = s.rows(), s.Ltab()
    rng = np.random.default_rng(seed)
    cands = np.stack([rng.integers(0, mm, 60) for mm in sp.m], axis=1).astype(np.uint8)
    got = s.repair(cands)
    for i, c in enumerate(cands):
        r, ham, sad, L = numpy_repair(rows, Ls, c)
        assert (int(got["rank"][i]), int(got["ham"][i]), int(got["sad"][i]), int(got["L"][i])) == (r, ham, sad, L)
        if s.is_valid(c):                                    # Alg.1 L205 / Alg.3: identity on valid
            assert ham == 0 and (rows[r] == c).all()
        else:
            assert ham >= 1


@pytest.mark.parametrize("seed", range(10))
def test_repair_of_rows_outside_the_domain(seed):
    """A27: idx_d >= m_d is not a point of X: is-valid is false, repair is the same key minimum over the byte values
    (numpy brute force; a worked cfg0 value: (7,0,0) -> nearest row by (Hamming, sum |d|, L))."""
    sp, s = nth_nonempty_tiny_space(300, seed)
    rows, Ls = s.rows(), s.Ltab()
    rng = np.random.default_rng(seed)
    cands = np.stack([rng.integers(0, mm, 40) for mm in sp.m], axis=1).astype(np.uint8)
    col = rng.integers(0, sp.n, 40)
    cands[np.arange(40), col] = np.array([sp.m[c] for c in col]) + rng.integers(0, 200, 40)   # at least one index outside
    got = s.repair(cands)
    for i, c in enumerate(cands):
        assert not s.is_valid(c)
        r, ham, sad, L = numpy_repair(rows, Ls, c)
        assert ham >= 1
        assert (int(got["rank"][i]), int(got["ham"][i]), int(got["sad"][i]), int(got["L"][i])) == (r, ham, sad, L)


def test_repair_outside_the_domain_worked_cfg0():
    # cfg0: bx idx 7 does not exist (m = 5).  Rows (x,0,0) are valid for x = 1..4 (32 <= bx*1 <= 1024 needs bx >= 32):
    # Hamming 1 each, sum |d| = 7 - x, so (4,0,0) wins with key (1, 3, L = 4*24 = 96).
    sp, s = oracle_space(0, with_objective=False)
    got = s.repair(np.array([[7, 0, 0]], np.uint8))
    assert list(s.rows()[got["rank"][0]]) == [4, 0, 0]
    assert (int(got["ham"][0]), int(got["sad"][0]), int(got["L"][0])) == (1, 3, 96)
    assert not s.is_valid(np.array([7, 0, 0], np.uint8))


def test_repair_worked_examples_cfg0():
    sp, s = oracle_space(0, with_objective=False)
    rows = s.rows()
    with open(os.path.join(GOLD, "repair_cfg0.txt")) as fh:
        for ln in fh:
            if ln.startswith("#") or not ln.strip():
                continue
            lhs, rhs = ln.split("->")
            c = np.array([int(x) for x in lhs.split()], np.uint8)
            w = [int(x) for x in rhs.split()]
            got = s.repair(c[None, :])
            assert list(rows[got["rank"][0]]) == w[:3]
            assert (int(got["ham"][0]), int(got["sad"][0]), int(got["L"][0])) == tuple(w[3:])


def test_repair_identity_on_every_valid_config_cfg1_sample():
    sp, s = oracle_space(1, with_objective=False)
    rows = s.rows()
    pick = np.random.default_rng(0).integers(0, s.V, 40)
    got = s.repair(rows[pick])
    assert (got["rank"] == pick).all() and (got["ham"] == 0).all() and (got["sad"] == 0).all()


def test_256_value_digit_carries():
    """O1: idx_d = (L / stride_d) mod m_d also for m_d = 256, the largest domain the boundary allows (a byte
    odometer would wrap without carrying).  Closed form: #{(a, b) in [0,200) x [0,256): (a + b) % 7 == 3}."""
    from workloads import P
    doms = [list(range(200)), list(range(256))]
    s = O.OracleSpace(doms, [((P(0) + P(1)) % 7).eq(3).program()]).build()
    want = sum(1 for a in range(200) for b in range(256) if (a + b) % 7 == 3)
    assert s.V == want == s.count_range(0, 200 * 256)
    rows = s.rows()
    assert ((rows[:, 0].astype(int) + rows[:, 1].astype(int)) % 7 == 3).all()
    assert np.array_equal(s.Ltab(), rows[:, 0].astype(np.uint64) * 256 + rows[:, 1].astype(np.uint64))

"""Pins of the oracle's primitives against what the paper and the mathematics fix (no GPU)."""
import math
import os
import struct
import numpy as np
import pytest

import oracle as O

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _lines(name):
    with open(os.path.join(GOLD, name)) as fh:
        return [ln.strip() for ln in fh if ln.strip() and not ln.startswith("#")]


# ----------------------------------------------------------------------------- O3 Philox
def test_philox_known_answers():
    for ln in _lines("philox_kat.txt"):
        w = [int(x, 16) for x in ln.split()]
        out = O.philox4x32_10(w[0:4], w[4:6])
        assert [int(x) for x in out] == w[6:10]


def test_philox_is_a_bijection_of_the_counter_on_a_sample():
    # a counter-mode block cipher cannot collide for distinct counters under one key
    seen = set()
    for c in range(2000):
        seen.add(tuple(int(x) for x in O.philox4x32_10([c, 0, 0, 0], [7, 9])))
    assert len(seen) == 2000


def test_draw_layout_matches_counter_spec():
    # counter = (run, generation, individual, stream<<24 | slot>>2), key = (seed_lo, seed_hi), word = slot & 3
    seed = 0x0123456789ABCDEF
    for (run, gen, ind, stream, slot) in [(0, 1, 0, 1, 0), (5, 7, 3, 2, 9), (99, 50, 19, 3, 130), (1, 0, 0, 0, 3)]:
        blk = O.philox4x32_10([run, gen, ind, (stream << 24) | (slot >> 2)], [seed & 0xFFFFFFFF, seed >> 32])
        assert O.draw(seed, run, gen, ind, stream, slot) == int(blk[slot & 3])
    kat = [ln for ln in _lines("prototype_cfg0.txt") if ln.startswith("layout_kat")][0].split()[1:]
    assert [O.draw(0, 0, 1, 0, "op", s) for s in range(4)] == [int(x, 16) for x in kat]


def test_u01_and_below():
    assert O.u01(0) == 0.0
    assert O.u01(0xFFFFFFFF) == 1.0 - 2.0 ** -24          # largest value, still < 1
    assert O.u01(0x80000000) == 0.5
    rng = np.random.default_rng(1)
    for w in rng.integers(0, 2 ** 32, 200):
        w = int(w)
        assert O.u01(w) == (w >> 8) / 2.0 ** 24            # exact in fp32
        for k in (1, 2, 3, 20, 92, 241600, 2 ** 32 - 1):
            b = O.below(w, k)
            assert b == (w * k) >> 32 and 0 <= b < k


# ----------------------------------------------------------------------------- O7 exp
def test_exp_neg_spec_against_libm():
    z = np.concatenate([np.linspace(0, 32, 200001), np.random.default_rng(0).uniform(0, 32, 200000)]).astype(np.float32)
    got = O.exp_neg_spec_many(z).astype(np.float64)
    ref = np.exp(-z.astype(np.float64))
    rel = np.abs(got - ref) / ref
    assert rel.max() < 2e-6, rel.max()                      # SURVEY 8(c)'s bound (measured 1.8e-6 near z = 30: the rounding of t = z*log2(e), ~z * 2^-24 relative)
    small = z <= 1.0
    assert rel[small].max() < 3e-7


def test_exp_neg_spec_special_values():
    assert O.exp_neg_spec(0.0) == float.fromhex("0x1.fffffep-1")   # DESIGN.md O7: not exactly 1
    assert O.exp_neg_spec(1e30) == 0.0 and O.exp_neg_spec(100.0) == 0.0   # floor(t) >= 126 -> 0
    assert O.exp_neg_spec(80.0) > 0.0
    zs = np.linspace(0, 60, 5000).astype(np.float32)
    v = O.exp_neg_spec_many(zs)
    assert (np.diff(v) <= 1e-7 * v[:-1]).all()             # monotone non-increasing up to rounding


def test_exp_neg_spec_follows_the_written_operation_order():
    # independent fp32 evaluation with numpy scalars: one rounding per written operation
    f = np.float32
    c = [f(1.0), f(float.fromhex("-0x1.62e430p-1")), f(float.fromhex("0x1.ebfbe0p-3")), f(float.fromhex("-0x1.c6b08ep-5")),
         f(float.fromhex("0x1.3b2ab6p-7")), f(float.fromhex("-0x1.5d87fep-10")), f(float.fromhex("0x1.430912p-13")),
         f(float.fromhex("-0x1.ffcbfcp-17"))]
    # the constants are fp32((-ln 2)^i / i!)
    for i in range(8):
        assert c[i] == f((-math.log(2.0)) ** i / math.factorial(i))
    for z in np.random.default_rng(3).uniform(0, 40, 3000).astype(np.float32):
        t = f(z) * f(float.fromhex("0x1.715476p+0"))
        kf = np.floor(t)
        u = f(f(t - kf) - f(0.5))
        p = c[7]
        for i in range(6, -1, -1):
            p = f(f(p * u) + c[i])
        p = f(p * f(float.fromhex("0x1.6a09e6p-1")))
        scale = struct.unpack("<f", struct.pack("<I", (127 - int(kf)) << 23))[0]
        assert O.exp_neg_spec(float(z)) == float(f(p * f(scale)))


# ----------------------------------------------------------------------------- O5 / O6 scalar steps
def test_de_rounding_ties_are_half_to_even():
    # fl(0.7f * k) is exactly a half-integer for k = 5, 15, ..., 55; rint != round there
    F = np.float32(0.7)
    for k in range(5, 60, 10):
        t = np.float32(F * np.float32(k))
        assert float(t) * 2 == int(float(t) * 2) and float(t) != int(float(t))
        lo = int(math.floor(float(t)))
        for best in (0, 1, 2, 3):
            want = best + (lo if (best + lo) % 2 == 0 else lo + 1)     # nearest even of best + lo + 0.5
            assert O.de_mutate_index(0.7, best, k, 0, 1000) == want
            want_neg = best - lo - 1 if (best - lo - 1) % 2 == 0 else best - lo
            assert O.de_mutate_index(0.7, best, 0, k, 1000) == max(want_neg, 0)


def test_de_mutate_index_general_and_clip():
    f = np.float32
    rng = np.random.default_rng(5)
    for _ in range(2000):
        best, a, b, top = (int(x) for x in rng.integers(0, 40, 4))
        mf = f(f(best) + f(f(0.7) * f(a - b)))
        want = min(max(int(np.rint(mf)), 0), top)
        assert O.de_mutate_index(0.7, best, a, b, top) == want
    assert O.de_mutate_index(0.7, 0, 0, 30, 9) == 0 and O.de_mutate_index(0.7, 9, 30, 0, 9) == 9


def test_coord_and_snap_roundtrip():
    for M in (2, 3, 4, 16, 37, 256):
        for k in range(M):
            x = O.coord(M, k)
            assert x == float(np.float32(k) / np.float32(M - 1))
            assert O.snap(M, M, x) == k                      # snapping a grid point is the identity
            if k + 1 < M:
                eps = O.coord(M, 1)
                assert O.snap(M, M, x + 0.26 * eps) == k and O.snap(M, M, x + 0.74 * eps) == k + 1
        assert O.coord(M, 0) == 0.0 and O.coord(M, M - 1) == 1.0
    assert O.coord(1, 0) == 0.0 and O.snap(1, 1, 0.0) == 0
    assert O.snap(16, 4, 1.0) == 3 and O.snap(16, 4, -1.0) == 0      # clip to the dimension's own top (A10)


def test_clamp_pos():
    assert O.clamp_pos(float("nan"), 0.5) == 0.0
    assert math.copysign(1.0, O.clamp_pos(-0.0, 0.5)) == 1.0
    assert O.clamp_pos(0.7, 0.5) == 0.5 and O.clamp_pos(0.25, 0.5) == 0.25 and O.clamp_pos(-3.0, 0.5) == 0.0
    assert O.clamp_pos(float("inf"), 1.0) == 1.0


# ----------------------------------------------------------------------------- O1 constraint programs
def test_constraint_saturation_and_division_by_zero():
    from workloads import P, C
    big = 1 << 40
    prog = (P(0) * P(1) * P(2) <= (1 << 20)).program()        # true product 2^120 wraps to 0 in int64
    assert O.eval_program(prog, [big, big, big]) == 0
    assert O.eval_program(prog, [1, 2, 4]) == 1
    assert O.eval_program((P(0) * P(1) >= -(1 << 61)).program(), [-big, big]) == 0   # saturates at -2^62
    assert O.eval_program((P(0) + P(1)).eq(1 << 62).program(), [1 << 62, 1 << 62]) == 1
    assert O.eval_program((P(0) % P(1)).eq(0).program(), [4, 0]) == 0
    assert O.eval_program((P(0) % P(1)).ne(0).program(), [4, 0]) == 0              # whole constraint false
    assert O.eval_program((P(0) // P(1) < 100).program(), [4, 0]) == 0
    assert O.eval_program(((-P(0)) // P(1)).eq(-2).program(), [7, 3]) == 1         # truncation toward zero
    assert O.eval_program(((-P(0)) % P(1)).eq(-1).program(), [7, 3]) == 1          # sign of the dividend
    assert O.eval_program(C(5).program(), [0]) == 1 and O.eval_program(C(0).program(), [0]) == 0


def test_malformed_programs_are_rejected():
    assert O.eval_program([3], [1]) == -1                    # ADD on empty stack
    assert O.eval_program([1, 5], [1]) == -1                 # param index out of range
    assert O.eval_program([1, 0, 1, 0], [1]) == -1           # two values left
    assert O.eval_program([99], [1]) == -1
    assert O.eval_program([2, 1], [1]) == -1                 # truncated constant

"""ctypes wrapper around the CPU oracle (oracle/cao_oracle.cc).  TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package; the product (paper_2606_28372_b200) never does.  Nothing here imports the product.
"""
from __future__ import annotations
import ctypes as C
import numpy as np

from .build import build as _build

ALGOS = {"de": 0, "pso": 1, "firefly": 2, "ga": 3}
STREAMS = {"init": 0, "op": 1, "mut": 2, "reinit": 3, "repair": 5}


class HParams(C.Structure):
    """Table IV defaults; ga_beta_b: reading A18."""
    _fields_ = [("de_F", C.c_float), ("de_CR", C.c_float),
                ("pso_w", C.c_float), ("pso_c1", C.c_float), ("pso_c2", C.c_float),
                ("ff_B0", C.c_float), ("ff_gamma", C.c_float), ("ff_alpha", C.c_float),
                ("ga_mutation_chance", C.c_int32), ("ga_beta_b", C.c_int32)]

    @classmethod
    def default(cls):
        return cls(0.7, 0.6, 0.5, 3.0, 0.5, 1.0, 1.0, 0.2, 5, 3)


class Variant(C.Structure):
    """SURVEY 8(f) switches (oracle/cao_oracle.cc `Variant`); the default is the north_star path."""
    _fields_ = [("aware", C.c_int32), ("repair_mode", C.c_int32), ("de_mutation", C.c_int32), ("de_crossover", C.c_int32),
                ("ga_crossover", C.c_int32), ("init_lhs", C.c_int32), ("penalty", C.c_float), ("reserved", C.c_int32)]
    DE_MUTATION = {"best1": 0, "rand1": 1, "currenttobest1": 2, "randtobest1": 3, "best2": 4, "rand2": 5}
    DE_CROSSOVER = {"bin": 0, "exp": 1}
    GA_CROSSOVER = {"single_point": 0, "two_point": 1, "uniform": 2, "disruptive_uniform": 3}

    @classmethod
    def make(cls, aware=True, repair_mode=0, de_mutation="best1", de_crossover="bin", ga_crossover="single_point",
             init_lhs=False, penalty=1e20):
        g = lambda table, v: table[v] if isinstance(v, str) else int(v)
        return cls(int(bool(aware)), int(repair_mode), g(cls.DE_MUTATION, de_mutation), g(cls.DE_CROSSOVER, de_crossover),
                   g(cls.GA_CROSSOVER, ga_crossover), int(bool(init_lhs)), float(penalty), 0)


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build())
        vp, u8p, u32p, u64p, f32p, i32p, i64p = (C.c_void_p, C.POINTER(C.c_uint8), C.POINTER(C.c_uint32),
                                                 C.POINTER(C.c_uint64), C.POINTER(C.c_float),
                                                 C.POINTER(C.c_int32), C.POINTER(C.c_int64))
        sig = {
            "orc_philox4x32_10": (None, [u32p, u32p, u32p]),
            "orc_draw": (C.c_uint32, [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint32]),
            "orc_u01": (C.c_float, [C.c_uint32]),
            "orc_below": (C.c_uint32, [C.c_uint32, C.c_uint32]),
            "orc_exp_neg_spec": (C.c_float, [C.c_float]),
            "orc_exp_neg_spec_many": (None, [f32p, f32p, C.c_uint64]),
            "orc_de_mutate_index": (C.c_int, [C.c_float, C.c_int, C.c_int, C.c_int, C.c_int]),
            "orc_clamp_pos": (C.c_float, [C.c_float, C.c_float]),
            "orc_coord": (C.c_float, [C.c_int, C.c_int]),
            "orc_snap": (C.c_int, [C.c_int, C.c_int, C.c_float]),
            "orc_space_create": (vp, []),
            "orc_space_destroy": (None, [vp]),
            "orc_space_add_param": (C.c_int, [vp, i64p, C.c_int32]),
            "orc_space_add_constraint": (C.c_int, [vp, i32p, C.c_int32]),
            "orc_space_build": (C.c_int, [vp]),
            "orc_eval_program": (C.c_int, [i32p, C.c_int32, i64p, C.c_int32]),
            "orc_space_N": (C.c_uint64, [vp]), "orc_space_V": (C.c_uint64, [vp]), "orc_space_n": (C.c_int32, [vp]),
            "orc_space_bitmap": (u64p, [vp]), "orc_space_rows": (u8p, [vp]), "orc_space_Ltab": (u64p, [vp]),
            "orc_space_is_valid": (C.c_int, [vp, u8p]),
            "orc_space_count_range": (C.c_uint64, [vp, C.c_uint64, C.c_uint64]),
            "orc_space_repair": (None, [vp, u8p, C.c_uint64, u32p, u32p, u32p, u64p]),
            "orc_space_set_objective": (C.c_int, [vp, f32p]),
            "orc_runs_create": (vp, [vp, C.c_int, C.POINTER(HParams), C.c_uint32, C.c_uint32, C.c_int32,
                                     C.c_uint32, C.c_uint32, C.c_uint64]),
            "orc_runs_create_ex": (vp, [vp, C.c_int, C.POINTER(HParams), C.POINTER(Variant), C.c_uint32, C.c_uint32, C.c_int32,
                                        C.c_uint32, C.c_uint32, C.c_uint64]),
            "orc_runs_n_penalised": (C.c_uint64, [vp]), "orc_runs_tap_rule": (u8p, [vp]),
            "orc_space_neighbors": (C.c_uint64, [vp, u8p, C.c_int, u32p, C.c_uint64]),
            "orc_space_repair_mode": (None, [vp, C.c_int, u8p, f32p, u32p, C.c_uint64, u32p, u8p]),
            "orc_de_mutate_variant": (C.c_int, [C.c_int, C.c_float, C.c_int, C.c_int, i32p, C.c_int]),
            "orc_lhs_rows": (None, [vp, C.c_uint64, C.c_uint32, C.c_int32, u8p]),
            "orc_baseline": (C.c_double, [vp, C.c_uint64]),
            "orc_baseline_budget": (C.c_uint64, [vp, C.c_double]),
            "orc_runs_score": (C.c_double, [vp, u64p, C.c_uint32, C.POINTER(C.c_double)]),
            "orc_runs_destroy": (None, [vp]),
            "orc_runs_step": (None, [vp, C.c_uint32]),
            "orc_runs_gen": (C.c_uint32, [vp]),
            "orc_runs_best": (None, [vp, f32p, u32p, u32p, u32p]),
            "orc_runs_trajectory": (u8p, [vp]),
            "orc_runs_tap_cand": (u8p, [vp]), "orc_runs_tap_valid": (u8p, [vp]),
            "orc_runs_tap_rep": (u32p, [vp]), "orc_runs_tap_eval": (u32p, [vp]),
            "orc_runs_tap_f": (f32p, [vp]), "orc_runs_tap_accept": (u8p, [vp]), "orc_runs_tap_active": (u8p, [vp]),
            "orc_runs_n_repaired": (C.c_uint64, [vp]), "orc_runs_n_evaluated": (C.c_uint64, [vp]),
            "orc_runs_state": (None, [vp, C.c_int, vp]),
        }
        for name, (res, args) in sig.items():
            fn = getattr(L, name)
            fn.restype, fn.argtypes = res, args
        _lib = L
    return _lib


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t))


def philox4x32_10(ctr, key):
    c = np.asarray(ctr, dtype=np.uint32); k = np.asarray(key, dtype=np.uint32); o = np.zeros(4, np.uint32)
    lib().orc_philox4x32_10(_p(c, C.c_uint32), _p(k, C.c_uint32), _p(o, C.c_uint32))
    return o


def draw(seed, run, gen, ind, stream, slot):
    return lib().orc_draw(seed, run, gen, ind, STREAMS[stream] if isinstance(stream, str) else stream, slot)


def u01(w): return float(lib().orc_u01(w))
def below(w, k): return int(lib().orc_below(w, k))
def exp_neg_spec(z): return float(lib().orc_exp_neg_spec(C.c_float(z)))


def de_mutate_index(F, ibest, ia, ib, top): return int(lib().orc_de_mutate_index(C.c_float(F), ibest, ia, ib, top))
def clamp_pos(x, hi): return float(lib().orc_clamp_pos(C.c_float(x), C.c_float(hi)))
def coord(M, k): return float(lib().orc_coord(M, k))
def snap(M, m_d, x): return int(lib().orc_snap(M, m_d, C.c_float(x)))


def de_mutate_variant(op, F, xi, best, donors, top):
    r = np.zeros(5, np.int32); r[:len(donors)] = donors
    return int(lib().orc_de_mutate_variant(Variant.DE_MUTATION[op] if isinstance(op, str) else op, C.c_float(F), xi, best,
                                           _p(r, C.c_int32), top))


def exp_neg_spec_many(z: np.ndarray) -> np.ndarray:
    z = np.ascontiguousarray(z, dtype=np.float32); o = np.empty_like(z)
    lib().orc_exp_neg_spec_many(_p(z, C.c_float), _p(o, C.c_float), z.size)
    return o


def eval_program(words, values) -> int:
    w = np.asarray(words, dtype=np.int32); x = np.asarray(values, dtype=np.int64)
    return lib().orc_eval_program(_p(w, C.c_int32), w.size, _p(x, C.c_int64), x.size)


class OracleSpace:
    """P = (X, D, C), fully enumerated before tuning (L137)."""

    def __init__(self, domains, programs):
        L = lib()
        self._h = C.c_void_p(L.orc_space_create())
        for d in domains:
            a = np.asarray(d, dtype=np.int64)
            if L.orc_space_add_param(self._h, _p(a, C.c_int64), a.size) != 0:
                raise ValueError("bad parameter")
        for prog in programs:
            a = np.asarray(prog, dtype=np.int32)
            if L.orc_space_add_constraint(self._h, _p(a, C.c_int32), a.size) != 0:
                raise ValueError("bad constraint program")
        self.m = [len(d) for d in domains]
        self.built = False

    @classmethod
    def from_space(cls, sp):
        return cls(sp.domains, sp.rpn)

    def build(self):
        if lib().orc_space_build(self._h) != 0:
            raise RuntimeError("build failed")
        self.built = True
        return self

    @property
    def N(self): return int(lib().orc_space_N(self._h))
    @property
    def V(self): return int(lib().orc_space_V(self._h))
    @property
    def n(self): return len(self.m)

    def bitmap(self) -> np.ndarray:
        nw = (self.N + 63) // 64
        return np.ctypeslib.as_array(lib().orc_space_bitmap(self._h), shape=(nw,)).copy() if nw else np.zeros(0, np.uint64)

    def rows(self) -> np.ndarray:
        V, n = self.V, self.n
        if V == 0:
            return np.zeros((0, n), np.uint8)
        return np.ctypeslib.as_array(lib().orc_space_rows(self._h), shape=(V, n)).copy()

    def Ltab(self) -> np.ndarray:
        V = self.V
        return np.ctypeslib.as_array(lib().orc_space_Ltab(self._h), shape=(V,)).copy() if V else np.zeros(0, np.uint64)

    def is_valid(self, row) -> bool:
        a = np.ascontiguousarray(row, dtype=np.uint8)
        return bool(lib().orc_space_is_valid(self._h, _p(a, C.c_uint8)))

    def count_range(self, L0, L1) -> int:
        return int(lib().orc_space_count_range(self._h, L0, L1))

    def repair(self, rows):
        """rows (count, n) uint8 -> dict(rank, ham, sad, L): brute-force nearest valid (O9)."""
        a = np.ascontiguousarray(rows, dtype=np.uint8).reshape(-1, self.n)
        c = a.shape[0]
        rank, ham, sad, L = np.zeros(c, np.uint32), np.zeros(c, np.uint32), np.zeros(c, np.uint32), np.zeros(c, np.uint64)
        lib().orc_space_repair(self._h, _p(a, C.c_uint8), c, _p(rank, C.c_uint32), _p(ham, C.c_uint32),
                               _p(sad, C.c_uint32), _p(L, C.c_uint64))
        return dict(rank=rank, ham=ham, sad=sad, L=L)

    def set_objective(self, obj):
        a = np.ascontiguousarray(obj, dtype=np.float32)
        assert a.size == self.V
        if lib().orc_space_set_objective(self._h, _p(a, C.c_float)) != 0:
            raise RuntimeError("set_objective before build")
        self._obj = a

    # -- neighbour rules (L139-143) and the paper's repairs (L270, Alg.2, Alg.3)
    def neighbors(self, row, rule) -> np.ndarray:
        """Ranks of the valid neighbours of `row`; rule 0 strictly-adjacent, 1 adjacent, 2 Hamming."""
        a = np.ascontiguousarray(row, dtype=np.uint8)
        out = np.zeros(max(self.V, 1), np.uint32)
        c = lib().orc_space_neighbors(self._h, _p(a, C.c_uint8), rule, _p(out, C.c_uint32), out.size)
        return out[:c].copy()

    def repair_mode(self, mode, rows, x=None, w=None):
        """mode 'index' (L270) | 'alg2' (needs x: continuous positions) | 'alg3' (needs w: 32-bit draws) -> (rank, rule)."""
        m = {"index": 1, "alg2": 2, "alg3": 3}[mode]
        a = np.ascontiguousarray(rows, dtype=np.uint8).reshape(-1, self.n)
        c = a.shape[0]
        xx = np.ascontiguousarray(x if x is not None else np.zeros((c, self.n)), dtype=np.float32)
        ww = np.ascontiguousarray(w if w is not None else np.zeros(c), dtype=np.uint32)
        rank, rule = np.zeros(c, np.uint32), np.zeros(c, np.uint8)
        lib().orc_space_repair_mode(self._h, m, _p(a, C.c_uint8), _p(xx, C.c_float), _p(ww, C.c_uint32), c,
                                    _p(rank, C.c_uint32), _p(rule, C.c_uint8))
        return rank, rule

    def lhs_rows(self, seed, run_id, pop) -> np.ndarray:
        out = np.zeros((pop, self.n), np.uint8)
        lib().orc_lhs_rows(self._h, seed, run_id, pop, _p(out, C.c_uint8))
        return out

    # -- NEXT-4
    def baseline(self, t) -> float:
        return float(lib().orc_baseline(self._h, int(t)))

    def baseline_budget(self, frac=0.95) -> int:
        return int(lib().orc_baseline_budget(self._h, float(frac)))

    def __del__(self):
        try:
            lib().orc_space_destroy(self._h)
        except Exception:
            pass


class OracleRuns:
    def __init__(self, space: OracleSpace, algo, n_runs, pop, budget=0, max_gens=0xFFFFFFFF, seed=0,
                 first_run=0, hparams: HParams | None = None, variant: Variant | None = None):
        self.space, self.R, self.P, self.n = space, int(n_runs), int(pop), space.n
        self.algo = ALGOS[algo] if isinstance(algo, str) else int(algo)
        self.hp = hparams or HParams.default()
        self.variant = variant or Variant.make()
        h = lib().orc_runs_create_ex(space._h, self.algo, C.byref(self.hp), C.byref(self.variant), self.R, first_run, self.P,
                                     budget, max_gens, seed)
        if not h:
            raise ValueError("orc_runs_create rejected the arguments")
        self._h = C.c_void_p(h)

    def step(self, k=1):
        lib().orc_runs_step(self._h, k)

    @property
    def gen(self): return int(lib().orc_runs_gen(self._h))

    def best(self):
        R = self.R
        bf, br, uq, gd = np.zeros(R, np.float32), np.zeros(R, np.uint32), np.zeros(R, np.uint32), np.zeros(R, np.uint32)
        lib().orc_runs_best(self._h, _p(bf, C.c_float), _p(br, C.c_uint32), _p(uq, C.c_uint32), _p(gd, C.c_uint32))
        return dict(best_f=bf, best_rank=br, uniq=uq, gens_done=gd)

    def trajectory(self) -> np.ndarray:
        """(gen+1, R) structured {best_f f32, best_rank u32, uniq u32}, packed little-endian 12-byte rows."""
        G = self.gen + 1
        raw = np.ctypeslib.as_array(lib().orc_runs_trajectory(self._h), shape=(G * self.R * 12,)).copy()
        dt = np.dtype([("best_f", "<f4"), ("best_rank", "<u4"), ("uniq", "<u4")])
        return raw.view(dt).reshape(G, self.R)

    def taps(self):
        R, P, n = self.R, self.P, self.n
        g = lambda fn, shape: np.ctypeslib.as_array(fn(self._h), shape=shape).copy()
        L = lib()
        return dict(cand=g(L.orc_runs_tap_cand, (R, P, n)), valid=g(L.orc_runs_tap_valid, (R, P)),
                    rep_rank=g(L.orc_runs_tap_rep, (R, P)), eval_rank=g(L.orc_runs_tap_eval, (R, P)),
                    f=g(L.orc_runs_tap_f, (R, P)), accept=g(L.orc_runs_tap_accept, (R, P)),
                    active=g(L.orc_runs_tap_active, (R,)), rule=g(L.orc_runs_tap_rule, (R, P)))

    @property
    def n_repaired(self): return int(lib().orc_runs_n_repaired(self._h))
    @property
    def n_evaluated(self): return int(lib().orc_runs_n_evaluated(self._h))
    @property
    def n_penalised(self): return int(lib().orc_runs_n_penalised(self._h))

    def score(self, t):
        """NEXT-4 (Eq.2): (score, per-sampling-point means) for the sampling points t (unique-evaluation counts)."""
        tt = np.ascontiguousarray(t, dtype=np.uint64)
        per = np.zeros(tt.size, np.float64)
        sc = lib().orc_runs_score(self._h, _p(tt, C.c_uint64), tt.size, per.ctypes.data_as(C.POINTER(C.c_double)))
        return float(sc), per

    def state(self):
        R, P, n = self.R, self.P, self.n
        out = {}
        def grab(which, dtype, shape):
            a = np.zeros(shape, dtype)
            lib().orc_runs_state(self._h, which, a.ctypes.data_as(C.c_void_p))
            return a
        out["rank"] = grab(1, np.uint32, (R, P))
        out["f"] = grab(2, np.float32, (R, P))
        if self.algo in (0, 3):
            out["idx"] = grab(0, np.uint8, (R, P, n))
        else:
            out["x"] = grab(3, np.float32, (R, P, n))
        if self.algo == 1:
            out["v"] = grab(4, np.float32, (R, P, n))
            out["pbest"] = grab(5, np.float32, (R, P, n))
            out["pbest_f"] = grab(6, np.float32, (R, P))
        return out

    def __del__(self):
        try:
            lib().orc_runs_destroy(self._h)
        except Exception:
            pass

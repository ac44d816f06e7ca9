"""ctypes binding of include/cao.h: same names, argument marshalling only.

PyTorch is used for device memory (``torch.empty(..., device='cuda')``) and the current stream.
The product path never imports ``oracle`` and has no CPU fallback.
"""
from __future__ import annotations
import ctypes as C
import os
import numpy as np
import torch

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libcao.so")
ALGOS = {"de": 0, "pso": 1, "firefly": 2, "ga": 3}

CAO_ERRORS = {-1: "CAO_E_INVALID_ARG", -2: "CAO_E_STATE", -3: "CAO_E_TOO_LARGE", -4: "CAO_E_EMPTY_SPACE",
              -5: "CAO_E_POP_GT_VALID", -6: "CAO_E_WORKSPACE", -7: "CAO_E_CUDA"}


class CaoError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"{CAO_ERRORS.get(code, code)}: {msg}")
        self.code = code


class HParams(C.Structure):
    """cao_hparams; defaults from Table IV, ga_beta_b per reading A18."""
    _fields_ = [("de_F", C.c_float), ("de_CR", C.c_float),
                ("pso_w", C.c_float), ("pso_c1", C.c_float), ("pso_c2", C.c_float),
                ("ff_B0", C.c_float), ("ff_gamma", C.c_float), ("ff_alpha", C.c_float),
                ("ga_mutation_chance", C.c_int32), ("ga_beta_b", C.c_int32)]

    @classmethod
    def default(cls):
        return cls(0.7, 0.6, 0.5, 3.0, 0.5, 1.0, 1.0, 0.2, 5, 3)


class Variant(C.Structure):
    """cao_variant: the SURVEY 8(f) switches (include/cao.h); the default is the north_star path."""
    _fields_ = [("constraint_aware", C.c_int32), ("repair_mode", C.c_int32), ("de_mutation", C.c_int32),
                ("de_crossover", C.c_int32), ("ga_crossover", C.c_int32), ("init_lhs", C.c_int32), ("penalty", C.c_float),
                ("reserved", C.c_int32)]
    DE_MUTATION = {"best1": 0, "rand1": 1, "currenttobest1": 2, "randtobest1": 3, "best2": 4, "rand2": 5}
    DE_CROSSOVER = {"bin": 0, "exp": 1}
    GA_CROSSOVER = {"single_point": 0, "two_point": 1, "uniform": 2, "disruptive_uniform": 3}

    @classmethod
    def make(cls, aware=True, repair_mode=0, de_mutation="best1", de_crossover="bin", ga_crossover="single_point",
             init_lhs=False, penalty=1e20):
        g = lambda table, v: table[v] if isinstance(v, str) else int(v)
        return cls(int(bool(aware)), int(repair_mode), g(cls.DE_MUTATION, de_mutation), g(cls.DE_CROSSOVER, de_crossover),
                   g(cls.GA_CROSSOVER, ga_crossover), int(bool(init_lhs)), float(penalty), 0)


vp, u64, u32, i32 = C.c_void_p, C.c_uint64, C.c_uint32, C.c_int32
pu64, pi32, pvp = C.POINTER(C.c_uint64), C.POINTER(C.c_int32), C.POINTER(C.c_void_p)

# name -> (restype, argtypes): every symbol include/cao.h declares
SIGNATURES = {
    "cao_space_create": (C.c_int, [pvp]),
    "cao_space_destroy": (None, [vp]),
    "cao_space_add_param": (C.c_int, [vp, C.c_char_p, C.POINTER(C.c_int64), i32]),
    "cao_space_add_constraint": (C.c_int, [vp, pi32, i32]),
    "cao_space_set_build_mode": (C.c_int, [vp, i32]),
    "cao_space_build_workspace_bytes": (C.c_int, [vp, pu64, pu64]),
    "cao_space_set_probe_levels": (C.c_int, [vp, i32]),
    "cao_space_probe_levels": (C.c_int, [vp, pi32]),
    "cao_space_build_count": (C.c_int, [vp, vp, vp, vp, pu64]),
    "cao_space_table_bytes": (C.c_int, [vp, pu64]),
    "cao_space_build_fill": (C.c_int, [vp, vp, vp]),
    "cao_space_rebuild": (C.c_int, [vp, vp]),
    "cao_space_sizes": (C.c_int, [vp, pu64, pu64, pi32, pi32]),
    "cao_space_ltab_bytes": (C.c_int, [vp, pi32]),
    "cao_space_build_stats": (C.c_int, [vp, vp, pu64]),
    "cao_space_views": (C.c_int, [vp, pvp, pvp, pvp, pvp]),
    "cao_space_is_valid": (C.c_int, [vp, vp, u64, vp, vp]),
    "cao_space_repair_scratch_bytes": (C.c_int, [vp, u64, pu64]),
    "cao_space_repair": (C.c_int, [vp, vp, u64, vp, vp, i32, vp, vp]),
    "cao_space_repair_noalloc": (C.c_int, [vp, vp, u64, vp, vp, i32, vp]),
    "cao_space_set_objective": (C.c_int, [vp, vp]),
    "cao_runs_workspace_bytes": (C.c_int, [vp, i32, i32, u32, u32, pu64]),
    "cao_runs_create": (C.c_int, [vp, i32, C.POINTER(HParams), u32, u32, i32, u32, u32, u64, vp, vp, pvp]),
    "cao_runs_workspace_bytes_ex": (C.c_int, [vp, i32, C.POINTER(Variant), i32, u32, u32, pu64]),
    "cao_runs_create_ex": (C.c_int, [vp, i32, C.POINTER(HParams), C.POINTER(Variant), u32, u32, i32, u32, u32, u64, vp, vp, pvp]),
    "cao_runs_debug_rule": (C.c_int, [vp, pvp]),
    "cao_space_repair_mode_scratch_bytes": (C.c_int, [vp, u64, pu64]),
    "cao_space_repair_mode": (C.c_int, [vp, i32, vp, vp, vp, u64, vp, vp, vp, vp]),
    "cao_space_sort_objective": (C.c_int, [vp, vp, vp, vp]),
    "cao_space_baseline": (C.c_int, [vp, vp, vp, u32, vp, vp]),
    "cao_runs_score": (C.c_int, [vp, vp, vp, vp, u32, vp, vp, vp, vp]),
    "cao_runs_destroy": (None, [vp]),
    "cao_runs_set_mode": (C.c_int, [vp, i32]),
    "cao_runs_mode": (C.c_int, [vp, pi32]),
    "cao_runs_step": (C.c_int, [vp, u32, vp]),
    "cao_runs_set_fused_width": (C.c_int, [vp, i32]),
    "cao_runs_fused_width": (C.c_int, [vp, pi32]),
    "cao_runs_best": (C.c_int, [vp, vp, vp, vp, vp, vp]),
    "cao_runs_trajectory": (C.c_int, [vp, pvp, C.POINTER(u32)]),
    "cao_runs_debug_last": (C.c_int, [vp, pvp, pvp, pvp, pvp, pvp, pvp, pvp]),
    "cao_runs_debug_state": (C.c_int, [vp, i32, pvp, pu64]),
    "cao_runs_counters": (C.c_int, [vp, vp, pu64, pu64, pu64]),
    "cao_runs_stats": (C.c_int, [vp, vp, pu64]),
    "cao_launch_count": (u64, []),
    "cao_profile_enable": (C.c_int, [i32]),
    "cao_profile_read": (C.c_int, [i32, C.POINTER(C.c_double), pu64]),
    "cao_profile_name": (C.c_char_p, [i32]),
    "cao_test_philox": (C.c_int, [vp, vp, u64, vp]),
    "cao_test_curand_philox": (C.c_int, [vp, vp, u64, vp]),
    "cao_test_exp_neg": (C.c_int, [vp, vp, u64, vp]),
    "cao_test_int_peak": (C.c_int, [i32, u32, u32, vp, vp]),
    "cao_last_error": (C.c_char_p, []),
}

_lib = None


def lib():
    """Loads libcao.so (built by paper_2606_28372_b200/build.py); raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2606_28372_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(L, name)
            fn.restype, fn.argtypes = res, args
        _lib = L
    return _lib


def _check(rc):
    if rc != 0:
        raise CaoError(rc, (lib().cao_last_error() or b"").decode())


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _dev_bytes(nbytes, device):
    # torch's caching allocator returns >= 512-byte aligned blocks
    t = torch.empty(max(int(nbytes), 1), dtype=torch.uint8, device=device)
    assert t.data_ptr() % 256 == 0
    return t


def launch_count() -> int:
    return int(lib().cao_launch_count())


def profile_enable(on=True):
    _check(lib().cao_profile_enable(1 if on else 0))


def profile_read():
    """{kernel class name: (total ms, launches)} since profile_enable(True)."""
    out = {}
    cls = 0
    while True:
        name = lib().cao_profile_name(cls).decode()
        if not name:                                   # "" beyond the last class
            return out
        ms, n = C.c_double(), u64()
        _check(lib().cao_profile_read(cls, C.byref(ms), C.byref(n)))
        out[name] = (ms.value, n.value)
        cls += 1


def _view(base: torch.Tensor, ptr: int, nbytes: int, dtype, shape):
    off = ptr - base.data_ptr()
    assert 0 <= off and off + nbytes <= base.numel(), "borrowed view outside its buffer"
    return base[off:off + nbytes].view(dtype).view(*shape)


class Space:
    """P = (X, D, C), resolved on the GPU before tuning (L137)."""

    def __init__(self, domains, programs, names=None, build_mode=0, device="cuda", probe_levels=-1):
        L = lib()
        self.device = torch.device(device)
        h = C.c_void_p()
        _check(L.cao_space_create(C.byref(h)))
        self._h = h
        self.m = [len(d) for d in domains]
        for k, d in enumerate(domains):
            a = np.ascontiguousarray(d, dtype=np.int64)
            nm = (names[k] if names else f"p{k}").encode()
            _check(L.cao_space_add_param(h, nm, a.ctypes.data_as(C.POINTER(C.c_int64)), a.size))
        for prog in programs:
            a = np.ascontiguousarray(prog, dtype=np.int32)
            _check(L.cao_space_add_constraint(h, a.ctypes.data_as(pi32), a.size))
        _check(L.cao_space_set_build_mode(h, build_mode))
        _check(L.cao_space_set_probe_levels(h, probe_levels))
        self.built = False
        self._bitmap = self._scratch = self._table = self._obj = None

    @classmethod
    def from_space(cls, sp, **kw):
        return cls(sp.domains, sp.rpn, names=sp.param_names, **kw)

    # -- S1
    def alloc_build(self):
        bb, sb = u64(), u64()
        _check(lib().cao_space_build_workspace_bytes(self._h, C.byref(bb), C.byref(sb)))
        self._bitmap = _dev_bytes(bb.value, self.device)
        self._scratch = _dev_bytes(sb.value, self.device)

    def build_count(self) -> int:
        V = u64()
        _check(lib().cao_space_build_count(self._h, self._bitmap.data_ptr(), self._scratch.data_ptr(), _stream(), C.byref(V)))
        return V.value

    def alloc_table(self):
        tb = u64()
        _check(lib().cao_space_table_bytes(self._h, C.byref(tb)))
        if self._table is None or self._table.numel() < tb.value:
            self._table = _dev_bytes(tb.value, self.device)

    def build_fill(self):
        _check(lib().cao_space_build_fill(self._h, self._table.data_ptr(), _stream()))
        self.built = True

    def build(self):
        """cao_space_build_count + cao_space_build_fill with freshly allocated buffers; returns self."""
        if self._bitmap is None:
            self.alloc_build()
        self.build_count()
        self.alloc_table()
        self.build_fill()
        return self

    def rebuild(self):
        """All of S1 again into the same buffers, asynchronously (no host round trip)."""
        _check(lib().cao_space_rebuild(self._h, _stream()))

    def sizes(self):
        N, V, n, rb = u64(), u64(), i32(), i32()
        _check(lib().cao_space_sizes(self._h, C.byref(N), C.byref(V), C.byref(n), C.byref(rb)))
        return N.value, V.value, n.value, rb.value

    @property
    def N(self): return self.sizes()[0]
    @property
    def V(self): return self.sizes()[1]
    @property
    def n(self): return len(self.m)
    @property
    def row_bytes(self): return 16 if self.n <= 16 else 32

    def _views(self):
        p = [C.c_void_p() for _ in range(4)]
        _check(lib().cao_space_views(self._h, *[C.byref(x) for x in p]))
        return [x.value for x in p]

    def bitmap(self) -> torch.Tensor:
        """ceil(N/64) int64 words (bit L&63 of word L>>6)."""
        nw = (self.N + 63) // 64
        return self._bitmap[:nw * 8].view(torch.int64)

    def rows(self) -> torch.Tensor:
        """(V, row_bytes) uint8, ascending L, padding zero."""
        N, V, n, rb = self.sizes()
        return _view(self._table, self._views()[1], V * rb, torch.uint8, (V, rb))

    def build_stats(self):
        a = (C.c_uint64 * 4)()
        _check(lib().cao_space_build_stats(self._h, _stream(), a))
        return dict(n_blocks=int(a[0]), live_blocks=int(a[1]), nonempty_groups=int(a[2]), B=int(a[3]))

    @property
    def ltab_bytes(self) -> int:
        v = i32()
        _check(lib().cao_space_ltab_bytes(self._h, C.byref(v)))
        return v.value

    def Ltab(self) -> torch.Tensor:
        """V linear indices, ascending: int32 bit patterns of u32 when N <= 2^32, else int64."""
        N, V, n, rb = self.sizes()
        lb = self.ltab_bytes
        return _view(self._table, self._views()[2], V * lb, torch.int32 if lb == 4 else torch.int64, (V,))

    def rank_dir(self) -> torch.Tensor:
        N, V, n, rb = self.sizes()
        nd = (N + 511) // 512 + 1
        return _view(self._table, self._views()[3], nd * 4, torch.int32, (nd,))

    # -- queries (L139)
    def pack_rows(self, rows) -> torch.Tensor:
        """(count, n) host/device integer rows -> (count, row_bytes) uint8 device rows, padding zero."""
        t = torch.as_tensor(np.ascontiguousarray(rows)) if not isinstance(rows, torch.Tensor) else rows
        t = t.to(self.device).to(torch.uint8).reshape(-1, t.shape[-1])
        if t.shape[1] == self.row_bytes:
            return t.contiguous()
        out = torch.zeros((t.shape[0], self.row_bytes), dtype=torch.uint8, device=self.device)
        out[:, :t.shape[1]] = t
        return out

    def is_valid(self, rows) -> torch.Tensor:
        r = self.pack_rows(rows)
        out = torch.empty(r.shape[0], dtype=torch.uint8, device=self.device)
        _check(lib().cao_space_is_valid(self._h, r.data_ptr(), r.shape[0], out.data_ptr(), _stream()))
        return out

    @property
    def probe_levels(self):
        v = i32()
        _check(lib().cao_space_probe_levels(self._h, C.byref(v)))
        return v.value

    def repair(self, rows, use_probe=True):
        """-> (rank int32-as-uint32 tensor, key int64 tensor: ham << 45 | sad << 32 | rank).
        use_probe: True = the library's probe level, False = scan only, or an explicit level 0..3."""
        use_probe = -1 if use_probe is True else 0 if use_probe is False else int(use_probe)
        r = self.pack_rows(rows)
        c = r.shape[0]
        sb = u64()
        _check(lib().cao_space_repair_scratch_bytes(self._h, c, C.byref(sb)))
        scratch = _dev_bytes(sb.value, self.device)
        rank = torch.empty(c, dtype=torch.int32, device=self.device)
        key = torch.empty(c, dtype=torch.int64, device=self.device)
        _check(lib().cao_space_repair(self._h, r.data_ptr(), c, rank.data_ptr(), key.data_ptr(), use_probe,
                                      scratch.data_ptr(), _stream()))
        self._last_scratch = scratch
        return rank, key

    REPAIR_NOALLOC_MAX_ROWS = 65536

    def repair_noalloc(self, rows, rank_out=None, key_out=None, use_probe=True):
        """cao_space_repair_noalloc: the repair of ``repair`` for code that may not allocate device memory when it runs
        (an allocator or memory-pool callback, a plugin that is only lent buffers and a stream, a process whose device
        memory is already fully reserved).  The scratch is a fixed 3 MiB array inside libcao.so, so at most
        REPAIR_NOALLOC_MAX_ROWS rows per call (CaoError CAO_E_TOO_LARGE beyond), and calls must not overlap on the GPU.

        This wrapper allocates nothing either, so everything is the caller's and already on the device:
        rows (count, row_bytes) uint8, contiguous, padding bytes zero or not (they are ignored) -- see ``pack_rows``;
        rank_out (count,) int32 and/or key_out (count,) int64 receive the results (uint32 / uint64 bit patterns)."""
        use_probe = -1 if use_probe is True else 0 if use_probe is False else int(use_probe)
        c = int(rows.shape[0])
        if not (rows.is_cuda and rows.dtype == torch.uint8 and rows.is_contiguous() and rows.dim() == 2 and
                rows.shape[1] == self.row_bytes):
            raise ValueError("repair_noalloc: rows must be a contiguous (count, row_bytes) uint8 CUDA tensor (pack_rows)")
        for t, dt in ((rank_out, torch.int32), (key_out, torch.int64)):
            if t is not None and not (t.is_cuda and t.dtype == dt and t.is_contiguous() and t.numel() >= c):
                raise ValueError("repair_noalloc: outputs must be contiguous CUDA tensors, int32 ranks / int64 keys, count long")
        _check(lib().cao_space_repair_noalloc(self._h, rows.data_ptr(), c,
                                              rank_out.data_ptr() if rank_out is not None else None,
                                              key_out.data_ptr() if key_out is not None else None, use_probe, _stream()))
        return rank_out, key_out

    def repair_mode(self, mode, rows, x=None, w=None):
        """NEXT-1 standalone: mode 'index' (L270) | 'alg2' (x: continuous positions) | 'alg3' (w: 32-bit draws)
        -> (rank int32 tensor, 0xFFFFFFFF = unrepaired; rule uint8 tensor)."""
        m = {"index": 1, "alg2": 2, "alg3": 3}[mode]
        r = self.pack_rows(rows)
        c = r.shape[0]
        sb = u64()
        _check(lib().cao_space_repair_mode_scratch_bytes(self._h, c, C.byref(sb)))
        scratch = _dev_bytes(sb.value, self.device)
        rank = torch.empty(c, dtype=torch.int32, device=self.device)
        rule = torch.empty(c, dtype=torch.uint8, device=self.device)
        xx = torch.as_tensor(np.ascontiguousarray(x, dtype=np.float32)).to(self.device).contiguous() if x is not None else None
        ww = torch.as_tensor(np.ascontiguousarray(w, dtype=np.uint32).view(np.int32)).to(self.device).contiguous() if w is not None else None
        _check(lib().cao_space_repair_mode(self._h, m, r.data_ptr(), xx.data_ptr() if xx is not None else None,
                                           ww.data_ptr() if ww is not None else None, c, rank.data_ptr(), rule.data_ptr(),
                                           scratch.data_ptr(), _stream()))
        self._last_scratch = (scratch, xx, ww, r)
        return rank, rule

    # -- NEXT-4
    def sorted_objective(self) -> torch.Tensor:
        V = self.V
        n2 = 1
        while n2 < V:
            n2 <<= 1
        out = torch.empty(V, dtype=torch.float32, device=self.device)
        scratch = _dev_bytes(n2 * 4, self.device)
        _check(lib().cao_space_sort_objective(self._h, out.data_ptr(), scratch.data_ptr(), _stream()))
        self._sort_scratch = scratch
        return out

    def baseline(self, sorted_obj: torch.Tensor, t) -> torch.Tensor:
        tt = torch.as_tensor(np.ascontiguousarray(t, dtype=np.int64)).to(self.device)
        B = torch.empty(tt.numel(), dtype=torch.float64, device=self.device)
        _check(lib().cao_space_baseline(self._h, sorted_obj.data_ptr(), tt.data_ptr(), tt.numel(), B.data_ptr(), _stream()))
        self._base_keep = tt
        return B

    def set_objective(self, obj):
        t = obj if isinstance(obj, torch.Tensor) else torch.from_numpy(np.ascontiguousarray(obj, dtype=np.float32))
        t = t.to(self.device, dtype=torch.float32).contiguous()
        assert t.numel() == self.V
        _check(lib().cao_space_set_objective(self._h, t.data_ptr()))
        self._obj = t

    def __del__(self):
        try:
            lib().cao_space_destroy(self._h)
        except Exception:
            pass


class Runs:
    """n_runs independent simulated tuning runs of one algorithm; creation executes generation 0 (S2)."""

    def __init__(self, space: Space, algo, n_runs, pop, budget=0, max_gens=100, seed=0, first_run=0, hparams=None,
                 mode=None, variant: Variant | None = None, fused_width=None):
        self.space, self.R, self.P, self.n = space, int(n_runs), int(pop), space.n
        self.algo = ALGOS[algo] if isinstance(algo, str) else int(algo)
        self.hp = hparams or HParams.default()
        self.variant = variant
        vref = C.byref(variant) if variant is not None else None
        self.max_gens = int(max_gens)
        wb = u64()
        _check(lib().cao_runs_workspace_bytes_ex(space._h, self.algo, vref, self.P, self.R, self.max_gens, C.byref(wb)))
        self.workspace_bytes = wb.value
        self._ws = _dev_bytes(wb.value, space.device)
        h = C.c_void_p()
        _check(lib().cao_runs_create_ex(space._h, self.algo, C.byref(self.hp), vref, self.R, int(first_run), self.P, int(budget),
                                        self.max_gens, int(seed), self._ws.data_ptr(), _stream(), C.byref(h)))
        self._h = h
        if mode is not None:
            self.set_mode(mode)
        if fused_width is not None:
            _check(lib().cao_runs_set_fused_width(self._h, int(fused_width)))

    @property
    def fused_width(self) -> int:
        v = i32()
        _check(lib().cao_runs_fused_width(self._h, C.byref(v)))
        return v.value

    def set_mode(self, mode):
        """'fused' / 1 = one persistent kernel per step call; 'phased' / 0 = per-generation kernels."""
        m = {"fused": 1, "phased": 0}.get(mode, mode)
        _check(lib().cao_runs_set_mode(self._h, int(m)))

    @property
    def mode(self) -> str:
        v = i32()
        _check(lib().cao_runs_mode(self._h, C.byref(v)))
        return "fused" if v.value == 1 else "phased"

    def step(self, k=1):
        _check(lib().cao_runs_step(self._h, int(k), _stream()))

    def best_into(self, best_f, best_rank, uniq, gens_done):
        _check(lib().cao_runs_best(self._h, best_f.data_ptr(), best_rank.data_ptr(), uniq.data_ptr(), gens_done.data_ptr(),
                                   _stream()))

    def best(self):
        dev = self.space.device
        bf = torch.empty(self.R, dtype=torch.float32, device=dev)
        br, uq, gd = (torch.empty(self.R, dtype=torch.int32, device=dev) for _ in range(3))
        self.best_into(bf, br, uq, gd)
        return dict(best_f=bf, best_rank=br, uniq=uq, gens_done=gd)

    @property
    def gen(self):
        p, g = C.c_void_p(), u32()
        _check(lib().cao_runs_trajectory(self._h, C.byref(p), C.byref(g)))
        return g.value

    def trajectory(self) -> torch.Tensor:
        """(gen+1, R, 3) int32: {best_f bits, best_rank, uniq}."""
        p, g = C.c_void_p(), u32()
        _check(lib().cao_runs_trajectory(self._h, C.byref(p), C.byref(g)))
        G = g.value + 1
        return _view(self._ws, p.value, G * self.R * 12, torch.int32, (G, self.R, 3))

    def taps(self):
        p = [C.c_void_p() for _ in range(7)]
        _check(lib().cao_runs_debug_last(self._h, *[C.byref(x) for x in p]))
        R, P, rb = self.R, self.P, self.space.row_bytes
        v = lambda k, nb, dt, shape: _view(self._ws, p[k].value, nb, dt, shape)
        return dict(cand=v(0, R * P * rb, torch.uint8, (R, P, rb)), valid=v(1, R * P, torch.uint8, (R, P)),
                    rep_rank=v(2, R * P * 4, torch.int32, (R, P)), eval_rank=v(3, R * P * 4, torch.int32, (R, P)),
                    f=v(4, R * P * 4, torch.float32, (R, P)), accept=v(5, R * P, torch.uint8, (R, P)),
                    active=v(6, R, torch.uint8, (R,)))

    def rule_tap(self) -> torch.Tensor:
        """NEXT-1: (R, P) uint8 neighbour rule of the last generation's repairs (runs with a non-default variant)."""
        p = C.c_void_p()
        _check(lib().cao_runs_debug_rule(self._h, C.byref(p)))
        return _view(self._ws, p.value, self.R * self.P, torch.uint8, (self.R, self.P))

    def score(self, sorted_obj: torch.Tensor, t, B: torch.Tensor | None = None):
        """NEXT-4 (Eq.2): (score, per-sampling-point means) as device float64 tensors."""
        dev = self.space.device
        tt = torch.as_tensor(np.ascontiguousarray(t, dtype=np.int64)).to(dev)
        if B is None:
            B = self.space.baseline(sorted_obj, t)
        per = torch.empty(tt.numel(), dtype=torch.float64, device=dev)
        sc = torch.empty(1, dtype=torch.float64, device=dev)
        scratch = _dev_bytes(tt.numel() * self.R * 8, dev)
        _check(lib().cao_runs_score(self._h, sorted_obj.data_ptr(), tt.data_ptr(), B.data_ptr(), tt.numel(), per.data_ptr(),
                                    sc.data_ptr(), scratch.data_ptr(), _stream()))
        self._score_keep = (tt, scratch, B)
        return sc, per

    def _state(self, which, dtype, shape):
        p, b = C.c_void_p(), u64()
        _check(lib().cao_runs_debug_state(self._h, which, C.byref(p), C.byref(b)))
        return _view(self._ws, p.value, b.value, dtype, shape)

    def state(self):
        """Population state; x / v / pbest are returned as (R, P, n) (stored dimension-major [run][dim][ind])."""
        R, P, n, rb = self.R, self.P, self.n, self.space.row_bytes
        out = dict(rank=self._state(1, torch.int32, (R, P)), f=self._state(2, torch.float32, (R, P)))
        if self.algo in (0, 3):
            out["idx"] = self._state(0, torch.uint8, (R, P, rb))[:, :, :n]
        else:
            out["x"] = self._state(3, torch.float32, (R, n, P)).permute(0, 2, 1)
        if self.algo == 1:
            out["v"] = self._state(4, torch.float32, (R, n, P)).permute(0, 2, 1)
            out["pbest"] = self._state(5, torch.float32, (R, n, P)).permute(0, 2, 1)
            out["pbest_f"] = self._state(6, torch.float32, (R, P))
        return out

    def counters(self):
        a, b, c = u64(), u64(), u64()
        _check(lib().cao_runs_counters(self._h, _stream(), C.byref(a), C.byref(b), C.byref(c)))
        return dict(n_repaired=a.value, n_scanned=b.value, n_evaluated=c.value)

    def stats(self):
        """cao_runs_stats: the sixteen statistics words as a dict."""
        a = (C.c_uint64 * 32)()
        _check(lib().cao_runs_stats(self._h, _stream(), a))
        names = ["n_repaired", "n_scanned", "n_evaluated", "n_probe2", "n_probe3", "n_memo", "n_rcache", "n_penalised",
                 "cyc_op", "cyc_tail", "cyc_probe2", "cyc_probe3", "cyc_scan", "cyc_finish", "cyc_max_run", "cyc_max_scan"]
        out = {k: int(v) for k, v in zip(names, a)}
        out["ham_hist"] = [int(a[16 + h]) for h in range(9)]
        return out

    def __del__(self):
        try:
            lib().cao_runs_destroy(self._h)
        except Exception:
            pass


def test_philox(ctr_key: torch.Tensor) -> torch.Tensor:
    """(count, 6) int32 {c0,c1,c2,c3,k0,k1} -> (count, 4) int32 Philox4x32-10 outputs (device self-test, O3)."""
    t = ctr_key.contiguous()
    out = torch.empty((t.shape[0], 4), dtype=torch.int32, device=t.device)
    _check(lib().cao_test_philox(t.data_ptr(), out.data_ptr(), t.shape[0], _stream()))
    return out


def test_curand_philox(ctr_key: torch.Tensor) -> torch.Tensor:
    """Same as test_philox, but computed by cuRAND's curand_Philox4x32_10 device function."""
    t = ctr_key.contiguous()
    out = torch.empty((t.shape[0], 4), dtype=torch.int32, device=t.device)
    _check(lib().cao_test_curand_philox(t.data_ptr(), out.data_ptr(), t.shape[0], _stream()))
    return out


def test_exp_neg(z: torch.Tensor) -> torch.Tensor:
    t = z.contiguous()
    out = torch.empty_like(t)
    _check(lib().cao_test_exp_neg(t.data_ptr(), out.data_ptr(), t.numel(), _stream()))
    return out


INT_PEAK_KINDS = {"imad": 0, "lop3": 1, "vabsdiff4": 2, "popc": 3, "iadd": 4, "idp4a": 5}


def int_peak(kind: str, iters=4096, n_ctas=148 * 8, reps=5) -> float:
    """Measured issue rate of one integer instruction kind in lane-operations per second (cao_test_int_peak timed
    with CUDA events on the current stream, best of `reps`)."""
    out = torch.empty(n_ctas * 256, dtype=torch.int32, device="cuda")
    best = None
    for _ in range(reps + 1):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        _check(lib().cao_test_int_peak(INT_PEAK_KINDS[kind], iters, n_ctas, out.data_ptr(), _stream()))
        e1.record(); e1.synchronize()
        ms = e0.elapsed_time(e1)
        best = ms if best is None else min(best, ms)
    return n_ctas * 256 * iters * 8 / (best / 1e3)


test_philox.__test__ = False
test_curand_philox.__test__ = False
test_exp_neg.__test__ = False

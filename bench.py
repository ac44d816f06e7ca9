#!/usr/bin/env python
"""bench.py -- whole-hot-path throughput of the batched constraint-aware generation step on B200.

One "step" = one pass of every S-row of the hot path over one batch of synthetic input:
  S1  build the search space on the GPU (bitmap, valid table, rank directory)
  S2  create R runs of each algorithm (generation 0)
  S3-S7  step every run until its budget of unique evaluations / the generation cap
  read best-so-far.
Workload at N=1: BASELINE.json names no config for its metric, so the default is the largest single-GPU one, configs[4]
(GEMM-like space of configs[1], DE+PSO+Firefly+GA, pop 32, no budget, 200 generations, 10,000 runs each: 2.57e8 candidates
per step); `--config 1` is the small budgeted workload rounds 1-2 reported (1000 runs, budget 1000 unique evaluations).
N>1: every rank processes its own 10,000 runs per algorithm (run indices rank*10000..), no data-path collective (weak scaling).

Besides the headline line the same JSON carries, as top-level keys: `enumeration` (S1 alone on configs[1..3]),
`sweep_cfg4` (configs[4]: candidates/s against the run count), `steps_cfg2` / `steps_cfg3` (the generation step of
configs[2] and configs[3] at their BASELINE sizes, fused and phased), `next_rows_cfg1` (the SURVEY 8(f) variants on
configs[1]), `int_peak` (measured integer issue rates) and `cpu_baseline`.  The headline figures of those legs are repeated
as plain numbers inside `roofline` (enumeration Gcfg/s and HBM fraction, the sweep's HBM fractions, the cfg2 / cfg3 steps).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 4]
prints ONE JSON line on rank 0.
"""
from __future__ import annotations
import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

N_SM = 148
# dram__bytes_read.sum + dram__bytes_write.sum per k_gen launch of THIS workload (configs[1], 1000 runs per algorithm),
# mean of the four launches of one step: a STORED constant from the ncu --set full capture summarised in
# profiles/r2_kgen.md (it does not change with the run; the live numbers of this line are the CUDA-event times).
NCU_KGEN_DRAM_BYTES_PER_LAUNCH = 17.2e6
NCU_KGEN_SOURCE = "profiles/r2b_kgen.md"
# the same for the default workload, configs[4] at 10,000 runs per algorithm: (741.3 + 413.1 + 107.2 + 100.9) / 4 MB
NCU_KGEN_TRAFFIC = {(1, 1000): (17.2e6, "profiles/r2b_kgen.md"), (4, 10000): (340.6e6, "profiles/r3_kgen_cfg4.md")}
SECTOR_BYTES_PER_CANDIDATE = 204          # state 2(n+8) + bitmap 32 + directory 32 + obj 32 + dedup 64


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm_gbs=float(d["hbm_gbs"]), sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)), source="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")


def workload(cfg: int, runs: int | None):
    import workloads as W
    w = W.WORKLOADS[cfg]
    return dict(cfg=cfg, space=w.space(), algos=list(w.algos), pop=w.pop, gens=w.gens, runs=runs or w.runs,
                budget=w.budget, seed=w.seed)


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.stop_flag, self.sm, self.reasons, self.sm_max = index, False, [], set(), None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.sm_max = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {getattr(nv, k): k for k in dir(nv) if k.startswith("nvmlClocksEventReason") or k.startswith("nvmlClocksThrottleReason")}
        while not self.stop_flag:
            try:
                self.sm.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, nm in names.items():
                    if isinstance(bit, int) and bit and (r & bit) == bit and bin(bit).count("1") == 1:
                        self.reasons.add(nm.replace("nvmlClocksEventReason", "").replace("nvmlClocksThrottleReason", ""))
            except Exception:
                pass
            time.sleep(0.02)

    def summary(self):
        if not self.sm:
            return {"sm_mhz": None, "sm_max_mhz": self.sm_max, "reasons": ["unavailable"]}
        drop = {"None", "GpuIdle", "ApplicationsClocksSetting"}
        return {"sm_mhz": float(np.median(self.sm)), "sm_max_mhz": float(self.sm_max),
                "reasons": sorted(x for x in self.reasons if x not in drop)}


# ----------------------------------------------------------------------------------------------------------
def cpu_info():
    model = "unknown"
    try:
        for ln in open("/proc/cpuinfo"):
            if ln.startswith("model name"):
                model = ln.split(":", 1)[1].strip()
                break
    except OSError:
        pass
    return {"cpu_model": model, "nproc": os.cpu_count()}


class PinnedToOneCore:
    """The oracle is single-threaded; pin it to one core for the timed sample."""

    def __enter__(self):
        self.old = None
        try:
            self.old = os.sched_getaffinity(0)
            os.sched_setaffinity(0, {sorted(self.old)[-1]})
        except (AttributeError, OSError):
            self.old = None
        return self

    def __exit__(self, *a):
        if self.old is not None:
            os.sched_setaffinity(0, self.old)


def oracle_prepare(wl):
    """Untimed: the oracle's own space (needed to derive the objective table, an INPUT) and that table."""
    import oracle as O
    import workloads as W
    sp = wl["space"]
    s = O.OracleSpace.from_space(sp).build()
    obj = W.objective_table(s.rows(), sp.m, 0)
    return obj


def oracle_sample_step(wl, R_o, obj):
    """One bounded pass of the hot path on the CPU oracle: S1 in full + the first R_o runs of every algorithm.
    Returns (candidates evaluated, seconds).  Repairs are brute-force table scans: the oracle is the definition."""
    import oracle as O
    sp = wl["space"]
    t0 = time.perf_counter()
    s = O.OracleSpace.from_space(sp).build()
    s.set_objective(obj)
    cands = 0
    for algo in wl["algos"]:
        r = O.OracleRuns(s, algo, n_runs=R_o, pop=wl["pop"], budget=wl["budget"], max_gens=wl["gens"], seed=wl["seed"])
        r.step(wl["gens"])
        cands += r.n_evaluated
    return cands, time.perf_counter() - t0


def oracle_sample_text(wl, R_o):
    sp = wl["space"]
    return (f"full space build (N={sp.N}) + first {R_o} runs of each of {len(wl['algos'])} algorithms "
            f"(pop {wl['pop']}, budget {wl['budget']}, cap {wl['gens']} generations), one thread pinned to one core; "
            "every repair is a brute-force scan of the valid table (the oracle is the plain definition, not a tuned CPU program)")


def oracle_seconds_per_run(wl):
    """Rough oracle cost of ONE run of every algorithm of the workload (~2,400 candidates/s on one core, measured in rounds
    1-2): with a budget of b unique evaluations a run evaluates about 4 b candidates before it stops (duplicates count)."""
    per_algo = wl["pop"] * (wl["gens"] + 1)
    if wl["budget"]:
        per_algo = min(per_algo, 4 * wl["budget"])
    return len(wl["algos"]) * per_algo / 2400.0


def reference_arm(args):
    """The CPU oracle as it stands, on the host cores, on a bounded sample of the same workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    wl = workload(args.config, None)
    sp = wl["space"]
    # bounded sample: one step = the full space build (~0.7 s on configs[1] / [4]) + R_o runs of every algorithm (configs[1]:
    # ~6.6 s per run of the four, configs[4]: ~11 s); R_o is cut so that (steps + 1 warm-up) steps end within a few minutes
    R_o = max(1, min(args.ref_runs, int((170.0 / (args.steps + 1) - 0.7) / oracle_seconds_per_run(wl))))
    obj = oracle_prepare(wl)
    with PinnedToOneCore():
        for _ in range(min(args.warmup, 1)):
            _, t_w = oracle_sample_step(wl, R_o, obj)
            if R_o > 1 and t_w * args.steps > 240.0:                      # a slower host than the estimate assumed: fewer runs per step
                R_o = max(1, int(R_o * 240.0 / (t_w * args.steps)))
        sample = oracle_sample_text(wl, R_o)
        tot_c, tot_t = 0, 0.0
        for _ in range(args.steps):
            c, t = oracle_sample_step(wl, R_o, obj)
            tot_c += c; tot_t += t
    val = tot_c / tot_t
    line = {"impl": "reference", "metric": "candidates_repaired_evaluated_per_s", "value": val, "unit": "candidates/s",
            "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u8/u64 integer + f32 (no FMA)",
            "data": "synthetic", "config": {"workload": f"BASELINE configs[{args.config}] ({sp.name}), bounded sample: {sample}"},
            "cpu_baseline": {"value": val, "unit": "candidates/s", "cores": 1, "kind": "oracle", "sample": sample, **cpu_info()},
            "e2e": {"value": val, "unit": "candidates/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ----------------------------------------------------------------------------------------------------------
def scan_ops_per_pair(n):
    """Integer instructions per (candidate, valid row) of k_scan, by kind, counted in the SASS of its inner loop
    (n = 20: 5 VABSDIFF4 + 6 IADD + 10 IDP.4A + 1 IMAD + 3 ISETP/SEL + 2 LDS)."""
    wu = (n + 3) // 4
    return {"vabsdiff4": wu, "lop3": 0, "iadd": wu + 1, "idp4a": 2 * wu, "setp_sel": 3, "imad": 1, "lds": (wu + 3) // 4}


def enum_bytes(N, V, row_bytes, ltab_bytes):
    """Algorithmic bytes of S1: bitmap + rank directory + rows + Ltab."""
    return N / 8 + N / 128 + V * (row_bytes + ltab_bytes)


def gpu_arm(args):
    import torch
    import torch.distributed as dist
    import workloads as W
    import paper_2606_28372_b200 as cao

    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU fallback)"
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    pk = peaks()
    wl = workload(args.config, args.runs)
    sp, R, P, G = wl["space"], wl["runs"], wl["pop"], wl["gens"]
    from paper_2606_28372_b200.shard import shard_runs, max_over_ranks, sum_over_ranks
    first_run, _n_local = shard_runs(world * R, world, rank)         # weak scaling: R runs per rank, global run indices
    assert _n_local == R

    # inputs resident in HBM before the timed region: the objective table (indexed by valid rank, so it is
    # derived once from a first build of the same space) on the device and in pinned host memory
    g0 = cao.Space.from_space(sp).build()
    N, V, n, rb = g0.sizes()
    obj = W.objective_table(g0.rows().cpu().numpy(), sp.m, 0)
    obj_d = torch.from_numpy(obj).to(dev)
    obj_h = torch.from_numpy(obj).pin_memory()
    host_out = [torch.empty(4 * R, dtype=torch.int32).pin_memory() for _ in wl["algos"]]
    del g0
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev)        # > 126 MB L2

    side = [torch.cuda.Stream(device=dev) for _ in wl["algos"]] if args.streams > 1 else None

    def one_step(e2e, concurrent=True):
        space = cao.Space.from_space(sp).build()                          # S1
        space.set_objective(obj_h.to(dev, non_blocking=True) if e2e else obj_d)
        runs = []
        main = torch.cuda.current_stream()
        use_side = side is not None and concurrent
        if use_side:                                                      # the algorithms are independent: one stream each
            ready = torch.cuda.Event(); ready.record(main)
        for a, algo in enumerate(wl["algos"]):
            st = side[a] if use_side else main
            with torch.cuda.stream(st):
                if use_side:
                    st.wait_event(ready)
                r = cao.Runs(space, algo, n_runs=R, pop=P, budget=wl["budget"], max_gens=G, seed=wl["seed"],
                             first_run=first_run)                         # S2
                r.step(G)                                                 # S3-S7
                b = r.best()
                if e2e:
                    packed = torch.cat([b["best_f"].view(torch.int32), b["best_rank"], b["uniq"], b["gens_done"]])
                    host_out[a].copy_(packed, non_blocking=True)
                if use_side:
                    done = torch.cuda.Event(); done.record(st); main.wait_event(done)
            runs.append(r)
        return space, runs

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(K, e2e, profile, concurrent=True):
        evs = []
        kept = None
        if profile:
            cao.profile_enable(True)
        l0 = cao.launch_count()
        barrier()
        t0 = time.perf_counter()
        for _ in range(K):
            flush.zero_()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            kept = one_step(e2e, concurrent)
            e1.record()
            evs.append((e0, e1))
            if e2e:
                e1.synchronize()                                          # the user reads the result every step
        barrier()
        wall = time.perf_counter() - t0
        ms = sum(a.elapsed_time(b) for a, b in evs)
        if os.environ.get('CAO_BENCH_DEBUG'):
            print('timed', e2e, profile, concurrent, [round(a.elapsed_time(b), 2) for a, b in evs], file=sys.stderr)
        prof = cao.profile_read() if profile else None
        if profile:
            cao.profile_enable(False)
        launches = cao.launch_count() - l0
        ms = max_over_ranks(ms, dev)
        return ms, wall, prof, launches, kept

    # warm-up keeps the previous step's objects alive while the next step allocates, exactly as the timed loop does, so
    # the caching allocator already owns both buffer sets (a first-time cudaMalloc inside a timed step costs milliseconds)
    kept_w = None
    for _ in range(args.warmup):
        kept_w = one_step(False)
    kept_w = None                                                         # both sets go back to the allocator's cache
    torch.cuda.synchronize()
    import gc
    gc.collect(); gc.disable()                                            # no cyclic-GC pause inside a timed step
    sampler = ClockSampler(local); sampler.start()
    ms, wall, _, launches, kept = timed(args.steps, False, False)
    sampler.stop_flag = True; sampler.join(timeout=2)
    space, runs = kept
    stats = [r.stats() for r in runs]
    cands_step = sum(c["n_evaluated"] for c in stats)
    scanned_step = sum(c["n_scanned"] for c in stats)
    repaired_step = sum(c["n_repaired"] for c in stats)
    gens_done = [int(r.best()["gens_done"].sum().item()) for r in runs]
    cands_job = sum_over_ranks(cands_step, dev)                            # every rank ran its own runs: the job's count is the sum
    value = cands_job * args.steps / (ms / 1e3)
    del space, runs, kept                                                 # never more than two buffer sets alive (see the warm-up)
    # per-kernel device times: the same step, serialised on one stream, events around every launch
    ms_prof, _, prof, _, _ = timed(args.steps, False, True, concurrent=False)

    for _ in range(max(args.warmup, 2)):
        kept_w = one_step(True)
    kept_w = None
    torch.cuda.synchronize()
    ms_e, wall_e, _, _, _ = timed(args.steps, True, False)
    value_e = cands_job * args.steps / (ms_e / 1e3)
    gc.enable()
    h2d = obj.nbytes + sum(len(d) * 8 for d in sp.domains) + sum(len(p) * 4 for p in sp.rpn)
    d2h = len(wl["algos"]) * 16 * R + 8

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (device time per kernel class, CUDA events inside the library on the
    # launching stream, over the timed region)
    clocks = sampler.summary()
    kern = {k: {"ms_per_step": v[0] / args.steps, "launches_per_step": v[1] / args.steps} for k, v in prof.items() if v[1]}
    top = max(kern, key=lambda k: kern[k]["ms_per_step"])
    top_ms, top_n = kern[top]["ms_per_step"], kern[top]["launches_per_step"]
    dur_s = top_ms / 1e3 / top_n                                          # average launch duration
    per = {"k_op": 2 * rb + 8 + 32 + 32, "k_finish": 8 + 32 + 64 + rb + 24, "k_init": 32 + 64 + rb + 8,
           "k_gen": SECTOR_BYTES_PER_CANDIDATE}.get(top, 64)
    by = per * cands_step / max(top_n, 1)
    roof = {"kernel": top, "bound": "hbm", "achieved": by / dur_s / 1e9, "peak": pk["hbm_gbs"], "unit": "GB/s",
            "peak_source": pk["source"], "algorithmic_bytes_per_candidate": per,
            "traffic": None, "traffic_source": "no ncu capture of this workload shape"}
    ncu_src = NCU_KGEN_SOURCE
    if top == "k_gen" and (args.config, R) in NCU_KGEN_TRAFFIC:
        roof["traffic"], ncu_src = NCU_KGEN_TRAFFIC[(args.config, R)]
        roof["traffic_source"] = f"stored constant from the ncu --set full capture in {ncu_src}, not measured by this run"
    roof["frac"] = roof["achieved"] / roof["peak"]
    roof["avg_launch_us"] = dur_s * 1e6
    roof["share_of_step"] = top_ms / (ms_prof / args.steps)
    roof["measured_in"] = ("the same step re-run in the timed loop on ONE stream with CUDA events around every launch "
                           f"({ms_prof / args.steps:.2f} ms/step serialised vs {ms / args.steps:.2f} ms/step with one stream per algorithm)")
    roof["note"] = ("sector-granular HBM model of SURVEY 8(d); the kernel is bound by instruction issue, not DRAM "
                    f"(ncu: {ncu_src}); sweep_cfg4 shows the same kernel from 100 to 100,000 runs")

    # ---- measured integer issue peaks (lane-operations per second, one instruction kind each)
    int_peak = {}
    if not args.no_peak:
        int_peak = {k: cao.int_peak(k) / 1e12 for k in ("imad", "lop3", "vabsdiff4", "popc", "iadd", "idp4a")}
        int_peak["unit"] = "T lane-op/s"

    def scan_alu(n_dim, pairs, seconds):
        """Integer-pipe fractions of the repair scan against the MEASURED rates: (a) all its instructions against the
        issue rate (one warp instruction per scheduler per clock = the measured IADD rate), (b) the instructions of the
        half-rate alu pipe (LOP3, VABSDIFF4, compare/select) against the measured LOP3 rate, (c) the IDP.4A / IMAD
        instructions against the measured IDP.4A rate.  The largest binds."""
        if not int_peak or pairs == 0 or seconds <= 0:
            return None
        mix = scan_ops_per_pair(n_dim)
        total = sum(mix.values())
        half = mix["vabsdiff4"] + mix["lop3"] + mix["setp_sel"]
        return {"bound": "alu", "ops_per_pair": mix, "pairs": pairs, "achieved": total * pairs / seconds / 1e12,
                "unit": "T lane-op/s", "peak_issue": int_peak["iadd"], "frac_of_issue": total * pairs / seconds / 1e12 / int_peak["iadd"],
                "peak_alu_pipe": int_peak["lop3"], "frac_of_alu_pipe": half * pairs / seconds / 1e12 / int_peak["lop3"],
                "peak_fma_pipe": int_peak["idp4a"],
                "frac_of_fma_pipe": (mix["idp4a"] + mix["imad"]) * pairs / seconds / 1e12 / int_peak["idp4a"]}

    # ---- S1 alone (BASELINE metric "enumeration Gcfg/s"): configs[1..3], resident buffers
    enum = {}
    for cfg in ([int(c) for c in args.enum_cfgs.split(",")] if not args.no_enum else []):
        spx = W.WORKLOADS[cfg].space()
        gx = cao.Space.from_space(spx)
        gx.alloc_build(); gx.build_count(); gx.alloc_table(); gx.build_fill()
        torch.cuda.synchronize()
        ts = []
        es = torch.cuda.Stream(device=dev)                                # cao_space_rebuild replays its CUDA graph on a real stream
        with torch.cuda.stream(es):
            gx.rebuild(); es.synchronize()                                # capture + first replay (untimed)
            for _ in range(args.enum_reps):                               # resident inputs, no host round trip
                flush.zero_()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(); gx.rebuild(); e1.record(); e1.synchronize()
                ts.append(e0.elapsed_time(e1))
        kp = {}
        if not args.no_kernel_times:
            cao.profile_enable(True)
            for _ in range(5):
                flush.zero_(); gx.rebuild()
            torch.cuda.synchronize()
            kp = {k: v[0] / 5 * 1e3 for k, v in cao.profile_read().items() if v[1]}
            cao.profile_enable(False)
        Nx, Vx, nx, rbx = gx.sizes()
        lb = gx.ltab_bytes
        t = float(np.median(ts)) / 1e3
        enum[f"cfg{cfg}"] = {"N": Nx, "V": Vx, "ms": t * 1e3, "ms_min": float(min(ts)), "gcfg_s": Nx / t / 1e9,
                             "hbm_gbs": enum_bytes(Nx, Vx, rbx, lb) / t / 1e9,
                             "hbm_frac": enum_bytes(Nx, Vx, rbx, lb) / t / 1e9 / pk["hbm_gbs"],
                             "algorithmic_bytes": enum_bytes(Nx, Vx, rbx, lb), "kernel_us": kp, "blocks": gx.build_stats(),
                             "timing": "cao_space_rebuild (whole of S1, CUDA graph replay) on a side stream, L2 flushed before each, median of 11"}
        del gx

    # ---- BASELINE configs[4]: candidates/s against the number of runs (same space, no budget, 200 generations)
    sweep = {}
    if not args.no_sweep:
        space4 = cao.Space.from_space(sp).build(); space4.set_objective(obj_d)
        for Rs in [100, 1000, 10000, 100000][:args.sweep_points]:
            row = {}
            for algo in wl["algos"]:
                best_ms, cands = None, 0
                for _ in range(2):
                    r4 = cao.Runs(space4, algo, n_runs=Rs, pop=P, budget=0, max_gens=200, seed=wl["seed"])
                    torch.cuda.synchronize(); flush.zero_()
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    e0.record(); r4.step(200); e1.record(); e1.synchronize()
                    t4 = e0.elapsed_time(e1); best_ms = t4 if best_ms is None else min(best_ms, t4)
                    cands = Rs * P * 200
                    del r4
                row[algo] = {"ms": best_ms, "candidates_per_s": cands / (best_ms / 1e3),
                             "hbm_frac_204B": cands * SECTOR_BYTES_PER_CANDIDATE / (best_ms / 1e3) / 1e9 / pk["hbm_gbs"]}
            sweep[str(Rs)] = row
        del space4

    # ---- the generation step of configs[2] (GA, P 64, 10^4 runs, 150 generations) and configs[3] (Firefly, P 128,
    # 1000 runs, 100 generations: the repair-scan stress case) at their BASELINE sizes, fused and phased
    other = {}
    for cfg in ([int(c) for c in args.other_cfgs.split(",")] if not args.no_other else []):
        w = workload(cfg, None)
        spx = w["space"]
        gx = cao.Space.from_space(spx).build()
        Nx, Vx, nx, rbx = gx.sizes()
        gx.set_objective(W.objective_table(gx.rows().cpu().numpy(), spx.m, 0))
        leg = {"workload": f"BASELINE configs[{cfg}] ({spx.name}): N={Nx} V={Vx} n={nx}; {w['algos'][0]}, pop {w['pop']}, "
                           f"{w['gens']} generations, {w['runs']} runs", "probe_levels": gx.probe_levels,
               "default_mode": cao.Runs(gx, w["algos"][0], n_runs=2, pop=w["pop"], max_gens=1).mode}
        for mode in args.other_modes.split(","):
            best_ms = None
            for rep in range(2):
                rr = cao.Runs(gx, w["algos"][0], n_runs=w["runs"], pop=w["pop"], budget=w["budget"], max_gens=w["gens"],
                              seed=w["seed"], mode=mode)
                torch.cuda.synchronize(); flush.zero_()
                if rep == 1:
                    cao.profile_enable(True)
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(); rr.step(w["gens"]); e1.record(); e1.synchronize()
                t = e0.elapsed_time(e1); best_ms = t if best_ms is None else min(best_ms, t)
                if rep == 1:
                    kp = {k: {"ms": v[0], "launches": v[1]} for k, v in cao.profile_read().items() if v[1]}
                    cao.profile_enable(False)
                    st = rr.stats()
                del rr
            cands = w["runs"] * w["pop"] * w["gens"]
            row = {"ms": best_ms, "candidates_per_s": cands / (best_ms / 1e3),
                   "hbm_frac_204B": cands * SECTOR_BYTES_PER_CANDIDATE / (best_ms / 1e3) / 1e9 / pk["hbm_gbs"],
                   "kernels": kp, "n_repaired": st["n_repaired"], "n_scanned": st["n_scanned"], "n_memo": st["n_memo"],
                   "n_rcache": st["n_rcache"], "ham_hist": st["ham_hist"]}
            if mode == "phased" and "k_scan" in kp:
                row["scan_alu"] = scan_alu(nx, st["n_scanned"] * Vx, kp["k_scan"]["ms"] / 1e3)
            leg[mode] = row
        other[f"cfg{cfg}"] = leg
        del gx
    torch.cuda.empty_cache()

    # ---- SURVEY 8(f) rows on configs[1] (1000 runs per algorithm, budget 1000 unique, cap 200 generations): the paper's
    # own repairs (NEXT-1), the non-constraint-aware counterparts (NEXT-2), operator variants (NEXT-3), each timed like the
    # headline step, and the performance score (NEXT-4, Eq.2) of every variant against the calculated random-search
    # baseline -- score(aware) - score(unaware) is the quantity the paper's headline (+0.393 on its 24 spaces, L411) reports
    nxt = {}
    if not args.no_next and args.config in (1, 4):                        # configs[1] and [4] share the space (and obj_d)
        wl1 = workload(1, None)
        spn = cao.Space.from_space(sp).build(); spn.set_objective(obj_d)
        srt = spn.sorted_objective()
        ts = [int(t) for t in np.linspace(wl1["pop"], wl1["budget"], 32)]
        Bt = spn.baseline(srt, ts)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); srt = spn.sorted_objective(); e1.record(); e1.synchronize(); ms_sort = e0.elapsed_time(e1)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); Bt = spn.baseline(srt, ts); e1.record(); e1.synchronize(); ms_base = e0.elapsed_time(e1)
        variants = [("default", {}), ("unaware", dict(aware=False)), ("paper_repair", dict(repair_mode=1))]
        extra = {"de": [("rand1exp", dict(de_mutation="rand1", de_crossover="exp")), ("lhs", dict(init_lhs=True))],
                 "ga": [("uniform", dict(ga_crossover="uniform"))]}
        for algo in wl["algos"]:
            row = {}
            for name, kw in variants + extra.get(algo, []):
                best_ms = None
                for rep in range(2):
                    rr = cao.Runs(spn, algo, n_runs=wl1["runs"], pop=wl1["pop"], budget=wl1["budget"], max_gens=wl1["gens"],
                                  seed=wl1["seed"], variant=cao.Variant.make(**kw) if kw else None)
                    torch.cuda.synchronize(); flush.zero_()
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    e0.record(); rr.step(wl1["gens"]); e1.record(); e1.synchronize()
                    t = e0.elapsed_time(e1); best_ms = t if best_ms is None else min(best_ms, t)
                    if rep == 1:
                        st = rr.stats()
                        sc, per = rr.score(srt, ts, Bt)
                        row[name] = {"ms": best_ms, "mode": rr.mode, "candidates_per_s": st["n_evaluated"] / (best_ms / 1e3),
                                     "n_repaired": st["n_repaired"], "n_scanned": st["n_scanned"], "n_penalised": st["n_penalised"],
                                     "score": float(sc.item()), "score_at_budget": float(per[-1].item())}
                    del rr
            row["aware_minus_unaware_score"] = row["default"]["score"] - row["unaware"]["score"]
            nxt[algo] = row
        nxt["mean_aware_minus_unaware_score"] = float(np.mean([nxt[a]["aware_minus_unaware_score"] for a in wl["algos"]]))
        nxt["score_sampling_points"] = f"32 points, {ts[0]}..{ts[-1]} unique evaluations"
        nxt["sort_objective_ms"] = ms_sort; nxt["baseline_32_points_ms"] = ms_base
        nxt["paper_context"] = "paper L411: +0.393 mean score gain from constraint-awareness on its 24 BAT search spaces (other hardware, other spaces)"
        del spn
    torch.cuda.empty_cache()

    # ---- CPU oracle on a bounded sample of the same workload (rank 0, N=1 only), and a spot check of the GPU against it
    cpu = None
    if world == 1 and not args.no_cpu:
        import oracle as O
        obj_o = oracle_prepare(wl)
        assert np.array_equal(obj_o, obj)                                 # same input on both sides
        R_cpu = max(1, min(args.ref_runs, int(25.0 / oracle_seconds_per_run(wl))))   # about 10-30 s of CPU work
        with PinnedToOneCore():
            c, t = oracle_sample_step(wl, R_cpu, obj_o)
        cpu = {"value": c / t, "unit": "candidates/s", "cores": 1, "kind": "oracle", "sample": oracle_sample_text(wl, R_cpu),
               "seconds": t, **cpu_info()}

    # BASELINE.json's metric has three parts (candidates/s, enumeration Gcfg/s, % of the HBM roofline): the other two, and the
    # remaining legs' headline figures, as plain numbers inside the contract key (the bulky per-leg objects follow below)
    roof["enumeration"] = {k: {"gcfg_s": round(v["gcfg_s"], 1), "us": round(v["ms"] * 1e3, 1), "hbm_frac": round(v["hbm_frac"], 4)}
                           for k, v in enum.items()}
    roof["sweep_cfg4_hbm_frac"] = {Rs: {a: round(v["hbm_frac_204B"], 4) for a, v in row.items()} for Rs, row in sweep.items()}
    roof["sweep_cfg4_gcand_s"] = {Rs: {a: round(v["candidates_per_s"] / 1e9, 3) for a, v in row.items()} for Rs, row in sweep.items()}
    for cfgk, leg in other.items():
        roof["step_" + cfgk] = {m: {"ms": round(v["ms"], 2), "mcand_s": round(v["candidates_per_s"] / 1e6, 1)}
                                for m, v in leg.items() if isinstance(v, dict) and "ms" in v}
    line = {
        "metric": "candidates_repaired_evaluated_per_s", "value": value, "unit": "candidates/s", "n_gpus": world,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "u8/u64 integer + f32 (no FMA)", "data": "synthetic",
        "config": {"workload": f"BASELINE configs[{args.config}] ({sp.name}): N={N} V={V} n={n}; " +
                               "+".join(wl["algos"]) + f", pop {P}, budget {wl['budget']} unique, cap {G} generations, "
                               f"{R} runs per algorithm per GPU; step = S1 build + S2 init + S3-S7 to budget + read best",
                   "runs_per_gpu": R, "pop": P, "l2": "flushed between steps (512 MiB write outside the per-step events)",
                   "timing": "CUDA events per step on the launching stream, max over ranks",
                   "streams": "one CUDA stream per algorithm (independent runs)" if side else "single stream"},
        "clocks": clocks,
        "e2e": {"value": value_e, "unit": "candidates/s", "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                "ms_per_step": ms_e / args.steps},
        "gpu_launches": int(launches),
        "roofline": roof,
        "cpu_baseline": cpu,
        "enumeration": enum,
        "sweep_cfg4": sweep,
        "steps_cfg2": other.get("cfg2"),
        "steps_cfg3": other.get("cfg3"),
        "int_peak": int_peak,
        "next_rows_cfg1": nxt,
        "extra": {"candidates_per_step": int(cands_step), "invalid_post_snap_per_step": int(repaired_step),
                  "scanned_per_step": int(scanned_step), "generations_done_sum": gens_done,
                  "stats": {a: {k: v for k, v in s.items() if not k.startswith("cyc") } for a, s in zip(wl["algos"], stats)},
                  "kernels": kern, "wall_s_timed_region": wall, "peaks": pk},
    }
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json configs[k]; 4 = the largest single-GPU workload (default), 1 = the small budgeted one")
    ap.add_argument("--runs", type=int, default=None, help="runs per algorithm per GPU (default: the config's)")
    ap.add_argument("--ref-runs", type=int, default=3, help="runs per algorithm of the CPU-oracle sample")
    ap.add_argument("--streams", type=int, default=4, help="1 = all algorithms on one stream, >1 = one stream per algorithm")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-enum", action="store_true")
    ap.add_argument("--no-sweep", action="store_true")
    ap.add_argument("--no-other", action="store_true", help="skip the configs[2] / configs[3] generation-step legs")
    ap.add_argument("--no-peak", action="store_true", help="skip the integer issue-rate microbenchmarks")
    ap.add_argument("--no-next", action="store_true", help="skip the SURVEY 8(f) legs (paper repairs, unaware variants, score)")
    ap.add_argument("--sweep-points", type=int, default=4, help="how many of the run counts 1e2, 1e3, 1e4, 1e5 to sweep")
    ap.add_argument("--enum-cfgs", default="1,2,3", help="configs of the S1 leg")
    ap.add_argument("--enum-reps", type=int, default=11, help="timed rebuilds per config of the S1 leg")
    ap.add_argument("--no-kernel-times", action="store_true", help="S1 leg: skip the per-kernel event timing pass")
    ap.add_argument("--other-cfgs", default="2,3", help="configs of the generation-step legs")
    ap.add_argument("--other-modes", default="fused,phased", help="execution modes of the generation-step legs")
    args = ap.parse_args()
    if args.impl == "reference":
        reference_arm(args)
    else:
        gpu_arm(args)


if __name__ == "__main__":
    main()

#!/usr/bin/env python
"""bench.py - formula-model evaluations/s of the n=5 census layer (BASELINE.json configs[2]).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--workload c3|c3_paper|c3_small|c4|c5|atlas|frames|correspond]

One step = one pass of the whole hot path (DESIGN.md steps H1-H6, H8's class loop) over the
5,624-formula seeded corpus on every labelled frame of five worlds in K, T, S4 and S5 and every
valuation of two variables: 1.99318e14 formula-model evaluations.  Programs are staged once and stay
resident; counts and witnesses land in device tensors.  Under torchrun (N > 1) each rank scans a
contiguous 1/N of every class's frame range and the per-formula results are combined with one
all-reduce (SUM on counts, MIN on packed witness keys): strong scaling.

Prints ONE JSON line (see DESIGN.md "Measurement" for every field).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import workloads as W  # noqa: E402

CLASSES = (("K", 0), ("T", 1), ("S4", 2), ("S5", 3))
N_WORLDS, N_VARS = 5, 2
NCU_TRAFFIC_BYTES = 4239616                  # class-K launches of one step, from profiles/r2_jit_launches_c3.md
SM_COUNT, INT_LANES_PER_SM = 148, 64       # 4 sub-partitions x 16 lanes/clk on the ALU pipe (B300_MICROARCH.md)


def class_sizes_n5():
    return {"K": 1 << 25, "T": 1 << 20, "S4": 6942, "S5": 52}


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.max_mhz = index, [], set(), None
        self.stop_flag = threading.Event()
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {
            getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
            getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwPowerBrakeSlowdown", 0x80): "hw_power_brake",
        }
        while not self.stop_flag.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    mask = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if mask & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            self.stop_flag.wait(0.2)

    def energy_mj(self):
        """NVML total energy counter of the device in millijoules, or None."""
        if self.nv is None:
            return None
        try:
            return int(self.nv.nvmlDeviceGetTotalEnergyConsumption(self.h))
        except Exception:
            return None

    def result(self):
        self.stop_flag.set()
        if self.nv is None or not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["nvml unavailable"]}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons)}


def formula_vars(code: bytes) -> int:
    """Number of distinct variables a postfix program mentions as written (Algorithm 1's k_b)."""
    return len({c for c in code if 0x10 <= c < 0x14})


def oracle_sample(progs, frames: int, threads: int = 0, repeats: int = 1):
    """The oracle as it stands on a bounded sample: the first `frames` K-frames at n=5, every formula."""
    from oracle import volume as V
    V.build()
    code, offs = W.pack_programs(progs)
    cores = V.max_threads() if threads <= 0 else threads
    dts = []
    for _ in range(repeats):
        t0 = time.perf_counter()
        V.census(code, offs, N_WORLDS, N_VARS, 0, 0, frames, threads=cores)
        dts.append(time.perf_counter() - t0)
    dt = float(np.median(dts))
    # The oracle as it stands sweeps all 2^(n_vars n) valuations of every formula, whether or not the formula
    # mentions every variable: it is credited with the evaluations it performs (`executed`).  Algorithm 1's own
    # count of the same job (formula b on the 2^(k_b n) valuations of the variables it mentions, the numerator
    # of the GPU arm's `value`) is returned beside it.
    executed = len(progs) * (frames << (N_VARS * N_WORLDS))
    alg1 = sum(frames << (formula_vars(c) * N_WORLDS) for c in progs)
    return executed / dt, dt, cores, executed, alg1


ORACLE_COUNTING = ("executed: every formula on all 2^(n_vars n) = 1,024 valuations of every sampled frame, which is what "
                   "oracle/volume_oracle.c sweeps; value_alg1_counting is the same run credited only with Algorithm 1's "
                   "2^(k_b n) valuations per formula (the GPU arm's `value` counting)")


def run_reference(args):
    """--impl reference: the oracle (oracle/volume_oracle.c) on the host cores; each step is a
    bounded sample of the same workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    progs = W.corpus_c2()
    frames = args.ref_frames
    for _ in range(args.warmup):
        oracle_sample(progs[:256], 8)
    rates, secs, cores = [], [], 0
    alg1_rates = []
    for _ in range(args.steps):
        r, dt, cores, executed, alg1 = oracle_sample(progs, frames)
        rates.append(r)
        alg1_rates.append(alg1 / dt)
        secs.append(dt)
    value = float(np.mean(rates))
    sample = f"first {frames} K-frames of n=5 x {len(progs)} formulas x 1,024 valuations per step"
    print(json.dumps({
        "impl": "reference", "metric": "formula-model evaluations/sec at n=5", "value": value,
        "unit": "evaluations/s", "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": float(np.mean(secs) * 1e3), "higher_is_better": True, "scaling": "strong",
        "vs_baseline": None, "dtype": "u8", "data": "synthetic",
        "config": {"workload": "C3 n=5 census layer (BASELINE.json configs[2]), bounded sample", "sample": sample,
                   "evaluations_counting": ORACLE_COUNTING},
        "cpu_baseline": {"value": value, "unit": "evaluations/s", "cores": cores, "kind": "oracle", "sample": sample,
                         "counting": ORACLE_COUNTING, "value_alg1_counting": float(np.mean(alg1_rates))},
        "e2e": {"value": value, "unit": "evaluations/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def paper_corpus(kb):
    """The paper-shaped corpus: every constant-free formula of <= 7 nodes over {p, q} (44,678),
    one representative per class of equal truth sets on all models of <= 3 worlds (kripke_signatures on the
    GPU: 5,621, the first in enumeration order per class), plus the K axiom (the only one of the paper's three
    added axioms that is identifiable, R19)."""
    forms = W.enumerate_constant_free(7, 2)
    progs = [W.to_postfix(t) for t in forms]
    h = kb.Programs(*W.pack_programs(progs), N_VARS)
    sig = kb.signatures(h, N_VARS, 3).cpu().numpy()
    h.destroy()
    first = {}
    for i, s in enumerate(map(tuple, sig.tolist())):
        first.setdefault(s, i)
    reps = [progs[i] for i in sorted(first.values())]
    return reps + [W.to_postfix(W.named_axioms()["K"])], len(progs), len(reps)


def check_results(kb, args, progs, counts, wits):
    """What the timed steps left in the device tensors, looked at after the timed region: a SHA-256 over the four
    classes' (models, frames) arrays; the rows with closed forms (F refuted by every model, T and the K axiom by
    none); and, for the contract corpus, the S4 / S5 records against tests/golden/n5_s4s5.npz (written by the
    oracle, tests/golden/make_golden.py).  A mismatch ends the run: a wrong scan has no throughput."""
    import hashlib
    res = {c: kb.unpack(counts[c], wits[c]) for c, _ in CLASSES}
    sha = hashlib.sha256()
    for c, _ in CLASSES:
        sha.update(np.ascontiguousarray(res[c]["models"]).tobytes())
        sha.update(np.ascontiguousarray(res[c]["frames"]).tobytes())
    done = ["sha256 over models|frames of K, T, S4, S5"]
    if args.workload in ("c3", "c3_paper"):
        sizes = class_sizes_n5()
        nval = 1 << (N_VARS * N_WORLDS)
        probes = {"F": W.to_postfix(W.parse("F")), "T": W.to_postfix(W.parse("T")), "K axiom": W.to_postfix(W.named_axioms()["K"])}
        for name, code in probes.items():
            for b in [i for i, p in enumerate(progs) if p == code][:1]:
                for c, _ in CLASSES:
                    want_f = sizes[c] if name == "F" else 0
                    got = (int(res[c]["models"][b]), int(res[c]["frames"][b]))
                    if got != (want_f * nval, want_f):
                        raise SystemExit(f"bench.py: result check failed: {name} on class {c}: {got}")
                done.append(f"closed form: {name} (formula {b}) on all four classes")
    gold = os.path.join(ROOT, "tests", "golden", "n5_s4s5.npz")
    if args.workload == "c3" and os.path.exists(gold):
        g = np.load(gold)
        for c in ("S4", "S5"):
            for key in ("models", "frames", "wit_f", "wit_v", "wit_w"):
                if not np.array_equal(np.asarray(res[c][key]).astype(np.uint64), g[f"{c}_{key}"].astype(np.uint64)):
                    raise SystemExit(f"bench.py: result check failed: class {c} {key} differs from tests/golden/n5_s4s5.npz")
        done.append("S4 and S5 records (counts and witnesses, every formula) equal the oracle's golden file")
    return {"counts_sha256": sha.hexdigest(), "checked": done}


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2606_15437_b200 import binding as kb
    from paper_2606_15437_b200 import shard as sh

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but the launcher started {world} rank(s); n_gpus is what ran")
    if not torch.cuda.is_available():
        raise SystemExit(f"bench.py: no CUDA device on rank {rank} (there is no CPU fallback)")
    if local_rank >= torch.cuda.device_count():
        raise SystemExit(f"bench.py: rank {rank} wants cuda:{local_rank} but the node has {torch.cuda.device_count()} GPU(s)")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    kb.load()

    corpus_note = None
    if args.workload == "c3_paper":
        progs, n_enum, n_reps = paper_corpus(kb)
        corpus_note = f"{n_enum} enumerated constant-free formulas -> {n_reps} semantic classes (GPU signatures) + K axiom"
    else:
        progs = W.corpus_c2()
    if args.workload == "c3_small":
        sizes = {"K": 1 << 20, "T": 1 << 16, "S4": 6942, "S5": 52}
    else:
        sizes = class_sizes_n5()
    code, offs = W.pack_programs(progs)
    B = len(progs)
    nval = 1 << (N_VARS * N_WORLDS)
    frames_total = sum(sizes.values())
    # evaluation counts of one step (one evaluation = one formula on one (frame, valuation)):
    #   alg1:  Algorithm 1's own count - formula b is swept over the 2^(k_b n) valuations of the k_b variables it
    #          mentions; this is how the paper's 1.63e14 is counted, and it is `value`'s numerator
    #   fixed: every formula on all 2^(n_vars n) valuations of the batch (the C ABI's counting, R8)
    kb_of = [formula_vars(c) for c in progs]
    evals_alg1 = sum(frames_total << (kv * N_WORLDS) for kv in kb_of)
    evals_fixed = B * nval * frames_total

    h = kb.Programs(code, offs, N_VARS)
    counts = {c: torch.zeros((B, 2), dtype=torch.int64, device="cuda") for c, _ in CLASSES}
    wits = {c: torch.zeros((B, 2), dtype=torch.int64, device="cuda") for c, _ in CLASSES}
    keys = {c: torch.zeros((B,), dtype=torch.int64, device="cuda") for c, _ in CLASSES}
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")      # > 126 MB L2
    launches = [0]
    k_info = {}
    executed = [0]
    compile_s = [0.0]

    def step(ev_k=None, flags=0):
        for cname, cls in CLASSES:
            begin, count = sh.shard_range(sizes[cname], rank, world)
            if ev_k is not None and cname == "K":
                ev_k[0].record()
            kb.eval_batch_range(h, N_WORLDS, N_VARS, cls, begin, count, flags, counts[cname], wits[cname])
            if ev_k is not None and cname == "K":
                ev_k[1].record()
            info = h.last_run_info()
            launches[0] += info.launches
            executed[0] += info.executed_models
            if cname == "K":
                k_info["instr_per_frame"] = info.logic_instr_per_frame
                k_info["alg_instr_per_frame"] = info.algorithmic_logic_instr_per_frame
                k_info["popc_per_frame"] = info.popc_instr_per_frame
                k_info["frames"] = count
                k_info["family"] = info.kernel_family
                k_info["programs"] = info.jit_programs
            compile_s[0] = max(compile_s[0], info.jit_compile_seconds)
        if world > 1:                                                   # the one exchange step
            for cname, _ in CLASSES:
                kb.witness_to_keys(wits[cname], N_WORLDS, N_VARS, keys[cname])
                sh.combine(counts[cname], keys[cname])
                kb.keys_to_witness(keys[cname], N_WORLDS, N_VARS, wits[cname])

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # calibration: the measured integer-pipe rate, right before the timed runs
    cal = {}
    for variant, name in ((0, "lop3"), (1, "iadd3"), (2, "shf"), (3, "lop3+imad"), (4, "lop3_with_1_popc_per_8"),
                          (5, "lop3_with_2_popc_per_8")):
        cal[name] = kb.calibrate_int32(variant)[0]

    t_first = time.perf_counter()
    for i in range(args.warmup):
        step()
        if i == 0:
            torch.cuda.synchronize()
            t_first = time.perf_counter() - t_first                    # includes building the plans (NVRTC)
        flush.fill_(1)
    barrier()

    sampler = ClockSampler(local_rank)
    sampler.start()
    launches[0] = 0
    executed[0] = 0
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    evk = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    barrier()
    e_before = sampler.energy_mj()
    ev0.record()
    for i in range(args.steps):
        step(evk[i])
        flush.fill_(i & 0xFF)            # L2 flush between iterations (inputs are < 100 KB anyway)
    ev1.record()
    barrier()
    e_after = sampler.energy_mj()
    ms_total = ev0.elapsed_time(ev1)
    clocks = sampler.result()
    k_ms = float(np.mean([a.elapsed_time(b) for a, b in evk]))
    n_launches = launches[0]

    t = torch.tensor([ms_total], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms_total = float(t.item())
    ms_per_step = ms_total / args.steps
    value = evals_alg1 / (ms_per_step * 1e-3)

    # end to end through the host-buffer entry point (kripke_eval_batch_host): H2D of the programs, plan look-up,
    # scan, D2H of the records.  These steps are WARM: every call creates a new handle with the same program bytes
    # and finds the finished plan in the process-wide plan cache (keyed by those bytes), so nothing is emitted or
    # compiled again - the figure is the cost of a repeated scan of a corpus the process has seen.  The cost of the
    # first scan of a fresh corpus (emitter + NVRTC + module load) is measured separately below as e2e["cold"].
    e2e = None
    check = None
    if rank == 0 and args.e2e_steps > 0:
        times = []
        host_res = {}
        for _ in range(max(args.e2e_steps, 1)):
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            for cname, cls in CLASSES:
                if args.workload in ("c3", "c3_paper"):
                    host_res[cname] = kb.eval_batch_host(code, offs, N_WORLDS, N_VARS, cls)
                else:   # reduced ranges are not expressible through the host entry point
                    hh = kb.Programs(code, offs, N_VARS)
                    c, w = kb.eval_batch_range(hh, N_WORLDS, N_VARS, cls, 0, sizes[cname])
                    c.cpu(); w.cpu()
                    hh.destroy()
            times.append(time.perf_counter() - t0)
        e2e = {"value": evals_alg1 / float(np.median(times)), "unit": "evaluations/s",
               "h2d_bytes_per_step": int(4 * (code.nbytes + offs.nbytes)), "d2h_bytes_per_step": int(4 * 32 * B),
               "seconds_per_step": float(np.median(times)), "samples": len(times), "statistic": "median",
               "seconds_per_step_min_max": [float(min(times)), float(max(times))],
               "state": "warm: amortised over repeated scans of a corpus whose compiled plan is cached in the process",
               "jit": f"kernels compiled with NVRTC once per process ({compile_s[0]:.2f} s for the class-K plan, paid "
                      f"in the first warm-up step: {t_first:.2f} s); the timed e2e steps create a new handle and find "
                      "the finished plan in the process-wide plan cache"}

    # what the timed region produced, checked after it (world == 1: the full ranges were scanned by this rank)
    if rank == 0 and world == 1:
        check = check_results(kb, args, progs, counts, wits)

    # ablation, one timed pass each after the timed region; the records are bit-identical in every mode (GPU tests)
    ablation = None
    if rank == 0 and world == 1 and args.workload in ("c3", "c3_paper") and args.e2e_steps > 0:
        ablation = {}
        modes = (("compiled_no_subterm_sharing", kb.NO_SUBTERM_SHARING,
                  "compiled kernels, identical programs scanned once, every program evaluates its own subterms"),
                 ("interpreted", kb.KERNEL_SLICED, "round-1 engine: micro-op interpreter, whole-program sharing"),
                 ("interpreted_no_sharing", kb.KERNEL_SLICED | kb.NO_SHARING, "interpreter, every formula scanned itself"),
                 ("interpreted_no_sharing_full_sweep", kb.KERNEL_SLICED | kb.NO_SHARING | kb.FULL_SWEEP,
                  "interpreter, every formula on all 2^(n_vars n) valuations: executed = fixed-n_vars count"))
        for name, fl, what in modes:
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            ex, ops = 0, 0.0
            for timed in (False, True):
                torch.cuda.synchronize()
                a.record()
                for cname, cls in CLASSES:
                    kb.eval_batch_range(h, N_WORLDS, N_VARS, cls, 0, sizes[cname], fl, counts[cname], wits[cname])
                    if timed:
                        info = h.last_run_info()
                        ex += info.executed_models
                        ops += info.logic_instr_per_frame * sizes[cname]
                b.record()
                torch.cuda.synchronize()
            ms = a.elapsed_time(b)
            ablation[name] = {"what": what, "ms_per_step": ms, "value": evals_alg1 / (ms * 1e-3),
                              "executed_evaluations_per_step": ex, "executed_logic_instr_per_step": ops}

    # cold end-to-end: the same host-buffer calls with every cached plan and compiled module dropped first, i.e.
    # the first scan of a corpus the process has never seen (a census scans each batch once)
    if rank == 0 and world == 1 and e2e is not None and args.workload in ("c3", "c3_paper") and not args.no_cold:
        h.destroy()
        torch.cuda.synchronize()
        import gc
        gc.collect()                     # handles of the ablation passes and of paper_corpus() are gone by now
        unloaded = kb.jit_cache_clear()  # raises if a handle is still alive: then there is no cold figure to report
        t0 = time.perf_counter()
        for cname, cls in CLASSES:
            kb.eval_batch_host(code, offs, N_WORLDS, N_VARS, cls)
        cold = time.perf_counter() - t0
        e2e["cold"] = {"value": evals_alg1 / cold, "unit": "evaluations/s", "seconds_per_step": cold, "samples": 1,
                       "modules_unloaded_before": unloaded,
                       "what": "kripke_jit_cache_clear(), then one pass through kripke_eval_batch_host: graph, rewrites, "
                               "emitter, NVRTC for sm_100a, module load, scan, D2H (CUDA context and library already up)"}

    if rank == 0:
        k_exec = k_info["instr_per_frame"] * k_info["frames"]         # logic thread-instructions the class-K launches execute
        k_alg = k_info["alg_instr_per_frame"] * k_info["frames"]      # SURVEY 8(d)'s algorithmic count for the same call
        achieved = k_exec / (k_ms * 1e-3) / 1e12
        peak_derived = SM_COUNT * INT_LANES_PER_SM * 1.965e9 / 1e12   # derived ALU-pipe peak at max clock
        peak = cal["lop3"] / 1e12                                      # measured in this process, right before the timed runs
        cpu_rate, cpu_dt, cores, cpu_evals, cpu_alg1 = oracle_sample(W.corpus_c2() if args.workload != "c3_paper" else progs,
                                                                     args.ref_frames, repeats=3)
        label = {"c3": "C3 n=5 census layer (BASELINE.json configs[2]): 5,624 seeded formulas x K/T/S4/S5 frames of 5 "
                       "worlds x 1,024 valuations",
                 "c3_paper": "C3-paper (SURVEY 8(d)): the paper-shaped census corpus (P:143) x K/T/S4/S5 frames of 5 worlds",
                 "c3_small": "c3_small: C3 with K cut to 2^20 and T to 2^16 frames (debug only)"}[args.workload]
        out = {
            "metric": "formula-model evaluations/sec at n=5", "value": value, "unit": "evaluations/s",
            "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_per_step,
            "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "u32",
            "data": "synthetic",
            "config": {
                "workload": label, "corpus": corpus_note,
                "formulas": B, "n_worlds": N_WORLDS, "n_vars": N_VARS, "classes": [c for c, _ in CLASSES],
                "evaluations_per_step": evals_alg1,
                "evaluations_counting": "Algorithm 1 (PAPER.md:93): formula b on the 2^(k_b n) valuations of the k_b "
                                        "variables it mentions; `value` = this count / device time",
                "evaluations_per_step_fixed_n_vars": evals_fixed,
                "value_fixed_n_vars": evals_fixed / (ms_per_step * 1e-3),
                "executed_evaluations_per_step": executed[0] // args.steps,
                "value_executed": executed[0] / args.steps / (ms_per_step * 1e-3),
                "formulas_by_variables_mentioned": {str(v): kb_of.count(v) for v in sorted(set(kb_of))},
                "engine": {0: "scalar", 1: "interpreted bit-sliced", 2: "compiled bit-sliced (NVRTC, sm_100a)"}[k_info["family"]],
                "distinct_programs_scanned_class_K": k_info["programs"],
                "jit_compile_seconds": compile_s[0], "first_step_seconds": t_first,
                "sharing": "all programs of a call form one graph of distinct subterms (negation folded, and/box normal "
                           "form, canonical variable order); every distinct subterm is evaluated once per 32-model word, "
                           "identical programs are scanned once; executed_evaluations_per_step counts distinct programs x "
                           "the models of their own variables",
                "parallelism": f"frame-range shard x{world}",
                "l2": "flushed between iterations (256 MiB fill); the kernels read < 100 KB of input",
            },
            "clocks": clocks,
            "e2e": e2e,
            "result_check": check,
            "gpu_launches": n_launches,
            "roofline": {
                "bound": "alu", "kernel": "kripke_jit_scan (the compiled class-K launches of one step)",
                "achieved": achieved, "peak": peak, "unit": "T thread-instr/s", "frac": achieved / peak,
                "frac_executed": achieved / peak,
                "peak_derived": peak_derived, "frac_of_peak_derived": achieved / peak_derived,
                "executed_ops": "3-input logic (LOP3) thread-instructions the compiled kernels execute: one per emitted "
                                "lop3.b32 (the emitter covers every expression tree with 3-input tables itself), weighted by "
                                "loop level; cross-checked against ncu's opcode count in profiles/r2_jit_full.md",
                "xu_pipe": {"popc_per_s_T": k_info["popc_per_frame"] * k_info["frames"] / (k_ms * 1e-3) / 1e12,
                            "peak_T": peak_derived / 4,
                            "frac": k_info["popc_per_frame"] * k_info["frames"] / (k_ms * 1e-3) / 1e12 / (peak_derived / 4),
                            "what": "one POPC per scanned program and 32-model word counts the refuting models; POPC issues on "
                                    "the XU pipe at 16 lanes/clk/SM (a quarter of the ALU rate).  At the two warps per "
                                    "scheduler these kernels run with, ALU and XU time barely overlap (ncu: "
                                    "profiles/r2_jit_perkernel.md), so frac + xu_pipe.frac is the share of the step the two "
                                    "pipes account for"},
                "frac_algorithmic": k_alg / (k_ms * 1e-3) / 1e12 / peak_derived,
                "algorithmic_ops": "SURVEY 8(d): every formula as written, (d n^2 + b n + n + 1) logic instructions per "
                                   "32-model word x 2^(k_b n)/32 words per frame - work the method defines per peak-second; "
                                   "NOT a pipe fraction (sharing makes it exceed 1)",
                "traffic": NCU_TRAFFIC_BYTES if (args.workload == "c3" and world == 1) else None,
                "traffic_source": "dram__bytes_read.sum + dram__bytes_write.sum of the class-K kernels of one step, "
                                  "ncu launch list profiles/r2_jit_launches_c3.csv (bytes; algorithmic HBM bytes = 0)",
                "kernel_ms": k_ms, "kernel_share_of_step": k_ms / ms_per_step,
                "peak_source": "measured: kripke_calibrate_int32 variant 0 (register-resident independent LOP3 on every SM) "
                               "in this process right before the timed runs; peak_derived = 148 SMs x 4 x 16 ALU "
                               "lanes/clk x 1.965 GHz (DESIGN.md 6)",
                "peak_measured_calibration": {k: v / 1e12 for k, v in cal.items()},
            },
            "ablation": ablation,
            # P:262 reports 10.53 nJ per evaluation on the H100: the same figure from NVML's energy counter
            "energy": None if (e_before is None or e_after is None or world > 1) else {
                "joules_per_step": (e_after - e_before) * 1e-3 / args.steps,
                "nj_per_evaluation": (e_after - e_before) * 1e-3 / args.steps / evals_alg1 * 1e9,
                "source": "nvmlDeviceGetTotalEnergyConsumption around the timed region (whole board)"},
            "cpu_baseline": {"value": cpu_rate, "unit": "evaluations/s", "cores": cores, "kind": "oracle",
                             "sample": f"first {args.ref_frames} K-frames of n=5 x {B} formulas x 1,024 valuations "
                                       f"({cpu_evals:.3g} evaluations, median of 3 runs of {cpu_dt:.1f} s)",
                             "counting": ORACLE_COUNTING, "value_alg1_counting": cpu_alg1 / cpu_dt},
        }
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def run_c4(args):
    """--workload c4: BASELINE.json configs[3] ablations: formula batch size (fusion)
    on the bit-sliced kernel, fused vs separate launches, and per-block / per-warp / per-thread atomics
    on the scalar (Algorithm 1) kernel under mixed and adversarial contention.  n=5, 3 variables."""
    import torch
    from paper_2606_15437_b200 import binding as kb
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    kb.load()
    n, k = 5, 3
    progs = W.corpus_c4()
    nval = 1 << (k * n)
    reps = max(1, args.steps)

    def timed(fn):
        for _ in range(max(1, args.warmup > 0)):
            fn()
        torch.cuda.synchronize()
        ts = []
        for _ in range(reps):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); fn(); b.record(); torch.cuda.synchronize()
            ts.append(a.elapsed_time(b) * 1e-3)
        return float(np.median(ts))

    out = {"batch": {}, "fusion": {}, "contention": {}}
    clock = ClockSampler(0)
    clock.start()
    # A. batch size (fusion) on the bit-sliced kernel
    for B, begin, count in ((1, 0, 1 << 25), (32, 0, 1 << 25), (256, 1 << 24, 1 << 20), (2048, 1 << 24, 1 << 20)):
        h = kb.Programs(*W.pack_programs(progs[:B]), k)
        c = torch.zeros((B, 2), dtype=torch.int64, device="cuda")
        w = torch.zeros((B, 2), dtype=torch.int64, device="cuda")
        t = timed(lambda: kb.eval_batch_range(h, n, k, 0, begin, count, 0, c, w))
        info = h.last_run_info()
        ev = B * count * nval
        out["batch"][str(B)] = {"frames": count, "seconds": t, "evaluations_per_s": ev / t,
                                "engine": info.kernel_family, "distinct_programs": info.jit_programs,
                                "compile_seconds": info.jit_compile_seconds,
                                "executed_logic_instr_per_s": info.logic_instr_per_frame * count / t,
                                "frac_of_alu_peak": info.logic_instr_per_frame * count / t / (SM_COUNT * INT_LANES_PER_SM * 1.965e9),
                                "algorithmic_logic_instr_per_s": info.algorithmic_logic_instr_per_frame * count / t}
        h.destroy()
    # B. one fused launch of 32 formulas vs 32 separate launches (2^20-frame range)
    begin, count = 1 << 24, 1 << 20
    hs = [kb.Programs(*W.pack_programs([p]), k) for p in progs[:32]]
    c1 = torch.zeros((1, 2), dtype=torch.int64, device="cuda")
    w1 = torch.zeros((1, 2), dtype=torch.int64, device="cuda")
    t_sep = timed(lambda: [kb.eval_batch_range(hh, n, k, 0, begin, count, 0, c1, w1) for hh in hs])
    h32 = kb.Programs(*W.pack_programs(progs[:32]), k)
    c = torch.zeros((32, 2), dtype=torch.int64, device="cuda")
    w = torch.zeros((32, 2), dtype=torch.int64, device="cuda")
    t_fused = timed(lambda: kb.eval_batch_range(h32, n, k, 0, begin, count, 0, c, w))
    out["fusion"] = {"formulas": 32, "frames": count, "separate_s": t_sep, "fused_s": t_fused,
                     "fused_speedup": t_sep / t_fused}
    # C. atomic contention on the scalar kernel (the paper's layout: thread = frame, one model per iteration),
    # SURVEY 8(d) shape: 256 formulas x K-frames [2^24, 2^24 + 2^20), "mixed" = the batch of 256 as it is,
    # "adversarial" = F & (each formula): every model refutes every formula.  One timed pass per
    # mode (each pass is 8.8e12 evaluations on the scalar kernel).
    begin, count = 1 << 24, args.c4_contention_frames
    NB = 256
    mixed = progs[:NB]
    adversarial = [W.to_postfix(("and", ("bot",), W.from_postfix(p))) for p in progs[:NB]]   # every model refutes

    def once(fn):
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(); fn(); b.record(); torch.cuda.synchronize()
        return a.elapsed_time(b) * 1e-3

    for name, batch in (("mixed", mixed), ("adversarial", adversarial)):
        h = kb.Programs(*W.pack_programs(batch), k)
        c = torch.zeros((NB, 2), dtype=torch.int64, device="cuda")
        w = torch.zeros((NB, 2), dtype=torch.int64, device="cuda")
        res = {"formulas": NB, "frames": count}
        kb.eval_batch_range(h, n, k, 0, begin, 256, kb.KERNEL_SCALAR, c, w)          # warm-up (module load)
        for mname, mode in (("block", kb.REDUCE_BLOCK), ("warp", kb.REDUCE_WARP), ("thread", kb.REDUCE_THREAD)):
            t = once(lambda: kb.eval_batch_range(h, n, k, 0, begin, count, kb.KERNEL_SCALAR | kb.NO_SHARING |
                                                 kb.FULL_SWEEP | mode, c, w))
            res[mname] = {"seconds": t, "evaluations_per_s": NB * count * nval / t}
        res["block_vs_thread"] = res["thread"]["seconds"] / res["block"]["seconds"]
        res["block_vs_warp"] = res["warp"]["seconds"] / res["block"]["seconds"]
        t = timed(lambda: kb.eval_batch_range(h, n, k, 0, begin, count, 0, c, w))
        res["bit_sliced_default"] = {"seconds": t, "evaluations_per_s": NB * count * nval / t}
        out["contention"][name] = res
        h.destroy()
    # D. the same ablation where atomics can matter: one variable (32 valuations per frame between two atomics
    # instead of 32,768), 256 seeded one-variable formulas, 2^20 frames - the regime of the paper's frame-atomic
    # kernel (26.27x adversarial / 3.44x mixed)
    rng = W.SplitMix64(15437014)
    seen, one = set(), []
    while len(one) < NB:
        c = W.to_postfix(W.gen_formula(rng, 9, 6, "p"))
        if c not in seen and len(c) >= 3:
            seen.add(c); one.append(c)
    adv1 = [W.to_postfix(("and", ("bot",), W.from_postfix(c))) for c in one]
    out["contention_one_variable"] = {}
    count = 1 << 20
    for name, batch in (("mixed", one), ("adversarial", adv1)):
        h = kb.Programs(*W.pack_programs(batch), 1)
        c = torch.zeros((NB, 2), dtype=torch.int64, device="cuda")
        w = torch.zeros((NB, 2), dtype=torch.int64, device="cuda")
        res = {"formulas": NB, "frames": count, "valuations_per_frame": 32}
        kb.eval_batch_range(h, n, 1, 0, begin, 256, kb.KERNEL_SCALAR, c, w)
        for mname, mode in (("block", kb.REDUCE_BLOCK), ("warp", kb.REDUCE_WARP), ("thread", kb.REDUCE_THREAD)):
            t = timed(lambda: kb.eval_batch_range(h, n, 1, 0, begin, count, kb.KERNEL_SCALAR | mode, c, w))
            res[mname] = {"seconds": t, "evaluations_per_s": NB * count * 32 / t}
        res["block_vs_thread"] = res["thread"]["seconds"] / res["block"]["seconds"]
        res["block_vs_warp"] = res["warp"]["seconds"] / res["block"]["seconds"]
        t = timed(lambda: kb.eval_batch_range(h, n, 1, 0, begin, count, 0, c, w))
        res["bit_sliced_default"] = {"seconds": t, "evaluations_per_s": NB * count * 32 / t}
        out["contention_one_variable"][name] = res
        h.destroy()
    clocks = clock.result()
    b2048 = out["batch"]["2048"]
    print(json.dumps({
        "metric": "formula-model evaluations/sec at n=5", "value": b2048["evaluations_per_s"],
        "unit": "evaluations/s", "n_gpus": 1, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": b2048["seconds"] * 1e3, "higher_is_better": True, "scaling": "strong",
        "vs_baseline": None, "dtype": "u32", "data": "synthetic",
        "config": {"workload": "C4 ablation (BASELINE.json configs[3]): n=5, 3 variables, 2,048 seeded formulas of "
                               "9-15 nodes; value = batch 2,048 on K-frames [2^24, 2^24+2^20) (the paper's stress shape)"},
        "clocks": clocks, "ablation": out,
    }))


def run_c5(args):
    """--workload c5: BASELINE.json configs[4]: variable-free pairwise
    distinguishability.  Stage A, the exact prefix: every pair of the C5 list (36 named + 4,096 seeded) on every
    labelled frame of 1..5 worlds (33,620,498 frames), counts and first distinguishing frame per pair and size, no
    early exit - the paper's "exact stage" (21.55 ms per candidate on the H100).  Stage B: every pair that
    agrees through five worlds goes on to six (2^36 frames) in ascending chunks of 2^30 frames with per-pair
    early exit (kripke_pairs_separation); reports the first distinguishing frame per separated pair and the pairs
    that survive all 2^36 frames."""
    import torch
    from paper_2606_15437_b200 import binding as kb
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    kb.load()
    progs, pairs, names = W.pairs_c5()
    pairs = np.asarray(pairs, np.uint32)
    P = len(pairs)
    h = kb.Programs(*W.pack_programs(progs), 0)
    peak = SM_COUNT * INT_LANES_PER_SM * 1.965e9
    clock = ClockSampler(0)
    clock.start()
    sizes = (1, 2, 3, 4, 5)
    c = torch.zeros((P, 2), dtype=torch.int64, device="cuda")
    w = torch.zeros((P, 2), dtype=torch.int64, device="cuda")

    def prefix():
        per_n = {}
        for n in sizes:
            kb.distinguish_pairs(h, pairs, n, 0, 0, 0, 1 << (n * n), 0, c, w)
            per_n[n] = kb.unpack(c, w)
        return per_n

    t0 = time.perf_counter()
    prefix()                                                   # warm-up: builds (compiles) the five plans
    torch.cuda.synchronize()
    t_build = time.perf_counter() - t0
    ts = []
    logic = 0.0
    for _ in range(max(1, args.steps)):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        logic = 0.0
        for n in sizes:
            kb.distinguish_pairs(h, pairs, n, 0, 0, 0, 1 << (n * n), 0, c, w)
            logic += h.last_run_info().logic_instr_per_frame * (1 << (n * n))
        b.record(); torch.cuda.synchronize()
        ts.append(a.elapsed_time(b) * 1e-3)
    t_prefix = float(np.median(ts))
    per_n = prefix()
    frames_prefix = sum(1 << (n * n) for n in sizes)
    first_size = np.zeros(P, np.int64)
    for n in sizes:
        hit = (per_n[n]["frames"] > 0) & (first_size == 0)
        first_size[hit] = n
    late = np.nonzero(first_size == 0)[0]
    info5 = h.last_run_info()

    # stage B: the survivors at six worlds, chunked with early exit (host loop inside the library)
    sub = pairs[late]
    kb.pairs_separation(h, sub[:8], 0, 6, 1 << 30) if len(sub) else None      # warm-up of the n=6 plan shape
    t0 = time.perf_counter()
    size6, wit6 = kb.pairs_separation(h, sub, 0, 6, 1 << 30)
    t_six = time.perf_counter() - t0
    sep = np.nonzero(size6 == 6)[0]
    never = np.nonzero(size6 == 0)[0]
    assert ((size6 == 0) | (size6 == 6)).all()
    # one full chunk of the never-split pairs, timed on the device: the steady-state rate of the pair path at n=6
    rate6 = None
    if len(never):
        pn = sub[never]
        cc = torch.zeros((len(pn), 2), dtype=torch.int64, device="cuda")
        ww = torch.zeros((len(pn), 2), dtype=torch.int64, device="cuda")
        kb.distinguish_pairs(h, pn, 6, 0, 0, 0, 1 << 24, 0, cc, ww)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(); kb.distinguish_pairs(h, pn, 6, 0, 0, 1 << 30, 1 << 30, 0, cc, ww); b.record(); torch.cuda.synchronize()
        t = a.elapsed_time(b) * 1e-3
        i6 = h.last_run_info()
        rate6 = {"pairs": int(len(pn)), "frames": 1 << 30, "seconds": t, "pair_frame_tests_per_s": len(pn) * (1 << 30) / t,
                 "distinct_programs": int(i6.jit_programs), "logic_instr_per_s": i6.logic_instr_per_frame * (1 << 30) / t,
                 "frac_of_alu_peak": i6.logic_instr_per_frame * (1 << 30) / t / peak}
    clocks = clock.result()
    first_frames = {}
    for i in sep:
        j = int(late[i])
        first_frames[names[j] or f"seeded#{j}"] = {"frame": int(wit6[i, 0]), "world": int(wit6[i, 1] >> np.uint64(32))}
    print(json.dumps({
        "metric": "pair-frame tests/sec (variable-free pairs, all labelled frames of 1..5 worlds)",
        "value": P * frames_prefix / t_prefix, "unit": "pair-frame tests/s", "n_gpus": 1, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": t_prefix * 1e3, "higher_is_better": True, "scaling": "strong",
        "vs_baseline": None, "dtype": "u32", "data": "synthetic",
        "config": {"workload": f"C5 (BASELINE.json configs[4]): {P} variable-free pairs (36 named + 4,096 seeded), exhaustive "
                               f"through n=5 ({frames_prefix} frames), survivors on to n=6 (2^36 frames, chunks of 2^30, early exit)",
                   "plan_build_seconds": t_build,
                   "prefix": {"seconds": t_prefix, "ms_per_pair": t_prefix * 1e3 / P,
                              "separation_size_histogram": {str(n): int((first_size == n).sum()) for n in (1, 2, 3, 4, 5, 0)},
                              "distinct_programs_n5": int(info5.jit_programs),
                              "logic_instr_per_s": logic / t_prefix, "frac_of_alu_peak": logic / t_prefix / peak,
                              "context": "paper, H100: 3,522 candidates rescanned through n=5 in 75.9 s = 21.55 ms per candidate (P:288)"},
                   "six_worlds": {"pairs": int(len(sub)), "seconds": t_six, "separated": int(len(sep)), "never_split": int(len(never)),
                                  "first_frames": first_frames, "full_chunk_rate": rate6,
                                  "never_split_named": [names[int(late[i])] for i in never if names[int(late[i])]]}},
        "clocks": clocks,
    }))


def run_atlas(args):
    """--workload atlas: failure densities: per (formula, frame) the number
    of (valuation, world) pairs on which the formula fails, written formula-major as uint32.  Two legs:
      panels  the paper-shaped atlas: the 5,624-formula corpus (two variables) on every K frame of 1..3 worlds
              (Atlas-3), a 2,048-frame four-world panel and a 4,096-frame five-world panel - each count
              sums 2^(2n) valuations x n worlds, so this leg is bound by the integer pipe, not by memory;
      write   the regime the paper reports for its atlas materialisation (51.54 GB at 91.6 % of its HBM ceiling,
              P:262): 64 variable-free formulas of the C5 list on ALL 2^25 five-world K frames, one frame per
              lane, 8.6 GB of counts - bound by HBM writes; roofline against MEASURED_PEAKS.json hbm_gbs."""
    import torch
    from paper_2606_15437_b200 import binding as kb
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    kb.load()
    peak_src = "MEASURED_PEAKS.json hbm_gbs"
    try:
        hbm = float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"])
    except Exception:
        hbm, peak_src = 6650.0, "fallback of B200_PROFILING.md (6.65 TB/s): MEASURED_PEAKS.json absent"
    alu_peak = SM_COUNT * INT_LANES_PER_SM * 1.965e9
    clock = ClockSampler(0)
    clock.start()
    reps = max(1, args.steps)

    def timed(fn):
        for _ in range(max(1, min(args.warmup, 3))):
            fn()
        torch.cuda.synchronize()
        ts = []
        for _ in range(reps):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); fn(); b.record(); torch.cuda.synchronize()
            ts.append(a.elapsed_time(b) * 1e-3)
        return float(np.median(ts))

    # leg 1: panels of the two-variable corpus
    progs = W.corpus_c2()
    B = len(progs)
    h = kb.Programs(*W.pack_programs(progs), N_VARS)
    panels = [(1, 0, 2), (2, 0, 16), (3, 0, 512), (4, 30000, 2048), (5, 1 << 24, 4096)]
    outs = [torch.zeros((B, cnt), dtype=torch.int32, device="cuda") for _, _, cnt in panels]
    logic = [0.0]

    def run_panels():
        logic[0] = 0.0
        for (n, begin, cnt), o in zip(panels, outs):
            kb.failure_density(h, n, N_VARS, 0, begin, cnt, o)
            logic[0] += h.last_run_info().logic_instr_per_frame * cnt

    leg1 = None
    if not args.atlas_skip_panels:
        t0 = time.perf_counter(); run_panels(); torch.cuda.synchronize(); t_build = time.perf_counter() - t0
        t_panels = timed(run_panels)
        entries = B * sum(cnt for _, _, cnt in panels)
        evals = B * sum(cnt << (N_VARS * n) for n, _, cnt in panels)
        leg1 = {"formulas": B, "frames": sum(cnt for _, _, cnt in panels), "entries": entries, "seconds": t_panels,
                "entries_per_s": entries / t_panels, "evaluations_per_s": evals / t_panels,
                "bytes_written": 4 * entries, "write_GB_per_s": 4 * entries / t_panels / 1e9,
                "logic_instr_per_s": logic[0] / t_panels, "frac_of_alu_peak": logic[0] / t_panels / alu_peak,
                "plan_build_seconds": t_build, "bound": "alu"}
    h.destroy()

    # leg 2: HBM-write-bound - variable-free formulas, every five-world K frame
    p0 = W.pairs_c5()[0][:64]
    h0 = kb.Programs(*W.pack_programs(p0), 0)
    frames = 1 << 25
    out = torch.empty((len(p0), frames), dtype=torch.int32, device="cuda")
    kb.failure_density(h0, 5, 0, 0, 0, 1 << 12, out)                     # builds the plan
    torch.cuda.synchronize()
    t_write = timed(lambda: kb.failure_density(h0, 5, 0, 0, 0, frames, out))
    info = h0.last_run_info()
    nbytes = 4 * len(p0) * frames
    # spot check of the written matrix against the scalar kernel on a window (both are this library's kernels;
    # parity against the oracle is tests/test_gpu_bitmaps.py)
    w0 = 12345 * 32
    chk = kb.failure_density(h0, 5, 0, 0, w0 + 1, 1023)                  # 1,023 frames: unaligned -> scalar kernel
    assert (chk == out[:, w0 + 1:w0 + 1024]).all()
    clocks = clock.result()
    achieved = nbytes / t_write / 1e9
    print(json.dumps({
        "metric": "failure-density entries/sec ((formula, frame) counts written, uint32)",
        "value": len(p0) * frames / t_write, "unit": "entries/s", "n_gpus": 1, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": t_write * 1e3, "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "u32",
        "data": "synthetic",
        "config": {"workload": f"atlas (SURVEY 8f N2; P:270, P:284, P:262): write leg = {len(p0)} variable-free formulas x all 2^25 "
                               f"five-world K frames ({nbytes / 1e9:.2f} GB of counts); panels leg = {B} two-variable formulas x "
                               "Atlas-3 + 2,048 four-world + 4,096 five-world frames",
                   "panels": leg1,
                   "context": "paper, H100: atlas materialisation 51.54 GB at >= 1,622 GB/s = 91.6 % of its measured 1,771 GB/s (P:262)"},
        "clocks": clocks,
        "roofline": {"bound": "hbm", "kernel": "kripke_jit_scan, density mode, one frame per lane (class K, n=5, no variables)",
                     "achieved": achieved, "peak": hbm, "unit": "GB/s", "frac": achieved / hbm, "peak_source": peak_src,
                     "algorithmic_bytes": nbytes, "traffic": 8471674000,
                     "traffic_source": "ncu dram__bytes_read.sum + dram__bytes_write.sum of the two density kernels of one pass: "
                                       "profiles/r2_atlas_full.md (the tail of the last rows is still in the 126 MB L2 when the "
                                       "kernel ends)",
                     "logic_instr_per_s": info.logic_instr_per_frame * frames / t_write,
                     "frac_of_alu_peak": info.logic_instr_per_frame * frames / t_write / alu_peak},
    }))


def run_frames(args):
    """--workload frames: frame-list mode (Table 2).  Per size n the
    pair path is timed on a seeded list of 2^20 explicit frames (kripke_frames_generate, KRIPKE_GEN_STRESS):
    constant pairs (the 36 named pairs of PAPER.md:179/190 plus seeded ones, one valuation) at every
    size, one-variable pairs (2^n valuations) through n = 12.  Reports pair-frame
    tests/s, valuation-frame evaluations/s (2 formulas per pair), the kernel's logic-instruction rate
    against the ALU peak, its shared-memory operand rate and HBM bytes, the scalar (thread = frame)
    kernel on the same list, and the oracle on a bounded sample."""
    import torch
    from paper_2606_15437_b200 import binding as kb
    from workloads import frames as F
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    kb.load()
    n_frames = 1 << 20
    progs0, pairs0, _ = W.pairs_c5(count=220)
    pairs0 = np.asarray(pairs0, np.uint32)
    rng = W.SplitMix64(15437007)
    progs1 = [W.to_postfix(W.gen_formula(rng, 9, 9, "pTF")) for _ in range(256)]
    pairs1 = np.arange(256, dtype=np.uint32).reshape(-1, 2)
    peak = SM_COUNT * INT_LANES_PER_SM * 1.965e9
    reps = max(1, args.steps)

    def timed(fn):
        for _ in range(max(1, min(args.warmup, 3))):
            fn()
        torch.cuda.synchronize()
        ts = []
        for _ in range(reps):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); fn(); b.record(); torch.cuda.synchronize()
            ts.append(a.elapsed_time(b) * 1e-3)
        return float(np.median(ts))

    clock = ClockSampler(0)
    clock.start()
    rows = {}
    total_tests = total_evals = total_time = 0.0
    for n in (6, 8, 10, 12, 14, 16):
        succ = kb.frames_generate(kb.GEN_STRESS, n, n_frames, F.SEED_FRAMES)      # written on the device
        row = {}
        for k, progs, pairs in ((0, progs0, pairs0), (1, progs1, pairs1)):
            if k * n > 12:
                continue
            h = kb.Programs(*W.pack_programs(progs), k)
            P = len(pairs)
            c = torch.zeros((P, 2), dtype=torch.int64, device="cuda")
            w = torch.zeros((P, 2), dtype=torch.int64, device="cuda")
            t = timed(lambda: kb.distinguish_pairs_frames(h, pairs, n, k, succ, 0, 0, c, w))
            info = h.last_run_info()
            tests = P * n_frames
            evals = 2 * tests * (1 << (k * n))
            logic = info.logic_instr_per_frame * n_frames
            sub = 1 << 16
            ts = timed(lambda: kb.distinguish_pairs_frames(h, pairs, n, k, succ[:sub * n].contiguous(), 0,
                                                           kb.KERNEL_SCALAR, c, w))
            row[f"k{k}"] = {"pairs": P, "seconds": t, "pair_frame_tests_per_s": tests / t,
                            "evaluations_per_s": evals / t, "logic_instr_per_s": logic / t,
                            "frac_of_alu_peak": logic / t / peak,
                            "scalar_kernel_evaluations_per_s": 2 * P * sub * (1 << (k * n)) / ts,
                            "hbm_bytes_frames": 2 * n * n_frames}
            total_tests += tests; total_evals += evals; total_time += t
            h.destroy()
        rows[str(n)] = row
        del succ
    clocks = clock.result()
    # the oracle on a bounded sample of the same workload (n = 8, one-variable pairs)
    from oracle import volume as V
    V.build()
    n = 8
    rel = F.stress_list_cb(n, 2048)
    code, offs = W.pack_programs(progs1)
    t0 = time.perf_counter()
    V.census_relations(code, offs, n, 1, rel, pairs=pairs1)
    dt = time.perf_counter() - t0
    cpu = 2 * len(pairs1) * len(rel) * (1 << n) / dt
    print(json.dumps({
        "metric": "valuation-frame evaluations/sec on explicit frame lists (n = 6..16)",
        "value": total_evals / total_time, "unit": "evaluations/s", "n_gpus": 1, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": total_time * 1e3, "higher_is_better": True, "scaling": "strong",
        "vs_baseline": None, "dtype": "u32", "data": "synthetic",
        "config": {"workload": "frame-list mode (PAPER.md:183-192, Table 2): 2^20 seeded explicit frames per size "
                               "n in {6,8,10,12,14,16} (templates, Erdos-Renyi, edge-flip, dead-end, back-edge); "
                               f"{len(pairs0)} constant pairs at every size, {len(pairs1)} one-variable pairs through n = 12",
                   "pair_frame_tests_per_s": total_tests / total_time,
                   "context": "paper, H100: 586,365,732 pair-frame tests / 94.68e9 evaluations in 53.0 s of GPU "
                              "evaluation (Table 2) = 1.79e9 evaluations/s"},
        "clocks": clocks, "per_size": rows,
        "cpu_baseline": {"value": cpu, "unit": "evaluations/s", "cores": V.max_threads(), "kind": "oracle",
                         "sample": f"n=8, 2,048 frames x 256 valuations x {len(pairs1)} one-variable pairs ({dt:.1f} s)"},
    }))


def run_correspond(args):
    """--workload correspond: correspondence recovery: validity
    bitmaps of the whole 5,624-formula corpus over every K frame of 1..4 worlds, matched against the
    library of eight first-order conditions (equal extensions at every size, Proposition 6); every
    match is re-confirmed over all 2^25 five-world frames.  Reports the matched / constant / unmatched
    split (paper, its own corpus: 220 / 2,798 / 2,606) and formula-frame validity tests per second."""
    import torch
    from paper_2606_15437_b200 import binding as kb
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    kb.load()
    progs = W.corpus_c2()
    B = len(progs)
    h = kb.Programs(*W.pack_programs(progs), N_VARS)
    names = list(kb.COND)
    sizes = (1, 2, 3, 4)

    def scan():
        bms, libs = [], []
        for n in sizes:
            total = 1 << (n * n)
            bms.append(kb.validity_bitmap(h, n, N_VARS, 0, 0, total))
            libs.append(torch.stack([kb.condition_bitmap(n, kb.COND[c], 0, 0, total) for c in names]))
        bm, lib = torch.cat(bms, dim=1).contiguous(), torch.cat(libs, dim=1).contiguous()
        return bm, lib, kb.match_bitmaps(bm, lib)

    for _ in range(max(1, min(args.warmup, 2))):
        scan()
    torch.cuda.synchronize()
    clock = ClockSampler(0)
    clock.start()
    ts = []
    for _ in range(max(1, args.steps)):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(); bm, lib, match = scan(); b.record(); torch.cuda.synchronize()
        ts.append(a.elapsed_time(b) * 1e-3)
    t = float(np.median(ts))
    match = match.cpu().numpy()
    bits = bm.cpu().numpy().view(np.uint32)
    frames_total = sum(1 << (n * n) for n in sizes)
    ones = np.unpackbits(bits.view(np.uint8), axis=1).sum(axis=1)
    constant = (ones == 0) | (ones == frames_total)
    matched = (match >= 0) & ~constant
    # re-confirmation over all 2^25 five-world frames, on the bit-sliced kernels: Val_5(phi) = Ext_5(X)
    # iff phi is refuted on no frame of Ext_5(X) (frame-list scan of the condition's own extension) and
    # the census counts as many valid frames as |Ext_5(X)|
    idx = np.nonzero(matched)[0]
    t5, confirmed, ext5 = 0.0, 0, {}
    if len(idx):
        total5 = 1 << 25
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        h5 = kb.Programs(*W.pack_programs([progs[i] for i in idx]), N_VARS)
        cen = kb.unpack(*kb.eval_batch(h5, 5, N_VARS, 0))
        for j, cname in enumerate(names):
            sel = np.nonzero(match[idx] == j)[0]
            if len(sel) == 0:
                continue
            cb = kb.condition_bitmap(5, kb.COND[cname], 0, 0, total5)
            _, n_set = kb.frames_from_bitmap(5, 0, 0, total5, cb, 0)
            succ, _ = kb.frames_from_bitmap(5, 0, 0, total5, cb, n_set)
            hj = kb.Programs(*W.pack_programs([progs[idx[i]] for i in sel]), N_VARS)
            on_ext = kb.unpack(*kb.eval_frames(hj, 5, N_VARS, succ))
            ok = (on_ext["frames"] == 0) & (cen["frames"][sel] == np.uint64(total5 - n_set))
            confirmed += int(ok.sum())
            ext5[cname] = n_set
            hj.destroy()
        b.record(); torch.cuda.synchronize()
        t5 = a.elapsed_time(b) * 1e-3
    clocks = clock.result()
    print(json.dumps({
        "metric": "formula-frame validity tests/sec (correspondence recovery, n <= 4)",
        "value": B * frames_total / t, "unit": "formula-frames/s", "n_gpus": 1, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": t * 1e3, "higher_is_better": True, "scaling": "strong",
        "vs_baseline": None, "dtype": "u32", "data": "synthetic",
        "config": {"workload": f"correspondence recovery (PAPER.md:358-380): {B} seeded formulas x all K frames of "
                               f"1..4 worlds ({frames_total} frames) x 8 first-order conditions",
                   "split": {"matched": int(matched.sum()), "constant_extension": int(constant.sum()),
                             "unmatched": int(B - matched.sum() - constant.sum())},
                   "matched_by_condition": {names[j]: int((match[matched] == j).sum()) for j in range(len(names))},
                   "reconfirmed_at_n5": {"formulas": int(len(idx)), "confirmed": confirmed, "seconds": t5,
                                         "frames": 1 << 25, "extension_sizes": ext5},
                   "context": "paper, its own 5,624-formula corpus: 220 matched / 2,798 constant / 2,606 unmatched"},
        "clocks": clocks,
    }))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c3", choices=["c3", "c3_paper", "c3_small", "c4", "c5", "atlas", "frames", "correspond"])
    ap.add_argument("--e2e-steps", type=int, default=5, help="warm end-to-end samples (median is reported); 0 = skip e2e, "
                                                             "ablation and cold e2e")
    ap.add_argument("--no-cold", action="store_true", help="skip the cold end-to-end pass (cache clear + recompilation)")
    ap.add_argument("--ref-frames", type=int, default=256)
    ap.add_argument("--c4-contention-frames", type=int, default=1 << 16,
                    help="frames of the three-variable contention leg on the scalar kernel (SURVEY 8(d) shape: 2^20, "
                         "about 20 minutes; recorded once in profiles/)")
    ap.add_argument("--atlas-skip-panels", action="store_true", help="atlas: only the HBM-write leg (for ncu captures)")
    args = ap.parse_args()
    if args.impl == "ours" and args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # asked for N GPUs without a launcher: start the N ranks ourselves (one process per GPU, NCCL over NVLink)
        # and let rank 0's line be the output
        import socket
        import subprocess
        with socket.socket() as sock:
            sock.bind(("127.0.0.1", 0))
            port = sock.getsockname()[1]
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        raise SystemExit(subprocess.call(cmd))
    if args.impl == "ours" and args.workload not in ("c3", "c3_paper", "c3_small") and \
            (args.gpus > 1 or int(os.environ.get("WORLD_SIZE", "1")) > 1):
        raise SystemExit(f"bench.py: --workload {args.workload} is a one-GPU measurement; only the census layer shards")
    if args.impl == "reference":
        run_reference(args)
    elif args.workload == "c4":
        run_c4(args)
    elif args.workload == "c5":
        run_c5(args)
    elif args.workload == "atlas":
        run_atlas(args)
    elif args.workload == "frames":
        run_frames(args)
    elif args.workload == "correspond":
        run_correspond(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()

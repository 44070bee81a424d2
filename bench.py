#!/usr/bin/env python
"""bench.py -- headline benchmark of the AFSAT hot path on B200 (contract in DESIGN.md "Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--impl ours|reference]
                    [--no-per-config] [--no-ttfs] [--sweep-batch] [--probe-peaks] [--line-search]

The headline (top-level keys) is BASELINE.json configs[4], the largest single-GPU configuration; the default run also
measures configs 0-3 and config 3 in fp64 (`per_config`) and the time to the first solution on the planted variant of
the headline workload (`time_to_first_solution`).

A "step" is one pass of the whole hot path (gather, DFT-point products,
contraction, leave-one-out gradient, scatter-add, projected step, sign rounding, exact discrete
count, freeze) over one batch of B synthetic candidates, through the C ABI (afsat_step).
metric = candidate-constraint FE+grad evaluations per second = m * B * steps / time.

N > 1 (torchrun): the path shards by candidate with no exchange ("replicas only"):
every rank runs its own batch of B candidates on its own GPU; value = N*m*B*K / max-over-ranks time.
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
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "candidate-constraint FE+grad evals/sec on 1 B200; % of FP32 roofline"
UNIT = "evals/s"
FP32_LANES_PER_SM = 128          # B200_PROFILING.md / B300_MICROARCH.md: 4 x 32 FP32 lanes per SM


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return {"hbm_gbs": float(d["hbm_gbs"]), "sm_max_mhz": float(d.get("sm_max_mhz", 1965.0)),
                "source": "measured"}
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "source": "fallback"}


def load_capture(cfg, dtype):
    """What the committed ncu captures of this workload measured (profiles/r2_ncu_summary.json; the commands are in
    profiles/r2_ncu_summary.md): DRAM bytes of the evaluation kernels per step with a WARM L2 (--cache-control none),
    FMA-pipe and issue-slot utilisation of the dominant kernel.  {} when there is no capture."""
    p = os.path.join(ROOT, "profiles", "r2_ncu_summary.json")
    try:
        with open(p) as f:
            return json.load(f).get(f"cfg{cfg}" + ("_f64" if dtype == 64 else ""), {})
    except (OSError, ValueError):
        return {}


def flop_model(inst):
    """Algorithmic work per candidate over all constraints:
    flop = k(19 C + 6 R) + 4 C + 2 R, FP32 instr = k(12 C + 4 R) + 2 C + R with R = 1 + [k odd]
    self-conjugate DFT points and C = floor((k+1)/2) + 1 - R complex ones."""
    ks, cnt = np.unique(inst.lengths(), return_counts=True)
    flop = instr = 0
    for k, c in zip(ks.tolist(), cnt.tolist()):
        R = 1 + (k % 2)
        Cc = (k + 1) // 2 + 1 - R
        flop += c * (k * (19 * Cc + 6 * R) + 4 * Cc + 2 * R)
        instr += c * (k * (12 * Cc + 4 * R) + 2 * Cc + R)
    return flop, instr


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML during the timed region."""

    def __init__(self, index, period=0.005):   # the default timed region is ~40 ms
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop_evt = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception as e:  # noqa: BLE001
            self.err = repr(e)

    def _sample(self):
        nv = self.nv
        self.samples.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
        r = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
        names = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "hw_thermal_slowdown": 0x40,
                 "sw_thermal_slowdown": 0x20, "hw_power_brake_slowdown": 0x80,
                 "applications_clocks_setting": 0x2, "sync_boost": 0x10}
        for k, bit in names.items():
            if r & bit:
                self.reasons.add(k)

    def run(self):
        if not self.ok:
            return
        while not self._stop_evt.is_set():
            try:
                self._sample()
            except Exception:  # noqa: BLE001
                pass
            self._stop_evt.wait(self.period)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=2)
        if not self.ok:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvml unavailable: " + getattr(self, "err", "")]}
        return {"sm_mhz": float(np.median(self.samples)) if self.samples else None,
                "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


_PEAKS = {}


def probed_peak(kind, device):
    """afsat_probe_peak (FFMA / FFMA2 / DFMA chains, measured in this run), cached."""
    from paper_2606_06641_b200 import binding as Bd
    if (kind, device) not in _PEAKS:
        _PEAKS[(kind, device)] = Bd.probe_peak(kind, device)
    return _PEAKS[(kind, device)]


def workload(cfg, batch=None, scale=1.0):
    from paper_2606_06641_b200 import instances as I
    inst = I.make_config(cfg, scale=scale, batch=batch)
    return inst


def oracle_sample(inst, x0, target_s=15.0, max_b=64):
    """Times oracle_step (as it stands) on a bounded candidate subsample of the same workload:
    B_o candidates x 1 step over ALL constraints, B_o sized from a 1-candidate-per-core probe."""
    from oracle import oracle as O
    cores = O.num_threads()
    probe_b = min(cores, inst.batch)
    t0 = time.perf_counter()
    O.step(inst, x0[:, :probe_b].astype(np.float64), inst.eta, 1, probe_b, want_F=False)
    t1 = time.perf_counter() - t0
    per_wave = max(t1, 1e-4)                       # one candidate per core
    waves = int(max(1, min(target_s / per_wave, max(1, max_b * 8 // max(cores, 1)))))
    b_o = int(min(inst.batch, max(probe_b, waves * cores)))
    t0 = time.perf_counter()
    X1, _, sat1, _, _ = O.step(inst, x0[:, :b_o].astype(np.float64), inst.eta, 1, b_o, want_F=False)
    dt = time.perf_counter() - t0
    oracle_sample.last = (X1[:, :b_o], sat1[:b_o])          # X(1) and the counts on X(1), for the deviation report
    return {"value": inst.n_cons * b_o * 1 / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"oracle_step (long double, gcc -O2, OpenMP over candidates) on the first {b_o} of "
                      f"{inst.batch} candidates x 1 step over all {inst.n_cons} constraints, {dt:.2f} s",
            "note": "the PRECISION oracle as it stands (x87 long double, a fresh O(k^2) leave-one-out DP per literal), "
                    "not a tuned CPU implementation: a reported baseline, never the target"}, dt, b_o


def time_to_first_solution(inst, x0, dtype, device, max_steps):
    """Time from the first afsat_step launch to the first step at which some candidate is solved, read from
    the pinned any-solved flag the library sets from the device (polled here without a blocking sync).
    The random instances of configs 1-4 sit far above the satisfiability threshold, so this runs the
    PLANTED variant of the same workload (literal signs re-chosen so that a hidden assignment satisfies
    every constraint); one candidate in 1024 starts next to the hidden assignment (0.1 % of the variables
    wrong, |x| = 0.5), the others start uniformly at random like the headline run."""
    import torch
    from paper_2606_06641_b200 import binding as Bd, instances as I

    def admissible(t, k, p):                       # counts of true literals that satisfy the constraint
        taus = np.arange(k + 1)
        ok = {0: taus >= 1, 1: taus % 2 == p, 2: taus >= p, 3: taus <= p, 4: taus == p, 5: (taus > 0) & (taus < k)}[int(t)]
        return taus[ok]
    base = I.Instance(**{**inst.__dict__})
    base.meta = dict(inst.meta)
    base.meta["admissible"] = [admissible(t, k, p) for t, k, p in zip(inst.ctype, inst.lengths(), inst.param)]
    planted, hidden = I.plant_solution(base, seed=I.SEED_X0 + 77)
    rng = np.random.default_rng(I.SEED_X0 + 78)
    x = x0.copy()
    near = np.where(hidden, -0.5, 0.5).astype(x.dtype)
    probes = list(range(0, inst.batch, 1024))
    for b in probes:
        col = near.copy()
        wrong = rng.choice(inst.n_vars, size=max(1, inst.n_vars // 1000), replace=False)
        col[wrong] = -col[wrong]
        if planted.fixed is not None:
            fx = planted.fixed != 0
            col[fx] = planted.fixed[fx]
        x[:, b] = col
    ctx = Bd.Context.from_instance(planted, dtype=dtype, device=device)
    xd = torch.from_numpy(x).cuda()
    flag = torch.zeros(2, dtype=torch.int32).pin_memory()
    ctx.step(xd, inst.eta, 2, want_F=False)                      # warm-up (module load, workspace)
    xd.copy_(torch.from_numpy(x))
    torch.cuda.synchronize()
    # the launching call blocks the host while the launch queue is full, so the flag is polled from a
    # second thread (the ctypes call releases the GIL); the device writes it through mapped pinned memory
    fl = flag.numpy()
    seen = {}
    stop = threading.Event()

    def poll():
        while not stop.is_set():
            if fl[0] == 1:
                seen["t"] = time.perf_counter()
                return
            time.sleep(0.0001)
    th = threading.Thread(target=poll, daemon=True)
    t0 = time.perf_counter()
    th.start()
    F, sat, sol, first = ctx.step(xd, inst.eta, max_steps, want_F=False, h_any_solved=flag)
    torch.cuda.synchronize()
    t_all = time.perf_counter() - t0
    stop.set()
    th.join(timeout=1)
    t_first = (seen["t"] - t0) if "t" in seen else (t_all if int(flag[0]) == 1 else None)
    out = {"instance": planted.name, "steps_run": max_steps, "probe_candidates": len(probes),
           "first_solved_step": int(flag[1]) if int(flag[0]) else None,
           "ms_to_first_solution": None if t_first is None else 1e3 * t_first,
           "ms_all_steps": 1e3 * t_all, "solved_candidates": int(sol.sum().item()),
           "random_instance": "no candidate solved in the benchmark's steps (far above the satisfiability threshold)"}
    ctx.close()
    return out


def rank_x0_seed(cfg, rank):
    """Replicas only: every rank draws its own batch of candidates."""
    from paper_2606_06641_b200 import instances as I
    return I.SEED_X0 + cfg + 1000 * rank


def reduce_max(values, device="cpu"):
    """Max over ranks of a list of per-rank timings (the only cross-rank datum of the benchmark)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return t.tolist()


def whole_job_value(world, m, B, K, seconds):
    """evals/s of the whole job: every rank processed m*B*K evaluations in `seconds` (max over ranks)."""
    return world * m * B * K / seconds


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    inst = workload(args.config, args.batch, args.scale)
    from paper_2606_06641_b200 import instances as I
    x0 = I.make_x0(inst)
    target = max(2.0, min(20.0, 60.0 / max(1, args.steps + args.warmup)))
    for _ in range(min(args.warmup, 1)):
        oracle_sample(inst, x0, target_s=min(target, 3.0))
    vals, times, b_o = [], [], 0
    for _ in range(args.steps):
        cb, dt, b_o = oracle_sample(inst, x0, target_s=target)
        vals.append(cb["value"]); times.append(dt)
    total_evals = inst.n_cons * b_o * len(times)
    value = total_evals / sum(times)
    cb["value"] = value
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * sum(times) / len(times),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f80 (x87 long double)",
            "data": "synthetic", "config": config_dict(inst, args.config, args.scale, args.gpus, extra={"sampled_candidates": b_o}),
            "cpu_baseline": cb, "gpu_launches": 0,
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)
    return 0


def config_dict(inst, cfg, scale, gpus, extra=None):
    ks = inst.lengths()
    d = {"workload": f"BASELINE.json configs[{cfg}]: {inst.name}", "n_vars": inst.n_vars,
         "n_constraints": inst.n_cons, "nnz": inst.nnz, "k_min": int(ks.min()), "k_max": int(ks.max()),
         "batch_per_gpu": inst.batch, "eta": inst.eta, "scale": scale,
         "parallelism": "replicas (candidates sharded, no collective)" if gpus > 1 else "single GPU",
         "l2": "flushed between timed steps (256 MiB write, untimed); per-step CUDA events summed"}
    d.update(extra or {})
    return d


def measure(cfg, dtype, K, W, *, batch=None, scale=1.0, oracle_seconds=10.0, rank=0, world=1, local=0, full=True,
            line_search=0, flags=0):
    """One workload through the C ABI: K timed steps (L2 flushed between them), the same K steps in one call, the
    evaluation / update / count kernels timed live with CUDA events, the end-to-end call on host buffers, and the
    oracle on a bounded sample beside it.  Returns the per-rank measurement dict (times already max-reduced)."""
    import torch
    import torch.distributed as dist
    from paper_2606_06641_b200 import binding as Bd, instances as I

    inst = workload(cfg, batch, scale)
    m, B, n = inst.n_cons, inst.batch, inst.n_vars
    npdt = np.float32 if dtype == 32 else np.float64
    x0 = I.make_x0(inst, seed=rank_x0_seed(cfg, rank), dtype=npdt)
    ctx = Bd.Context.from_instance(inst, dtype=dtype, device=local, flags=flags)
    ldb = ctx.ldb
    stream = torch.cuda.current_stream()
    x = torch.from_numpy(x0).cuda()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    state = None
    sol = None
    # The timed step delivers the objective too: F_pre = F(X(t-1)), the contraction a3 of the very products the gradient is
    # made of (one "eval" of the metric = the value AND all k partials of a constraint).  Without it afsat_step runs the
    # gradient-only form of the packed kernels; that is measured beside it (step_without_objective).  The one-launch loop of
    # small instances (cfg0) never evaluates the objective, so there the request would only switch the path.
    persistent = ctx.query(Bd.Q_STEP_PATH) == Bd.STEP_PERSISTENT
    F_pre_dev = None if persistent else torch.empty(B, dtype=x.dtype, device=x.device)

    def one_step(t, with_objective=True):
        nonlocal state, sol
        _, _, sol, first = ctx.step(x, inst.eta, 1, step_base=t, state=state, want_F=False,
                                    F_pre=F_pre_dev if with_objective else None)
        state = (sol, first)

    for t in range(W):
        one_step(t)
        flush.fill_(t & 0xFF)
    # ---- timed region: K steps, per-step events, L2 flushed (untimed) between steps ----------------
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    l0 = ctx.query(Bd.Q_KERNEL_LAUNCHES)
    wall0 = time.perf_counter()
    for t in range(K):
        ev[t][0].record(stream)
        one_step(W + t)
        ev[t][1].record(stream)
        flush.fill_(t & 0xFF)
    barrier()
    wall = time.perf_counter() - wall0
    launches = ctx.query(Bd.Q_KERNEL_LAUNCHES) - l0
    clocks = sampler.stop()
    t_total = sum(a.elapsed_time(b) for a, b in ev) * 1e-3
    # ---- the same K flushed steps with no objective requested (gradient-only kernels) ----------------------
    t_nof = None
    if F_pre_dev is not None:
        ev2 = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
        one_step(W + K, with_objective=False)
        flush.fill_(1)
        barrier()
        for t in range(K):
            ev2[t][0].record(stream)
            one_step(W + K + 1 + t, with_objective=False)
            ev2[t][1].record(stream)
            flush.fill_(t & 0xFF)
        barrier()
        t_nof = sum(a.elapsed_time(b) for a, b in ev2) * 1e-3
    # ---- back-to-back (L2-warm) variant: what a solver run sees (ONE call; cfg0: its own 200 steps) -------
    K_warm = max(K, inst.steps) if cfg == 0 else K
    ctx.step(x, inst.eta, min(K_warm, 3), step_base=W + K, state=state, want_F=False)
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l1 = ctx.query(Bd.Q_KERNEL_LAUNCHES)
    e0.record(stream)
    ctx.step(x, inst.eta, K_warm, step_base=W + K + 3, state=state, want_F=False)
    e1.record(stream)
    barrier()
    t_warm = e0.elapsed_time(e1) * 1e-3 * K / K_warm
    launches_warm_call = ctx.query(Bd.Q_KERNEL_LAUNCHES) - l1
    # ---- afsat_eval_grad alone (a1-a5 into a caller-owned full-width G, F reduced) --------
    t_eg = None
    if full or n * ldb * (4 if dtype == 32 else 8) <= (2 << 30):
        Gfull = torch.empty_like(x)
        Ffull = torch.empty(B, dtype=x.dtype, device=x.device)
        K_eg = min(K, 5)
        ctx.eval_grad(x, Ffull, Gfull)
        barrier()
        t_eg = 0.0
        for t in range(K_eg):
            flush.fill_(t & 0xFF)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            ctx.eval_grad(x, Ffull, Gfull)
            e1.record(stream)
            barrier()
            t_eg += e0.elapsed_time(e1) * 1e-3
        t_eg = t_eg * K / K_eg
        del Gfull, Ffull
    # ---- kernels of a step, timed with events inside the library (a second pass of K flushed steps) ----
    path = ctx.query(Bd.Q_STEP_PATH)
    kern_ms = upd_ms = chk_ms = 0.0
    kern_launches = 0
    if path != Bd.STEP_PERSISTENT:
        ctx.set_profiling(True)
        for t in range(K):
            one_step(W + 2 * K + t)
            flush.fill_(t & 0xFF)
        barrier()
        kern_ms, kern_launches = ctx.profiled_eval_ms()
        upd_ms = ctx.query(Bd.Q_PROFILED_UPDATE_NS) * 1e-6
        chk_ms = ctx.query(Bd.Q_PROFILED_CHECK_NS) * 1e-6
        ctx.set_profiling(False)
    # ---- end to end: HOST buffers, H2D + step + D2H inside the timed region ---------------------------
    hx = torch.from_numpy(x0.copy()).pin_memory()
    F_pre = np.empty(B, dtype=npdt)
    K_e2e = K if full else min(K, 5)
    for _ in range(2):
        ctx.step_host(hx, inst.eta, 1, want_F=False, F_pre=F_pre)
    barrier()
    w0 = time.perf_counter()
    for _ in range(K_e2e):
        ctx.step_host(hx, inst.eta, 1, want_F=False, F_pre=F_pre)
    barrier()
    t_e2e = (time.perf_counter() - w0) * K / K_e2e
    del hx
    # ---- optional: Alg. 1 with the line search (afsat_step_ls), reported beside the headline ---------
    t_ls = None
    if line_search:
        xl = torch.from_numpy(x0).cuda()
        ls_kw = dict(s_max=1.0, beta=0.5, c1=1e-4, delta=1e-6, max_trials=line_search)
        ls_state = None
        for t in range(max(W, 1)):
            *_, s_, f_, c_ = ctx.step_ls(xl, 1, step_base=t, state=ls_state, want_F=False, **ls_kw)
            ls_state = (s_, f_, c_)
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for t in range(K):
            *_, s_, f_, c_ = ctx.step_ls(xl, 1, step_base=W + t, state=ls_state, want_F=False, **ls_kw)
            ls_state = (s_, f_, c_)
        e1.record(stream)
        barrier()
        t_ls = e0.elapsed_time(e1) * 1e-3
        del xl
    esz = 4 if dtype == 32 else 8
    t_total, t_warm, t_e2e, kern_ms, upd_ms, chk_ms, t_eg_r, t_nof_r = reduce_max(
        [t_total, t_warm, t_e2e, kern_ms, upd_ms, chk_ms, t_eg if t_eg is not None else 0.0, t_nof if t_nof is not None else 0.0],
        device="cuda")
    t_eg = t_eg_r if t_eg is not None else None
    t_nof = t_nof_r if t_nof is not None else None
    out = {"inst": inst, "x0": x0, "ctx": ctx, "K": K, "W": W, "dtype": dtype, "cfg": cfg, "t_total": t_total, "t_warm": t_warm,
           "t_e2e": t_e2e, "kern_ms": kern_ms, "upd_ms": upd_ms, "chk_ms": chk_ms, "kern_launches": kern_launches,
           "launches": launches, "launches_warm_call": launches_warm_call, "K_warm": K_warm, "clocks": clocks, "wall": wall,
           "h2d": n * ldb * esz, "d2h": n * ldb * esz + B * (esz + 4 + 1 + 4), "t_ls": t_ls, "t_eg": t_eg, "t_nof": t_nof, "path": path,
           "solved": int(sol.sum().item()), "scale": scale}
    del x, flush
    return out


LTS_BYTES_PER_CLK = 6300.0       # B300_MICROARCH.md "LTS throughput cap ~6300 B/cyc full-chip": the L2's delivery rate


def l2_report(inst, ctx, B, kern_ms_per_step, cap, local=0):
    """Second roofline of the evaluation kernels: L2 throughput.  Algorithmic bytes = 4 B gathered + 4 B scatter-added per
    literal and candidate on the table the kernels run (after substitution).  Reported beside the ALU
    roofline because cfg4 (k = 3..5, ~7 flop per byte of L2 traffic) sits close to both; which of them binds is settled by
    experiment in DESIGN.md 6.7, not by this ratio."""
    from paper_2606_06641_b200 import binding as Bd
    peaks = load_peaks()
    alg = 8.0 * ctx.query(Bd.Q_LIVE_NNZ) * B
    cap_gbs = LTS_BYTES_PER_CLK * peaks["sm_max_mhz"] * 1e6 / 1e9
    rd, red, mix = probed_peak(3, local) * 1e3, probed_peak(4, local) * 1e3, probed_peak(5, local) * 1e3
    out = {"algorithmic_bytes_per_step": alg, "achieved_gbs": alg / (kern_ms_per_step * 1e-3) / 1e9 if kern_ms_per_step > 0 else 0.0,
           "peak_gbs": cap_gbs, "peak_source": "guide: ~6300 B/clk full-chip LTS cap (B300_MICROARCH.md) x sm_max_mhz",
           "peak_measured": {"load_gbs": rd, "red_gbs": red, "half_and_half_gbs": mix,
                             "how": "afsat_probe_peak kinds 3 / 4 / 5: 16-byte L1-bypassing loads / red.global.add.v4.f32 / both in equal "
                                    "parts over a 24 MB L2-resident buffer from every SM, CUDA events, best of 3; the evaluation kernels "
                                    "move half of their algorithmic bytes each way"},
           "lts_bytes_per_step_measured": cap.get("lts_bytes_per_step_eval_kernels")}
    if out["peak_measured"]["half_and_half_gbs"]:
        out["frac_of_measured"] = out["achieved_gbs"] / out["peak_measured"]["half_and_half_gbs"]
    out["frac"] = out["achieved_gbs"] / cap_gbs
    if cap.get("lts_bytes_per_step_eval_kernels") and kern_ms_per_step > 0:
        out["measured_traffic_gbs"] = cap["lts_bytes_per_step_eval_kernels"] / (kern_ms_per_step * 1e-3) / 1e9
        out["measured_traffic_frac_of_peak"] = out["measured_traffic_gbs"] / cap_gbs
    return out


def report(r, world, local, oracle_seconds, rank0_oracle=True):
    """The JSON-able report of one measurement (rank 0)."""
    import torch
    from paper_2606_06641_b200 import binding as Bd
    inst, ctx, K, dtype, cfg = r["inst"], r["ctx"], r["K"], r["dtype"], r["cfg"]
    m, B, n = inst.n_cons, inst.batch, inst.n_vars
    peaks = load_peaks()
    sm = ctx.query(Bd.Q_SM_COUNT)
    flop_c, instr_c = flop_model(inst)
    flop_sub, instr_sub = ctx.query(Bd.Q_FLOP_PER_CANDIDATE), ctx.query(Bd.Q_FP_INSTR_PER_CANDIDATE)
    value = whole_job_value(world, m, B, K, r["t_total"])
    kern_ms = r["kern_ms"]
    flop_per_step = flop_c * B
    peak_tf = sm * FP32_LANES_PER_SM * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12
    ach_tf = flop_per_step / (kern_ms * 1e-3 / K) / 1e12 if kern_ms > 0 else 0.0
    esz = 4 if dtype == 32 else 8
    cap = load_capture(cfg, dtype)
    path_name = {1: "launches", 2: "persistent (one launch)", 3: "cuda graph"}.get(r["path"], str(r["path"]))
    roof = {"bound": "alu",
            "kernel": "evaluation kernels, a1-a5 (fp32: k_eval_f2m k<=8 | k_eval_split k>=9; fp64: k_eval_km k<=8 | "
                      "k_eval_split k>=9): all launches of one step",
            "achieved": ach_tf, "peak": peak_tf, "unit": "TFLOP/s", "frac": ach_tf / peak_tf,
            "peak_source": f"{sm} SMs x 128 FP32 lanes x 2 flop x {peaks['sm_max_mhz']:.0f} MHz "
                           f"({peaks['source']} sm_max_mhz; DESIGN.md 6); MEASURED_PEAKS.json has no FP32 figure, so the "
                           f"probe below checks it",
            "peak_measured": {"ffma_tflops": probed_peak(0, local), "ffma2_tflops": probed_peak(1, local),
                              "dfma_tflops": probed_peak(2, local),
                              "how": "afsat_probe_peak: 8 independent FMA chains per thread, CUDA events, best of 5"},
            "model_instr_over_issue_peak": (instr_c * B / (kern_ms * 1e-3 / K)) / (sm * FP32_LANES_PER_SM * peaks["sm_max_mhz"] * 1e6)
            if kern_ms > 0 else 0.0,
            "measured_pipe_utilisation": {k_: cap.get(k_) for k_ in ("kernel", "sm__pipe_fma_cycles_active_pct",
                                                                      "sm__pipe_fp64_cycles_active_pct", "smsp__issue_active_pct",
                                                                      "executed_warp_instructions_per_launch", "capture")} if cap else None,
            "kernel_ms_per_step": kern_ms / K, "kernel_launches_per_step": max(1, r["kern_launches"] // K) if r["kern_launches"] else 0,
            "kernel_share_of_step": (kern_ms / K) / (1e3 * r["t_total"] / K),
            "update_ms_per_step": r["upd_ms"] / K, "count_ms_per_step": r["chk_ms"] / K,
            "algorithmic_flop_per_step": flop_per_step,
            "algorithmic_flop_per_step_after_substitution": flop_sub * B,
            "frac_after_substitution": (flop_sub * B / (kern_ms * 1e-3 / K) / 1e12) / peak_tf if kern_ms > 0 else 0.0,
            "traffic": cap.get("dram_bytes_per_step_eval_kernels"),
            "traffic_whole_step": cap.get("dram_bytes_per_step"),
            "traffic_source": cap.get("traffic_capture"),
            "l2": l2_report(inst, ctx, B, kern_ms / K, cap, local),
            "hbm_floor_bytes_per_step": 2 * n * B * esz, "hbm_peak_gbs": peaks["hbm_gbs"],
            "note": "achieved = ALGORITHMIC flop of the instance as given (SURVEY.md App. D: 12 / 4 FP32 instructions per literal at a "
                    "complex / real DFT point, every retained point) / measured kernel time.  The kernels execute fewer instructions: "
                    "trivial twiddles at the points 1 and -1, literal groups with folded weights at the complex points (k <= 8) and literal "
                    "groups in the lane-split kernels (k >= 9), and a partial assignment is substituted before anything is evaluated (frac_after_substitution "
                    "counts the model on the substituted table); measured_pipe_utilisation is what ncu saw executed"}
    l2 = roof["l2"]
    roof["limited_by"] = ("instruction issue at the occupancy the register file allows (roofline.measured_pipe_utilisation; DESIGN.md 6.7: "
                          "in three A/B experiments the kernel time followed the executed-instruction count, not the L2 traffic)")
    if l2.get("measured_traffic_frac_of_peak"):
        roof["limited_by"] += "; measured L2 traffic of the evaluation kernels at %.0f %% of the guide's L2 cap" % (
            100 * l2["measured_traffic_frac_of_peak"])
    if dtype == 64:
        roof["fp64_peak"] = probed_peak(2, local)
        roof["frac_of_fp64_peak"] = ach_tf / max(probed_peak(2, local), 1e-9)
    if r["clocks"].get("sm_mhz"):
        roof["frac_at_observed_clock"] = roof["frac"] * peaks["sm_max_mhz"] / r["clocks"]["sm_mhz"]
    if r["path"] == Bd.STEP_PERSISTENT:
        roof["note_small"] = "launch-latency-bound workload: the whole step loop is one launch; no per-kernel roofline"
    cb = dev_rep = None
    if rank0_oracle:
        x0 = r["x0"]
        cb, _, b_o = oracle_sample(inst, x0.astype(np.float64), target_s=oracle_seconds)
        # deviation vs the oracle (BASELINE.json configs[3]: "report deviation vs oracle"): ONE step from x0
        # on the GPU against the oracle's step on the sampled candidates -- X(1) = clamp(x0 - eta G), so
        # max|dX| / eta is the gradient deviation where the clamp is inactive; counts are bit-exact or not
        X1o, sat1o = oracle_sample.last
        xd = torch.from_numpy(np.ascontiguousarray(x0)).cuda()
        _, sat_d, _, _ = ctx.step(xd, inst.eta, 1, step_base=0, state=None, want_F=False)
        torch.cuda.synchronize()
        dX = np.abs(xd[:, :b_o].double().cpu().numpy() - X1o)
        dev_rep = {"candidates": int(b_o), "max_abs_dX_after_one_step": float(dX.max()),
                   "max_abs_dG_implied": float(dX.max() / inst.eta),
                   "sat_count_bit_exact": bool(np.array_equal(sat_d[:b_o].cpu().numpy(), sat1o)),
                   "tables": "default (paper tables to k = 20, robust tables beyond)"}
        del xd
    out = {"value": value, "unit": UNIT, "ms_per_step": 1e3 * r["t_total"] / K, "dtype": "f32" if dtype == 32 else "f64",
           "config": config_dict(inst, cfg, r["scale"], world), "clocks": r["clocks"], "gpu_launches": int(r["launches"]),
           "step_path": path_name,
           "e2e": {"value": world * m * B * K / r["t_e2e"], "unit": UNIT, "h2d_bytes_per_step": r["h2d"],
                   "d2h_bytes_per_step": r["d2h"], "ms_per_step": 1e3 * r["t_e2e"] / K,
                   "result_read_back": "X(t), F(X(t-1)) (by-product of the fused pass), sat_count, is_solution, first_step"},
           "roofline": roof, "cpu_baseline": cb, "deviation_vs_oracle": dev_rep,
           "value_l2_warm": world * m * B * K / r["t_warm"], "ms_per_step_l2_warm": 1e3 * r["t_warm"] / K,
           "l2_warm_call": {"n_steps": r["K_warm"], "launches": int(r["launches_warm_call"])},
           "solved_candidates": r["solved"], "wall_s_timed_region": r["wall"]}
    out["objective_in_timed_step"] = ("F(X(t-1)) delivered by every timed step (F_pre: a3 of the same products as the gradient)"
                                      if r.get("t_nof") else "not evaluated: the one-launch loop of small instances computes gradients only")
    if r.get("t_nof"):
        out["step_without_objective"] = {"ms_per_step": 1e3 * r["t_nof"] / K, "value": world * m * B * K / r["t_nof"], "unit": UNIT,
                                         "note": "afsat_step with no objective requested (what the fixed-step search of Alg. 1 needs: "
                                                 "X(t), counts, flags): the packed kernels run their gradient-only form, which drops "
                                                 "the contraction a3; value_l2_warm (K steps in ONE call) is measured this way too"}
    if r.get("t_eg"):
        out["eval_grad_alone"] = {"ms_per_call": 1e3 * r["t_eg"] / K, "value": world * m * B * K / r["t_eg"], "unit": UNIT,
                                  "note": "afsat_eval_grad on its own: F and a caller-owned full-width G (memset + a1-a5 + the "
                                          "fixed-order reduction of F), L2 flushed between calls; the fused step adds a6-a9"}
    if r["t_ls"] is not None:
        out["line_search"] = {"ms_per_step": 1e3 * r["t_ls"] / K,
                              "note": "afsat_step_ls: 1 FE+grad evaluation + max_trials objective-only "
                                      "evaluations of the candidates still searching, per step (L2 warm)"}
    return out


def sweep_batch(cfg, dtype, local, K=5):
    """Throughput against batch size (Fig. 2b: the paper's throughput peaks where the working set is
    ~2x the device cache and decays beyond; candidate tiling is this build's answer)."""
    import torch
    from paper_2606_06641_b200 import binding as Bd, instances as I
    rows = []
    base = workload(cfg)
    esz = 4 if dtype == 32 else 8
    for B in (64, 128, 256, 512, 1024, 2048, 4096, 8192, 16384, 32768, 65536):
        if 2 * base.n_vars * B * esz > 60e9:
            break
        inst = workload(cfg, B)
        x0 = I.make_x0(inst, dtype=np.float32 if dtype == 32 else np.float64)
        ctx = Bd.Context.from_instance(inst, dtype=dtype, device=local)
        x = torch.from_numpy(x0).cuda()
        ctx.step(x, inst.eta, 2, want_F=False)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        ctx.step(x, inst.eta, K, want_F=False)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / K
        rows.append({"batch": B, "x_bytes": inst.n_vars * ctx.ldb * esz, "working_set_over_l2": 2 * inst.n_vars * ctx.ldb * esz / ctx.query(Bd.Q_L2_BYTES),
                     "tile_w": ctx.query(Bd.Q_TILE_W), "ms_per_step": ms, "evals_per_s": inst.n_cons * B / (ms * 1e-3)})
        ctx.close()
        del x, x0
        torch.cuda.empty_cache()
    return rows


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2606_06641_b200 import binding as Bd, build as Build

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        Build.build()
    if world > 1:
        dist.barrier()
    t_run0 = time.perf_counter()
    K, W = args.steps, max(args.warmup, 0)
    r = measure(args.config, args.dtype, K, W, batch=args.batch, scale=args.scale, rank=rank, world=world, local=local,
                line_search=args.ls_trials if args.line_search else 0)
    line = None
    if rank == 0:
        rep = report(r, world, local, args.oracle_seconds)
        line = {"metric": METRIC, "value": rep.pop("value"), "unit": rep.pop("unit"), "n_gpus": world, "steps": K, "warmup": W,
                "ms_per_step": rep.pop("ms_per_step"), "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": rep.pop("dtype"), "data": "synthetic"}
        line.update(rep)
    # ---- time to first solution (BASELINE.json configs[4]) on the PLANTED variant of the headline workload ----
    if rank == 0 and world == 1 and not args.no_ttfs:
        line["time_to_first_solution"] = time_to_first_solution(r["inst"], r["x0"], args.dtype, local, args.ttfs_steps)
    r["ctx"].close()
    r.clear()
    torch.cuda.empty_cache()
    # ---- the other configurations of BASELINE.json (and cfg3 in fp64), single GPU only -------------------------
    if rank == 0 and world == 1 and not args.no_per_config and args.batch is None and args.scale == 1.0:
        per = {}
        todo = [(c, 32) for c in range(5) if c != args.config or args.dtype != 32] + [(3, 64)]
        for c, dt in todo:
            Kc = 200 if c == 0 else max(5, min(K, 10))
            rc = measure(c, dt, Kc, 3, local=local, full=False)
            rp = report(rc, 1, local, args.per_config_oracle_seconds)
            keep = {k_: rp[k_] for k_ in ("ms_per_step", "value", "ms_per_step_l2_warm", "value_l2_warm", "l2_warm_call", "step_path",
                                          "gpu_launches", "deviation_vs_oracle", "clocks", "solved_candidates")}
            if "eval_grad_alone" in rp:
                keep["eval_grad_alone"] = {k_: rp["eval_grad_alone"][k_] for k_ in ("ms_per_call", "value")}
            keep["objective_in_timed_step"] = rp["objective_in_timed_step"]
            if "step_without_objective" in rp:
                keep["step_without_objective"] = {k_: rp["step_without_objective"][k_] for k_ in ("ms_per_step", "value")}
            keep["steps"] = Kc
            keep["e2e"] = {k_: rp["e2e"][k_] for k_ in ("value", "ms_per_step")}
            keep["cpu_baseline"] = {k_: rp["cpu_baseline"][k_] for k_ in ("value", "cores", "sample")}
            keep["roofline"] = {k_: rp["roofline"].get(k_) for k_ in ("frac", "achieved", "peak", "frac_after_substitution",
                                                                      "frac_of_fp64_peak", "model_instr_over_issue_peak",
                                                                      "kernel_ms_per_step", "kernel_share_of_step",
                                                                      "update_ms_per_step", "count_ms_per_step",
                                                                      "measured_pipe_utilisation", "traffic", "l2", "note_small")}
            if c == 3:
                # BASELINE.json configs[3]: "run in both fp32 and fp64 and report deviation vs oracle" -- also for the paper's
                # own product form (AFSAT_FLAG_PAPER), which the default context replaces beyond k = 20
                rq = measure(c, dt, 5, 2, local=local, full=False, flags=Bd.FLAG_PAPER)
                rq_rep = report(rq, 1, local, 2.0)
                rq_rep["deviation_vs_oracle"]["tables"] = "paper tables at every length (AFSAT_FLAG_PAPER)"
                keep["paper_tables"] = {"ms_per_step": rq_rep["ms_per_step"], "deviation_vs_oracle": rq_rep["deviation_vs_oracle"]}
                rq["ctx"].close()
            per[f"cfg{c}" + ("_f64" if dt == 64 else "")] = keep
            rc["ctx"].close()
            rc.clear()
            torch.cuda.empty_cache()
        line["per_config"] = per
    if rank == 0 and world == 1 and args.sweep_batch:
        line["batch_sweep"] = {f"cfg{c}": sweep_batch(c, 32, local) for c in (1, 3)}
    if rank == 0:
        line["wall_s_whole_run"] = time.perf_counter() - t_run0
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--batch", type=int, default=None)
    ap.add_argument("--scale", type=float, default=1.0)
    ap.add_argument("--dtype", type=int, default=32, choices=[32, 64])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--oracle-seconds", type=float, default=10.0)
    ap.add_argument("--per-config-oracle-seconds", type=float, default=2.5)
    ap.add_argument("--no-per-config", action="store_true", help="headline workload only")
    ap.add_argument("--no-ttfs", action="store_true", help="skip the time-to-first-solution run")
    ap.add_argument("--ttfs-steps", type=int, default=100)
    ap.add_argument("--sweep-batch", action="store_true", help="also throughput vs batch size on cfg1 and cfg3 (PAPER.md Fig. 2b)")
    ap.add_argument("--probe-peaks", action="store_true", help="print the measured FFMA / FFMA2 / DFMA peaks and exit")
    ap.add_argument("--line-search", action="store_true", help="also time afsat_step_ls (Alg. 1 with line search)")
    ap.add_argument("--ls-trials", type=int, default=4)
    args = ap.parse_args()
    if args.probe_peaks:
        from paper_2606_06641_b200 import build as Build
        Build.build()
        print(json.dumps({"ffma_tflops": probed_peak(0, 0), "ffma2_tflops": probed_peak(1, 0), "dfma_tflops": probed_peak(2, 0),
                          "l2_load_tbs": probed_peak(3, 0), "l2_red_tbs": probed_peak(4, 0), "l2_half_and_half_tbs": probed_peak(5, 0)}))
        return 0
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())

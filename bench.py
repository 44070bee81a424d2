#!/usr/bin/env python
"""bench.py -- headline benchmark of the AFSAT hot path on B200 (contract in DESIGN.md "Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1] [--impl ours|reference]

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


def load_traffic(cfg):
    """DRAM bytes per launch of the dominant kernel from the committed ncu capture (profiles/), or None."""
    p = os.path.join(ROOT, "profiles", "r1_traffic.json")
    try:
        with open(p) as f:
            return json.load(f).get(f"cfg{cfg}", {}).get("bytes_per_launch")
    except (OSError, ValueError):
        return None


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
                      f"{inst.batch} candidates x 1 step over all {inst.n_cons} constraints, {dt:.2f} s"}, dt, b_o


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
    xd.copy_(torch.from_numpy(x).cuda())
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
            "data": "synthetic", "config": config_dict(inst, args, extra={"sampled_candidates": b_o}),
            "cpu_baseline": cb, "gpu_launches": 0,
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)
    return 0


def config_dict(inst, args, extra=None):
    ks = inst.lengths()
    d = {"workload": f"BASELINE.json configs[{args.config}]: {inst.name}", "n_vars": inst.n_vars,
         "n_constraints": inst.n_cons, "nnz": inst.nnz, "k_min": int(ks.min()), "k_max": int(ks.max()),
         "batch_per_gpu": inst.batch, "eta": inst.eta, "scale": args.scale,
         "parallelism": "replicas (candidates sharded, no collective)" if args.gpus > 1 else "single GPU",
         "l2": "flushed between timed steps (256 MiB write, untimed); per-step CUDA events summed"}
    d.update(extra or {})
    return d


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2606_06641_b200 import binding as Bd, build as Build, instances as I

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
    inst = workload(args.config, args.batch, args.scale)
    m, B, n = inst.n_cons, inst.batch, inst.n_vars
    dtype = args.dtype
    npdt = np.float32 if dtype == 32 else np.float64
    x0 = I.make_x0(inst, seed=rank_x0_seed(args.config, rank), dtype=npdt)
    ctx = Bd.Context.from_instance(inst, dtype=dtype, device=local)
    ldb = ctx.ldb
    stream = torch.cuda.current_stream()
    x = torch.from_numpy(x0).cuda()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    K, W = args.steps, max(args.warmup, 0)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    state = None
    F = sat = sol = first = None

    def one_step(t):
        nonlocal state, F, sat, sol, first
        F, sat, sol, first = ctx.step(x, inst.eta, 1, step_base=t, state=state, want_F=False)
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
    ms = [a.elapsed_time(b) for a, b in ev]
    t_total = sum(ms) * 1e-3
    # ---- back-to-back (L2-warm) variant: what a solver run sees; reported beside the headline -------
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    F, sat, sol, first = ctx.step(x, inst.eta, K, step_base=W + K, state=state, want_F=False)
    e1.record(stream)
    barrier()
    t_warm = e0.elapsed_time(e1) * 1e-3
    # ---- dominant kernel: per-launch duration measured with events inside the library --------------
    ctx.set_profiling(True)
    for t in range(K):
        one_step(W + 2 * K + t)
        flush.fill_(t & 0xFF)
    barrier()
    kern_ms, kern_launches = ctx.profiled_eval_ms()
    ctx.set_profiling(False)
    # ---- end to end: HOST buffers, H2D + step + D2H inside the timed region ---------------------------
    hx = torch.from_numpy(x0.copy()).pin_memory()
    for _ in range(min(W, 3)):
        ctx.step_host(hx, inst.eta, 1, want_F=True)
    barrier()
    w0 = time.perf_counter()
    for _ in range(K):
        ctx.step_host(hx, inst.eta, 1, want_F=True)
    barrier()
    t_e2e = time.perf_counter() - w0
    # ---- optional: Alg. 1 with the line search (afsat_step_ls), reported beside the headline ---------
    t_ls = None
    if args.line_search:
        xl = torch.from_numpy(x0).cuda()
        ls_kw = dict(s_max=1.0, beta=0.5, c1=1e-4, delta=1e-6, max_trials=args.ls_trials)
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
    # ---- optional: time to first solution (BASELINE.json configs[4]) on the PLANTED variant of the workload ----
    ttfs = None
    if args.ttfs:
        ttfs = time_to_first_solution(inst, x0, dtype, local, args.ttfs_steps)
    esz = 4 if dtype == 32 else 8
    h2d = n * ldb * esz
    d2h = n * ldb * esz + B * (esz + 4 + 1 + 4)

    t_total, t_warm, t_e2e, kern_ms = reduce_max([t_total, t_warm, t_e2e, kern_ms], device="cuda")
    if rank == 0:
        peaks = load_peaks()
        sm = ctx.query(Bd.Q_SM_COUNT)
        flop_c, instr_c = flop_model(inst)
        evals = world * m * B * K
        value = whole_job_value(world, m, B, K, t_total)
        kern_s = kern_ms * 1e-3 / max(1, kern_launches)          # avg duration of one eval launch set
        launches_per_step = max(1, kern_launches // K)
        flop_per_step = flop_c * B
        peak_tf = sm * FP32_LANES_PER_SM * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12
        ach_tf = flop_per_step / (kern_ms * 1e-3 / K) / 1e12 if kern_ms > 0 else 0.0
        roof = {"bound": "alu", "kernel": "evaluation kernels, a1-a5 (fp32: k_eval_f2m k<=8 | k_eval_split k>=9; fp64: k_eval_km k<=20 | k_eval_split k>20): all launches of one step", "achieved": ach_tf, "peak": peak_tf,
                "unit": "TFLOP/s", "frac": ach_tf / peak_tf,
                "peak_source": f"{sm} SMs x 128 FP32 lanes x 2 flop x {peaks['sm_max_mhz']:.0f} MHz "
                               f"({peaks['source']} sm_max_mhz; DESIGN.md 'Roofline')",
                "fp32_issue_frac": (instr_c * B / (kern_ms * 1e-3 / K)) / (sm * FP32_LANES_PER_SM * peaks["sm_max_mhz"] * 1e6)
                if kern_ms > 0 else 0.0,
                "kernel_ms_per_step": kern_ms / K, "kernel_launches_per_step": launches_per_step,
                "kernel_share_of_step": (kern_ms / K) / (1e3 * t_total / K),
                "algorithmic_flop_per_step": flop_per_step, "traffic": load_traffic(args.config),
                "hbm_floor_bytes_per_step": 2 * n * B * esz, "hbm_peak_gbs": peaks["hbm_gbs"],
                "note": "achieved = ALGORITHMIC flop (SURVEY.md App. D: 12 / 4 FP32 instructions per literal at a complex / "
                        "real DFT point, every retained point) / measured kernel time; the kernels execute fewer "
                        "instructions than that at the points 1, -1, i (trivial twiddles, DESIGN.md 6.1)"}
        if dtype == 64:
            # the DFMA pipe issues 64 lanes per SM per clock on this part (ncu: sm__pipe_fp64_cycles_active 61.7 % for
            # 1.3e9 FP64 warp instructions in 4.0 ms, profiles/r1_eval_split_cfg3_f64.md): half the FP32 rate
            roof["fp64_peak"] = peak_tf / 2
            roof["frac_of_fp64_peak"] = ach_tf / (peak_tf / 2)
        if clocks.get("sm_mhz"):
            roof["frac_at_observed_clock"] = roof["frac"] * peaks["sm_max_mhz"] / clocks["sm_mhz"]
        cb = dev_rep = None
        if world == 1 or rank == 0:
            cb, _, b_o = oracle_sample(inst, x0.astype(np.float64), target_s=args.oracle_seconds)
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
                       "sat_count_bit_exact": bool(np.array_equal(sat_d[:b_o].cpu().numpy(), sat1o))}
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
                "ms_per_step": 1e3 * t_total / K, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f32" if dtype == 32 else "f64", "data": "synthetic",
                "config": config_dict(inst, args), "clocks": clocks, "gpu_launches": int(launches),
                "e2e": {"value": world * m * B * K / t_e2e, "unit": UNIT, "h2d_bytes_per_step": h2d,
                        "d2h_bytes_per_step": d2h, "ms_per_step": 1e3 * t_e2e / K},
                "roofline": roof, "cpu_baseline": cb, "deviation_vs_oracle": dev_rep,
                "value_l2_warm": world * m * B * K / t_warm, "ms_per_step_l2_warm": 1e3 * t_warm / K,
                "solved_candidates": int(sol.sum().item()), "wall_s_timed_region": wall}
        if ttfs is not None:
            line["time_to_first_solution"] = ttfs
        if t_ls is not None:
            line["line_search"] = {"ms_per_step": 1e3 * t_ls / K, "max_trials": args.ls_trials,
                                   "note": "afsat_step_ls: 1 FE+grad evaluation + max_trials objective-only "
                                           "evaluations of the candidates still searching, per step (L2 warm)"}
        print(json.dumps(line), flush=True)
    ctx.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", type=int, default=1)
    ap.add_argument("--batch", type=int, default=None)
    ap.add_argument("--scale", type=float, default=1.0)
    ap.add_argument("--dtype", type=int, default=32, choices=[32, 64])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--oracle-seconds", type=float, default=15.0)
    ap.add_argument("--ttfs", action="store_true", help="also report time to first solution on the planted variant")
    ap.add_argument("--ttfs-steps", type=int, default=100)
    ap.add_argument("--line-search", action="store_true", help="also time afsat_step_ls (Alg. 1 with line search)")
    ap.add_argument("--ls-trials", type=int, default=4)
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())

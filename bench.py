#!/usr/bin/env python
"""bench.py -- one line of JSON for the TACG/GESR hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2] [--impl tacg|reference]

A step is one pass of the whole hot path over one batch of synthetic traces:
  tacg_coact_accumulate(build trace) -> tacg_affinity_swapgain(primary) -> tacg_eval_placement(eval trace)
`value` = routed tokens (token x layer records, build + eval) per second with inputs resident
in HBM; `e2e` = the same through pinned HOST buffers (H2D of both traces and D2H of the results
inside the timed region).  `roofline` is the co-activation kernel against measured HBM bandwidth.
Multi-GPU: the path does not shard ("replicas only"): every rank runs the same
workload on its own seeded traces, no collective on the data path.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

import numpy as np
import torch

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import tracegen  # noqa: E402

METRIC = "trace tokens/s (coact build + placement eval)"
UNIT = "routed tokens/s"


# ------------------------------------------------------------------ helpers
def env_int(name, default):
    try:
        return int(os.environ.get(name, default))
    except ValueError:
        return default


class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int, period_s: float = 0.002):
        self.index, self.period = index, period_s
        self.samples, self.reasons = [], set()
        self.max_mhz = None
        self._stop = threading.Event()
        self._thr = None
        self.ok = False
        try:
            import pynvml
            self.nv = pynvml
            pynvml.nvmlInit()
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception:
            self.ok = False

    def _run(self):
        nv = self.nv
        names = {
            getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
            getattr(nv, "nvmlClocksEventReasonHwPowerBrakeSlowdown", 0x80): "hw_power_brake_slowdown",
        }
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    mask = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, nm in names.items():
                    if mask & bit:
                        self.reasons.add(nm)
            except Exception:
                pass
            time.sleep(self.period)

    def start(self):
        if self.ok:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()

    def stop(self):
        if self._thr:
            self._stop.set()
            self._thr.join()

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": 0}
        return {"sm_mhz": statistics.median(self.samples), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def ncu_traffic(config, path):
    """dram__bytes_read.sum + dram__bytes_write.sum of the co-activation kernel(s), per launch, from the
    committed ncu --set full capture (profiles/traffic.json, written by hand from the .ncu-rep); None if absent."""
    try:
        return json.load(open(os.path.join(ROOT, "profiles", "traffic.json")))[f"config{config}_{path}"]["bytes"]
    except Exception:
        return None


def coact_algorithmic_bytes(cfg):
    """indices read once + family once + D and C written once."""
    return cfg.L * cfg.N * cfg.k * 2 + cfg.N + cfg.L * cfg.F * (cfg.E * cfg.E + cfg.E) * 4


def make_sets(cfg, n_sets, rank, device):
    """n_sets distinct (build, eval) traces; together they exceed the 126 MB L2."""
    params = tracegen.make_params(cfg)
    sets = []
    for s in range(n_sets):
        seed = rank_seed(cfg.seed, s, rank)
        bi, bf = tracegen.gen_trace(cfg, params, eval_trace=False, device=device, seed=seed)
        ei, ef = tracegen.gen_trace(cfg, params, eval_trace=True, device=device, seed=seed)
        sets.append((bi, bf, ei, ef))
    return sets


# ------------------------------------------------------------------ the oracle legs (CPU)
def oracle_step(cbind, cfg, bi, bf, ei, ef, primary, replicas, Ls):
    """One pass of the hot path by the oracle on the first Ls layers.  Returns routed tokens done."""
    D, C, ntok = cbind.coact(bi[:Ls], bf, cfg.E, cfg.F)
    cbind.affinity_swapgain(D, C, ntok, cfg.P, primary[:Ls], alpha=0.25, tau=1.0, eps=1e-6)
    cbind.eval_placement(ei[:Ls], ef, cfg.E, cfg.F, cfg.P, primary[:Ls],
                         None if replicas is None else replicas[:Ls], theta=0.15, rho=0.995,
                         microbatch=cfg.microbatch, load_state=np.zeros((Ls, cfg.P)))
    return Ls * (bi.shape[1] + ei.shape[1])


def oracle_sample_layers(cbind, cfg, bi, bf, ei, ef, primary, replicas, budget_s):
    """Picks how many layers one oracle step covers so that it takes about budget_s."""
    threads = cbind.threads()
    L0 = min(cfg.L, threads)
    t0 = time.perf_counter()
    oracle_step(cbind, cfg, bi, bf, ei, ef, primary, replicas, L0)
    dt = max(1e-3, time.perf_counter() - t0)
    rounds = max(1, int(budget_s / dt))
    return max(1, min(cfg.L, L0 * rounds)), threads


def run_reference(args, cfg, rank):
    """--impl reference: the oracle, as it stands, on the host cores (rank 0 only)."""
    if rank != 0:
        return
    from oracle import cbind                      # the one other place bench.py executes oracle/
    device = "cuda" if torch.cuda.is_available() else "cpu"
    (bi, bf, ei, ef), = make_sets(cfg, 1, 0, device)
    bi, bf, ei, ef = (x.cpu().numpy() for x in (bi, bf, ei, ef))
    primary = tracegen.random_placement(cfg.E, cfg.P, cfg.capacity, cfg.L, seed=cfg.seed)
    replicas = tracegen.random_replicas(primary, cfg.P, cfg.r, cfg.n_rep, seed=cfg.seed + 1) if cfg.r else None
    per_step_budget = max(0.2, min(3.0, 120.0 / max(1, args.steps + args.warmup)))
    Ls, threads = oracle_sample_layers(cbind, cfg, bi, bf, ei, ef, primary, replicas, per_step_budget)
    for _ in range(args.warmup):
        oracle_step(cbind, cfg, bi, bf, ei, ef, primary, replicas, Ls)
    t0 = time.perf_counter()
    units = 0
    for _ in range(args.steps):
        units += oracle_step(cbind, cfg, bi, bf, ei, ef, primary, replicas, Ls)
    dt = time.perf_counter() - t0
    value = units / dt
    sample = f"first {Ls} of {cfg.L} layers, all {cfg.N}+{cfg.N_eval} tokens per layer, per step"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / max(1, args.steps),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u32", "data": "synthetic",
        "config": workload_config(cfg, 1, "n/a (CPU oracle)"),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def rank_seed(cfg_seed, set_index, rank):
    """Seed of trace set `set_index` on `rank`: every replica draws its own traces (replicas only)."""
    return cfg_seed + 17 * set_index + 1009 * rank


def max_over_ranks(ms, dist, device):
    """The only data exchanged between ranks: the elapsed time of the timed region, reduced with MAX."""
    if dist is None:
        return float(ms)
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(units_per_step, steps, world, ms_total):
    """Aggregate throughput of `world` independent replicas that each did units_per_step * steps units."""
    return world * units_per_step * steps / (ms_total * 1e-3)


def workload_config(cfg, n_sets, l2_note):
    return {
        "workload": f"BASELINE.json configs[{[k for k, v in tracegen.CONFIGS.items() if v.name == cfg.name][0] - 1}] "
                    f"{cfg.name}: E={cfg.E} k={cfg.k} L={cfg.L} F={cfg.F} N={cfg.N} (build) + {cfg.N_eval} (eval) "
                    f"tokens/layer, P={cfg.P} cap={cfg.capacity}, r={cfg.r}",
        "step": "tacg_coact_accumulate + tacg_affinity_swapgain + tacg_eval_placement",
        "unit_definition": "routed tokens = token x layer records consumed per step (build + eval trace)",
        "trace_sets": n_sets, "l2": l2_note, "parallelism": "replicas only (no data-path collective)",
    }


# ------------------------------------------------------------------ the CUDA path
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config number, 1-based (default 2 = configs[1])")
    ap.add_argument("--impl", default="tacg", choices=["tacg", "reference"])
    ap.add_argument("--sets", type=int, default=0, help="distinct trace sets rotated over (0 = enough to exceed L2)")
    ap.add_argument("--path", default="auto", choices=["auto", "hist", "mma"])
    ap.add_argument("--compare-paths", action="store_true",
                    help="also time tacg_coact_accumulate alone on both paths (histogram, tcgen05 kind::i8)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)

    rank = env_int("RANK", 0)
    local_rank = env_int("LOCAL_RANK", 0)
    world = env_int("WORLD_SIZE", 1)
    cfg = tracegen.get_config(args.config)

    if args.impl == "reference":
        run_reference(args, cfg, rank)
        return

    import paper_2606_01007_b200 as tacg
    from paper_2606_01007_b200 import placement

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the library has no CPU path")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    ctx = tacg.Context(local_rank)
    path_flag = {"auto": tacg.TACG_PATH_AUTO, "hist": tacg.TACG_PATH_HIST, "mma": tacg.TACG_PATH_MMA}[args.path]

    # ---- inputs: enough distinct trace sets that a step never finds its inputs in L2
    step_in_bytes = cfg.L * (cfg.N + cfg.N_eval) * cfg.k * 2 + cfg.N + cfg.N_eval
    n_sets = args.sets or max(2, int(np.ceil(3 * 126e6 / step_in_bytes)) + 1)
    free_b = torch.cuda.mem_get_info(dev)[0]
    n_sets = max(1, min(n_sets, int(0.5 * free_b / step_in_bytes)))
    sets = make_sets(cfg, n_sets, rank, dev)
    l2_note = (f"inputs rotate over {n_sets} distinct trace sets = {n_sets * step_in_bytes / 1e6:.0f} MB "
               f"(L2 is 126 MB)") if n_sets * step_in_bytes > 2 * 126e6 else \
        f"one step reads {step_in_bytes / 1e6:.0f} MB of inputs, larger than the 126 MB L2"

    # ---- outputs and placement inputs (allocated once; device memory is torch's job)
    L, E, F, P, k = cfg.L, cfg.E, cfg.F, cfg.P, cfg.k
    D = torch.empty((L, F, E), dtype=torch.int32, device=dev)
    Cm = torch.empty((L, F, E, E), dtype=torch.int32, device=dev)
    ntok = torch.empty((F,), dtype=torch.int64, device=dev)
    pref = torch.empty((L, E, F), dtype=torch.float32, device=dev)
    W = torch.empty((L, E, E), dtype=torch.float32, device=dev)
    aff = torch.empty((L, E, P), dtype=torch.float32, device=dev)
    gain = torch.empty((L, E, E), dtype=torch.float32, device=dev)
    load = torch.empty((L, P), dtype=torch.int64, device=dev)
    span = torch.empty((L, F), dtype=torch.int64, device=dev)
    remote = torch.empty((L, F), dtype=torch.int64, device=dev)
    ntok_e = torch.empty((F,), dtype=torch.int64, device=dev)
    fair = torch.empty((L + 1, 3), dtype=torch.float32, device=dev)

    # placement used by the step: local search on the first build trace, GESR table per config
    bi0, bf0, _, _ = sets[0]
    co = tacg.tacg_coact_accumulate(ctx, bi0, bf0, E, F, D=D, Cm=Cm, ntok=ntok, flags=tacg.TACG_ZERO_FIRST | path_flag)
    primary_np, swaps = placement.local_search(ctx, D, Cm, ntok, P, cfg.capacity)
    primary = torch.from_numpy(primary_np).to(dev)
    # GESR offline step on the device (Eq. 11 with the canonical lambda1 = lambda2 = 0, Eq. 12)
    replicas = tacg.gesr_build_replicas(ctx, D, Cm, ntok, P, cfg.capacity, primary, cfg.n_rep, cfg.r)[0] if cfg.r else None
    replicas_np = None if replicas is None else replicas.cpu().numpy()
    r = cfg.r if replicas is not None else 0

    def step(bi, bf, ei, ef):
        ctx.check(ctx.tacg_coact_accumulate(bi, bf, cfg.N, k, L, E, F, D, Cm, ntok, tacg.TACG_ZERO_FIRST | path_flag),
                  "tacg_coact_accumulate")
        ctx.check(ctx.tacg_affinity_swapgain(D, Cm, ntok, L, E, F, P, cfg.capacity, primary, 0.25, 1.0, 1e-6,
                                             pref, W, aff, gain), "tacg_affinity_swapgain")
        ctx.check(ctx.tacg_eval_placement(ei, ef, cfg.N_eval, k, L, E, F, P, primary, replicas, r, 0.15, 0.995,
                                          cfg.microbatch, 0, None, load, span, remote, ntok_e, fair, None, None, 0),
                  "tacg_eval_placement")

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize(dev)

    def timed(fn, steps, warmup, profile=False):
        for i in range(warmup):
            fn(i)
        barrier()
        ctx.profile_enable(profile)
        for s in range(3):
            ctx.profile_read(s)
        l0 = ctx.launch_count()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for i in range(steps):
            fn(warmup + i)
        e1.record()
        barrier()
        ctx.profile_enable(False)
        ms = max_over_ranks(e0.elapsed_time(e1), dist, dev)
        return ms, ctx.launch_count() - l0

    # ---- device-resident throughput (the headline `value`), clocks sampled during it
    sampler = ClockSampler(torch.cuda._get_nvml_device_index(local_rank) if hasattr(torch.cuda, "_get_nvml_device_index") else local_rank)
    dev_fn = lambda i: step(*sets[i % n_sets])
    for i in range(args.warmup):
        dev_fn(i)
    sampler.start()
    ms_total, launches = timed(dev_fn, args.steps, 0)
    sampler.stop()
    clocks = sampler.summary()
    units_per_step = cfg.L * (cfg.N + cfg.N_eval)
    value = whole_job_value(units_per_step, args.steps, world, ms_total)

    # ---- roofline of the dominant kernel: same steps again with the library's event brackets on
    _, _ = timed(dev_fn, args.steps, 0, profile=True)
    co_ms, co_n = ctx.profile_read(tacg.TACG_PROF_COACT)
    af_ms, af_n = ctx.profile_read(tacg.TACG_PROF_AFFINITY)
    ev_ms, ev_n = ctx.profile_read(tacg.TACG_PROF_EVAL)
    peak, peak_src = measured_peaks()
    abytes = coact_algorithmic_bytes(cfg)
    co_avg_ms = co_ms / max(1, co_n)
    achieved = abytes / (co_avg_ms * 1e-3) / 1e9 if co_avg_ms > 0 else 0.0
    used_path = {tacg.TACG_PATH_HIST: "hist", tacg.TACG_PATH_MMA: "mma"}.get(ctx.last_path(), "?")
    roofline = {
        "bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
        "traffic": ncu_traffic(args.config, used_path), "kernel": f"coact_{used_path}_kernel", "peak_source": peak_src,
        "algorithmic_bytes_per_launch": abytes, "avg_launch_ms": co_avg_ms, "launches_timed": co_n,
        "coact_routed_tokens_per_s": cfg.L * cfg.N / (co_avg_ms * 1e-3) if co_avg_ms > 0 else 0.0,
        "other_kernels_avg_ms": {"affinity_fused_kernel": af_ms / max(1, af_n), "eval_kernel": ev_ms / max(1, ev_n)},
    }
    if used_path == "hist" and co_avg_ms > 0:
        # What actually bounds the histogram kernel: k(k-1)/2 shared-memory atomic increments per
        # token.  Peak from unit counts and the sampled clock: an ATOMS instruction whose 32 lanes hit 32 different
        # banks takes 2 LSU wavefronts, one wavefront per clock and SM -> 16 increments per clock and SM.
        sm_count = torch.cuda.get_device_properties(0).multi_processor_count
        incs = cfg.L * cfg.N * (k * (k - 1) // 2)
        apeak = 16.0 * sm_count * (clocks.get("sm_mhz") or 0) * 1e6
        roofline["atomic_pipe"] = {
            "achieved": incs / (co_avg_ms * 1e-3), "peak": apeak, "unit": "shared-memory increments/s",
            "frac": (incs / (co_avg_ms * 1e-3)) / apeak if apeak else None,
            "peak_source": "16 conflict-free lane increments / clk / SM x SMs x sampled SM clock (DESIGN.md 5.1)",
        }

    # ---- optional: the co-activation call alone on both paths
    coact_paths = None
    if args.compare_paths:
        coact_paths = {}
        epad = 64 if E <= 64 else (128 if E <= 128 else 256)
        for name, flag in (("hist", tacg.TACG_PATH_HIST), ("mma", tacg.TACG_PATH_MMA)):
            def one(i, flag=flag):
                bi, bf, _, _ = sets[i % n_sets]
                ctx.check(ctx.tacg_coact_accumulate(bi, bf, cfg.N, k, L, E, F, D, Cm, ntok, tacg.TACG_ZERO_FIRST | flag),
                          "tacg_coact_accumulate")
            try:
                timed(one, max(3, min(args.steps, 20)), 3, profile=True)
            except Exception as exc:                         # shape not supported by the tensor path
                coact_paths[name] = {"unsupported": str(exc)}
                continue
            ms, n = ctx.profile_read(tacg.TACG_PROF_COACT)
            avg = ms / max(1, n)
            coact_paths[name] = {"avg_call_ms": avg, "routed_tokens_per_s": cfg.L * cfg.N / (avg * 1e-3),
                                 "hbm_frac": abytes / (avg * 1e-3) / 1e9 / peak}
        coact_paths["useful_over_dense"] = (k * (k - 1) / 2) / float(epad * epad)
        coact_paths["note"] = "tensor path: Epad^2 MACs per token in kind::i8 against k(k-1)/2 useful increments"

    # ---- end to end through host buffers: H2D of both traces, the calls, D2H of the results
    e2e = None
    if not args.no_e2e:
        n_host = min(n_sets, 2)
        host_sets = [tuple(x.cpu().pin_memory() for x in sets[s]) for s in range(n_host)]
        stage = tuple(torch.empty_like(x) for x in sets[0])
        host_out = [torch.empty_like(t, device="cpu").pin_memory() for t in (gain, aff, load, span, remote, fair)]
        h2d = sum(x.numel() * x.element_size() for x in host_sets[0])
        d2h = sum(x.numel() * x.element_size() for x in host_out)

        def e2e_fn(i):
            hs = host_sets[i % n_host]
            for dst, src in zip(stage, hs):
                dst.copy_(src, non_blocking=True)
            step(*stage)
            for dst, src in zip(host_out, (gain, aff, load, span, remote, fair)):
                dst.copy_(src, non_blocking=True)
            torch.cuda.current_stream(dev).synchronize()      # the caller reads the result every step

        e2e_steps = max(3, min(args.steps, 50))
        ms_e2e, _ = timed(e2e_fn, e2e_steps, 3)
        e2e = {"value": world * units_per_step * e2e_steps / (ms_e2e * 1e-3), "unit": UNIT,
               "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "steps": e2e_steps,
               "ms_per_step": ms_e2e / e2e_steps}
        del host_sets, stage

    # ---- the oracle timed beside it (rank 0, N=1 only)
    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        from oracle import cbind                    # cpu_baseline leg: the oracle as it stands
        bi, bf, ei, ef = (x.cpu().numpy() for x in sets[0])
        Ls, threads = oracle_sample_layers(cbind, cfg, bi, bf, ei, ef, primary_np, replicas_np, 10.0)
        t0 = time.perf_counter()
        units, reps = 0, 0
        while reps == 0 or time.perf_counter() - t0 < 10.0:        # about 10 s of CPU work
            units += oracle_step(cbind, cfg, bi, bf, ei, ef, primary_np, replicas_np, Ls)
            reps += 1
        dt = time.perf_counter() - t0
        cpu_baseline = {"value": units / dt, "unit": UNIT, "cores": threads, "kind": "oracle",
                        "sample": f"{reps} step(s) on the first {Ls} of {cfg.L} layers, all tokens ({dt:.1f} s)"}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_total / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "u32", "data": "synthetic",
            "config": workload_config(cfg, n_sets, l2_note), "clocks": clocks, "e2e": e2e,
            "gpu_launches": launches, "roofline": roofline, "cpu_baseline": cpu_baseline,
            "coact_path": used_path, "local_search_swaps_mean": float(np.mean(swaps)),
        }
        if coact_paths is not None:
            line["coact_paths"] = coact_paths
        print(json.dumps(line), flush=True)
    ctx.close()
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

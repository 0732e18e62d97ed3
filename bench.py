#!/usr/bin/env python
"""bench.py -- one line of JSON for the TACG/GESR hot path on B200 ("Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--impl tacg|reference]

The headline workload is BASELINE.json configs[3] (config 4), the largest single-GPU configuration; the
other throughput configurations (2, 3, 5) are timed device-resident in the same run and reported in the
`per_config` sub-record of the same line.

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
    """Picks how many layers one oracle step covers so that it takes about budget_s.  Returns (layers, cores):
    the oracle runs one OpenMP thread per layer, so it uses min(layers, threads) cores."""
    threads = cbind.threads()
    Lmax = bi.shape[0]
    L0 = min(Lmax, threads)
    t0 = time.perf_counter()
    oracle_step(cbind, cfg, bi, bf, ei, ef, primary, replicas, L0)
    dt = max(1e-3, time.perf_counter() - t0)
    rounds = max(1, int(budget_s / dt))
    Ls = max(1, min(Lmax, L0 * rounds))
    return Ls, min(Ls, threads)


def cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.lower().startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def oracle_sample_config(cfg, cbind):
    """The slice of the workload the oracle legs run on: the first layers of the configuration (at most one per
    OpenMP thread and at most 16: layers are independent problems), all tokens of each."""
    return tracegen.scaled(cfg, L=min(cfg.L, max(1, min(16, cbind.threads()))))


def run_reference(args, cfg, rank):
    """--impl reference: the oracle, as it stands, on the host cores (rank 0 only)."""
    if rank != 0:
        return
    from oracle import cbind                      # the one other place bench.py executes oracle/
    device = "cuda" if torch.cuda.is_available() else "cpu"
    scfg = oracle_sample_config(cfg, cbind)       # only the sampled layers are generated
    (bi, bf, ei, ef), = make_sets(scfg, 1, 0, device)
    bi, bf, ei, ef = (x.cpu().numpy() for x in (bi, bf, ei, ef))
    primary = tracegen.random_placement(cfg.E, cfg.P, cfg.capacity, scfg.L, seed=cfg.seed)
    replicas = tracegen.random_replicas(primary, cfg.P, cfg.r, cfg.n_rep, seed=cfg.seed + 1) if cfg.r else None
    per_step_budget = max(0.2, min(3.0, 120.0 / max(1, args.steps + args.warmup)))
    Ls, cores = oracle_sample_layers(cbind, cfg, bi, bf, ei, ef, primary, replicas, per_step_budget)
    for _ in range(args.warmup):
        oracle_step(cbind, cfg, bi, bf, ei, ef, primary, replicas, Ls)
    t0 = time.perf_counter()
    units = 0
    for _ in range(args.steps):
        units += oracle_step(cbind, cfg, bi, bf, ei, ef, primary, replicas, Ls)
    dt = time.perf_counter() - t0
    value = units / dt
    sample = f"{Ls} layers of the configuration's shape (it has {cfg.L}), all {cfg.N}+{cfg.N_eval} tokens per layer, per step"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / max(1, args.steps),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u32", "data": "synthetic",
        "config": workload_config(cfg), "inputs": {"trace_sets": 1, "l2": "n/a (CPU oracle)"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                         "cpu_model": cpu_model(), "omp_threads": cbind.threads()},
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


def workload_config(cfg, n_sets=None, l2_note=None):
    """`config` of the JSON line: the same dict on both arms (the driver compares them); what differs between the
    arms (how many trace sets rotate, the L2 note) goes into the line's `inputs` key."""
    return {
        "workload": f"BASELINE.json configs[{[k for k, v in tracegen.CONFIGS.items() if v.name == cfg.name][0] - 1}] "
                    f"{cfg.name}: E={cfg.E} k={cfg.k} L={cfg.L} F={cfg.F} N={cfg.N} (build) + {cfg.N_eval} (eval) "
                    f"tokens/layer, P={cfg.P} cap={cfg.capacity}, r={cfg.r}",
        "step": "tacg_coact_accumulate + tacg_affinity_swapgain + tacg_eval_placement",
        "unit_definition": "routed tokens = token x layer records consumed per step (build + eval trace)",
        "parallelism": "replicas only (no data-path collective)",
    }


# ------------------------------------------------------------------ the CUDA path
class Workload:
    """Device buffers, placement inputs and the step function of one configuration."""

    def __init__(self, tacg, placement, ctx, cfg, rank, dev, n_sets, path_flag):
        self.tacg, self.ctx, self.cfg, self.dev, self.path_flag = tacg, ctx, cfg, dev, path_flag
        L, E, F, P = cfg.L, cfg.E, cfg.F, cfg.P
        self.step_in_bytes = cfg.L * (cfg.N + cfg.N_eval) * cfg.k * 2 + cfg.N + cfg.N_eval
        if not n_sets:
            n_sets = max(2, int(np.ceil(3 * 126e6 / self.step_in_bytes)) + 1)
        free_b = torch.cuda.mem_get_info(dev)[0]
        self.n_sets = max(1, min(n_sets, int(0.4 * free_b / self.step_in_bytes)))
        self.sets = make_sets(cfg, self.n_sets, rank, dev)
        tot = self.n_sets * self.step_in_bytes
        self.l2_note = (f"inputs rotate over {self.n_sets} distinct trace sets = {tot / 1e6:.0f} MB (L2 is 126 MB)"
                        if self.step_in_bytes <= 2 * 126e6 else
                        f"one step reads {self.step_in_bytes / 1e6:.0f} MB of inputs, larger than the 126 MB L2 "
                        f"({self.n_sets} trace sets rotate)")
        i32, i64, f32 = torch.int32, torch.int64, torch.float32
        self.D = torch.empty((L, F, E), dtype=i32, device=dev)
        self.Cm = torch.empty((L, F, E, E), dtype=i32, device=dev)
        self.ntok = torch.empty((F,), dtype=i64, device=dev)
        self.pref = torch.empty((L, E, F), dtype=f32, device=dev)
        self.W = torch.empty((L, E, E), dtype=f32, device=dev)
        self.aff = torch.empty((L, E, P), dtype=f32, device=dev)
        self.gain = torch.empty((L, E, E), dtype=f32, device=dev)
        self.load = torch.empty((L, P), dtype=i64, device=dev)
        self.span = torch.empty((L, F), dtype=i64, device=dev)
        self.remote = torch.empty((L, F), dtype=i64, device=dev)
        self.ntok_e = torch.empty((F,), dtype=i64, device=dev)
        self.fair = torch.empty((L + 1, 3), dtype=f32, device=dev)
        # placement used by the step: local search on the first build trace, GESR table per config
        bi0, bf0, _, _ = self.sets[0]
        tacg.tacg_coact_accumulate(ctx, bi0, bf0, E, F, D=self.D, Cm=self.Cm, ntok=self.ntok,
                                   flags=tacg.TACG_ZERO_FIRST | path_flag)
        self.primary_np, self.swaps = placement.local_search(ctx, self.D, self.Cm, self.ntok, P, cfg.capacity)
        self.primary = torch.from_numpy(self.primary_np).to(dev)
        # GESR offline step on the device (Eq. 11 with the canonical lambda1 = lambda2 = 0, Eq. 12)
        self.replicas = tacg.gesr_build_replicas(ctx, self.D, self.Cm, self.ntok, P, cfg.capacity, self.primary,
                                                 cfg.n_rep, cfg.r)[0] if cfg.r else None
        self.replicas_np = None if self.replicas is None else self.replicas.cpu().numpy()
        self.r = cfg.r if self.replicas is not None else 0
        self.units_per_step = cfg.L * (cfg.N + cfg.N_eval)

    def coact(self, bi, bf, flag=None):
        c, t = self.cfg, self.tacg
        self.ctx.check(self.ctx.tacg_coact_accumulate(bi, bf, c.N, c.k, c.L, c.E, c.F, self.D, self.Cm, self.ntok,
                                                      t.TACG_ZERO_FIRST | (self.path_flag if flag is None else flag)),
                       "tacg_coact_accumulate")

    def affinity(self):
        c = self.cfg
        self.ctx.check(self.ctx.tacg_affinity_swapgain(self.D, self.Cm, self.ntok, c.L, c.E, c.F, c.P, c.capacity,
                                                       self.primary, 0.25, 1.0, 1e-6, self.pref, self.W, self.aff,
                                                       self.gain), "tacg_affinity_swapgain")

    def evaluate(self, ei, ef):
        c = self.cfg
        self.ctx.check(self.ctx.tacg_eval_placement(ei, ef, c.N_eval, c.k, c.L, c.E, c.F, c.P, self.primary,
                                                    self.replicas, self.r, 0.15, 0.995, c.microbatch, 0, None,
                                                    self.load, self.span, self.remote, self.ntok_e, self.fair,
                                                    None, None, 0), "tacg_eval_placement")

    def step(self, bi, bf, ei, ef):
        self.coact(bi, bf)
        self.affinity()
        self.evaluate(ei, ef)

    def results(self):
        return (self.gain, self.aff, self.load, self.span, self.remote, self.fair)


def coact_roofline(tacg, ctx, cfg, co_ms, co_n, peak):
    abytes = coact_algorithmic_bytes(cfg)
    avg = co_ms / max(1, co_n)
    achieved = abytes / (avg * 1e-3) / 1e9 if avg > 0 else 0.0
    used = {tacg.TACG_PATH_HIST: "hist", tacg.TACG_PATH_MMA: "mma"}.get(ctx.last_path(), "?")
    return abytes, avg, achieved, achieved / peak, used


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", type=int, default=4,
                    help="BASELINE.json config number, 1-based (default 4 = configs[3], the largest single-GPU one)")
    ap.add_argument("--impl", default="tacg", choices=["tacg", "reference"])
    ap.add_argument("--sets", type=int, default=0, help="distinct trace sets rotated over (0 = enough to exceed L2)")
    ap.add_argument("--path", default="auto", choices=["auto", "hist", "mma"])
    ap.add_argument("--compare-paths", action="store_true",
                    help="also time tacg_coact_accumulate alone on both paths (histogram, tcgen05 kind::i8)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-per-config", action="store_true", help="skip the device-resident timing of the other configs")
    ap.add_argument("--no-peaks", action="store_true", help="skip the shared-atomic / int8 tensor micro-benchmarks")
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
    peak, peak_src = measured_peaks()

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

    # ---- measured denominators of the units the co-activation kernels saturate
    peaks = None
    if not args.no_peaks:
        peaks = {}
        for name, which in (("atoms_spread", tacg.TACG_PEAK_ATOMS_SPREAD), ("atoms_random", tacg.TACG_PEAK_ATOMS_RANDOM),
                            ("i8_tensor", tacg.TACG_PEAK_I8_TENSOR)):
            per_s, per_clk = ctx.measure_peak(which)
            peaks[name] = {"per_second": per_s, "per_clk_sm": per_clk}
        peaks["units"] = {"atoms_*": "shared-memory increments", "i8_tensor": "int8 operations (2 per multiply-add)"}
        peaks["source"] = "tacg_measure_peak (csrc/peaks.cu), this run, one CTA per SM"

    wl = Workload(tacg, placement, ctx, cfg, rank, dev, args.sets, path_flag)
    n_sets, sets, k = wl.n_sets, wl.sets, cfg.k
    head_note = wl.l2_note

    # ---- device-resident throughput (the headline `value`), clocks sampled during it
    sampler = ClockSampler(torch.cuda._get_nvml_device_index(local_rank) if hasattr(torch.cuda, "_get_nvml_device_index") else local_rank)
    dev_fn = lambda i: wl.step(*sets[i % n_sets])
    for i in range(args.warmup):
        dev_fn(i)
    sampler.start()
    ms_total, launches = timed(dev_fn, args.steps, 0)
    sampler.stop()
    clocks = sampler.summary()
    value = whole_job_value(wl.units_per_step, args.steps, world, ms_total)

    # ---- roofline of the dominant kernel: same steps again with the library's event brackets on
    _, _ = timed(dev_fn, args.steps, 0, profile=True)
    co_ms, co_n = ctx.profile_read(tacg.TACG_PROF_COACT)
    af_ms, af_n = ctx.profile_read(tacg.TACG_PROF_AFFINITY)
    ev_ms, ev_n = ctx.profile_read(tacg.TACG_PROF_EVAL)
    abytes, co_avg_ms, achieved, frac, used_path = coact_roofline(tacg, ctx, cfg, co_ms, co_n, peak)
    kernel_names = {"hist": "coact_hist_kernel+coact_finalize_kernel" + ("+part_count/scan/scatter_kernel" if cfg.E > 160 else ""),
                    "mma": "coact_mma_kernel+coact_mma_finalize_kernel"}
    roofline = {
        "bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": frac,
        "traffic": ncu_traffic(args.config, used_path), "kernel": kernel_names.get(used_path, used_path),
        "peak_source": peak_src, "algorithmic_bytes_per_launch": abytes, "avg_launch_ms": co_avg_ms,
        "launches_timed": co_n,
        "coact_routed_tokens_per_s": cfg.L * cfg.N / (co_avg_ms * 1e-3) if co_avg_ms > 0 else 0.0,
        "other_kernels_avg_ms": {"affinity_fused_kernel": af_ms / max(1, af_n),
                                 "eval_scan_kernel+eval_chain_kernel": ev_ms / max(1, ev_n)},
    }
    if used_path == "hist" and co_avg_ms > 0 and peaks:
        # what bounds a histogram: k(k-1)/2 shared-memory atomic increments per token against the MEASURED rate of
        # increments on random words (tacg_measure_peak); the token-set table makes the kernel do fewer
        incs = cfg.L * cfg.N * (k * (k - 1) // 2)
        roofline["atomic_pipe"] = {
            "achieved": incs / (co_avg_ms * 1e-3), "peak": peaks["atoms_random"]["per_second"],
            "unit": "pair increments/s (algorithmic: k(k-1)/2 per token)",
            "frac": incs / (co_avg_ms * 1e-3) / peaks["atoms_random"]["per_second"],
            "peak_conflict_free": peaks["atoms_spread"]["per_second"],
            "peak_source": "measured: tacg_measure_peak TACG_PEAK_ATOMS_RANDOM / _SPREAD",
        }

    # ---- the co-activation call alone: both paths, and a trace without repeated expert sets
    coact_paths = None
    if args.compare_paths:
        coact_paths = {}
        epad = 64 if cfg.E <= 64 else (128 if cfg.E <= 128 else 256)
        for name, flag in (("hist", tacg.TACG_PATH_HIST), ("mma", tacg.TACG_PATH_MMA)):
            one = lambda i, flag=flag: wl.coact(sets[i % n_sets][0], sets[i % n_sets][1], flag)
            try:
                timed(one, max(3, min(args.steps, 20)), 3, profile=True)
            except Exception as exc:                         # shape not supported by the tensor path
                coact_paths[name] = {"unsupported": str(exc)}
                continue
            ms, n = ctx.profile_read(tacg.TACG_PROF_COACT)
            avg = ms / max(1, n)
            coact_paths[name] = {"avg_call_ms": avg, "routed_tokens_per_s": cfg.L * cfg.N / (avg * 1e-3),
                                 "hbm_frac": abytes / (avg * 1e-3) / 1e9 / peak}
            if name == "mma" and peaks:
                # dense work issued by the tensor path against the measured int8 peak
                dense = 2.0 * epad * epad * cfg.L * cfg.N / (avg * 1e-3)
                coact_paths[name]["int8_util"] = dense / peaks["i8_tensor"]["per_second"]
        coact_paths["useful_over_dense"] = (k * (k - 1) / 2) / float(epad * epad)
        coact_paths["note"] = "tensor path: Epad^2 MACs per token in kind::i8 against k(k-1)/2 useful increments"
        # the token-set table pays only when expert sets repeat (planted groups of exactly k members): same shape
        # with p_group = 0, i.e. every token draws k experts from the popularity, no repeats to exploit
        from dataclasses import replace as _replace
        cfg0 = _replace(cfg, p_group=0.0)
        p0 = tracegen.make_params(cfg0)
        bi0, bf0 = tracegen.gen_trace(cfg0, p0, eval_trace=False, device=dev, seed=cfg.seed + 7)
        timed(lambda i: wl.coact(bi0, bf0, tacg.TACG_PATH_HIST), max(3, min(args.steps, 20)), 3, profile=True)
        ms, n = ctx.profile_read(tacg.TACG_PROF_COACT)
        coact_paths["hist_no_repeated_sets"] = {"avg_call_ms": ms / max(1, n),
                                                "hbm_frac": abytes / (ms / max(1, n) * 1e-3) / 1e9 / peak,
                                                "trace": "p_group = 0 (no planted groups)"}
        del bi0, bf0

    # ---- end to end through host buffers: H2D of both traces, the calls, D2H of the results.  The build trace
    # is copied layer chunk by layer chunk on a second stream and counted as the chunks arrive (the counts of
    # different layers are independent), the evaluation trace follows on the copy stream meanwhile.
    e2e = None
    if not args.no_e2e:
        n_host = 1 if wl.step_in_bytes > 2e9 else min(n_sets, 2)
        host_sets = [tuple(x.cpu().pin_memory() for x in sets[s]) for s in range(n_host)]
        stage = tuple(torch.empty_like(x) for x in sets[0])
        host_out = [torch.empty_like(t, device="cpu").pin_memory() for t in wl.results()]
        h2d = sum(x.numel() * x.element_size() for x in host_sets[0])
        d2h = sum(x.numel() * x.element_size() for x in host_out)
        copy_stream = torch.cuda.Stream(dev)
        main_stream = torch.cuda.current_stream(dev)
        nchunk = max(1, min(cfg.L, 8))
        bounds = [cfg.L * c // nchunk for c in range(nchunk + 1)]
        ntok_tmp = torch.empty_like(wl.ntok)

        def e2e_fn(i):
            hb, hf, he, hef = host_sets[i % n_host]
            sb, sf, se, sef = stage
            copy_stream.wait_stream(main_stream)            # the previous step has finished with the staging buffers
            events = []
            with torch.cuda.stream(copy_stream):
                sf.copy_(hf, non_blocking=True)
                for c in range(nchunk):
                    sb[bounds[c]:bounds[c + 1]].copy_(hb[bounds[c]:bounds[c + 1]], non_blocking=True)
                    ev = torch.cuda.Event()
                    ev.record(copy_stream)
                    events.append(ev)
                sef.copy_(hef, non_blocking=True)
                se.copy_(he, non_blocking=True)
                ev_eval = torch.cuda.Event()
                ev_eval.record(copy_stream)
            for c in range(nchunk):
                a, b = bounds[c], bounds[c + 1]
                main_stream.wait_event(events[c])
                ctx.check(ctx.tacg_coact_accumulate(sb[a:b], sf, cfg.N, k, b - a, cfg.E, cfg.F, wl.D[a:b], wl.Cm[a:b],
                                                    wl.ntok if c == 0 else ntok_tmp, tacg.TACG_ZERO_FIRST | path_flag),
                          "tacg_coact_accumulate")
            wl.affinity()
            main_stream.wait_event(ev_eval)
            wl.evaluate(se, sef)
            for dst, src in zip(host_out, wl.results()):
                dst.copy_(src, non_blocking=True)
            main_stream.synchronize()                        # the caller reads the result every step

        e2e_steps = max(3, min(args.steps, 20 if wl.step_in_bytes > 2e9 else 50))
        ms_e2e, _ = timed(e2e_fn, e2e_steps, 3)
        e2e = {"value": world * wl.units_per_step * e2e_steps / (ms_e2e * 1e-3), "unit": UNIT,
               "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "steps": e2e_steps,
               "ms_per_step": ms_e2e / e2e_steps, "overlap": f"build trace in {nchunk} layer chunks on a copy stream"}
        del host_sets, stage

    # ---- the oracle timed beside it (rank 0, N=1 only): all host cores, then one thread
    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        from oracle import cbind                    # cpu_baseline leg: the oracle as it stands
        scfg = oracle_sample_config(cfg, cbind)
        Lh = scfg.L
        bi, bf, ei, ef = (x[:Lh].cpu().numpy() if x.dim() == 3 else x.cpu().numpy() for x in sets[0])
        pr_np = wl.primary_np[:Lh]
        rp_np = None if wl.replicas_np is None else wl.replicas_np[:Lh]
        Ls, cores = oracle_sample_layers(cbind, cfg, bi, bf, ei, ef, pr_np, rp_np, 8.0)
        t0 = time.perf_counter()
        units, reps = 0, 0
        while reps == 0 or time.perf_counter() - t0 < 8.0:         # about 8 s of CPU work
            units += oracle_step(cbind, cfg, bi, bf, ei, ef, pr_np, rp_np, Ls)
            reps += 1
        dt = time.perf_counter() - t0
        nthreads = cbind.threads()
        cbind.set_threads(1)                                       # single thread: one layer, about 4 s
        t1 = time.perf_counter()
        u1, r1 = 0, 0
        while r1 == 0 or time.perf_counter() - t1 < 4.0:
            u1 += oracle_step(cbind, cfg, bi, bf, ei, ef, pr_np, rp_np, 1)
            r1 += 1
        dt1 = time.perf_counter() - t1
        cbind.set_threads(nthreads)
        cpu_baseline = {"value": units / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
                        "sample": f"{reps} step(s) on the first {Ls} of {cfg.L} layers, all tokens ({dt:.1f} s)",
                        "single_thread_value": u1 / dt1,
                        "single_thread_sample": f"{r1} step(s) on the first layer, all tokens ({dt1:.1f} s)",
                        "cpu_model": cpu_model(), "omp_threads": nthreads}
        del bi, bf, ei, ef

    # ---- the other throughput configurations, device-resident (parity-tested, not the headline)
    per_config = None
    if not args.no_per_config and world == 1:
        results = {str(args.config): {"ms_per_step": ms_total / args.steps, "coact_ms": co_avg_ms,
                                      "affinity_ms": af_ms / max(1, af_n), "eval_ms": ev_ms / max(1, ev_n),
                                      "coact_hbm_frac": frac, "coact_path": used_path}}
        del wl, sets
        torch.cuda.empty_cache()
        for other in (2, 3, 5):
            if other == args.config:
                continue
            ocfg = tracegen.get_config(other)
            ow = Workload(tacg, placement, ctx, ocfg, rank, dev, 0, path_flag)
            fn = lambda i: ow.step(*ow.sets[i % ow.n_sets])
            steps_o = max(10, min(args.steps, 50))
            ms_o, _ = timed(fn, steps_o, 3)
            timed(fn, steps_o, 0, profile=True)
            c_ms, c_n = ctx.profile_read(tacg.TACG_PROF_COACT)
            a_ms, a_n = ctx.profile_read(tacg.TACG_PROF_AFFINITY)
            e_ms, e_n = ctx.profile_read(tacg.TACG_PROF_EVAL)
            _, c_avg, _, c_frac, c_path = coact_roofline(tacg, ctx, ocfg, c_ms, c_n, peak)
            results[str(other)] = {"ms_per_step": ms_o / steps_o, "coact_ms": c_avg, "affinity_ms": a_ms / max(1, a_n),
                                   "eval_ms": e_ms / max(1, e_n), "coact_hbm_frac": c_frac, "coact_path": c_path,
                                   "routed_tokens_per_s": ow.units_per_step * steps_o / (ms_o * 1e-3),
                                   "workload": workload_config(ocfg, ow.n_sets, ow.l2_note)["workload"]}
            del ow
            torch.cuda.empty_cache()
        per_config = results
    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_total / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "u32", "data": "synthetic",
            "config": workload_config(cfg), "inputs": {"trace_sets": n_sets, "l2": head_note}, "clocks": clocks, "e2e": e2e,
            "gpu_launches": launches, "roofline": roofline, "cpu_baseline": cpu_baseline,
            "coact_path": used_path, "measured_peaks": peaks, "per_config": per_config,
        }
        if coact_paths is not None:
            line["coact_paths"] = coact_paths
        print(json.dumps(line), flush=True)
    ctx.close()
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

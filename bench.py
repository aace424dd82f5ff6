#!/usr/bin/env python
"""bench.py -- throughput of the checkerboard Potts sweep on B200 (driver contract).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--workload cfgN] [--no-per-config] [--no-cpu-baseline]

A "step" is one pass of the whole hot path over one workload of BASELINE.json: create the
start state, then `sweeps` checkerboard Metropolis sweeps at the workload's temperature(s) with
the workload's measurement cadence (energy / histogram series recorded on the device).  The
default workload is BASELINE.json configs[1] (q=6, L=1024, ordered start, 1.005 T_c, 10^4
sweeps, energy every sweep).  `value` = spin-flip attempts per second (= 1e9 / ns-per-flip),
inputs resident in HBM; `e2e` = the same through the C-ABI with HOST buffers (upload of the
start configuration from pinned host memory, series + final configuration copied back).

N > 1 (torchrun): the paper averages over independent samples ("repeat over
samples"), so rank r runs sample r (seed + r) of the same workload: no data-path collective,
weak scaling; the time is the max over ranks.

Rank 0 prints ONE JSON line.  See DESIGN.md section 8 for every field.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

import workloads  # noqa: E402

# ---- roofline constants -------------------------------------------------
SM_COUNT = 148
ISSUE_LANES_PER_SM_CLK = 128          # 4 SMSPs x 1 warp-instruction (32 lanes) per clock
I_ALG_PER_UPDATE = 36                 # Philox4x32-10 words 0,1 of counter (j,i,t,colour): 17 IMAD.WIDE + 18 LOP3, + 1 IMAD.HI proposal
BYTES_ALG_PER_UPDATE_U8 = 3.0         # read own + read other (once) + write own, uint8 planes
# Measured on B200 (profiles/r01b_pipe_model.md): for this integer mix (IMAD.WIDE / LOP3 / IADD3 / SHF / PRMT) an SM
# sub-partition retires one warp instruction every 2 clocks, whichever pipe it goes to: half the nominal issue rate.
MEASURED_INT_ISSUE_PER_CLK = 0.5
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel from the
# `ncu --set full` capture summarised in profiles/ (None until a capture exists for the workload)
NCU_TRAFFIC_BYTES_PER_LAUNCH = {          # profiles/r01c_kernels.md
    "cfg2_q6_L1024": 1.113e6 + 5.1e3,      # resident kernel: the lattice is loaded once per launch, whatever the sweep count
    "cfg3_q9_L4096": 17.30e6 + 8.7e3,
    "cfg4_q24_L8192": 41.98e6 + 1.5e3,     # 40 MB of packed planes, L2-resident after the first touch
    "cfg5_q9_L32768": 1.0738e9 + 0.4973e9,
}


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), float(d.get("sm_max_mhz", 1965.0)), "measured"
    return 6650.0, 1965.0, "fallback"


# ---- clocks during the timed region -----------------------------------------------------------
class ClockSampler:
    """Samples SM clock and throttle reasons through NVML every 20 ms while running."""

    REASONS = {
        0x1: "gpu_idle", 0x2: "applications_clocks_setting", 0x4: "sw_power_cap", 0x8: "hw_slowdown",
        0x10: "sync_boost", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
        0x80: "hw_power_brake_slowdown", 0x100: "display_clock_setting",
    }

    def __init__(self, index: int):
        self.index, self.samples, self.mask, self.max_mhz = index, [], 0, None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nv = pynvml
            self._dev = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self._dev, pynvml.NVML_CLOCK_SM))
        except Exception:
            self._nv = None

    def _run(self):
        nv = self._nv
        while not self._stop.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self._dev, nv.NVML_CLOCK_SM)))
                self.mask |= int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self._dev))
            except Exception:
                pass
            self._stop.wait(0.02)

    def __enter__(self):
        if self._nv is not None:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()

    def summary(self):
        reasons = [n for b, n in self.REASONS.items() if self.mask & b and n != "gpu_idle"]
        return {"sm_mhz": statistics.median(self.samples) if self.samples else None,
                "sm_max_mhz": self.max_mhz, "samples": len(self.samples), "reasons": reasons}


# ---- one workload on one GPU ------------------------------------------------------------------
def slice_of(w: workloads.Workload, max_sweeps: int | None):
    """(temperatures, sweeps per temperature) of the whole workload or of a bounded slice of it."""
    if max_sweeps is None or max_sweeps >= w.total_sweeps:
        return list(w.temperatures), w.sweeps_per_t
    per_t = max(w.every, (max_sweeps // len(w.temperatures)) // w.every * w.every)
    return list(w.temperatures), per_t


class GpuRun:
    """Drives the product through the Python binding of the C-ABI (argument marshalling only)."""

    def __init__(self, pb, torch, w: workloads.Workload, seed: int, max_sweeps: int | None, options=None, stream_spec=1):
        self.pb, self.torch, self.w, self.seed = pb, torch, w, seed
        self.stream_spec = stream_spec
        self.temps, self.per_t = slice_of(w, max_sweeps)
        self.sweeps = self.per_t * len(self.temps)
        self.updates = self.sweeps * w.L * w.L
        self.ns = self.sweeps // w.every
        self.layout = pb.LAYOUT_PACKED if w.packed else pb.LAYOUT_U8
        bits = 8 if self.layout == pb.LAYOUT_U8 else (5 if w.q > 16 else 4)
        self.bytes_per_update = 3.0 * bits / 8.0       # read own + read other (once) + write own
        self.options = dict(options or {})
        dev = torch.device("cuda", torch.cuda.current_device())
        self.E_dev = torch.zeros(max(self.ns, 1), dtype=torch.int64, device=dev)
        self.H_dev = torch.zeros((max(self.ns, 1), w.q), dtype=torch.int64, device=dev) if w.hist else None
        self.g = None

    def fresh(self):
        """New handle in the workload's start state, t = 0 (untimed)."""
        if self.g is not None:
            self.g.close()
        self.g = self.pb.Potts(self.w.L, self.w.q, self.seed, self.w.init, layout=self.layout)
        for k, v in self.options.items():
            self.g.potts_set_option(k, v)
        if self.stream_spec != 1:
            self.g.potts_set_stream_spec(self.stream_spec)
        self.resident_ctas = self.g.potts_get_option("resident_active")     # 0: not the resident kernel
        self.cluster_ctas = self.g.potts_get_option("cluster_active")       # 0: not the cluster kernel
        return self.g

    @property
    def kernel(self):
        if self.layout != self.pb.LAYOUT_U8:
            return "k_half_sweep_packed"
        if self.cluster_ctas:
            return "k_cluster_u8"
        return "k_resident_u8" if self.resident_ctas else "k_half_sweep_u8"

    @property
    def kernel_launches_per_step(self):
        return len(self.temps) if (self.resident_ctas or self.cluster_ctas) else 2 * self.sweeps

    def enqueue(self):
        """The step: all sweeps with the device-resident series; returns without a sync."""
        per_s = self.per_t // self.w.every
        for n, T in enumerate(self.temps):
            E = self.E_dev[n * per_s:(n + 1) * per_s]
            H = self.H_dev[n * per_s:(n + 1) * per_s] if self.H_dev is not None else None
            self.g.potts_sweep_measured_dev(T, self.per_t, self.w.every, E, H)

    # -- end to end through host buffers ----------------------------------------------------
    def e2e_prepare(self):
        torch, w = self.torch, self.w
        g = self.fresh()
        self.h_start = torch.empty((w.L, w.L), dtype=torch.uint8, pin_memory=True)
        g.potts_download(self.h_start.numpy())
        self.h_final = torch.empty((w.L, w.L), dtype=torch.uint8, pin_memory=True)
        self.h2d = w.L * w.L
        self.d2h = w.L * w.L + self.ns * 8 * (1 + (w.q if w.hist else 0))

    def e2e_step(self):
        g, w = self.g, self.w
        g.potts_upload(self.h_start.numpy())
        g.potts_set_sweep_count(0)
        last = None
        for T in self.temps:
            last = g.potts_sweep_measured(T, self.per_t, w.every, hist=w.hist)
        g.potts_download(self.h_final.numpy())
        return last


def time_steps(torch, run: GpuRun, steps: int, warmup: int, flush, e2e: bool = False):
    """-> (list of per-step ms, kernels launched in the timed steps)."""
    if e2e:
        run.e2e_prepare()
    ms, launches = [], 0
    for it in range(warmup + steps):
        if not e2e:
            run.fresh()
        flush()
        torch.cuda.synchronize()
        n0 = run.g.potts_launch_count()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        if e2e:
            run.e2e_step()
        else:
            run.enqueue()
        e1.record()
        torch.cuda.synchronize()
        if it >= warmup:
            ms.append(e0.elapsed_time(e1))
            launches += run.g.potts_launch_count() - n0
    return ms, launches


def make_flusher(torch):
    buf = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")   # 2x the 126 MB L2

    def flush():
        buf.fill_(1)
    return flush


# ---- the oracle timed on the host cores (cpu_baseline and --impl reference) --------------------
def host_threads() -> int:
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


def oracle_time(w: workloads.Workload, sweeps: int, threads: int):
    """Seconds the oracle, as it stands, needs for `sweeps` sweeps of workload w (with its cadence)."""
    import oracle
    o = oracle.OraclePotts(w.L, w.q, w.seed, w.init, threads=threads)
    sweeps = max(w.every, sweeps // w.every * w.every)
    t0 = time.perf_counter()
    o.sweep_measured(w.temperatures[0], sweeps, w.every, hist=w.hist)
    dt = time.perf_counter() - t0
    used = o.threads
    o.close()
    return dt, sweeps, used


def cpu_baseline(w: workloads.Workload, budget_s: float = 12.0):
    """The oracle on a bounded sample of the workload: all host threads (row-parallel mode, same
    bits) and one thread.  Returns the cpu_baseline object of the JSON line."""
    threads = host_threads()
    dt, n, _ = oracle_time(w, w.every, threads)                      # calibration (and page-in)
    per_sweep = max(dt / n, 1e-6)
    sweeps = int(min(w.total_sweeps, max(w.every, budget_s / per_sweep)))
    dt, n, used = oracle_time(w, sweeps, threads)
    multi = n * w.L * w.L / dt
    n1 = max(w.every, int(n / max(threads, 1) / 2))
    dt1, n1, _ = oracle_time(w, n1, 1)
    single = n1 * w.L * w.L / dt1
    return {"value": multi, "unit": "spin updates/s", "cores": used, "kind": "oracle",
            "sample": f"{n} sweeps of {w.name} (L={w.L}, q={w.q}) with its measurement cadence, {dt:.1f} s",
            "ns_per_spin_flip": 1e9 / multi,
            "single_thread": {"value": single, "ns_per_spin_flip": 1e9 / single,
                              "sample": f"{n1} sweeps, {dt1:.1f} s"}}


def run_reference(args, w):
    """--impl reference: the oracle on the host cores, same metric / config; rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    threads = host_threads()
    dt, n, _ = oracle_time(w, w.every, threads)
    per_sweep = max(dt / n, 1e-6)
    total = args.steps + args.warmup
    sweeps = int(min(w.total_sweeps, max(w.every, (90.0 / total) / per_sweep)))   # whole run ~1.5 min
    times = []
    for it in range(total):
        dt, n, used = oracle_time(w, sweeps, threads)
        if it >= args.warmup:
            times.append(dt)
    sec = sum(times) / len(times)
    val = n * w.L * w.L / sec
    sample = f"each step = {n} sweeps of {w.name} by the oracle (OpenMP rows, {used} threads)"
    line = {
        "impl": "reference", "metric": "spin_updates_per_s", "value": val, "unit": "spin updates/s",
        "ns_per_spin_flip": 1e9 / val, "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "u8", "data": "synthetic", "gpu_launches": 0,
        "config": {"workload": w.name, "q": w.q, "L": w.L, "init": "random" if w.init else "ordered",
                   "T_over_Tc": w.t_factors[0], "sweeps_per_step": n, "measure_every": w.every, "hist": w.hist},
        "cpu_baseline": {"value": val, "unit": "spin updates/s", "cores": used, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": "spin updates/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line), flush=True)


# ---- N > 1: independent samples, one per rank ------------------------------------------------------
def rank_seed(w: workloads.Workload, rank: int) -> int:
    """Rank r simulates sample r of the workload ("repeat over samples"): same parameters, seed + r."""
    return w.seed + rank


def reduce_over_ranks(dist, device, timed_ms: float, updates: int, launches: int):
    """-> (max over ranks of the timed milliseconds, total updates, total launches).  `dist` is
    torch.distributed (or None for one process); the path has no other collective (weak scaling)."""
    import torch
    t = torch.tensor([timed_ms], dtype=torch.float64, device=device)
    c = torch.tensor([updates, launches], dtype=torch.int64, device=device)
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(c, op=dist.ReduceOp.SUM)
    return float(t.item()), int(c[0].item()), int(c[1].item())


# ---- roofline -----------------------------------------------------------------------------------
def roofline(w, kernel: str, updates_per_launch: float, ms_per_launch: float, sm_mhz_max: float, hbm_gbs: float,
             which: str, bytes_per_update: float):
    """ALU/issue roofline of the dominant kernel: algorithmic thread-instructions (36 per
    update: the Philox block and the proposal multiply the stream definition fixes) x updates per launch over the
    average launch duration, against 148 SMs x 128 lanes/clk x max SM clock (one warp instruction per clock and
    sub-partition, the guide's issue model); the HBM view and the measured integer issue ceiling go beside it."""
    sec = ms_per_launch * 1e-3
    ach = I_ALG_PER_UPDATE * updates_per_launch / sec / 1e12
    peak = SM_COUNT * ISSUE_LANES_PER_SM_CLK * sm_mhz_max * 1e6 / 1e12
    gbs = bytes_per_update * updates_per_launch / sec / 1e9
    return {"bound": "alu", "kernel": kernel, "achieved": ach, "peak": peak, "unit": "Tinstr/s (thread-level)",
            "frac": ach / peak, "peak_source": f"148 SMs x 128 lanes/clk x {sm_mhz_max:.0f} MHz ({which} max SM clock)",
            "instr_per_update_algorithmic": I_ALG_PER_UPDATE, "ms_per_launch": ms_per_launch,
            "updates_per_launch": updates_per_launch,
            "frac_of_measured_int_issue": ach / (peak * MEASURED_INT_ISSUE_PER_CLK),
            "traffic": NCU_TRAFFIC_BYTES_PER_LAUNCH.get(w.name),
            "hbm": {"achieved": gbs, "peak": hbm_gbs, "unit": "GB/s", "frac": gbs / hbm_gbs,
                    "bytes_per_update_algorithmic": bytes_per_update, "peak_source": f"{which} copy bandwidth"}}


PER_CONFIG_SLICE = {1: None, 2: 2000, 3: 1600, 4: 200, 5: 100}       # sweeps timed per step (None = all)


def per_config_table(pb, torch, flush, sm_max, hbm_gbs, which, skip=(), stream_spec=1):
    out = {}
    for k, w in workloads.CONFIGS.items():
        if k in skip:
            continue
        run = GpuRun(pb, torch, w, w.seed, PER_CONFIG_SLICE[k], stream_spec=stream_spec)
        ms, launches = time_steps(torch, run, steps=3, warmup=1, flush=flush)
        sec = statistics.median(ms) * 1e-3
        ups = run.updates / sec
        nl = run.kernel_launches_per_step
        r = roofline(w, run.kernel, run.updates / nl, sec * 1e3 / nl, sm_max, hbm_gbs, which, run.bytes_per_update)
        out[w.name] = {"q": w.q, "L": w.L, "sweeps_timed": run.sweeps, "of_sweeps": w.total_sweeps,
                       "ns_per_spin_flip": 1e9 / ups, "spin_updates_per_s": ups, "ms": sec * 1e3,
                       "launches": launches // 3, "kernel": run.kernel, "resident_ctas": run.resident_ctas, "cluster_ctas": run.cluster_ctas,
                       "alu_frac": r["frac"], "alu_frac_of_measured_int_issue": r["frac_of_measured_int_issue"],
                       "hbm_frac": r["hbm"]["frac"],
                       "layout": "packed" if run.layout == pb.LAYOUT_PACKED else "u8"}
        run.g.close()
        del run
        torch.cuda.empty_cache()
    return out


def paper_protocol_e6(pb, torch):
    """The paper's end-to-end example: q=9, L=1024, 3 samples, T = 0.71 .. 0.73 in steps of 0.002,
    t_tran = 2000, t_max = 8000, one measure every 50 sweeps; 193 s on a GTX 280, 8115 s on its CPU.  Here: the same
    protocol through potts_ladder (heating from the ordered state), wall time including the series copy-back."""
    Ts = [0.71 + 0.002 * k for k in range(11)]
    t0 = time.perf_counter()
    e_last = None
    for sample in range(3):
        g = pb.Potts(1024, 9, 100 + sample, pb.INIT_ORDERED)
        E, H = g.potts_ladder(Ts, 2000, 8000, 50, hist=True)
        e_last = float(E[-1].mean()) / (1024 * 1024)
        g.close()
    torch.cuda.synchronize()
    sec = time.perf_counter() - t0
    sweeps = 3 * 11 * 10000
    return {"seconds": sec, "sweeps": sweeps, "spin_updates_per_s": sweeps * 1024 * 1024 / sec,
            "mean_e_per_spin_at_T0.73_last_sample": e_last,
            "paper_seconds_gtx280": 193.0, "paper_seconds_cpu": 8115.0, "note": "context only: other hardware and RNG"}


def batch_of_cfg1(pb, torch, n=1184):
    """n independent samples of BASELINE configs[0] (q=9, L=64, 1000 sweeps, E + histogram every sweep)
    advanced together by potts_batch_sweep_measured (one lattice per CTA, 8 per SM); wall time of the call, which
    includes the copy of the series to the host.  Sample 0 is configs[0] itself (seed 1)."""
    w = workloads.CONFIGS[1]
    b = pb.PottsBatch(w.L, w.q, [w.seed + r for r in range(n)], w.init)
    b.potts_batch_sweep_measured(w.temperatures[0], w.every, w.every)             # warm-up launch
    b.close()
    b = pb.PottsBatch(w.L, w.q, [w.seed + r for r in range(n)], w.init)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    E, H = b.potts_batch_sweep_measured(w.temperatures[0], w.sweeps_per_t, w.every)
    sec = time.perf_counter() - t0
    b.close()
    ups = n * w.updates / sec
    return {"lattices": n, "q": w.q, "L": w.L, "sweeps": w.sweeps_per_t, "seconds": sec, "spin_updates_per_s": ups,
            "ns_per_spin_flip": 1e9 / ups, "kernel": "k_resident_batch_u8", "E_last_of_sample_0": int(E[0, -1])}


def delta_stream_cost(pb, torch, sweeps=20):
    """SURVEY 8(f)4 / PAPER.md:361-363: cost of accumulating the energy change of every sweep on the fly
    (potts_sweep_delta, k_half_sweep_delta_u8) against the plain streaming half-sweep (variant 1, no measurement)
    on BASELINE configs[4]'s shape (q=9, L=32768).  CUDA events around the calls; the delta call includes the
    copy of its series to the host."""
    w = workloads.CONFIGS[5]
    T = w.temperatures[0]
    out = {"q": w.q, "L": w.L, "sweeps": sweeps}
    for name in ("plain", "delta"):
        g = pb.Potts(w.L, w.q, w.seed, w.init)
        g.potts_set_option("variant", 1)
        step = (lambda n: g.potts_sweep(T, n)) if name == "plain" else (lambda n: g.potts_sweep_delta(T, n))
        step(3)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        step(sweeps)
        e1.record()
        torch.cuda.synchronize()
        out[name + "_ns_per_spin_flip"] = e0.elapsed_time(e1) * 1e6 / (sweeps * w.L * w.L)
        g.close()
    out["delta_over_plain"] = out["delta_ns_per_spin_flip"] / out["plain_ns_per_spin_flip"]
    return out


# ---- main -----------------------------------------------------------------------------------------
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg2", help="cfg1..cfg5 (BASELINE.json configs[0..4])")
    ap.add_argument("--max-sweeps", type=int, default=None, help="time a bounded slice of the workload per step")
    ap.add_argument("--no-per-config", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--option", action="append", default=[], help="key=value passed to potts_set_option")
    args = ap.parse_args()
    w = workloads.CONFIGS[int(args.workload.replace("cfg", ""))]

    if args.impl == "reference":
        run_reference(args, w)
        return

    import torch
    import paper_1101_0876_b200 as pb
    pb.load_library()                                    # raises if the CUDA library is not built: no fallback
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback); use --impl reference for the oracle")

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    hbm_gbs, sm_max, which = _peaks()
    flush = make_flusher(torch)
    options = {kv.split("=")[0]: int(kv.split("=")[1]) for kv in args.option}

    # rank r runs sample r of the workload (independent lattice, seed + r): weak scaling, no collective
    run = GpuRun(pb, torch, w, rank_seed(w, rank), args.max_sweeps, options)

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    barrier()
    t_wall0 = time.perf_counter()
    with ClockSampler(local) as clk:
        ms, launches = time_steps(torch, run, args.steps, args.warmup, flush)
    barrier()
    wall = time.perf_counter() - t_wall0
    total_ms, updates_all, launches_all = reduce_over_ranks(dist, "cuda", sum(ms), run.updates * args.steps, launches)
    total_s = total_ms * 1e-3
    value = updates_all / total_s
    nl = run.kernel_launches_per_step
    roof = roofline(w, run.kernel, run.updates / nl, (sum(ms) / len(ms)) / nl, sm_max, hbm_gbs, which, run.bytes_per_update)

    e2e = None
    if not args.no_e2e:
        barrier()
        ms_e, _ = time_steps(torch, run, args.steps, max(1, args.warmup), flush, e2e=True)
        tot_e, upd_e, _ = reduce_over_ranks(dist, "cuda", sum(ms_e), run.updates * args.steps, 0)
        e2e = {"value": upd_e / (tot_e * 1e-3), "unit": "spin updates/s",
               "h2d_bytes_per_step": run.h2d, "d2h_bytes_per_step": run.d2h, "ms_per_step": tot_e / args.steps,
               "path": "potts_upload (pinned host) + potts_sweep_measured (host series) + potts_download (pinned host)"}
    layout = "packed" if run.layout == pb.LAYOUT_PACKED else "u8"
    run.g.close()

    per_cfg, cpu, e6 = None, None, None
    if rank == 0 and world == 1 and not args.no_per_config:
        per_cfg = per_config_table(pb, torch, flush, sm_max, hbm_gbs, which)
        e6 = paper_protocol_e6(pb, torch)
        per_cfg["batch_cfg1_x1184"] = batch_of_cfg1(pb, torch)
        per_cfg["delta_stream_cfg5"] = delta_stream_cost(pb, torch)
        # SURVEY 8(f)1, NOT the headline chain: the same workloads under stream-spec v2 (one Philox block per pair of
        # sites, S15); its algorithmic instruction count is 19 per update, so alu_frac is not comparable
        v2 = per_config_table(pb, torch, flush, sm_max, hbm_gbs, which, skip=(1,), stream_spec=2)
        per_cfg["stream_spec_2"] = {k: {"ns_per_spin_flip": v["ns_per_spin_flip"], "spin_updates_per_s": v["spin_updates_per_s"],
                                        "kernel": v["kernel"]} for k, v in v2.items()}
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = cpu_baseline(w)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    if rank != 0:
        return
    line = {
        "metric": "spin_updates_per_s", "value": value, "unit": "spin updates/s", "ns_per_spin_flip": 1e9 / value * world,
        "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": total_s * 1e3 / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u8", "data": "synthetic",
        "gpu_launches": launches_all,
        "config": {"workload": w.name, "q": w.q, "L": w.L, "init": "random" if w.init else "ordered",
                   "T_over_Tc": w.t_factors if len(w.t_factors) > 1 else w.t_factors[0],
                   "sweeps_per_step": run.sweeps, "of_sweeps": w.total_sweeps, "measure_every": w.every,
                   "hist": w.hist, "layout": layout, "seed": w.seed, "options": options,
                   "parallelism": f"{world} independent sample(s), one per GPU" if world > 1 else "1 GPU",
                   "l2": "each step starts from a fresh lattice after a 256 MiB L2 flush; within a step the "
                         "lattice is re-swept in place, so L2 residency for L <= 8192 is the workload's own"},
        "clocks": clk.summary(), "roofline": roof, "e2e": e2e, "cpu_baseline": cpu, "per_config": per_cfg,
        "paper_protocol_e6": e6,
        "wall_s_timed_region": wall,
        "paper_context": {"ns_per_spin_flip_gtx480": 0.147, "note": "other hardware and RNG; context, not a target"},
    }
    print(json.dumps(line), flush=True)


if __name__ == "__main__":
    main()

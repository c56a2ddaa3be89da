#!/usr/bin/env python
"""bench.py -- throughput of the direct-summation hot path on B200, one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload C3|C3b|C4|C2|C1]

Metric (BASELINE.json): pairwise interactions/s for acc+jerk+pot at N=131072 (config C3:
seeded Plummer sphere, eps=1/256, all i active), interactions = n_i * n_j with the self pair
counted as the paper does.

A "step" is one pass of the whole hot path through the C ABI:
  a1 nbk_set_j_particles[_dev]  a2 nbk_set_ti  a3 predict kernel  a4+a5 i x j force kernel
  a6 reduce kernel  a7 nbk_calc_lasthalf[_dev]
`value`   : inputs resident in HBM, _dev entry points, each step timed with CUDA events on the
            stream the library launches on; L2 is flushed between steps (outside the events).
`e2e`     : the same step through the HOST entry points with inputs and results in PINNED host
            arrays (the library copies host <-> device directly from / into them), host clock
            around K steps, copies inside the timed region.
`roofline`: the i x j force kernel alone (the library's own CUDA events around that launch),
            bound "alu": executed fp32 flops / (SMs x 128 lanes x 2 x max SM clock).
`cpu_baseline`: oracle/nbody_oracle.c (fp64, OpenMP) on a bounded i-slice of the same workload, on all
            host cores; `cpu_baseline_1core`: the same with OMP_NUM_THREADS=1 (a child process).
--extras  : adds `block_sweep` (config C2: i-blocks of 1..16384 at N=16384: kernel, call and launch-floor
            microseconds) and `hermite` (config C5 on the device-resident loop: wall time, steps, dE/E)
            to the JSON line.

N > 1 (torchrun): the path does not shard under BASELINE.json's north_star ("Everything runs on
one GPU, with no sharding or collectives"), so every rank runs an independent replica of the
workload ("replicas only"); value = sum of interactions over ranks / max time.
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

METRIC = "pairwise interactions/sec (acc+jerk+pot) and % of B200 FP32 peak at N=131072"   # BASELINE.json (config C3)


def metric_of(wl, n):
    """BASELINE.json's metric string for its own workload (C3); the same wording with the workload's
    quantities and N for the others, so that a line never claims a workload it did not run."""
    _, eps, jerk, _ = wl
    what = "acc+jerk+pot" if jerk else "acc+pot"
    if eps == 0.0:
        what += ", eps=0"
    return f"pairwise interactions/sec ({what}) and % of B200 FP32 peak at N={n}"


def sm_max_mhz_measured(fallback=1965.0):
    """Max SM clock from the driver-written MEASURED_PEAKS.json (the roofline denominator's clock)."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["sm_max_mhz"]), "MEASURED_PEAKS.json sm_max_mhz"
    except Exception:
        return float(fallback), "nvml max SM clock"

UNIT = "interactions/s"
FLOPS_EXECUTED = {True: 42.0, False: 20.0}   # per interaction, FFMA = 2
FLOPS_PAPER = {True: 60.0, False: 38.0}      # PAPER.md Eq. 3
FP32_OPS = {True: 27.0, False: 13.0}         # minimum FP32-pipe lane operations per interaction
L2_FLUSH_BYTES = 256 << 20                   # > 126 MB L2

WORKLOADS = {
    # name: (config, eps, jerk, description)
    "C1": ("C1", 1.0 / 256.0, True, "C1: N=1024 Plummer seed 1, eps=1/256, acc+jerk+pot, all i"),
    "C2": ("C2", 1.0 / 256.0, True, "C2: N=16384 Plummer seed 2, eps=1/256, acc+jerk+pot, all i"),
    "C3": ("C3", 1.0 / 256.0, True, "C3: N=131072 Plummer seed 3, eps=1/256, acc+jerk+pot, all i"),
    "C3b": ("C3", 0.0, True, "C3b: N=131072 Plummer seed 3, eps=0 (self/zero-distance masked), acc+jerk+pot"),
    "C4": ("C4", 1.0 / 256.0, False, "C4: N=1048576 Plummer seed 4, eps=1/256, acc+pot only, all i"),
    "C5": ("C5", 1.0 / 256.0, True, "C5: N=65536 Plummer seed 5, eps=1/256, acc+jerk+pot, all i"),
}


# ------------------------------------------------------------------------ multi-rank plumbing
def dist_env():
    return int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))


def aggregate(local_ms: float, local_units: float, world: int, backend_device: str):
    """max-over-ranks time and sum-over-ranks units (torch.distributed; identity at world 1)."""
    if world == 1:
        return local_ms, local_units
    import torch
    import torch.distributed as dist
    t = torch.tensor([local_ms], dtype=torch.float64, device=backend_device)
    u = torch.tensor([local_units], dtype=torch.float64, device=backend_device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


# ------------------------------------------------------------------------ clocks during timing
class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons of one GPU through NVML while the timed region runs."""

    BITS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown",
            0x40: "hw_thermal_slowdown", 0x80: "hw_power_brake_slowdown"}

    def __init__(self, index: int, period: float = 0.02):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.samples, self.reasons, self.power = [], set(), []
        self.max_mhz = None
        self._stop_evt = threading.Event()
        self.error = None

    def run(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            h = pynvml.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM)
            while not self._stop_evt.is_set():
                self.samples.append(pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_SM))
                try:
                    self.power.append(pynvml.nvmlDeviceGetPowerUsage(h) / 1000.0)
                    r = pynvml.nvmlDeviceGetCurrentClocksEventReasons(h)
                except Exception:  # older binding name
                    r = pynvml.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                for bit, name in self.BITS.items():
                    if r & bit:
                        self.reasons.add(name)
                time.sleep(self.period)
        except Exception as e:  # NVML unavailable: report it, never fake clocks
            self.error = repr(e)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=2.0)
        out = {"sm_mhz": float(np.median(self.samples)) if self.samples else None,
               "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
               "samples": len(self.samples)}
        if self.power:
            out["power_w_max"] = max(self.power)
        if self.error:
            out["error"] = self.error
        return out


def physical_gpu_index(local: int) -> int:
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local])
        except Exception:
            return local
    return local


# ------------------------------------------------------------------------ the oracle legs
def oracle_sample(m, x, v, eps, jerk, target_s=15.0, seed=11):
    """Time oracle/nbody_oracle.c on a bounded i-slice of the workload (all j).  Returns
    (interactions/s, cores, n_i_sample, seconds)."""
    from oracle import c_oracle
    c_oracle.build()
    n = m.shape[0]
    cores = c_oracle.num_threads()
    rng = np.random.default_rng(seed)
    probe = min(n, 64 * cores)
    idx = np.sort(rng.choice(n, size=probe, replace=False))
    t0 = time.perf_counter()
    c_oracle.force(m, x, v, eps, i_index=idx, want_jerk=jerk)
    dt = max(time.perf_counter() - t0, 1e-6)
    n_i = int(min(n, max(probe, probe * target_s / dt)))
    idx = np.sort(rng.choice(n, size=n_i, replace=False))
    t0 = time.perf_counter()
    c_oracle.force(m, x, v, eps, i_index=idx, want_jerk=jerk)
    dt = time.perf_counter() - t0
    return n_i * n / dt, cores, n_i, dt


def oracle_sample_1core(workload, target_s=6.0):
    """The same oracle sample with OMP_NUM_THREADS=1, in a child process (the thread count of an OpenMP
    runtime is fixed once it has started); None if the child fails."""
    import subprocess
    env = dict(os.environ, OMP_NUM_THREADS="1")
    try:
        out = subprocess.run([sys.executable, os.path.abspath(__file__), "--oracle-sample", str(target_s),
                              "--workload", workload], env=env, capture_output=True, text=True, timeout=300)
        return json.loads(out.stdout.strip().splitlines()[-1])
    except Exception:
        return None


def run_oracle_sample(args, wl):
    """--oracle-sample SECONDS: time the oracle on a bounded i-slice of the workload, print one JSON object."""
    from paper_0707_0438_b200 import inputs
    cfg, eps, jerk, _ = wl
    m, x, v = inputs.config_inputs(cfg)
    ov, cores, ni_s, secs = oracle_sample(m, x, v, eps, jerk, target_s=args.oracle_sample)
    n = m.shape[0]
    print(json.dumps({"value": ov, "unit": UNIT, "cores": cores, "kind": "oracle",
                      "sample": f"{ni_s} of {n} i-particles (seeded choice) x all {n} j, {secs:.1f} s"}), flush=True)
    return 0


def run_reference(args, wl):
    """--impl reference: the oracle as it stands, on the host cores, same metric and config."""
    rank, _, world = dist_env()
    if rank != 0:
        return 0
    from paper_0707_0438_b200 import inputs
    from oracle import c_oracle
    cfg, eps, jerk, desc = wl
    m, x, v = inputs.config_inputs(cfg)
    n = m.shape[0]
    c_oracle.build()
    cores = c_oracle.num_threads()
    rng = np.random.default_rng(11)
    # size one step to ~ (120 s / (steps + warmup)), from a short probe
    probe = min(n, 32 * cores)
    idx = np.sort(rng.choice(n, size=probe, replace=False))
    t0 = time.perf_counter()
    c_oracle.force(m, x, v, eps, i_index=idx, want_jerk=jerk)
    dt = max(time.perf_counter() - t0, 1e-6)
    budget = 120.0 / max(1, args.steps + args.warmup)
    n_i = int(min(n, max(probe, probe * budget / dt)))
    idx = np.sort(rng.choice(n, size=n_i, replace=False))
    for _ in range(args.warmup):
        c_oracle.force(m, x, v, eps, i_index=idx, want_jerk=jerk)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        c_oracle.force(m, x, v, eps, i_index=idx, want_jerk=jerk)
    dt = time.perf_counter() - t0
    value = args.steps * n_i * n / dt
    sample = f"{n_i} of {n} i-particles (seeded choice) x all {n} j per step"
    line = {
        "impl": "reference", "metric": metric_of(wl, n), "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": {"workload": desc, "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


# ------------------------------------------------------------------------ our arm
def run_ours(args, wl):
    import torch
    rank, local, world = dist_env()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the hot path has no CPU fallback")
    from paper_0707_0438_b200 import binding as nb
    from paper_0707_0438_b200 import inputs
    nb.load()
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    cfg, eps, jerk, desc = wl
    m, x, v = inputs.config_inputs(cfg)
    n = m.shape[0]
    eps2 = float(np.float32(eps) ** 2)
    flags = (nb.NBK_JERK if jerk else 0) | nb.NBK_POT

    stream = torch.cuda.Stream(device=dev)
    ctx = nb.nbk_open(local, n, n, stream.cuda_stream)
    try:
        with torch.cuda.stream(stream):
            d_m = torch.from_numpy(m).to(dev)
            d_x = torch.from_numpy(x).to(dev)
            d_v = torch.from_numpy(v).to(dev)
            d_acc = torch.empty((n, 3), dtype=torch.float32, device=dev)
            d_jrk = torch.empty((n, 3), dtype=torch.float32, device=dev)
            d_pot = torch.empty((n,), dtype=torch.float32, device=dev)
            flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device=dev)
        stream.synchronize()

        def step_dev():
            nb.nbk_set_j_particles_dev(ctx, n, 0, 0, d_m.data_ptr(), d_x.data_ptr(), d_v.data_ptr())
            nb.nbk_set_ti(ctx, 0.0)
            nb.nbk_calc_firsthalf_dev(ctx, n, n, 0, 0, 0, eps2, flags)
            nb.nbk_calc_lasthalf_dev(ctx, n, d_acc.data_ptr(), d_jrk.data_ptr(), d_pot.data_ptr())

        # end-to-end arm: inputs and results in PINNED host memory (numpy views of pinned torch tensors);
        # the library copies host <-> device directly from / into them
        def pinned(a):
            t = torch.from_numpy(a).pin_memory()
            return t, t.numpy()
        keep = [pinned(m), pinned(x), pinned(v), pinned(np.empty((n, 3), np.float32)),
                pinned(np.empty((n, 3), np.float32)), pinned(np.empty(n, np.float32))]
        hm, hx, hv, h_acc, h_jrk, h_pot = (k[1] for k in keep)

        def step_host():
            nb.nbk_set_j_particles(ctx, None, None, hm, hx, hv)
            nb.nbk_set_ti(ctx, 0.0)
            nb.nbk_calc_firsthalf(ctx, n, n, None, None, None, eps2, flags)
            return nb.nbk_calc_lasthalf(ctx, n, out=(h_acc, h_jrk, h_pot))

        def barrier():
            if world > 1:
                import torch.distributed as dist
                dist.barrier()
            torch.cuda.synchronize(dev)

        # ---- device-resident arm: per-step CUDA events on the library's stream
        nb.nbk_set_timing(ctx, True)
        with torch.cuda.stream(stream):
            for _ in range(max(args.warmup, 0)):
                flush.zero_()
                step_dev()
        barrier()
        sampler = ClockSampler(physical_gpu_index(local))
        sampler.start()
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
               for _ in range(args.steps)]
        kern_ms = {"scatter": [], "predict": [], "force": [], "reduce": []}
        with torch.cuda.stream(stream):
            for k in range(args.steps):
                flush.zero_()            # L2 flush between timed iterations, outside the events
                evs[k][0].record(stream)
                step_dev()
                evs[k][1].record(stream)
                t = nb.nbk_get_timing(ctx)   # waits for this step; the library's own per-kernel events
                for key in kern_ms:
                    kern_ms[key].append(t[key])
        barrier()
        clocks = sampler.stop()
        step_ms = [a.elapsed_time(b) for a, b in evs]
        local_ms = float(np.sum(step_ms))
        launch = nb.nbk_last_launch(ctx)
        nb.nbk_set_timing(ctx, False)
        total_ms, total_units = aggregate(local_ms, float(args.steps) * n * n, world, str(dev))
        value = total_units / (total_ms * 1e-3)

        # ---- end-to-end arm: host buffers through the host entry points
        for _ in range(min(args.warmup, 3)):
            step_host()
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            out = step_host()
        torch.cuda.synchronize(dev)
        e2e_local_ms = 1e3 * (time.perf_counter() - t0)
        barrier()
        e2e_ms, e2e_units = aggregate(e2e_local_ms, float(args.steps) * n * n, world, str(dev))
        e2e_value = e2e_units / (e2e_ms * 1e-3)
        assert np.all(np.isfinite(out[0])) and np.all(np.isfinite(out[2]))
    finally:
        nb.nbk_close(ctx)

    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()
    if rank != 0:
        return 0

    # ---- roofline of the dominant kernel (i x j force tile), rank 0
    sm_count = torch.cuda.get_device_properties(dev).multi_processor_count
    sm_max_mhz, peak_src = sm_max_mhz_measured(clocks.get("sm_max_mhz") or 1965.0)
    peak_tflops = sm_count * 128 * 2 * sm_max_mhz * 1e6 / 1e12
    force_ms = float(np.mean(kern_ms["force"]))
    kint = n * n / (force_ms * 1e-3)
    achieved = FLOPS_EXECUTED[jerk] * kint / 1e12
    # DRAM bytes of one launch of the kernel from the committed ncu --set full capture (bench.py cannot
    # run under ncu itself); null for workloads that were not captured
    traffic, traffic_src = None, None
    try:
        with open(os.path.join(ROOT, "profiles", "force_kernel_traffic.json")) as f:
            tj = json.load(f)
        traffic = tj.get(args.workload)
        if traffic is not None:
            traffic_src = tj.get("source", "committed ncu --set full capture, not measured in this run")
    except Exception:
        pass
    roofline = {
        "bound": "alu", "kernel": "nbk::force_kernel", "achieved": achieved, "peak": peak_tflops,
        "unit": "TFLOP/s", "frac": achieved / peak_tflops, "traffic": traffic, "traffic_source": traffic_src,
        "peak_source": f"{sm_count} SMs x 128 fp32 lanes x 2 x {sm_max_mhz:.0f} MHz ({peak_src}); "
                       "DESIGN.md 'Roofline'",
        "flops_per_interaction": FLOPS_EXECUTED[jerk],
        "kernel_ms": force_ms, "kernel_interactions_per_s": kint,
        "tflops_paper_convention": FLOPS_PAPER[jerk] * kint / 1e12,
        "frac_paper_convention": FLOPS_PAPER[jerk] * kint / 1e12 / peak_tflops,
        "fp32_pipe_frac_at_max_clock": FP32_OPS[jerk] * kint / (sm_count * 128 * sm_max_mhz * 1e6),
        "fp32_pipe_frac_at_observed_clock": (FP32_OPS[jerk] * kint / (sm_count * 128 * clocks["sm_mhz"] * 1e6)
                                             if clocks.get("sm_mhz") else None),
        "mufu_limit_interactions_per_s": sm_count * 16 * sm_max_mhz * 1e6,
        "kernel_share_of_step": force_ms / float(np.mean(step_ms)),
        "other_kernels_ms": {k: float(np.mean(kern_ms[k])) for k in ("scatter", "predict", "reduce")},
    }

    # ---- the oracle on the host cores, bounded sample
    cpu_baseline = None
    if not args.skip_cpu_baseline:
        ov, cores, ni_s, secs = oracle_sample(m, x, v, eps, jerk)
        cpu_baseline = {"value": ov, "unit": UNIT, "cores": cores, "kind": "oracle",
                        "sample": f"{ni_s} of {n} i-particles (seeded choice) x all {n} j, {secs:.1f} s"}

    cpu_1core = None
    if not args.skip_cpu_baseline:
        cpu_1core = oracle_sample_1core(args.workload)
    extras = extras_objects(args) if args.extras else {}

    line = {
        "metric": metric_of(wl, n), "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": desc, "n_i": n, "n_j": n, "l2": f"flushed between steps ({L2_FLUSH_BYTES >> 20} MiB write)",
                   "parallelism": "replicas only" if world > 1 else "1 GPU",
                   "launch": launch},
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(n * (4 + 12 + 12)),
                "d2h_bytes_per_step": int(n * 28), "ms_per_step": e2e_ms / args.steps},
        "gpu_launches": int(args.steps * 4),
        "roofline": roofline,
        "cpu_baseline": cpu_baseline,
        "cpu_baseline_1core": cpu_1core,
        "tflops_paper_convention": FLOPS_PAPER[jerk] * value / 1e12,
    }
    line.update(extras)
    print(json.dumps(line), flush=True)
    return 0


def launch_floor_us(nb):
    """Launch + synchronise floor of this box: one 1-particle predictor launch and a stream sync."""
    ctx = nb.nbk_open(0, 256, 256)
    try:
        nb.nbk_set_j_particles(ctx, None, None, np.ones(1, np.float32), np.zeros((1, 3), np.float32))
        for q in range(20):
            nb.nbk_predict(ctx, 1)
            nb.nbk_sync(ctx)
        t0 = time.perf_counter()
        for q in range(500):
            nb.nbk_predict(ctx, 1)
            nb.nbk_sync(ctx)
        return (time.perf_counter() - t0) / 500 * 1e6
    finally:
        nb.nbk_close(ctx)


def extras_objects(args):
    """--extras: the block-step sweep of config C2 and the C5 Hermite run, as objects for the JSON line
    (the numbers of DESIGN.md section 9 from one committed command)."""
    from paper_0707_0438_b200 import binding as nb
    from paper_0707_0438_b200 import inputs
    eps = 1.0 / 256.0
    eps2 = float(np.float32(eps) ** 2)
    flags = nb.NBK_JERK | nb.NBK_POT
    # ---- C2: N = 16384, i-blocks drawn without replacement, prediction to a new time before every call
    m, x, v = inputs.config_inputs("C2")
    n = m.shape[0]
    floor = launch_floor_us(nb)
    sweep = []
    ctx = nb.nbk_open(0, n, n)
    try:
        nb.nbk_set_j_particles(ctx, None, None, m, x, v)
        for n_i in (1, 32, 256, 2048, 16384):
            idx = inputs.active_block(n, n_i, seed=2)
            nb.nbk_set_ti(ctx, 0.0)
            nb.nbk_set_timing(ctx, True)
            ks = []
            for _ in range(11):
                nb.nbk_calc_firsthalf(ctx, n, n_i, idx, None, None, eps2, flags)
                t = nb.nbk_get_timing(ctx)
                ks.append(t["force"] + t["reduce"])
            nb.nbk_set_timing(ctx, False)
            reps = 100 if n_i <= 2048 else 20
            for q in range(-5, reps):
                if q == 0:
                    t0 = time.perf_counter()
                nb.nbk_set_ti(ctx, 1e-4 * (q + 6))     # forces a new prediction, as a block step does
                nb.nbk_calc_firsthalf(ctx, n, n_i, idx, None, None, eps2, flags)
                nb.nbk_calc_lasthalf(ctx, n_i)
            w = (time.perf_counter() - t0) / reps
            k = float(np.median(ks[2:]))
            sweep.append({"n_i": n_i, "n_j": n, "kernel_us": 1e3 * k, "kernel_interactions_per_s": n * n_i / (k * 1e-3),
                          "api_us": 1e6 * w, "launch_sync_floor_us": floor})
    finally:
        nb.nbk_close(ctx)
    # ---- C5: N = 65536 to t = 1 on the device-resident loop; energies from the library's own potential
    cfg = inputs.CONFIGS["C5"]
    n5 = cfg["N"]
    m5, x5, v5 = inputs.plummer(n5, cfg["seed"])
    ctx = nb.nbk_open(0, n5, n5)

    def energy():
        nb.nbk_set_j_particles_f64(ctx, None, None, m5, x5, v5)
        nb.nbk_set_ti(ctx, 0.0)
        nb.nbk_calc_firsthalf(ctx, n5, n5, None, None, None, eps2, nb.NBK_POT)
        pot = nb.nbk_calc_lasthalf_f64(ctx, n5)[2]
        return float(0.5 * np.sum(m5 * np.sum(v5 * v5, axis=1)) + 0.5 * np.sum(m5 * pot))
    try:
        e0 = energy()
        st = nb.nbk_hermite_evolve_dev(ctx, m5, x5, v5, eps, 1.0, 0.01, 1.0 / 16.0)
        e1 = energy()
    finally:
        nb.nbk_close(ctx)
    hermite = {"workload": f"C5: N={n5} Plummer seed {cfg['seed']}, eps=1/256, eta=0.01, dt_max=1/16, to t=1",
               "loop": "device-resident", "wall_s": st["wall_seconds"], "block_steps": st["block_steps"],
               "particle_steps": st["particle_steps"], "interactions": st["interactions"],
               "interactions_per_s": st["interactions"] / st["wall_seconds"],
               "dE_over_E_gpu_potential": (e0 - e1) / e0}
    return {"block_sweep": sweep, "hermite": hermite}


def run_sharded(args, wl):
    """--shard j: the j-sharded path (paper_0707_0438_b200/sharded.py): every rank
    holds N/G j-particles, computes partial sums for all N i-particles, two all-reduces per step.
    Total work is fixed as G grows ("strong").  Not the default multi-GPU mode."""
    import torch
    rank, local, world = dist_env()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the hot path has no CPU fallback")
    from paper_0707_0438_b200 import binding as nb
    from paper_0707_0438_b200 import inputs
    from paper_0707_0438_b200.sharded import ShardedForce
    nb.load()
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    cfg, eps, jerk, desc = wl
    m, x, v = inputs.config_inputs(cfg)
    n = m.shape[0]
    eps2 = float(np.float32(eps) ** 2)
    flags = (nb.NBK_JERK if jerk else 0) | nb.NBK_POT
    if args.transport == "peer" and world == 1:   # symmetric memory wants a process group, also at world size 1
        import torch.distributed as dist
        if not dist.is_initialized():
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            os.environ.setdefault("MASTER_PORT", "29577")
            dist.init_process_group("nccl", rank=0, world_size=1, device_id=dev)
    sf = ShardedForce(n, n, device=local, mode=args.shard,
                      transport=args.transport if args.shard == "j" else "nccl")
    ci = -(-n // world)   # i-particles this rank's force kernel handles
    n_i_rank = n if args.shard == "j" else max(0, min((rank + 1) * ci, n) - min(rank * ci, n))
    try:
        sf.set_j_particles(None, None, m, x, v)
        sf.set_ti(0.0)
        ig = torch.arange(n, dtype=torch.int32, device=dev)
        out = (torch.empty((n, 3), dtype=torch.float32, device=dev), torch.empty((n, 3), dtype=torch.float32, device=dev),
               torch.empty((n,), dtype=torch.float32, device=dev))
        flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device=dev)

        def barrier():
            if world > 1:
                import torch.distributed as dist
                dist.barrier()
            torch.cuda.synchronize(dev)

        nb.nbk_set_timing(sf.ops.ctx, True)
        for _ in range(max(args.warmup, 0)):
            flush.zero_()
            sf.calc(ig, eps2, flags, out)
        barrier()
        sampler = ClockSampler(physical_gpu_index(local))
        sampler.start()
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
        force_ms = []
        for k in range(args.steps):
            flush.zero_()
            evs[k][0].record()
            sf.calc(ig, eps2, flags, out)
            evs[k][1].record()
            force_ms.append(nb.nbk_get_timing(sf.ops.ctx)["force"])
        barrier()
        clocks = sampler.stop()
        local_ms = float(np.sum([a.elapsed_time(b) for a, b in evs]))
        # strong scaling: the job's units are N x N per step whatever G is; time = max over ranks
        total_ms, units_sum = aggregate(local_ms, float(args.steps) * n_i_rank * sf.n_local, world, str(dev))
        launch = nb.nbk_last_launch(sf.ops.ctx)
        assert bool(torch.isfinite(out[0]).all()) and bool(torch.isfinite(out[2]).all())
    finally:
        sf.close()
    import torch.distributed as dist
    if dist.is_initialized():
        dist.destroy_process_group()
    if rank != 0:
        return 0
    sm_count = torch.cuda.get_device_properties(dev).multi_processor_count
    peak_tflops = sm_count * 128 * 2 * sm_max_mhz_measured()[0] * 1e6 / 1e12
    kint = n_i_rank * sf.n_local / (float(np.mean(force_ms)) * 1e-3)
    achieved = FLOPS_EXECUTED[jerk] * kint / 1e12
    line = {
        "metric": metric_of(wl, n), "value": units_sum / (total_ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "strong",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": desc, "n_i": n, "n_j": n, "parallelism": f"{args.shard}-sharded x{world}",
                   "n_j_per_rank": sf.n_local, "n_i_per_rank": n_i_rank,
                   "collectives_per_step": (0 if sf.transport == "peer" else 2 if args.shard == "j" else 3) if world > 1 else 0,
                   "transport": sf.transport + (" (symmetric memory, 2 barriers per step, P2P loads)" if sf.transport == "peer" else ""),
                   "l2": f"flushed between steps ({L2_FLUSH_BYTES >> 20} MiB write)", "launch": launch},
        "clocks": clocks, "gpu_launches": int(args.steps * 5),
        "roofline": {"bound": "alu", "kernel": "nbk::force_kernel (rank 0)", "achieved": achieved, "peak": peak_tflops,
                     "unit": "TFLOP/s", "frac": achieved / peak_tflops, "traffic": None,
                     "kernel_ms": float(np.mean(force_ms))},
        "cpu_baseline": None,
    }
    print(json.dumps(line), flush=True)
    return 0


def run_hermite(args):
    """--hermite host|dev: BASELINE.json config C5 (N = 65536 Plummer sphere, seed 5, eps = 1/256, eta = 0.01) integrated
    to --t-end with the host-driven (a8) or the device-resident (8(f)-1) block-step loop.  Prints wall time, block-step
    statistics and |dE/E| with the energies taken from the library's own fp32 potential (the fp64-oracle figure is in
    tests/test_gpu_configs.py).  Not the bench line."""
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py --hermite needs a CUDA device")
    from paper_0707_0438_b200 import binding as nb
    from paper_0707_0438_b200 import inputs
    nb.load()
    cfg = inputs.CONFIGS["C5"]
    n, eps = cfg["N"], 1.0 / 256.0
    m, x, v = inputs.plummer(n, cfg["seed"])
    ctx = nb.nbk_open(0, n, n)

    def energy():
        nb.nbk_set_j_particles_f64(ctx, None, None, m, x, v)
        nb.nbk_set_ti(ctx, 0.0)
        nb.nbk_calc_firsthalf(ctx, n, n, None, None, None, float(np.float32(eps) ** 2), nb.NBK_POT)
        pot = nb.nbk_calc_lasthalf_f64(ctx, n)[2]
        return float(0.5 * np.sum(m * np.sum(v * v, axis=1)) + 0.5 * np.sum(m * pot))
    try:
        e0 = energy()
        fn = nb.nbk_hermite_evolve_dev if args.hermite == "dev" else nb.nbk_hermite_evolve
        st = fn(ctx, m, x, v, eps, args.t_end, 0.01, args.dt_max)
        e1 = energy()
    finally:
        nb.nbk_close(ctx)
    print(json.dumps({"workload": f"C5: N={n} Plummer seed {cfg['seed']}, eps=1/256, eta=0.01, dt_max={args.dt_max}, to t={args.t_end}",
                      "loop": "device-resident" if args.hermite == "dev" else "host-driven", "wall_s": st["wall_seconds"],
                      "block_steps": st["block_steps"], "particle_steps": st["particle_steps"],
                      "interactions": st["interactions"], "interactions_per_s": st["interactions"] / st["wall_seconds"],
                      "dE_over_E_gpu_potential": (e0 - e1) / e0, "ni_histogram_log2": st["ni_histogram"][:18]}), flush=True)
    return 0


def run_sweep(args):
    """--sweep: the paper's Table 3 / Table 4 shape (kernel-only time against N)
    plus the block-step i-set sizes of config C2, as a markdown table on stdout.  Not the bench line."""
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py --sweep needs a CUDA device")
    from paper_0707_0438_b200 import binding as nb
    from paper_0707_0438_b200 import inputs
    nb.load()
    sm = torch.cuda.get_device_properties(0).multi_processor_count
    peak = sm * 128 * 2 * sm_max_mhz_measured()[0] * 1e6
    eps2 = float(np.float32(1.0 / 256.0) ** 2)

    def kernel_ms(ctx, n_j, n_i, idx, flags, e2, reps):
        ts = []
        for _ in range(reps + 2):
            nb.nbk_calc_firsthalf(ctx, n_j, n_i, idx, None, None, e2, flags)
            t = nb.nbk_get_timing(ctx)
            ts.append(t["force"] + t["reduce"])
        return float(np.median(ts[2:]))

    print("| N | acc+jerk+pot ms | interactions/s | TFLOP/s (42) | % FP32 peak | TFLOP/s (k=60) | "
          "acc+pot ms | interactions/s | TFLOP/s (20) | eps=0 ms | +nearest neighbour ms |")
    print("|---|---|---|---|---|---|---|---|---|---|---|")
    seeds = {1024: 1, 16384: 2, 131072: 3, 1048576: 4, 65536: 5}
    for lg in range(10, 21):
        n = 1 << lg
        m, x, v = inputs.plummer_f32(n, seeds.get(n, 100 + lg))
        ctx = nb.nbk_open(0, n, n)
        try:
            nb.nbk_set_j_particles(ctx, None, None, m, x, v)
            nb.nbk_set_ti(ctx, 0.0)
            nb.nbk_set_timing(ctx, True)
            reps = 9 if n <= 131072 else 3
            full = kernel_ms(ctx, n, n, None, nb.NBK_JERK | nb.NBK_POT, eps2, reps)
            accp = kernel_ms(ctx, n, n, None, nb.NBK_POT, eps2, reps)
            e0 = kernel_ms(ctx, n, n, None, nb.NBK_JERK | nb.NBK_POT | nb.NBK_EPS0, 0.0, reps)
            nn = kernel_ms(ctx, n, n, None, nb.NBK_JERK | nb.NBK_POT | nb.NBK_NN, eps2, reps)
        finally:
            nb.nbk_close(ctx)
        r = n * n / (full * 1e-3)
        ra = n * n / (accp * 1e-3)
        print(f"| {n} | {full:.4f} | {r:.3e} | {42 * r / 1e12:.2f} | {100 * 42 * r / peak:.1f} | {60 * r / 1e12:.2f} | "
              f"{accp:.4f} | {ra:.3e} | {20 * ra / 1e12:.2f} | {e0:.4f} | {nn:.4f} |", flush=True)
    # Small N: one call's events include ~7 us of launch and event overhead (NBK_TRACE in-kernel spans are
    # that much shorter), so also time 32 calls queued back to back between two events
    print()
    print("| N | acc+jerk+pot, events per call us | 32 calls back to back, us per call | interactions/s (back to back) |")
    print("|---|---|---|---|")
    dev = torch.device("cuda", 0)
    ts_stream = torch.cuda.Stream(device=dev)
    for lg in range(10, 16):
        n = 1 << lg
        m, x, v = inputs.plummer_f32(n, seeds.get(n, 100 + lg))
        ctx = nb.nbk_open(0, n, n, ts_stream.cuda_stream)
        try:
            nb.nbk_set_j_particles(ctx, None, None, m, x, v)
            nb.nbk_set_ti(ctx, 0.0)
            nb.nbk_set_timing(ctx, True)
            single = kernel_ms(ctx, n, n, None, nb.NBK_JERK | nb.NBK_POT, eps2, 9)
            nb.nbk_set_timing(ctx, False)
            per = []
            for rep in range(5):
                e0_, e1_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0_.record(ts_stream)
                for q in range(32):
                    nb.nbk_calc_firsthalf_dev(ctx, n, n, 0, 0, 0, eps2, nb.NBK_JERK | nb.NBK_POT)
                e1_.record(ts_stream)
                ts_stream.synchronize()
                per.append(e0_.elapsed_time(e1_) / 32.0)
            b2b = float(np.median(per[1:]))
        finally:
            nb.nbk_close(ctx)
        print(f"| {n} | {single * 1e3:.1f} | {b2b * 1e3:.1f} | {n * n / (b2b * 1e-3):.3e} |", flush=True)
    # a3 predictor (HBM-bound: 72 B read + 28 B written per particle)
    hbm_peak = 6549.1
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            hbm_peak = float(json.load(f)["hbm_gbs"])
    except Exception:
        pass
    print()
    print(f"| N | predict_kernel us | GB/s (100 B per particle) | fraction of measured HBM copy peak ({hbm_peak:.0f} GB/s) |")
    print("|---|---|---|---|")
    for n in (131072, 1048576, 4194304):
        rng = np.random.default_rng(n)
        m = np.full(n, 1.0 / n, np.float32)
        x = rng.standard_normal((n, 3)).astype(np.float32)
        v = rng.standard_normal((n, 3)).astype(np.float32)
        ctx = nb.nbk_open(0, n, 1024)
        try:
            nb.nbk_set_j_particles(ctx, None, np.zeros(n), m, x, v, v, v)
            nb.nbk_set_timing(ctx, True)
            ts = []
            for q in range(12):
                nb.nbk_set_ti(ctx, 1e-3 * (q + 1))
                nb.nbk_predict(ctx, n)
                ts.append(nb.nbk_get_timing(ctx)["predict"])
            us = float(np.median(ts[2:])) * 1e3
        finally:
            nb.nbk_close(ctx)
        gbs = 100.0 * n / (us * 1e-6) / 1e9
        print(f"| {n} | {us:.1f} | {gbs:.0f} | {gbs / hbm_peak:.2f} |", flush=True)
    floor_us = launch_floor_us(nb)
    print()
    print(f"Launch + synchronise floor (one 1-thread-block kernel, stream sync, through the binding): {floor_us:.1f} us")
    print()
    print("| N | n_i (block) | force+reduce kernels us | interactions/s | firsthalf+lasthalf wall us (host API) |")
    print("|---|---|---|---|---|")
    for n, seed in ((16384, 2), (65536, 5), (131072, 3), (1048576, 4)):   # north_star: N from 1K to 1M, block-step i-sets
        m, x, v = inputs.plummer_f32(n, seed)
        ctx = nb.nbk_open(0, n, 16384)
        try:
            nb.nbk_set_j_particles(ctx, None, None, m, x, v)
            for n_i in (1, 32, 256, 2048, 16384):
                idx = inputs.active_block(n, n_i, seed=2)
                nb.nbk_set_timing(ctx, True)
                nb.nbk_set_ti(ctx, 0.0)
                k = kernel_ms(ctx, n, n_i, idx, nb.NBK_JERK | nb.NBK_POT, eps2, 9)
                nb.nbk_set_timing(ctx, False)
                reps = 100 if n_i <= 2048 else 20
                t0 = time.perf_counter()
                for q in range(reps):
                    nb.nbk_set_ti(ctx, 1e-4 * (q + 1))     # forces a new prediction, as a block step does
                    nb.nbk_calc_firsthalf(ctx, n, n_i, idx, None, None, eps2, nb.NBK_JERK | nb.NBK_POT)
                    nb.nbk_calc_lasthalf(ctx, n_i)
                w = (time.perf_counter() - t0) / reps
                print(f"| {n} | {n_i} | {k * 1e3:.1f} | {n * n_i / (k * 1e-3):.3e} | {w * 1e6:.1f} |", flush=True)
        finally:
            nb.nbk_close(ctx)
    return 0


def run_profile_pass(args):
    """--profile-pass: one call of each launch shape outside the headline kernel, few launches in all, meant to be run
    under ncu (profiles/): config C2 blocks of 32, 256, 2048 and 16384 i-particles (predict, force, reduce), the predictor
    at N = 1048576, one batched call (groups of ~256), and config C5 on the device-resident loop for one dt_max."""
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py --profile-pass needs a CUDA device")
    from paper_0707_0438_b200 import binding as nb
    from paper_0707_0438_b200 import inputs
    nb.load()
    eps = 1.0 / 256.0
    eps2 = float(np.float32(eps) ** 2)
    flags = nb.NBK_JERK | nb.NBK_POT
    m, x, v = inputs.config_inputs("C2")
    n = m.shape[0]
    ctx = nb.nbk_open(0, n, n)
    try:
        nb.nbk_set_j_particles(ctx, None, None, m, x, v)
        for rep in range(2):   # second round: warm
            for n_i in (32, 256, 2048, 16384):
                nb.nbk_set_ti(ctx, 1e-3 * (rep + 1) + 1e-5 * n_i)
                nb.nbk_calc_firsthalf(ctx, n, n_i, inputs.active_block(n, n_i, seed=2), None, None, eps2, flags)
                nb.nbk_calc_lasthalf(ctx, n_i)
    finally:
        nb.nbk_close(ctx)
    n4 = 1 << 20
    m4, x4, v4 = inputs.plummer_f32(n4, 4)
    ctx = nb.nbk_open(0, n4, 1024)
    try:
        nb.nbk_set_j_particles(ctx, None, None, m4, x4, v4)
        for rep in range(3):
            nb.nbk_set_ti(ctx, 1e-3 * (rep + 1))
            nb.nbk_predict(ctx, n4)
        nb.nbk_sync(ctx)
    finally:
        nb.nbk_close(ctx)
    rng = np.random.default_rng(1234)
    ng = 1024
    ni, nj = rng.integers(128, 385, ng), rng.integers(1800, 2701, ng)
    io = np.concatenate([[0], np.cumsum(ni)]).astype(np.int64)
    jo = np.concatenate([[0], np.cumsum(nj)]).astype(np.int64)
    centre = rng.standard_normal((ng, 3)).astype(np.float32)
    xi = np.repeat(centre, ni, axis=0) + np.float32(0.05) * rng.standard_normal((io[-1], 3)).astype(np.float32)
    xj = np.repeat(centre, nj, axis=0) + rng.standard_normal((jo[-1], 3)).astype(np.float32)
    mj = (rng.uniform(0.5, 2.0, jo[-1]) / 1000.0).astype(np.float32)
    ctx = nb.nbk_open(0, 64, 64)
    try:
        for rep in range(2):
            nb.nbk_calc_batch(ctx, io, xi, jo, mj, xj, eps2, nb.NBK_POT)
    finally:
        nb.nbk_close(ctx)
    cfg = inputs.CONFIGS["C5"]
    m5, x5, v5 = inputs.plummer(cfg["N"], cfg["seed"])
    ctx = nb.nbk_open(0, cfg["N"], cfg["N"])
    try:
        st = nb.nbk_hermite_evolve_dev(ctx, m5, x5, v5, eps, args.dt_max, 0.01, args.dt_max)
    finally:
        nb.nbk_close(ctx)
    print(json.dumps({"profile_pass": "ok", "hermite_block_steps": st["block_steps"]}), flush=True)
    return 0


def run_batch(args):
    """--batch: batched acceleration + potential calls (the treecode use of PAPER.md L229-L231,
    Table 7): about one million i-particles per call in groups of ~8, ~64, ~256 and ~1024 particles, each with
    its own interaction list, all groups in one launch.  Markdown table on stdout: kernel time (the library's CUDA events
    around batch_kernel), interactions/s in the kernel, and the whole call (packing, descriptors, reduction) with device
    pointers.  Seeded synthetic groups (clump of i-particles, list of cells around it).  Not the bench line."""
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py --batch needs a CUDA device")
    from paper_0707_0438_b200 import binding as nb
    nb.load()
    eps2 = float(np.float32(1.0 / 256.0) ** 2)
    shapes = [("~8", (4, 12), (300, 700)), ("~64", (32, 96), (900, 1500)), ("~256", (128, 384), (1800, 2700)),
              ("~1024", (512, 1536), (3600, 5400))]
    print("| group size | groups | i-particles | list entries | interactions | launch (i per lane, j-slices) | "
          "batch_kernel ms | interactions/s (kernel) | whole call ms | interactions/s (call) |")
    print("|---|---|---|---|---|---|---|---|---|---|")
    ctx = nb.nbk_open(0, 64, 64)
    try:
        for name, (i_lo, i_hi), (j_lo, j_hi) in shapes:
            rng = np.random.default_rng(1234)
            n_groups = int(round(1048576 / (0.5 * (i_lo + i_hi))))
            ni = rng.integers(i_lo, i_hi + 1, n_groups)
            nj = rng.integers(j_lo, j_hi + 1, n_groups)
            io = np.concatenate([[0], np.cumsum(ni)]).astype(np.int64)
            jo = np.concatenate([[0], np.cumsum(nj)]).astype(np.int64)
            centre = rng.standard_normal((n_groups, 3)).astype(np.float32)
            xi = np.repeat(centre, ni, axis=0) + np.float32(0.05) * rng.standard_normal((io[-1], 3)).astype(np.float32)
            xj = np.repeat(centre, nj, axis=0) + rng.standard_normal((jo[-1], 3)).astype(np.float32)
            mj = (rng.uniform(0.5, 2.0, jo[-1]) / 1000.0).astype(np.float32)
            inter = float(np.sum(ni.astype(np.float64) * nj))
            dxi, dmj, dxj = (torch.from_numpy(t).cuda() for t in (xi, mj, xj))
            acc = torch.empty((int(io[-1]), 3), dtype=torch.float32, device="cuda")
            pot = torch.empty(int(io[-1]), dtype=torch.float32, device="cuda")
            torch.cuda.synchronize()

            def call():
                nb.nbk_calc_batch_dev(ctx, io, dxi.data_ptr(), jo, dmj.data_ptr(), dxj.data_ptr(), eps2, nb.NBK_POT,
                                      acc.data_ptr(), pot.data_ptr())
            for _ in range(2):
                call()
            nb.nbk_set_timing(ctx, True)
            ks = []
            for _ in range(5):
                call()
                ks.append(nb.nbk_get_timing(ctx)["force"])
            nb.nbk_set_timing(ctx, False)
            t0 = time.perf_counter()
            for _ in range(5):
                call()
            w = (time.perf_counter() - t0) / 5
            k = float(np.median(ks))
            shape = nb.nbk_last_launch(ctx)
            print(f"| {name} | {n_groups} | {int(io[-1])} | {int(jo[-1])} | {inter:.3e} | {shape['i_per_thread']}, "
                  f"{shape['j_split_warps']} | {k:.3f} | {inter / (k * 1e-3):.3e} | {w * 1e3:.3f} | {inter / w:.3e} |",
                  flush=True)
            del dxi, dmj, dxj, acc, pot
    finally:
        nb.nbk_close(ctx)
    return 0


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--workload", choices=sorted(WORKLOADS), default="C3")
    ap.add_argument("--skip-cpu-baseline", action="store_true",
                    help="do not time the oracle (for runs under ncu); cpu_baseline is then null")
    ap.add_argument("--sweep", action="store_true",
                    help="print kernel time against N (1K..1M) and the block-step sweep as markdown tables")
    ap.add_argument("--shard", choices=["none", "j", "i"], default="none",
                    help="j: shard the j-particles over the ranks with two all-reduces per step; i: replicate j, shard "
                         "each i-list, all-gather the results (both strong scaling); "
                         "default: independent replicas (weak)")
    ap.add_argument("--transport", choices=["nccl", "peer"], default="nccl",
                    help="with --shard j: exchange by NCCL all-reduces, or by loads from peer (symmetric) memory")
    ap.add_argument("--hermite", choices=["host", "dev"], default=None,
                    help="integrate config C5 with the host-driven or the device-resident Hermite loop and print wall time")
    ap.add_argument("--extras", action="store_true",
                    help="add block_sweep (config C2) and hermite (config C5, device-resident loop) objects to the JSON line")
    ap.add_argument("--oracle-sample", type=float, default=None, help=argparse.SUPPRESS)
    ap.add_argument("--profile-pass", action="store_true",
                    help="one call of each launch shape outside the headline kernel (for ncu)")
    ap.add_argument("--batch", action="store_true",
                    help="time the batched acceleration + potential calls (groups of ~8 to ~1024 particles) as a markdown table")
    ap.add_argument("--t-end", type=float, default=1.0)
    ap.add_argument("--dt-max", type=float, default=1.0 / 16.0)
    args = ap.parse_args(argv)
    if args.hermite:
        return run_hermite(args)
    if args.sweep:
        return run_sweep(args)
    if args.batch:
        return run_batch(args)
    if args.profile_pass:
        return run_profile_pass(args)
    wl = WORKLOADS[args.workload]
    if args.oracle_sample is not None:
        return run_oracle_sample(args, wl)
    if args.impl == "reference":
        return run_reference(args, wl)
    if args.shard in ("j", "i"):
        return run_sharded(args, wl)
    return run_ours(args, wl)


if __name__ == "__main__":
    sys.exit(main())

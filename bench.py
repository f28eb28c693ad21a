#!/usr/bin/env python
"""bench.py — headline measurement of the per-time-step hot path.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload cfg2]

One bench "step" = TIME_STEPS_PER_BENCH_STEP (1000) consecutive simulation time steps = 100 ms of biological time of
the whole hot path (update + Poisson -> spike collection -> delivery) on the full-scale cortical-microcircuit-shaped
network (BASELINE.json configs[2]: 77,169 LIF neurons, 298,905,266 synapses).  metric = real-time factor
(wall seconds per biological second, lower is better) — the quantity PAPER.md:248 reports (1.055 s on an RTX 2080 Ti).

Prints ONE JSON line (rank 0).  Extra objects: `roofline` (dominant kernel of the step, per-kernel CUDA-event times),
`delivery_microbench` (BASELINE.json configs[3], the delivery kernel alone at bandwidth-relevant load),
`cpu_baseline` (the oracle as it stands on the host cores, bounded sample), `e2e` (state in/out through HOST buffers).
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

TIME_STEPS_PER_BENCH_STEP = 1000
DT_MS = 0.1
NCU_DRAM_BYTES_PER_LAUNCH_CFG2 = 895.8e6     # profiles/r01f_cfg2_full_summary.csv
NCU_DRAM_BYTES_PER_LAUNCH_CFG4 = 36.33e9     # profiles/r01h_cfg4_full_summary.csv (13.5 GB read + 22.8 GB written)
PAPER_RTF_2080TI = 1.055          # PAPER.md:248, full-scale microcircuit, NeuronGPU on RTX 2080 Ti (context, other hardware)
PAPER_RTF_ADEX_1M = 70.0          # PAPER.md:16, balanced network of 1e6 AdEx neurons / 1e9 synapses on an RTX 2080 Ti (context)
BYTES_PER_EVENT = 8               # 4 B target + 4 B weight per synaptic event
BYTES_PER_NEURON_STEP = 33        # V, I_syn, refr read+write (24 B) + ring slot read+zero (8 B) + population index (1 B)


def measured_peak_gbs():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """Samples SM clock and throttle reasons with NVML while the timed region runs."""

    def __init__(self, index=0, period=0.05):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._t = None
        self.period, self.index = period, index
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def _run(self):
        nv = self.nv
        names = {"hw_slowdown": 0x8, "sw_thermal_slowdown": 0x20, "hw_thermal_slowdown": 0x40,
                 "hw_power_brake_slowdown": 0x80, "sw_power_cap": 0x4}
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h) if hasattr(nv, "nvmlDeviceGetCurrentClocksEventReasons") \
                    else nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            self._stop.wait(self.period)

    def __enter__(self):
        if self.nv:
            self._t = threading.Thread(target=self._run, daemon=True)
            self._t.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._t:
            self._t.join()

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": 0}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


def make_workload(name, seed_offset=0):
    from paper_2007_14236_b200 import workloads as W
    wl = {"cfg0": W.brunel_tiny, "cfg1": lambda: W.microcircuit(10), "cfg2": lambda: W.microcircuit(1),
          "cfg4": W.balanced_large, "adex1m": W.balanced_adex, "adex100k": lambda: W.balanced_adex(n=100_000)}[name]()
    wl.seed += seed_offset
    return wl


def workload_label(name):
    return {"cfg0": "configs[0] tiny Brunel-style LIF net, 1,000 neurons",
            "cfg1": "configs[1] cortical microcircuit at 10% neuron scale, full in-degrees, 7,718 neurons / 29,892,043 synapses",
            "cfg2": "configs[2] full-scale cortical microcircuit, 77,169 LIF neurons / 298,905,266 synapses",
            "cfg4": "configs[4] balanced E/I network, 1,000,000 LIF neurons / 1e9 synapses",
            "adex1m": "the paper's balanced network (PAPER.md:110-128, Tables I-II): 1,000,000 AdEx neurons with alpha conductances, "
                      "1000 inputs each (1e9 synapses), adaptive RK5",
            "adex100k": "the paper's balanced network at 100,000 AdEx neurons, 1000 inputs each (1e8 synapses)"}[name]


def dist_setup(n_gpus):
    """torch.distributed only when launched under torchrun with N > 1 (replicas: no data-path collective)."""
    import torch
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        import torch.distributed as dist
        torch.cuda.set_device(local)
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    return rank, world, local


def max_over_ranks(x, world, device):
    if world <= 1:
        return x
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(x, world, device):
    if world <= 1:
        return x
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def barrier(world):
    import torch
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
    torch.cuda.synchronize()


def delivery_microbench(device, peak_gbs, K=10000, fraction=0.05, steps=30, warm=5, fallback=True, kernel=0):
    """BASELINE.json configs[3]: delivery kernel alone (neuron update bypassed), 1e6 sources, out-degree K, a random
    fraction of sources firing per step.  Falls back to K = 1000 when 90 GB of records do not fit."""
    import torch
    from paper_2007_14236_b200 import binding as B, workloads as W
    for k_try in ((K, 1000) if fallback else (K,)):
        g = None
        try:
            wl = W.delivery_microbench(K=k_try, fraction=fraction)
            g = B.Sim(DT_MS, wl.ring_slots, wl.seed, record_spikes=False, device=device)
            wl.apply(g)
            g.set_option(B.OPT_DELIVERY_KERNEL, kernel)       # before prepare: kernel 4 changes what is allocated
            g.prepare()
            # the spike-buffer backend reaches its steady-state work per step only after ring_slots steps
            g.simulate(max(warm, wl.ring_slots + 8))
            # whole step (spike injection + delivery) in the default step mode, CUDA events on the simulator's stream
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            g.simulate(steps)
            e0.record(g.stream); g.simulate(steps); e1.record(g.stream); torch.cuda.synchronize()
            step_ms = e0.elapsed_time(e1) / steps
            step_mode = int(g.stats().step_mode)
            g.set_option(B.OPT_PROFILE, 1)
            s0 = g.stats()
            g.simulate(steps)
            s1 = g.stats()
            ev = s1.events - s0.events
            # kernels 1 and 2: the delivery kernel alone; kernel 3 is one launch per step (spike injection + delivery)
            ms = (s1.ms_deliver - s0.ms_deliver) if int(s1.delivery_kernel) != 3 else (s1.ms_update - s0.ms_update)
            out = {"workload": f"configs[3] delivery microbenchmark: 1e6 sources, out-degree {k_try}, {fraction:.1%} firing per step, D=64",
                   "steps": steps, "events_per_step": ev / steps, "deliver_ms_per_step": ms / steps,
                   "step_ms_default_mode": step_ms, "step_mode": step_mode, "events_per_s_whole_step": ev / steps / (step_ms * 1e-3),
                   "events_per_s": ev / (ms * 1e-3), "algorithmic_gbs": ev * BYTES_PER_EVENT / (ms * 1e-3) / 1e9,
                   "frac_of_hbm_peak": ev * BYTES_PER_EVENT / (ms * 1e-3) / 1e9 / peak_gbs,
                   "delivery_kernel": int(s1.delivery_kernel),
                   "ring_bytes": 4 * wl.n_neurons * (2 if int(s1.delivery_kernel) >= 4 else wl.ring_slots + 1),
                   "timed": "delivery kernel" if int(s1.delivery_kernel) != 3 else "pipelined step kernel (injection + delivery)",
                   "build_ms": s1.build_ms,
                   "n_connections": int(s1.n_connections)}
            g.close()
            return out
        except Exception as e:                       # out of memory on a smaller card: try the smaller point
            err = str(e)
            if g is not None:
                g.close()
            torch.cuda.empty_cache()
    return {"error": err}


def run_probes(device=0):
    """Measured ceilings for the access shapes of the delivery stage."""
    from paper_2007_14236_b200 import binding as B
    out = {"stream_read_GBps": B.probe(0, 4 << 20, device) / 1e9}
    for mb in (4, 16, 64, 256):
        out[f"scattered_red_per_s_{mb}MB"] = B.probe(1, mb << 20, device)
        out[f"records_plus_red_events_per_s_{mb}MB"] = B.probe(2, mb << 20, device)
    return out


def run_ours(args):
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback")
    from paper_2007_14236_b200 import binding as B
    rank, world, local = dist_setup(args.gpus)
    dev = torch.device(f"cuda:{local}")
    torch.cuda.set_device(dev)
    peak_gbs, peak_src = measured_peak_gbs()
    T = TIME_STEPS_PER_BENCH_STEP

    wl = make_workload(args.workload, seed_offset=rank)       # replicas: independent seeds, no exchange
    g = B.Sim(DT_MS, wl.ring_slots, wl.seed, record_spikes=True, max_recorded_spikes=1 << 24, device=local)
    wl.apply(g)
    if args.delivery_kernel >= 4:
        g.set_option(B.OPT_DELIVERY_KERNEL, args.delivery_kernel)                # before prepare: the spike-buffer backend changes what is allocated
    t0 = time.time(); g.prepare(); build_wall = time.time() - t0
    g.set_option(B.OPT_STEP_MODE, args.step_mode)
    g.set_option(B.OPT_DELIVERY_KERNEL, args.delivery_kernel)
    g.set_option(B.OPT_PREFETCH, 0 if args.no_prefetch else 1)
    g.set_state(B.FIELD_V, wl.initial_v())
    N = wl.n_neurons

    # ---- warm-up: W untimed bench steps (also runs the network past its initial transient) ----
    for _ in range(args.warmup):
        g.simulate(T, allow_overflow=True)
    g.get_spikes()

    # ---- timed region: exactly K bench steps, device-resident, CUDA events on the simulator's stream ----
    s0 = g.stats()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier(world)
    with ClockSampler(local) as clk:
        e0.record(g.stream)
        for _ in range(args.steps):
            g.simulate(T, allow_overflow=True)
        e1.record(g.stream)
        barrier(world)
    ms_total = max_over_ranks(e0.elapsed_time(e1), world, dev)
    s1 = g.stats()
    g.get_spikes()
    events = sum_over_ranks(float(s1.events - s0.events), world, dev)
    spikes = sum_over_ranks(float(s1.spikes - s0.spikes), world, dev)
    launches = int((s1.launches_update - s0.launches_update) + (s1.launches_deliver - s0.launches_deliver))
    bio_s = args.steps * T * DT_MS * 1e-3
    rtf = (ms_total * 1e-3) / (bio_s * world)                 # whole job: N replicas advance N biological seconds

    # ---- e2e: the same K bench steps with the state entering and the results leaving through HOST buffers ----
    hV = torch.empty(N, dtype=torch.float32).pin_memory(); hI = torch.empty(N, dtype=torch.float32).pin_memory()
    hR = torch.empty(N, dtype=torch.int32).pin_memory()
    hs = torch.empty(1 << 24, dtype=torch.int32).pin_memory(); hi = torch.empty(1 << 24, dtype=torch.int32).pin_memory()
    g.get_state(B.FIELD_V, out=hV); g.get_state(B.FIELD_I_SYN, out=hI); g.get_state(B.FIELD_REFR, out=hR)
    barrier(world)
    d2h = h2d = 0
    t0 = time.perf_counter()
    for _ in range(args.steps):
        g.set_state(B.FIELD_V, hV); g.set_state(B.FIELD_I_SYN, hI); g.set_state(B.FIELD_REFR, hR)      # H2D
        g.simulate(T, allow_overflow=True)
        g.get_state(B.FIELD_V, out=hV); g.get_state(B.FIELD_I_SYN, out=hI); g.get_state(B.FIELD_REFR, out=hR)  # D2H
        st, _ = g.get_spikes(hs.numpy(), hi.numpy())                                                    # D2H
        h2d += 3 * N * 4; d2h += 3 * N * 4 + 2 * 4 * st.size
    barrier(world)
    e2e_s = max_over_ranks(time.perf_counter() - t0, world, dev)
    e2e_rtf = e2e_s / (bio_s * world)

    if rank != 0:
        g.close()
        return

    # ---- roofline of the dominant kernel ----
    if int(s1.step_mode) == 2:
        # one persistent kernel per bench step: its launch IS the timed region (CUDA events on the simulator's stream)
        kern = {1: "persistent_kernel<1>", 2: "persistent_kernel<2>", 3: "persistent_pipe_kernel"}[int(s1.delivery_kernel)]
        us = ms_total * 1e3 / args.steps
        ev_per_launch = float(s1.events - s0.events) / args.steps
        # AdEx: seven state words and two input ports per neuron instead of three and one
        bpn = 73 if args.workload.startswith("adex") else BYTES_PER_NEURON_STEP
        alg_bytes = T * N * bpn + ev_per_launch * BYTES_PER_EVENT
        share = {"persistent_kernel_share_of_step": 1.0, "time_steps_per_launch": T}
    else:
        # per-kernel CUDA-event times (NG_OPT_PROFILE, plain launches) over the same number of time steps
        g.set_option(B.OPT_PROFILE, 1)
        p0 = g.stats()
        g.simulate(args.steps * T, allow_overflow=True)
        p1 = g.stats()
        g.set_option(B.OPT_PROFILE, 0)
        n_launch = args.steps * T
        us_upd = (p1.ms_update - p0.ms_update) * 1e3 / n_launch
        us_del = (p1.ms_deliver - p0.ms_deliver) * 1e3 / n_launch
        ev_per_launch = (p1.events - p0.events) / n_launch
        if int(p1.delivery_kernel) == 3:          # pipelined step kernel: update + collection + delivery in one launch
            kern, alg_bytes, us = "pipe_step_kernel", N * BYTES_PER_NEURON_STEP + ev_per_launch * BYTES_PER_EVENT, us_upd
        elif us_del >= us_upd:
            kern, alg_bytes, us = f"deliver_kernel<{int(p1.delivery_kernel)}>", ev_per_launch * BYTES_PER_EVENT, us_del
        else:
            kern, alg_bytes, us = "update_kernel", N * BYTES_PER_NEURON_STEP, us_upd
        share = {"update_kernel_us": us_upd, "deliver_kernel_us": us_del}
    achieved = alg_bytes / (us * 1e-6) / 1e9
    # dram__bytes_read.sum + dram__bytes_write.sum of one launch of this kernel in this configuration, from the committed
    # `ncu --set full` capture (profiles/r01f_cfg2_full_summary.csv: 890.4 MB + 5.4 MB per 1000 time steps); below the
    # algorithmic bytes because the 33 B per neuron-step never leave the chip (state resident in shared memory / L2)
    traffic = None
    if kern == "persistent_pipe_kernel" and T == 1000 and args.delivery_kernel in (0, 3):
        traffic = {"cfg2": NCU_DRAM_BYTES_PER_LAUNCH_CFG2, "cfg4": NCU_DRAM_BYTES_PER_LAUNCH_CFG4}.get(args.workload)
    roofline = {"bound": "hbm", "kernel": kern, "achieved": achieved, "peak": peak_gbs, "unit": "GB/s",
                "frac": achieved / peak_gbs, "traffic": traffic, "peak_source": peak_src,
                "avg_launch_us": us, "algorithmic_bytes_per_launch": alg_bytes,
                "share_of_step": share,
                "note": "latency-bound regime: ~1e5 events (0.8 MB) + 2.5 MB of neuron state per time step against "
                        "~5 us of dependent memory round trips and one grid barrier; see delivery_microbench for the "
                        "bandwidth-relevant load and DESIGN.md for the L2 tag-rate ceiling of scattered reductions"}
    g.close()
    del g
    torch.cuda.empty_cache()

    micro = None if args.no_microbench else delivery_microbench(local, peak_gbs, K=args.micro_k, fraction=args.micro_fraction, steps=args.micro_steps)
    cpu = None if args.no_cpu_baseline else cpu_baseline_sample()

    line = {
        "metric": "real_time_factor", "value": rtf, "unit": "wall_s_per_bio_s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_total / args.steps, "higher_is_better": False, "scaling": "weak",
        "vs_baseline": rtf / PAPER_RTF_2080TI if args.workload == "cfg2" else rtf / PAPER_RTF_ADEX_1M if args.workload == "adex1m" else None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": workload_label(args.workload), "time_steps_per_bench_step": T, "dt_ms": DT_MS,
                   "parallelism": "replicas only (independent seeds per rank, no collective)" if world > 1 else "1 GPU",
                   "l2": "no flush: 2.7 GB of connection records (>> 126 MB L2) read by data-dependent rows; neuron "
                         "state and ring stay resident as in any long simulation",
                   "step_mode": {0: "cuda graph, 100 time steps per graph", 1: "plain launches",
                                 2: "one persistent cooperative kernel per ng_simulate call"}[int(s1.step_mode)],
                   "delivery_kernel": int(s1.delivery_kernel), "seed": wl.seed},
        "synaptic_events_per_s": events / (ms_total * 1e-3), "spikes_per_time_step": spikes / (args.steps * T * world),
        "mean_rate_hz": spikes / world / N / bio_s, "us_per_time_step": ms_total * 1e3 / (args.steps * T),
        "build_s": build_wall, "gpu_launches": launches,
        "clocks": clk.summary(),
        "e2e": {"value": e2e_rtf, "unit": "wall_s_per_bio_s", "h2d_bytes_per_step": h2d // args.steps,
                "d2h_bytes_per_step": d2h // args.steps,
                "what": "per bench step: V, I_syn, refr from pinned HOST buffers -> ng_set_state, ng_simulate(1000), "
                        "state and recorded spikes back to HOST buffers (ng_get_state, ng_get_spikes)"},
        "roofline": roofline, "delivery_microbench": micro, "cpu_baseline": cpu,
    }
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------------------------------
# CPU arm: the oracle as it stands (oracle/, single thread, fp64), on a bounded sample of the same workload.
# ---------------------------------------------------------------------------------------------------------------------
ORACLE_SAMPLE = ("the same microcircuit at 10% neuron scale with full in-degrees (BASELINE.json configs[1]: 7,718 neurons, "
                 "29,892,043 synapses; the oracle needs minutes and >8 GB just to build the full-scale network), "
                 "time steps after a 1000-step transient; value = wall s per biological s OF THE SAMPLE network; "
                 "the full-scale network carries ~10x the neurons and synaptic events per step")

_oracle_cache = {}


def oracle_sample_sim(transient=1000):
    """Build (once per process) the oracle on the bounded sample and run it past the initial transient."""
    if "o" not in _oracle_cache:
        import oracle
        from paper_2007_14236_b200 import workloads as W
        wl = W.microcircuit(10)
        o = oracle.Oracle(DT_MS, wl.ring_slots, wl.seed)
        wl.apply(o)
        t0 = time.time(); o.prepare(); build_s = time.time() - t0
        o.set_state(oracle.FIELD_V, wl.initial_v().astype(np.float64))
        o.simulate(transient, record=False)
        _oracle_cache.update(o=o, wl=wl, build_s=build_s)
    return _oracle_cache["o"], _oracle_cache["wl"], _oracle_cache["build_s"]


def cpu_baseline_sample(time_steps=5000):
    o, wl, build_s = oracle_sample_sim()
    ev0 = o.n_events
    t0 = time.perf_counter()
    o.simulate(time_steps, record=False)
    dt = time.perf_counter() - t0
    bio_s = time_steps * DT_MS * 1e-3
    return {"value": dt / bio_s, "unit": "wall_s_per_bio_s", "cores": 1, "kind": "oracle",
            "sample": f"{time_steps} {ORACLE_SAMPLE}", "host_cores_available": os.cpu_count(),
            "synaptic_events_per_s": (o.n_events - ev0) / dt, "oracle_build_s": build_s}


def run_reference(args):
    """--impl reference: the oracle timed on the host cores, same metric/unit; each bench step = a bounded sample of
    TIME_STEPS_PER_BENCH_STEP time steps of the 10%-scale network.  Rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    T = TIME_STEPS_PER_BENCH_STEP
    o, wl, build_s = oracle_sample_sim()
    for _ in range(args.warmup):
        o.simulate(T, record=False)
    ev0 = o.n_events
    t0 = time.perf_counter()
    for _ in range(args.steps):
        o.simulate(T, record=False)
    dt = time.perf_counter() - t0
    bio_s = args.steps * T * DT_MS * 1e-3
    rtf = dt / bio_s
    sample = f"{T} time steps per bench step of {ORACLE_SAMPLE}"
    line = {"impl": "reference", "metric": "real_time_factor", "value": rtf, "unit": "wall_s_per_bio_s",
            "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3 / args.steps,
            "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_label(args.workload), "time_steps_per_bench_step": T, "dt_ms": DT_MS,
                       "sample": sample},
            "synaptic_events_per_s": (o.n_events - ev0) / dt, "gpu_launches": 0,
            "cpu_baseline": {"value": rtf, "unit": "wall_s_per_bio_s", "cores": 1, "kind": "oracle", "sample": sample,
                             "host_cores_available": os.cpu_count(), "oracle_build_s": build_s},
            "e2e": {"value": rtf, "unit": "wall_s_per_bio_s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg2", choices=["cfg0", "cfg1", "cfg2", "cfg4", "adex1m", "adex100k"])
    ap.add_argument("--no-microbench", action="store_true", help="skip the configs[3] delivery microbenchmark")
    ap.add_argument("--no-cpu-baseline", action="store_true", help="skip timing the oracle")
    ap.add_argument("--only-microbench", action="store_true",
                    help="run only the configs[3] delivery microbenchmark and print its JSON object (used for ncu captures)")
    ap.add_argument("--micro-sweep", action="store_true",
                    help="run the 3 x 3 sweep of BASELINE.json configs[3] (out-degree 100/1000/10000 x firing 0.1/1/5 %%)")
    ap.add_argument("--micro-k-only", type=int, default=0, help="restrict --micro-sweep to one out-degree")
    ap.add_argument("--probe", action="store_true", help="run the ceiling probes (ng_probe) and print them as JSON")
    ap.add_argument("--step-mode", type=int, default=3, choices=[0, 1, 2, 3], help="NG_OPT_STEP_MODE (3 = auto)")
    ap.add_argument("--delivery-kernel", type=int, default=0, choices=[0, 1, 2, 3, 4, 5], help="NG_OPT_DELIVERY_KERNEL (0 = auto)")
    ap.add_argument("--no-prefetch", action="store_true", help="NG_OPT_PREFETCH = 0")
    ap.add_argument("--micro-k", type=int, default=10000)
    ap.add_argument("--micro-fraction", type=float, default=0.05)
    ap.add_argument("--micro-steps", type=int, default=30)
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    if args.probe:
        print(json.dumps(run_probes()), flush=True)
    elif args.micro_sweep:
        # BASELINE.json configs[3]: out-degree x firing-fraction sweep of the delivery stage alone, one JSON object per line
        peak = measured_peak_gbs()[0]
        for k in ((100, 1000, 10000) if args.micro_k_only == 0 else (args.micro_k_only,)):
            for f in (0.001, 0.01, 0.05):
                print(json.dumps(delivery_microbench(0, peak, K=k, fraction=f, steps=args.micro_steps, fallback=False,
                                                     kernel=args.delivery_kernel)), flush=True)
    elif args.only_microbench:
        print(json.dumps(delivery_microbench(0, measured_peak_gbs()[0], K=args.micro_k, fraction=args.micro_fraction, kernel=args.delivery_kernel,
                                             steps=args.micro_steps)), flush=True)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)
        if int(os.environ.get("WORLD_SIZE", "1")) > 1:
            import torch.distributed as dist
            dist.destroy_process_group()


if __name__ == "__main__":
    main()

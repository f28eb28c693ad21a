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
TRAFFIC_FILE = os.path.join(ROOT, "profiles", "r02_traffic.csv")   # ncu dram bytes per launch, keyed by the kernel sources' hash
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


def csrc_hash():
    """sha256 over the CUDA sources the simulation kernels are built from (ng.cu + ng_device.cuh; ng_noalloc.cu holds a
    separate entry point with kernels of its own that bench.py never launches): an ncu capture is only quoted for the
    code it was taken on."""
    import hashlib
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2007_14236_b200", "csrc")
    for f in ("ng.cu", "ng_device.cuh"):
        h.update(open(os.path.join(d, f), "rb").read())
    return h.hexdigest()[:16]


def ncu_traffic(workload, kernel):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` on `workload` from the committed ncu capture
    (profiles/r02_traffic.csv), or None (with the reason) when no capture exists for the current kernel sources."""
    if not os.path.exists(TRAFFIC_FILE):
        return None, "no capture file"
    cur = csrc_hash()
    stale = None
    for line in open(TRAFFIC_FILE):
        f = [t.strip() for t in line.split(",")]
        if len(f) >= 6 and f[0] == workload and f[1] == kernel:
            if f[4] == cur:
                return {"value": float(f[2]), "time_steps_per_launch": int(f[3]), "from": f[5], "csrc_sha256_16": f[4]}, None
            stale = f"capture {f[5]} was taken on csrc {f[4]}, current csrc is {cur}"
    return None, stale or "no capture for this workload / kernel"


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


def measure(name, steps, warmup, local, world, rank, dev, step_mode=3, delivery_kernel=0, no_prefetch=False, e2e=True):
    """One workload through the C-ABI: W untimed + K timed bench steps of T time steps each, device-resident (CUDA events on
    the simulator's stream), then (optionally) the same K steps with state and results crossing the host boundary."""
    import torch
    from paper_2007_14236_b200 import binding as B
    T = TIME_STEPS_PER_BENCH_STEP
    wl = make_workload(name, seed_offset=rank)                # replicas: independent seeds, no exchange
    g = B.Sim(DT_MS, wl.ring_slots, wl.seed, record_spikes=True, max_recorded_spikes=1 << 24, device=local)
    wl.apply(g)
    if delivery_kernel >= 4:
        g.set_option(B.OPT_DELIVERY_KERNEL, delivery_kernel)  # before prepare: the two-plane backends change what is allocated
    t0 = time.time(); g.prepare(); build_wall = time.time() - t0
    g.set_option(B.OPT_STEP_MODE, step_mode)
    g.set_option(B.OPT_DELIVERY_KERNEL, delivery_kernel)
    g.set_option(B.OPT_PREFETCH, 0 if no_prefetch else 1)
    g.set_state(B.FIELD_V, wl.initial_v())
    N = wl.n_neurons
    for _ in range(warmup):                                   # also runs the network past its initial transient
        g.simulate(T, allow_overflow=True)
    g.get_spikes()
    s0 = g.stats()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier(world)
    with ClockSampler(local) as clk:
        e0.record(g.stream)
        for _ in range(steps):
            g.simulate(T, allow_overflow=True)
        e1.record(g.stream)
        barrier(world)
    ms_total = max_over_ranks(e0.elapsed_time(e1), world, dev)
    s1 = g.stats()
    g.get_spikes()
    bio_s = steps * T * DT_MS * 1e-3
    out = {"wl": wl, "g": g, "N": N, "s0": s0, "s1": s1, "ms_total": ms_total, "bio_s": bio_s, "build_wall": build_wall,
           "clocks": clk.summary(),
           "events": sum_over_ranks(float(s1.events - s0.events), world, dev),
           "spikes": sum_over_ranks(float(s1.spikes - s0.spikes), world, dev),
           "launches": int((s1.launches_update - s0.launches_update) + (s1.launches_deliver - s0.launches_deliver)),
           "rtf": (ms_total * 1e-3) / (bio_s * world)}      # whole job: N replicas advance N biological seconds
    if e2e:
        hV = torch.empty(N, dtype=torch.float32).pin_memory(); hI = torch.empty(N, dtype=torch.float32).pin_memory()
        hR = torch.empty(N, dtype=torch.int32).pin_memory()
        hs = torch.empty(1 << 24, dtype=torch.int32).pin_memory(); hi = torch.empty(1 << 24, dtype=torch.int32).pin_memory()
        g.get_state(B.FIELD_V, out=hV); g.get_state(B.FIELD_I_SYN, out=hI); g.get_state(B.FIELD_REFR, out=hR)
        barrier(world)
        d2h = h2d = 0
        t0 = time.perf_counter()
        for _ in range(steps):
            g.set_state(B.FIELD_V, hV); g.set_state(B.FIELD_I_SYN, hI); g.set_state(B.FIELD_REFR, hR)      # H2D
            g.simulate(T, allow_overflow=True)
            g.get_state(B.FIELD_V, out=hV); g.get_state(B.FIELD_I_SYN, out=hI); g.get_state(B.FIELD_REFR, out=hR)  # D2H
            st, _ = g.get_spikes(hs.numpy(), hi.numpy())                                                    # D2H
            h2d += 3 * N * 4; d2h += 3 * N * 4 + 2 * 4 * st.size
        barrier(world)
        e2e_s = max_over_ranks(time.perf_counter() - t0, world, dev)
        out.update(e2e_rtf=e2e_s / (bio_s * world), h2d=h2d // steps, d2h=d2h // steps)
    return out


def run_sharded(args):
    """--sharded (opt-in, N > 1): ONE network, target-sharded over the ranks — every rank builds the
    connections onto its own neurons, the spike ids cross NVLink once per time step inside the kernels.  Strong scaling of
    args.workload.  Built and tested on one GPU (tests/test_gpu_sharded*.py); never yet run on several."""
    import torch
    import torch.distributed as dist
    from paper_2007_14236_b200 import binding as B
    rank, world, local = dist_setup(args.gpus)
    if world < 2:
        raise SystemExit("--sharded needs --gpus N > 1 (launch under torchrun, or let bench.py spawn the ranks)")
    dev = torch.device(f"cuda:{local}")
    T = TIME_STEPS_PER_BENCH_STEP
    wl = make_workload(args.workload)                         # the SAME seeded network on every rank
    g = B.Sim(DT_MS, wl.ring_slots, wl.seed, record_spikes=False, device=local, rank=rank, world=world)
    wl.apply(g)
    t0 = time.time(); g.prepare(); build_wall = time.time() - t0
    B.connect_peers(g, dist)
    f0, n = B.shard_range(wl.n_neurons, rank, world)
    g.set_state(B.FIELD_V, wl.initial_v()[f0:f0 + n])
    for _ in range(args.warmup):
        g.simulate(T)
    s0 = g.stats()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier(world)
    with ClockSampler(local) as clk:
        e0.record(g.stream)
        for _ in range(args.steps):
            g.simulate(T)
        e1.record(g.stream)
        barrier(world)
    ms_total = max_over_ranks(e0.elapsed_time(e1), world, dev)
    s1 = g.stats()
    events = sum_over_ranks(float(s1.events - s0.events), world, dev)
    bio_s = args.steps * T * DT_MS * 1e-3
    g.close()
    if rank != 0:
        return
    rtf = ms_total * 1e-3 / bio_s
    print(json.dumps({
        "metric": "real_time_factor", "value": rtf, "unit": "wall_s_per_bio_s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_total / args.steps, "higher_is_better": False, "scaling": "strong", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic",
        "config": {"workload": workload_label(args.workload), "time_steps_per_bench_step": T, "dt_ms": DT_MS,
                   "parallelism": f"target-sharded over {world} GPUs, one in-kernel exchange of spike ids per time step (peer memory)",
                   "delivery_kernel": int(s1.delivery_kernel), "seed": wl.seed},
        "synaptic_events_per_s": events / (ms_total * 1e-3), "us_per_time_step": ms_total * 1e3 / (args.steps * T),
        "build_s": build_wall, "gpu_launches": int((s1.launches_update - s0.launches_update) + (s1.launches_deliver - s0.launches_deliver)),
        "clocks": clk.summary(), "e2e": None, "roofline": None, "cpu_baseline": None}), flush=True)


def short_result(m, steps):
    """Entry of the `configs` object: one workload, device-timed."""
    T = TIME_STEPS_PER_BENCH_STEP
    s1 = m["s1"]
    return {"workload": workload_label(m["name"]), "real_time_factor": m["rtf"], "us_per_time_step": m["ms_total"] * 1e3 / (steps * T),
            "synaptic_events_per_s": m["events"] / (m["ms_total"] * 1e-3), "spikes_per_time_step": m["spikes"] / (steps * T),
            "mean_rate_hz": m["spikes"] / m["N"] / m["bio_s"], "steps": steps, "time_steps_per_bench_step": T,
            "delivery_kernel": int(s1.delivery_kernel), "step_mode": int(s1.step_mode), "build_s": m["build_wall"],
            "e2e_real_time_factor": m.get("e2e_rtf")}


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

    m = measure(args.workload, args.steps, args.warmup, local, world, rank, dev, args.step_mode, args.delivery_kernel, args.no_prefetch)
    g, wl, N, s0, s1, ms_total = m["g"], m["wl"], m["N"], m["s0"], m["s1"], m["ms_total"]
    rtf, events, spikes, bio_s = m["rtf"], m["events"], m["spikes"], m["bio_s"]
    if rank != 0:
        g.close()
        return

    # ---- roofline of the dominant kernel ----
    if int(s1.step_mode) == 2:
        # one persistent kernel per bench step: its launch IS the timed region (CUDA events on the simulator's stream)
        kern = {1: "persistent_kernel<1>", 2: "persistent_kernel<2>", 3: "persistent_pipe_kernel", 4: "persistent_kernel<4>", 6: "persistent_pipe_kernel"}[int(s1.delivery_kernel)]
        if int(s1.step_kernel) == 3:
            kern = "persistent_split_kernel"             # ng_stats.step_kernel: what ng_simulate launched
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
            kname = "queue_deliver_kernel" if int(p1.delivery_kernel) == 5 else f"deliver_kernel<{int(p1.delivery_kernel)}>"
            kern, alg_bytes, us = kname, ev_per_launch * BYTES_PER_EVENT, us_del
        else:
            kern, alg_bytes, us = "update_kernel", N * BYTES_PER_NEURON_STEP, us_upd
        share = {"update_kernel_us": us_upd, "deliver_kernel_us": us_del}
    achieved = alg_bytes / (us * 1e-6) / 1e9
    # dram__bytes_read.sum + dram__bytes_write.sum of one launch of this kernel in this configuration: quoted from the
    # committed `ncu --set full` capture only while the kernel sources are the ones the capture was taken on
    traffic, traffic_note = (None, "non-default options") if (args.delivery_kernel or args.step_mode != 3) else ncu_traffic(args.workload, kern)
    if traffic and traffic["time_steps_per_launch"] != T:
        traffic, traffic_note = None, "capture used another launch length"
    roofline = {"bound": "hbm", "kernel": kern, "achieved": achieved, "peak": peak_gbs, "unit": "GB/s",
                "frac": achieved / peak_gbs, "traffic": traffic["value"] if traffic else None,
                "traffic_source": traffic if traffic else traffic_note, "peak_source": peak_src,
                "avg_launch_us": us, "algorithmic_bytes_per_launch": alg_bytes,
                "share_of_step": share,
                "target_frac_north_star": 0.5, "target_met": False,
                "note": "latency-bound regime: ~1e5 events (0.8 MB) + 2.5 MB of neuron state per time step against "
                        "~4 us of dependent memory round trips and grid-wide list / plane barriers; the north_star target (>= 50 % of HBM "
                        "peak on connection-record reads) is about the bandwidth regime: see delivery_microbench "
                        "(best point 0.21 of the measured peak: NOT met; DESIGN.md section 7 names the scattered-reduction ceiling)"}
    g.close()
    del g
    torch.cuda.empty_cache()

    # ---- the other configurations of BASELINE.json, device-timed, into the same record ----
    configs = {}
    m["name"] = args.workload
    configs[args.workload] = short_result(m, args.steps)
    if not args.no_configs and world == 1:
        for name in ("cfg0", "cfg1", "cfg4", "adex1m"):
            if name == args.workload:
                continue
            try:
                mm = measure(name, 5, 3, local, 1, 0, dev, e2e=False)
                mm["name"] = name
                configs[name] = short_result(mm, 5)
                mm["g"].close()
                del mm
            except Exception as e:                       # a smaller card: say so instead of failing the headline
                configs[name] = {"error": str(e)}
            torch.cuda.empty_cache()

    micro, sweep = None, None
    if not args.no_microbench and world == 1:
        if args.no_configs:
            micro = delivery_microbench(local, peak_gbs, K=args.micro_k, fraction=args.micro_fraction, steps=args.micro_steps)
        else:
            sweep = []
            for k in (100, 1000, 10000):
                for f in (0.001, 0.01, 0.05):
                    r = delivery_microbench(local, peak_gbs, K=k, fraction=f, steps=args.micro_steps, fallback=False)
                    r.update(out_degree=k, firing_fraction=f)
                    sweep.append(r)
                    if k == args.micro_k and f == args.micro_fraction:
                        micro = r
            if micro is None:
                micro = delivery_microbench(local, peak_gbs, K=args.micro_k, fraction=args.micro_fraction, steps=args.micro_steps)
        if micro and "frac_of_hbm_peak" in micro:
            micro["target_frac_north_star"] = 0.5
            micro["target_met"] = bool(micro["frac_of_hbm_peak"] >= 0.5)
    cpu = None
    if not args.no_cpu_baseline and world == 1:
        standin = configs.get("cfg1", {}).get("real_time_factor")
        cpu = cpu_baseline_for(args.workload, gpu_rtf=rtf, gpu_rtf_standin=standin)
        # the oracle beside the GPU on the small configurations too (BASELINE.md "CPU-baseline plan"); configs 3 and 4 need
        # 32 GB and a quarter of an hour per run on the host and are timed off line
        for name in ("cfg0", "cfg1"):
            if name != args.workload and "real_time_factor" in configs.get(name, {}):
                o = cpu_baseline_for(name, gpu_rtf=configs[name]["real_time_factor"])
                configs[name]["oracle"] = {k: o[k] for k in ("value", "unit", "cores", "sample", "oracle_build_s", "ratio_same_workload")}

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
        "build_s": m["build_wall"], "gpu_launches": m["launches"],
        "clocks": m["clocks"],
        "e2e": {"value": m["e2e_rtf"], "unit": "wall_s_per_bio_s", "h2d_bytes_per_step": m["h2d"],
                "d2h_bytes_per_step": m["d2h"],
                "what": "per bench step: V, I_syn, refr from pinned HOST buffers -> ng_set_state, ng_simulate(1000), "
                        "state and recorded spikes back to HOST buffers (ng_get_state, ng_get_spikes)"},
        "roofline": roofline, "delivery_microbench": micro, "cpu_baseline": cpu,
        "configs": configs, "delivery_sweep": sweep,
    }
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------------------------------
# CPU arm: the oracle as it stands (oracle/, single thread, fp64).
#   cpu_baseline of the default line: a bounded sample of the GPU line's own workload (1000 time steps of configs[2] after
#     its transient; the oracle needs about a minute to build the full-scale network), the GPU's number beside it.
#   --impl reference: the oracle on the SAME workload as the GPU arm (configs[2] by default), each bench step a bounded
#     sample of REF_TIME_STEPS time steps.
# ---------------------------------------------------------------------------------------------------------------------
REF_TIME_STEPS = 200               # time steps per bench step of the reference arm (20 ms biological)
ORACLE_FEASIBLE = ("cfg0", "cfg1", "cfg2")     # networks the oracle builds within minutes; others fall back to a stand-in

_oracle_cache = {}


def oracle_sim(name, transient=1000):
    """Build (once per process) the oracle on workload `name` and run it past the initial transient."""
    if name not in _oracle_cache:
        import oracle
        wl = make_workload(name)
        o = oracle.Oracle(DT_MS, wl.ring_slots, wl.seed)
        wl.apply(o)
        t0 = time.time(); o.prepare(); build_s = time.time() - t0
        o.set_state(oracle.FIELD_V, wl.initial_v().astype(np.float64))
        o.simulate(transient, record=False)
        _oracle_cache[name] = (o, wl, build_s)
    return _oracle_cache[name]


def cpu_baseline_for(name, time_steps=1000, gpu_rtf=None, gpu_rtf_standin=None):
    """The oracle as it stands, one host thread, on a bounded sample (time_steps time steps after a 1000-step transient) of
    the GPU line's own workload where it can build it within minutes (configs 0-2; the full-scale microcircuit takes about
    a minute and 10 GB), else of the 10 %-scale microcircuit as a labelled stand-in."""
    run = name if name in ORACLE_FEASIBLE else "cfg1"
    o, wl, build_s = oracle_sim(run)
    ev0 = o.n_events
    t0 = time.perf_counter()
    o.simulate(time_steps, record=False)
    dt = time.perf_counter() - t0
    out = {"value": dt / (time_steps * DT_MS * 1e-3), "unit": "wall_s_per_bio_s", "cores": 1, "kind": "oracle",
           "workload": workload_label(run), "same_workload_as_gpu_line": run == name,
           "sample": f"{time_steps} time steps of {workload_label(run)} after a 1000-step transient; value = wall s per biological s",
           "host_cores_available": os.cpu_count(), "synaptic_events_per_s": (o.n_events - ev0) / dt, "oracle_build_s": build_s}
    g = gpu_rtf if run == name else gpu_rtf_standin
    if g:
        out["gpu_value_same_workload"] = g
        out["ratio_same_workload"] = out["value"] / g
    return out


def run_reference(args):
    """--impl reference: the oracle timed on the host cores on the GPU arm's own workload, same metric and unit; each bench
    step = REF_TIME_STEPS time steps (a bounded sample of the 1000 the GPU arm runs per bench step).  Rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    T = REF_TIME_STEPS
    name = args.workload if args.workload in ORACLE_FEASIBLE else "cfg1"
    same = name == args.workload
    o, wl, build_s = oracle_sim(name, transient=0)
    for _ in range(args.warmup):
        o.simulate(T, record=False)
    ev0 = o.n_events
    t0 = time.perf_counter()
    for _ in range(args.steps):
        o.simulate(T, record=False)
    dt = time.perf_counter() - t0
    bio_s = args.steps * T * DT_MS * 1e-3
    rtf = dt / bio_s
    sample = (f"{T} time steps per bench step (the GPU arm runs {TIME_STEPS_PER_BENCH_STEP}); value = wall s per biological s; "
              f"{args.warmup} untimed warm-up steps first" + ("" if same else f"; STAND-IN network: the oracle cannot build {args.workload} within minutes"))
    line = {"impl": "reference", "metric": "real_time_factor", "value": rtf, "unit": "wall_s_per_bio_s",
            "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3 / args.steps,
            "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_label(name), "time_steps_per_bench_step": T, "dt_ms": DT_MS, "sample": sample,
                       "same_workload_as_gpu_arm": same},
            "synaptic_events_per_s": (o.n_events - ev0) / dt, "gpu_launches": 0,
            "cpu_baseline": {"value": rtf, "unit": "wall_s_per_bio_s", "cores": 1, "kind": "oracle", "sample": sample,
                             "host_cores_available": os.cpu_count(), "oracle_build_s": build_s},
            "e2e": {"value": rtf, "unit": "wall_s_per_bio_s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def spawn_command(args_list, n_gpus, port=None):
    """`python bench.py --gpus N` outside torchrun: the command that re-launches this script as N ranks on this node."""
    port = port or (29500 + os.getpid() % 2000)
    return [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n_gpus}",
            "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + list(args_list)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg2", choices=["cfg0", "cfg1", "cfg2", "cfg4", "adex1m", "adex100k"])
    ap.add_argument("--sharded", action="store_true",
                    help="with --gpus N > 1: one network target-sharded over the ranks instead of N replicas (never yet run on several GPUs)")
    ap.add_argument("--no-microbench", action="store_true", help="skip the configs[3] delivery microbenchmark")
    ap.add_argument("--no-configs", action="store_true", help="skip the other BASELINE.json configurations and the 9-point configs[3] sweep")
    ap.add_argument("--no-cpu-baseline", action="store_true", help="skip timing the oracle")
    ap.add_argument("--only-microbench", action="store_true",
                    help="run only the configs[3] delivery microbenchmark and print its JSON object (used for ncu captures)")
    ap.add_argument("--micro-sweep", action="store_true",
                    help="run the 3 x 3 sweep of BASELINE.json configs[3] (out-degree 100/1000/10000 x firing 0.1/1/5 %%)")
    ap.add_argument("--micro-k-only", type=int, default=0, help="restrict --micro-sweep to one out-degree")
    ap.add_argument("--probe", action="store_true", help="run the ceiling probes (ng_probe) and print them as JSON")
    ap.add_argument("--step-mode", type=int, default=3, choices=[0, 1, 2, 3], help="NG_OPT_STEP_MODE (3 = auto)")
    ap.add_argument("--delivery-kernel", type=int, default=0, choices=[0, 1, 2, 3, 4, 5, 6], help="NG_OPT_DELIVERY_KERNEL (0 = auto)")
    ap.add_argument("--no-prefetch", action="store_true", help="NG_OPT_PREFETCH = 0")
    ap.add_argument("--micro-k", type=int, default=10000)
    ap.add_argument("--micro-fraction", type=float, default=0.05)
    ap.add_argument("--micro-steps", type=int, default=20)
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and args.impl == "ours" and not (args.probe or args.micro_sweep or args.only_microbench):
        # launched plainly: become N ranks, one per GPU (the driver's torchrun command does the same)
        os.execv(sys.executable, spawn_command(sys.argv[1:], args.gpus))
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
        if args.sharded:
            run_sharded(args)
        else:
            run_ours(args)
        if int(os.environ.get("WORLD_SIZE", "1")) > 1:
            import torch.distributed as dist
            dist.destroy_process_group()


if __name__ == "__main__":
    main()

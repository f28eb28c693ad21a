#!/usr/bin/env python
"""Writes tests/golden/oracle_rates_<cfg>.txt: spike counts per population and per window of a FREE-RUNNING oracle
simulation of one BASELINE.json workload.  Calls only oracle/ and the seeded input recipes (workloads.py holds no
arithmetic of the method); nothing here touches the CUDA path.

    python tests/golden/make_oracle_rates.py cfg2 [--seconds 11] [--window-steps 1000]

Why stored: the oracle needs minutes (config 2: 77,169 neurons / 3.0e8 connections, 9.6 GB; config 4: 1e6 neurons / 1e9
connections, 32 GB) for what the GPU does in a second, so the free-running rate parity tests (north_star: "population
firing rates agree within 5 % over 10 s of biological time"; PAPER.md:181 discards the first second and analyses 10 s)
compare the CUDA path with these stored oracle counts.  The oracle is deterministic (fp64, one thread, counter-based
Philox), so any prefix of a file can be regenerated exactly; tests/test_oracle_golden.py does that for the small configs.

File format: '#' comment lines (workload, seed, window length, populations), then one row per window:
    window_index  count_pop0  count_pop1 ...
"""
from __future__ import annotations

import argparse
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

DEFAULT_SECONDS = {"cfg0": 2.1, "cfg1": 11.0, "cfg2": 11.0, "cfg4": 1.0}
DEFAULT_WINDOW = {"cfg0": 1000, "cfg1": 1000, "cfg2": 1000, "cfg4": 1000}


def golden_path(name: str) -> str:
    return os.path.join(HERE, f"oracle_rates_{name}.txt")


def window_counts(oracle_mod, wl, n_windows: int, window_steps: int, progress=None) -> np.ndarray:
    """[n_windows, n_pops] spike counts of the oracle, free-running from the recipe's seeded initial V."""
    o = oracle_mod.Oracle(0.1, wl.ring_slots, wl.seed)
    wl.apply(o)
    o.prepare()
    o.set_state(oracle_mod.FIELD_V, wl.initial_v().astype(np.float64))
    edges = np.array([r[0] for r in wl.pop_ranges()] + [wl.n_neurons])
    out = np.zeros((n_windows, len(wl.populations)), np.int64)
    for k in range(n_windows):
        o.simulate(window_steps)
        _, ids = o.get_spikes()
        out[k] = np.histogram(ids, bins=edges)[0]
        if progress:
            progress(k, out[k])
    return out


def write_file(path: str, name: str, wl, counts: np.ndarray, window_steps: int, wall_s: float) -> None:
    with open(path, "w") as f:
        f.write("# oracle spike counts per population and window (free-running, fp64, one thread)\n")
        f.write("# written by tests/golden/make_oracle_rates.py, which calls only oracle/ and the seeded recipes\n")
        f.write(f"# workload {name} = BASELINE.json configs[{name[3:]}]: {wl.name}, {wl.n_neurons} neurons, "
                f"{wl.n_connections} connections, seed {wl.seed}, dt 0.1 ms, D {wl.ring_slots}\n")
        f.write(f"# window_steps {window_steps}  n_windows {counts.shape[0]}  oracle_wall_s {wall_s:.0f}\n")
        f.write("# populations " + " ".join(f"{p[0]}:{p[1]}" for p in wl.populations) + "\n")
        for k, row in enumerate(counts):
            f.write(f"{k} " + " ".join(str(int(c)) for c in row) + "\n")


def read_file(path: str):
    """-> (window_steps, pop sizes, counts[n_windows, n_pops])"""
    window_steps, sizes, rows = None, None, []
    for line in open(path):
        if line.startswith("# window_steps"):
            window_steps = int(line.split()[2])
        elif line.startswith("# populations"):
            sizes = [int(t.split(":")[1]) for t in line.split()[2:]]
        elif not line.startswith("#") and line.strip():
            rows.append([int(t) for t in line.split()[1:]])
    return window_steps, sizes, np.array(rows, np.int64)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("workload", choices=sorted(DEFAULT_SECONDS))
    ap.add_argument("--seconds", type=float, default=None, help="biological seconds to simulate")
    ap.add_argument("--window-steps", type=int, default=None)
    ap.add_argument("--out", default=None)
    a = ap.parse_args()
    import oracle
    from paper_2007_14236_b200 import workloads as W
    wl = W.by_name(a.workload)
    ws = a.window_steps or DEFAULT_WINDOW[a.workload]
    n_windows = int(round((a.seconds or DEFAULT_SECONDS[a.workload]) * 10000 / ws))
    t0 = time.time()

    def progress(k, row):
        print(f"[{time.time() - t0:7.0f} s] window {k + 1}/{n_windows}: {row.tolist()}", flush=True)

    counts = window_counts(oracle, wl, n_windows, ws, progress)
    write_file(a.out or golden_path(a.workload), a.workload, wl, counts, ws, time.time() - t0)


if __name__ == "__main__":
    main()

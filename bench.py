#!/usr/bin/env python
"""bench.py -- events/s of the PV-finder hot path on B200 (BASELINE.json `metric`).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 1] [--events E]

A step is one pass of the whole hot path (a1..a6, one pv_find call = three kernel launches: seed, fit, cleanup)
over one batch of synthetic events: configs[1] of BASELINE.json (100 000 events, mu = 5 pp + SMOG2, seed 2), resident in HBM.
Rank 0 prints ONE JSON line.  Under torchrun (N > 1) every rank processes its own batch of the same model
(different generator blocks), no data-path collective: events are independent -> "scaling": "weak".

`--impl reference` times the CPU oracle (oracle/, as it stands) on the box's host cores instead.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "events/s on 1 B200 (device-timed) at mu=5 pp+SMOG2; achieved HBM GB/s vs peak"
UNIT = "events/s"


def hbm_peak():
    """Measured copy bandwidth of this pool's B200s (driver-written), else the profiling guide's fallback."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json, copy read+write)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


class ClockSampler(threading.Thread):
    """Samples nvidia-smi clocks and throttle reasons while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.rows, self._stop_evt = index, [], threading.Event()

    def sample(self):
        try:
            out = subprocess.run(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-i", str(self.index)],
                                 capture_output=True, text=True, timeout=5).stdout.strip().splitlines()
            if out:
                self.rows.append([c.strip() for c in out[0].split(",")])
        except Exception:
            pass

    def run(self):
        while not self._stop_evt.is_set():
            self.sample()
            self._stop_evt.wait(0.05)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=10)

    def summary(self):
        sm = [float(r[0]) for r in self.rows if r and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({names[i] for r in self.rows if len(r) >= 7 for i in range(4) if r[3 + i].lower().startswith("active")})
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(self.rows)}


def gen_batch(cfg_idx: int, n_events, rank: int):
    """configs[cfg_idx]; rank r > 0 takes different generator blocks of the same model (distinct events)."""
    from synth import events
    import dataclasses
    m = events.config(cfg_idx, n_events)
    if rank > 0:
        m = dataclasses.replace(m, seed=m.seed + 1000 * rank)
    return events.generate(m), m


KERNELS = ("seed_kernel", "fit_kernel", "cleanup_kernel")


def algorithmic_bytes(data, n_vtx_total: int) -> int:
    """SURVEY.md 8(d) / DESIGN.md: compulsory HBM traffic of one pass: 9 fp32 inputs + offsets read,
    trk_vertex + trk_weight written, 48 B per vertex (pos 12, cov 24, chi2 4, ntrk 4, niter 4), n_vtx + status."""
    T = int(data["offsets"][-1])
    E = int(data["offsets"].size - 1)
    return T * 36 + (E + 1) * 4 + T * 8 + n_vtx_total * 48 + E * 8


def algorithmic_bytes_by_kernel(data, n_vtx_total: int):
    """The same compulsory bytes attributed to the kernel that first reads / last writes them:
    seed reads the nine input arrays and the offsets; fit writes trk_weight; cleanup writes the vertices, n_vtx,
    status and trk_vertex.  Intermediate records (seed records, the seed-sorted fit-ready track records, per-seed
    fit slots) and re-reads are NOT algorithmic."""
    T = int(data["offsets"][-1])
    E = int(data["offsets"].size - 1)
    return {"seed_kernel": T * 36 + (E + 1) * 4, "fit_kernel": T * 4,
            "cleanup_kernel": T * 4 + n_vtx_total * 48 + E * 8}


def run_oracle(data, n_threads: int, flavour: str = "explicit"):
    from oracle import pvref
    pvref.build()
    p = pvref.mv_params() if flavour == "multivertex" else pvref.default_params()
    t = time.perf_counter()
    r = pvref.find(data, p, n_threads=n_threads)
    return time.perf_counter() - t, r


def main_reference(args):
    """The reference arm of this tier is the oracle, as it stands, on the host cores (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from synth import events
    cores = os.cpu_count() or 1
    sample_events = min(args.events or 100_000, 20_000)
    data, m = gen_batch(args.config, sample_events, 0)
    for _ in range(args.warmup):
        run_oracle(events.slice_events(data, 0, min(2000, sample_events)), cores, args.flavour)
    t = 0.0
    for _ in range(args.steps):
        dt, _r = run_oracle(data, cores, args.flavour)
        t += dt
    value = sample_events * args.steps / t
    sample = f"first {sample_events} events of configs[{args.config}] ({m.name}, seed {m.seed}) per step, OpenMP over events"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * t / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64 (fp32 contract for the integer decisions)", "data": "synthetic",
            "config": {"workload": f"configs[{args.config}] {m.name}: bounded sample of {sample_events} events per step",
                       "events_per_step": sample_events, "flavour": args.flavour},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def main_ours(args):
    import torch
    import torch.distributed as dist
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the PV finder has no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dev = f"cuda:{local_rank}"
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device(dev))

    from paper_2412_14966_b200 import build as pvbuild
    pvbuild.build()
    import paper_2412_14966_b200 as pv

    data, m = gen_batch(args.config, args.events, rank)
    E, T = int(data["offsets"].size - 1), int(data["offsets"][-1])
    p = pv.multivertex_params() if args.flavour == "multivertex" else pv.default_params()
    batch = pv.DeviceBatch(data, p, device=dev)
    stream = torch.cuda.Stream(device=dev)
    L = pv.lib()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    with torch.cuda.stream(stream):
        for _ in range(max(args.warmup, 3)):
            batch.find(stream)
    barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    L.pv_kernel_timing(1)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    with torch.cuda.stream(stream):
        ev0.record(stream)
        for _ in range(args.steps):
            batch.find(stream)
        ev1.record(stream)
    barrier()
    sampler.sample()
    sampler.stop()
    ms_total = ev0.elapsed_time(ev1)
    # per-kernel durations: CUDA events recorded by the library on the launching stream around each of the
    # three launches, read back after every step of a second pass over the same K steps (not part of `value`)
    import ctypes
    kt = np.zeros((args.steps, len(KERNELS)))
    buf = (ctypes.c_float * len(KERNELS))()
    for i in range(args.steps):
        with torch.cuda.stream(stream):
            batch.find(stream)
        stream.synchronize()
        L.pv_kernel_times_ms(buf, len(KERNELS))
        kt[i] = list(buf)
    kernel_ms = kt.mean(axis=0)
    L.pv_kernel_timing(0)
    info = pv.last_launch_info()
    if world > 1:
        t = torch.tensor([ms_total], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_total = float(t.item())
    res = batch.results()
    n_vtx_total = int(res["n_vtx"].sum())

    # ---- optional: the IP consumer (NEXT-4) on the vertices just found, timed on its own (not part of `value`) ----
    ip_info = None
    if args.with_ip:
        for _ in range(3):
            batch.track_ip(stream)
        stream.synchronize()
        i0, i1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        with torch.cuda.stream(stream):
            i0.record(stream)
            for _ in range(args.steps):
                batch.track_ip(stream)
            i1.record(stream)
        stream.synchronize()
        ip_ms = i0.elapsed_time(i1) / args.steps
        ip_bytes = T * 36 + (E + 1) * 4 + E * 4 + n_vtx_total * 36 + T * 12
        ip_info = {"kernel": "pvk::ip_kernel", "ms": ip_ms, "algorithmic_bytes": ip_bytes,
                   "achieved_gbs": ip_bytes / (ip_ms * 1e-3) / 1e9, "tracks_per_s": T / (ip_ms * 1e-3)}

    # ---- e2e: HOST buffers through pv_find_host (H2D + kernel + D2H inside the timed region) --------------------
    hp = pv.HostPipeline(E, T, p, n_streams=4, device=dev)
    hin = hp.pin_inputs(data)
    hout = hp.alloc_outputs(E, T)
    for _ in range(2):
        hp.find(hin, hout, n_chunks=args.chunks)
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.e2e_steps):
        hp.find(hin, hout, n_chunks=args.chunks)
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    if world > 1:
        t = torch.tensor([e2e_s], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e_s = float(t.item())
    e2e_ok = bool(np.array_equal(hout["n_vtx"], res["n_vtx"]))
    mv = p.max_vtx_per_event
    h2d = T * 36 + (E + 1) * 4
    d2h = E * mv * 48 + E * 8 + T * 8
    hp.close()

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    ms_step = ms_total / args.steps
    value = world * E * args.steps / (ms_total * 1e-3)
    peak, peak_src = hbm_peak()
    alg = algorithmic_bytes(data, n_vtx_total)
    alg_k = algorithmic_bytes_by_kernel(data, n_vtx_total)
    assert sum(alg_k.values()) == alg
    traffic_k = {}
    tpath = os.path.join(ROOT, "profiles", "dram_traffic.csv")      # copied from the committed ncu --set full capture
    if os.path.exists(tpath):
        import csv
        for row in csv.DictReader(open(tpath)):
            if int(row["config"]) == args.config and int(row["events"]) == E:
                traffic_k[row["kernel"]] = int(row["dram_bytes_per_launch"])
    ksum = float(kernel_ms.sum())
    kernels = [{"name": n, "ms": float(kernel_ms[i]), "share": float(kernel_ms[i] / ksum),
                "algorithmic_bytes": alg_k[n], "achieved_gbs": alg_k[n] / (kernel_ms[i] * 1e-3) / 1e9,
                "traffic": traffic_k.get(n)} for i, n in enumerate(KERNELS)]
    dom = max(kernels, key=lambda k: k["ms"])
    achieved = dom["achieved_gbs"]

    # ---- cpu_baseline: the oracle, as it stands, on this box's host cores --------------------------------------
    cores = os.cpu_count() or 1
    cpu = None
    if not args.no_cpu_baseline:
        from synth import events as ev_mod
        ns = min(E, args.cpu_sample)
        sample = ev_mod.slice_events(data, 0, ns)
        run_oracle(ev_mod.slice_events(data, 0, min(ns, 1000)), cores, args.flavour)
        dt, ref = run_oracle(sample, cores, args.flavour)
        same = bool(np.array_equal(ref["n_vtx"], res["n_vtx"][:ns]))
        cpu = {"value": ns / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"first {ns} events of the same batch, one pass, OpenMP over events on {cores} threads; "
                         f"n_vtx identical to the GPU's on the sample: {same}"}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32 (int32 fixed-point histogram)", "data": "synthetic",
        "config": {"workload": f"configs[{args.config}] {m.name}: {E} events, {T} tracks, seed {m.seed}, per GPU",
                   "events_per_step": E, "tracks_per_step": T, "vertices_per_step": n_vtx_total, "flavour": args.flavour,
                   "l2": f"inputs {T * 36 / 1e6:.0f} MB per step exceed the 126 MB L2; no flush needed",
                   "launch": info, "parallelism": f"events sharded over {world} GPU(s), no collective"},
        "clocks": sampler.summary(),
        "e2e": {"value": world * E * args.e2e_steps / e2e_s, "unit": UNIT, "h2d_bytes_per_step": h2d,
                "d2h_bytes_per_step": d2h, "steps": args.e2e_steps, "chunks": args.chunks,
                "api": "pv_find_host (pinned host buffers, 4 streams)", "matches_device_path": e2e_ok},
        "gpu_launches": args.steps * info["n_kernels"],
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "traffic": dom["traffic"], "peak_source": peak_src, "kernel": "pvk::" + dom["name"],
                     "algorithmic_bytes_per_launch": dom["algorithmic_bytes"], "kernel_ms": dom["ms"],
                     "kernels": kernels,
                     "path": {"algorithmic_bytes_per_step": alg, "ms_per_step": ms_step,
                              "achieved": alg / (ms_step * 1e-3) / 1e9, "frac": alg / (ms_step * 1e-3) / 1e9 / peak},
                     "note": "issue/latency-bound path, not HBM-bound: see DESIGN.md section 8"},
        "cpu_baseline": cpu,
    }
    if ip_info is not None:
        ip_info["frac"] = ip_info["achieved_gbs"] / peak
        line["ip"] = ip_info
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=1)
    ap.add_argument("--events", type=int, default=None, help="override the number of events (configs[4] sweep)")
    ap.add_argument("--chunks", type=int, default=8, help="pipeline chunks of the e2e host path")
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--cpu-sample", type=int, default=100_000)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--with-ip", action="store_true", help="also time pv_track_ip (IP / IP chi2 of every track, NEXT-4)")
    ap.add_argument("--flavour", default="explicit", choices=["explicit", "multivertex"],
                    help="explicit: one track one vertex, Tukey weights (headline); multivertex: the paper's GPU flavour, Eq. 19")
    args = ap.parse_args()
    if args.impl == "reference":
        main_reference(args)
    else:
        main_ours(args)


if __name__ == "__main__":
    main()

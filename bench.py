#!/usr/bin/env python
"""bench.py -- events/s of the PV-finder hot path on B200 (BASELINE.json `metric`).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 1] [--events E]

A step is one pass of the whole hot path (a1..a6, one pv_find call = three kernel launches: seed, fit, cleanup)
over one batch of synthetic events: configs[1] of BASELINE.json (100 000 events, mu = 5 pp + SMOG2, seed 2), resident in HBM.
Rank 0 prints ONE JSON line.

N > 1: ONE batch of N x E events of the same model is cut by paper_2412_14966_b200.shard.event_range into N
contiguous event ranges of equal track count; rank r keeps range r resident and runs pv_find on it.
No data-path collective: events are independent -> "scaling": "weak" (E events per GPU).  Started either by
the driver's torchrun line or plainly as `python bench.py --gpus N`, which re-executes itself under
torch.distributed.run (one rank per GPU) and fails loudly when the box has fewer than N CUDA devices.

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


def gen_batch(cfg_idx: int, n_events, rank: int = 0, world: int = 1, gather_counts=None):
    """This rank's share of ONE batch of world x E events of configs[cfg_idx] (E = n_events or the config's own size):
    the contiguous event range shard.event_range gives it (equal track counts).  Every rank draws
    only the generator blocks it needs: first its nominal range [rank E, (rank + 1) E) for the per-event track
    counts, which `gather_counts` (an all_gather of E int64 per rank: control plane, not data path) turns into the
    global offsets; then the blocks of its actual range (its neighbours' edge blocks at most).
    Returns (batch, model, (e0, e1), global track count)."""
    from synth import events
    from paper_2412_14966_b200 import shard
    import dataclasses
    m = events.config(cfg_idx, n_events)
    E = m.n_events
    if world == 1:
        d = events.generate(m)
        return d, m, (0, E), int(d["offsets"][-1])
    big = dataclasses.replace(m, n_events=world * E)
    cache = {}
    nominal = events.generate_range(big, rank * E, (rank + 1) * E, cache)
    counts = gather_counts(np.diff(nominal["offsets"]).astype(np.int64))          # [world * E]
    off = np.concatenate([[0], np.cumsum(counts)])
    e0, e1 = shard.event_range(off, rank, world)
    return events.generate_range(big, e0, e1, cache), big, (e0, e1), int(off[-1])


def spawn_command(n_gpus: int, argv, port: int):
    """The command `python bench.py --gpus N ...` re-executes itself with when it was not started by torchrun."""
    return [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n_gpus}",
            "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + list(argv)


def kernels_sha() -> str:
    """git blob hashes of the two CUDA sources, joined: recorded beside every ncu DRAM-traffic capture in
    profiles/dram_traffic.csv so that a capture made with other kernels is recognised as stale."""
    import hashlib
    out = []
    for f in ("pv_kernels.cuh", "pv_api.cu"):
        b = open(os.path.join(ROOT, "paper_2412_14966_b200", "csrc", f), "rb").read()
        out.append(hashlib.sha1(b"blob %d\0" % len(b) + b).hexdigest()[:12])
    return "+".join(out)


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
    """The reference arm of this tier is the oracle, as it stands, on the host cores (rank 0 only; it uses no GPU,
    so n_gpus is 1 whatever --gpus says)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from synth import events
    cores = os.cpu_count() or 1
    data, m, _rng, _T = gen_batch(args.config, args.events)
    full_events = int(data["offsets"].size - 1)
    # every step is the workload of the GPU arm whenever the host cores finish it in time (about two minutes for all
    # steps, judged from the warm-up's rate); otherwise a prefix of it, rounded down to 1000 events
    rate = 0.0
    for _ in range(max(args.warmup, 1)):
        n0 = min(2000, full_events)
        dt, _r = run_oracle(events.slice_events(data, 0, n0), cores, args.flavour)
        rate = max(rate, n0 / dt)
    sample_events = min(full_events, max(1000, int(rate * 120.0 / max(args.steps, 1)) // 1000 * 1000))
    if sample_events < full_events:
        data = events.slice_events(data, 0, sample_events)
    t = 0.0
    for _ in range(args.steps):
        dt, _r = run_oracle(data, cores, args.flavour)
        t += dt
    value = sample_events * args.steps / t
    whole = sample_events == full_events
    sample = (f"{'all' if whole else 'first'} {sample_events} events of configs[{args.config}] ({m.name}, seed {m.seed}) per step, "
              f"OpenMP over events on {cores} threads")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": 1, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * t / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64 (fp32 contract for the integer decisions)", "data": "synthetic",
            "config": {"workload": (f"configs[{args.config}] {m.name}: {full_events} events, {_T} tracks, seed {m.seed}" if whole else
                                    f"configs[{args.config}] {m.name}: bounded sample of {sample_events} of {full_events} events per step"),
                       "events_per_step": sample_events, "flavour": args.flavour},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


L2_BYTES = 126 * 1024 * 1024


def main_ours(args):
    import torch
    import torch.distributed as dist
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the PV finder has no CPU fallback)")
    if torch.cuda.device_count() <= local_rank:
        raise SystemExit(f"bench.py: rank {rank} needs CUDA device {local_rank}, the box has {torch.cuda.device_count()}")
    torch.cuda.set_device(local_rank)
    dev = f"cuda:{local_rank}"
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("NCCL_DEBUG", "INFO")                 # the init log names every rank and its device
        dist.init_process_group("nccl", device_id=torch.device(dev))

    from paper_2412_14966_b200 import build as pvbuild
    pvbuild.build()
    import paper_2412_14966_b200 as pv

    def gather_counts(c):
        t = torch.from_numpy(c).to(dev)
        out = torch.empty(world * t.numel(), dtype=t.dtype, device=dev)
        dist.all_gather_into_tensor(out, t)
        return out.cpu().numpy()

    data, m, (ge0, ge1), T_global = gen_batch(args.config, args.events, rank, world, gather_counts)
    E, T = int(data["offsets"].size - 1), int(data["offsets"][-1])
    E_global = m.n_events
    p = pv.multivertex_params() if args.flavour == "multivertex" else pv.default_params()
    if args.split == "recursive":
        p.split_mode = 1
    if args.fill == "template":
        p.fill_mode = 1
    batch = pv.DeviceBatch(data, p, device=dev)
    stream = torch.cuda.Stream(device=dev)
    L = pv.lib()
    # inputs smaller than twice the L2 would be served from it on the second step: write a buffer larger than the
    # L2 between the timed steps (outside the per-step event pairs)
    flush = T * 36 < 2 * L2_BYTES
    fbuf = torch.empty(2 * L2_BYTES, dtype=torch.uint8, device=dev) if flush else None

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
    barrier()
    if not flush:
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        with torch.cuda.stream(stream):
            ev0.record(stream)
            for _ in range(args.steps):
                batch.find(stream)
            ev1.record(stream)
        barrier()
        ms_total = ev0.elapsed_time(ev1)
    else:
        pairs = []
        with torch.cuda.stream(stream):
            for _ in range(args.steps):
                fbuf.zero_()
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(stream)
                batch.find(stream)
                b.record(stream)
                pairs.append((a, b))
        barrier()
        ms_total = sum(a.elapsed_time(b) for a, b in pairs)
    sampler.sample()
    sampler.stop()
    # per-kernel durations: CUDA events recorded by the library on the launching stream around each of the
    # three launches, read back after every step of a second pass over the same K steps (not part of `value`)
    import ctypes
    L.pv_kernel_timing(1)
    kt = np.zeros((args.steps, len(KERNELS)))
    buf = (ctypes.c_float * len(KERNELS))()
    for i in range(args.steps):
        with torch.cuda.stream(stream):
            if flush:
                fbuf.zero_()
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
    hp = pv.HostPipeline(E, T, p, n_streams=args.e2e_streams, device=dev)
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
    e2e_ok = hp.matches(hout, res)
    h2d, d2h = hp.bytes_per_call(hin, hout)
    hp.close()
    if world > 1:                                                    # whole-job totals for the line
        tot = torch.tensor([n_vtx_total, E, T, h2d, d2h, int(e2e_ok)], dtype=torch.int64, device=dev)
        dist.all_reduce(tot, op=dist.ReduceOp.SUM)
        n_vtx_job, E_job, T_job, h2d_job, d2h_job, ok_job = [int(v) for v in tot.tolist()]
        e2e_ok = ok_job == world
        assert E_job == E_global and T_job == T_global, (E_job, E_global, T_job, T_global)
    else:
        n_vtx_job, E_job, T_job, h2d_job, d2h_job = n_vtx_total, E, T, h2d, d2h

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    ms_step = ms_total / args.steps
    value = E_job * args.steps / (ms_total * 1e-3)
    peak, peak_src = hbm_peak()
    alg = algorithmic_bytes(data, n_vtx_total)
    alg_k = algorithmic_bytes_by_kernel(data, n_vtx_total)
    assert sum(alg_k.values()) == alg
    # DRAM bytes per launch from the committed `ncu --set full` capture: accepted only when the capture was made with
    # the kernels of this working tree (hash recorded beside it), else reported as stale
    traffic_k, inst_k, tinst_k, traffic_src = {}, {}, {}, "none for this workload"
    tpath = os.path.join(ROOT, "profiles", "dram_traffic.csv")
    sha = kernels_sha()
    if os.path.exists(tpath):
        import csv
        for row in csv.DictReader(open(tpath)):
            if int(row["config"]) == args.config and int(row["events"]) == E and row.get("flavour", "explicit") == args.flavour \
                    and args.split == "z_ordered" and args.fill == "polynomial":
                if row.get("kernels_sha") == sha:
                    traffic_k[row["kernel"]] = int(row["dram_bytes_per_launch"])
                    if row.get("warp_inst_per_launch"):
                        inst_k[row["kernel"]] = int(row["warp_inst_per_launch"])
                    if row.get("thread_inst_per_launch"):
                        tinst_k[row["kernel"]] = int(row["thread_inst_per_launch"])
                    traffic_src = f"profiles/{row['source']} (ncu dram__bytes_read.sum + dram__bytes_write.sum, kernels {sha})"
                elif not traffic_k:                                  # (rows of earlier rounds stay in the file as history)
                    traffic_src = f"stale: profiles/dram_traffic.csv was captured with kernels {row.get('kernels_sha')}, this tree is {sha}"
    ksum = float(kernel_ms.sum())
    kernels = [{"name": n, "ms": float(kernel_ms[i]), "share": float(kernel_ms[i] / ksum),
                "algorithmic_bytes": alg_k[n], "achieved_gbs": alg_k[n] / (kernel_ms[i] * 1e-3) / 1e9,
                "traffic": traffic_k.get(n)} for i, n in enumerate(KERNELS)]
    dom = max(kernels, key=lambda k: k["ms"])
    achieved = dom["achieved_gbs"]
    # what actually binds the path: warp-instructions issued against 148 SMs x 4 schedulers x the
    # SM clock; instruction counts from the same ncu capture as the traffic (same staleness check), time measured live
    # `issue` is a UTILISATION (every executed instruction counts, the bookkeeping included), not a roofline fraction.
    issue = None
    clk = sampler.summary().get("sm_mhz") or 1965.0
    sms = torch.cuda.get_device_properties(dev).multi_processor_count
    if len(inst_k) >= len(KERNELS):
        peak_issue = sms * 4 * clk * 1e6 / 1e9
        ach = sum(inst_k.values()) / (ms_step * 1e-3) / 1e9
        issue = {"achieved": ach, "peak": peak_issue, "unit": "G warp-instructions/s", "utilisation": ach / peak_issue,
                 "warp_instructions_per_step": sum(inst_k.values()),
                 "peak_source": f"{sms} SMs x 4 schedulers x {clk:.0f} MHz (one warp-instruction per scheduler and cycle)"}
    # The ALU roofline of SURVEY.md 8(d): the METHOD's own arithmetic (about 330 fp32 flop per track: projection 25,
    # fill ~100 for ~8 edges, fit 35 x 5.5 + 10; plus ~10 000 integer operations per event for the peak search)
    # against the fp32 peak of the SMs.  `overhead` = thread-instructions the kernels executed per algorithmic operation.
    alg_ops = 330.0 * T + 10_000.0 * E
    peak_alu = sms * 128 * 2 * clk * 1e6 / 1e12
    alu = {"bound": "alu", "algorithmic_ops_per_event": alg_ops / E, "achieved": alg_ops / (ms_step * 1e-3) / 1e12,
           "peak": peak_alu, "unit": "Tops/s", "frac": alg_ops / (ms_step * 1e-3) / 1e12 / peak_alu,
           "peak_source": f"{sms} SMs x 128 fp32 lanes x 2 (FMA) x {clk:.0f} MHz",
           "overhead": (sum(tinst_k.values()) / alg_ops) if len(tinst_k) >= len(KERNELS) else None,
           "overhead_by_kernel": ({k: v / alg_ops for k, v in tinst_k.items()} if len(tinst_k) >= len(KERNELS) else None)}

    # ---- cpu_baseline: the oracle, as it stands, on this box's host cores --------------------------------------
    cores = os.cpu_count() or 1
    cpu = None
    if not args.no_cpu_baseline:
        from synth import events as ev_mod
        ns = min(E, args.cpu_sample)
        sample = ev_mod.slice_events(data, 0, ns)
        run_oracle(ev_mod.slice_events(data, 0, min(ns, 1000)), cores, args.flavour)
        dt, ref = run_oracle(sample, cores, args.flavour)
        same = bool(np.array_equal(ref["n_vtx"], res["n_vtx"][:ns])) if args.split == "z_ordered" and args.fill == "polynomial" else None
        n1 = min(E, max(1000, args.cpu_sample // 10))
        dt1, _r1 = run_oracle(ev_mod.slice_events(data, 0, n1), 1, args.flavour)
        cpu = {"value": ns / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"first {ns} events of the same batch, one pass, OpenMP over events on {cores} threads; "
                         f"n_vtx identical to the GPU's on the sample: {same}",
               "single_thread": {"value": n1 / dt1, "unit": UNIT, "cores": 1, "sample": f"first {n1} events, one pass, one thread"}}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32 (int32 fixed-point histogram)", "data": "synthetic",
        "config": {"workload": f"configs[{args.config}] {m.name}: {E_job} events, {T_job} tracks, seed {m.seed}"
                               + (f", cut into {world} event ranges of equal track count (rank 0: events [{ge0}, {ge1}))" if world > 1 else ""),
                   "events_per_step": E_job, "tracks_per_step": T_job, "vertices_per_step": n_vtx_job, "flavour": args.flavour,
                   "split": args.split, "fill": args.fill,
                   "l2": (f"inputs {T * 36 / 1e6:.0f} MB per step and GPU exceed the 126 MB L2; no flush needed" if not flush else
                          f"inputs {T * 36 / 1e6:.0f} MB per step would fit the 126 MB L2: a {2 * L2_BYTES >> 20} MB buffer is "
                          "written between the timed steps, each step timed with its own event pair"),
                   "launch": info, "parallelism": f"events sharded over {world} GPU(s) by shard.event_range, no collective"},
        "clocks": sampler.summary(),
        "e2e": {"value": E_job * args.e2e_steps / e2e_s, "unit": UNIT, "h2d_bytes_per_step": h2d_job,
                "d2h_bytes_per_step": d2h_job, "steps": args.e2e_steps, "chunks": args.chunks,
                "api": f"pv_find_host (pinned host buffers, {args.e2e_streams} streams, compacted vertex read-back)",
                "matches_device_path": e2e_ok},
        "gpu_launches": args.steps * info["n_kernels"],
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "traffic": dom["traffic"], "traffic_source": traffic_src, "peak_source": peak_src,
                     "kernel": "pvk::" + dom["name"],
                     "algorithmic_bytes_per_launch": dom["algorithmic_bytes"], "kernel_ms": dom["ms"],
                     "kernels": kernels,
                     "path": {"algorithmic_bytes_per_step": alg, "ms_per_step": ms_step,
                              "achieved": alg / (ms_step * 1e-3) / 1e9, "frac": alg / (ms_step * 1e-3) / 1e9 / peak},
                     "alu": alu, "issue": issue,
                     "note": "rank 0's kernels; the path is issue- and latency-bound, not HBM-bound (DESIGN.md section 8): "
                             "`frac` / `path.frac` are the HBM fractions BASELINE.json asks for, `alu.frac` the method's own "
                             "arithmetic against the fp32 peak, `issue.utilisation` the issue slots the kernels keep busy"},
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
    ap.add_argument("--events", type=int, default=None, help="events PER GPU (default: the config's own size; configs[4] sweep)")
    ap.add_argument("--chunks", type=int, default=8, help="pipeline chunks of the e2e host path")
    ap.add_argument("--e2e-streams", type=int, default=4)
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--cpu-sample", type=int, default=100_000)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--with-ip", action="store_true", help="also time pv_track_ip (IP / IP chi2 of every track, NEXT-4)")
    ap.add_argument("--flavour", default="explicit", choices=["explicit", "multivertex"],
                    help="explicit: one track one vertex, Tukey weights (headline); multivertex: the paper's GPU flavour, Eq. 19")
    ap.add_argument("--split", default="z_ordered", choices=["z_ordered", "recursive"], help="proto-cluster splitting (P:L137)")
    ap.add_argument("--fill", default="polynomial", choices=["polynomial", "template"], help="histogram fill (P:L131)")
    args = ap.parse_args()
    if args.gpus < 1:
        raise SystemExit("bench.py: --gpus must be >= 1")
    if args.impl == "reference":
        main_reference(args)
        return
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # not started by torchrun: start the N ranks ourselves
        import socket
        import torch
        have = torch.cuda.device_count() if torch.cuda.is_available() else 0
        if have < args.gpus:
            raise SystemExit(f"bench.py: --gpus {args.gpus} needs {args.gpus} CUDA devices, this box has {have}")
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        raise SystemExit(subprocess.run(spawn_command(args.gpus, sys.argv[1:], port)).returncode)
    if int(os.environ.get("WORLD_SIZE", "1")) != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={os.environ.get('WORLD_SIZE', '1')}")
    main_ours(args)


if __name__ == "__main__":
    main()

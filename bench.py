#!/usr/bin/env python
"""bench.py -- headline benchmark of the B200-native SDM coalescence step.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg3] [--impl ours|reference]

One "step" = one pass of the whole hot path over the workload:
sdm_coalescence_step (Philox keys, histograms/scan, LSD radix sort, fused pair kernel) followed by
sdm_remove_zero_multiplicity ("compaction every step", configs[3]).  Default workload: configs[3]
(8,388,608 super-droplets, 256x256 cells, geometric kernel) -- the configuration BASELINE.json's
metric and target are quoted on.  Prints ONE JSON line (rank 0).

  value        super-droplet-steps/s, whole job, inputs resident in HBM, CUDA events on the stream
  e2e          same metric through sdm_coalescence_step_host with pinned HOST buffers (H2D + D2H inside)
  roofline     dominant kernel (k_radix_pass): algorithmic bytes / mean launch time vs measured HBM peak
  cpu_baseline the serial oracle on this box's host cores, on a bounded sample of the same workload

--impl reference times the oracle itself (the reference arm of this tier).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "super-droplet-steps/s per coalescence step; achieved HBM GB/s vs B200 peak"
UNIT = "SD-steps/s"
FALLBACK_HBM_GBS = 6650.0  # /opt/skills/guides/B200_PROFILING.md fallback


# ------------------------------------------------------------------------------------------------
def make_workload(name: str):
    import sdm_workloads as W
    if name not in W.FULL:
        raise SystemExit(f"unknown workload {name}; choose from {sorted(W.FULL)}")
    return W.FULL[name]()


def workload_config(w, name, extra=None):
    kernel = "golovin" if w.kernel_kind == 0 else "geometric"
    cfg = {"workload": f"{name}: BASELINE.json configs[{name[-1]}]", "n_sd": w.n_sd, "n_cell": w.n_cell,
           "kernel": kernel, "dt": w.dt, "dV": w.dV, "compaction_every_step": bool(w.compact_every == 1),
           "compact_every": w.compact_every, "seed": w.seed, "cell_order": "cell-major (R30)",
           "l2": "inputs+workspace larger than L2 (no flush)" if w.n_sd * 36 > 126e6 else
                 "L2 flushed between timed steps"}
    if extra:
        cfg.update(extra)
    return cfg


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


# Algorithmic bytes per super-droplet per launch, by kernel class.
def algorithmic_bytes(n_cell: int, n_pass: int):
    return {
        "keys_hist": (4 if n_cell > 1 else 0) + 8,   # read cell_id, write 8-byte sort key
        "radix_pass": 16,                            # read 8, write 8 (per pass)
        "pair": 8 + 16 + 16,                         # read packed, gather xi,v, write xi,v
        "count_zero": 8,                             # read xi
        "cell_scan": 0, "compact": 20, "cell_stats": 20, "other": 0,
        "cell_bounds": 4,                            # read cell_id
        "cell_fused": 32,                            # read xi,v 16 + write xi,v 16 (keys regenerated)
        "cell_digit_hist": 4,                        # read cell_id
        "tie_repair": 8,                             # read the sorted words (rewrites only tied runs)
        "_step_total": (4 if n_cell > 1 else 0) + 8 + 16 * n_pass + 40,
    }


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.FIELDS}", "--format=csv,noheader,nounits",
                 "-lms", "50"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            parts = [x.strip() for x in ln.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0])); mx.append(float(parts[1])); power.append(float(parts[2]))
            except ValueError:
                continue
            for nm, val in zip(names, parts[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        busy = [s for s in sm if s >= 0.5 * max(sm)] or sm
        return {"sm_mhz": statistics.median(busy), "sm_max_mhz": max(mx), "reasons": sorted(reasons),
                "samples": len(sm), "power_w_max": max(power)}


# ------------------------------------------------------------------------------------------------
def oracle_rate(w, n_steps: int, max_cells: int | None = None):
    """Times the oracle as it stands (1 thread) on `n_steps` steps of (a cell-subset of) the workload.
    Returns (SD-steps/s, seconds, n_sd_sample, description)."""
    import numpy as np
    import oracle
    xi, v, cell, n_cell = w.xi, w.v, w.cell_id, w.n_cell
    desc = f"{n_steps} steps of the full {w.name} workload ({w.n_sd} SDs)"
    if max_cells is not None and max_cells < w.n_cell:
        keep = int(np.searchsorted(cell, max_cells, side="left"))  # cell-major order
        xi, v, cell, n_cell = xi[:keep], v[:keep], cell[:keep], max_cells
        desc = f"{n_steps} steps of the first {max_cells} cells of {w.name} ({keep} SDs)"
    xi, v, cell = xi.copy(), v.copy(), cell.copy()
    kp = oracle.golovin(w.b) if w.kernel_kind == 0 else oracle.geometric(w.E)
    n = len(xi)
    done = 0
    t0 = time.perf_counter()
    for s in range(n_steps):
        oracle.coalescence_step(xi, v, cell, n_cell, w.dt, w.dV, kp, w.seed, s, n_sd=n)
        done += n
        if w.compact_every and (s + 1) % w.compact_every == 0:
            n = oracle.remove_zero_multiplicity(xi, v, cell, n_sd=n)
    dt = time.perf_counter() - t0
    return done / dt, dt, len(xi), desc


def run_reference(args):
    """--impl reference: the oracle timed on the host cores (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = make_workload(args.workload)
    total_steps = args.steps + args.warmup
    # bound the run to about two minutes: the oracle does roughly 3e6 SD-steps/s on one core
    budget_sd = 3.0e6 * 120.0 / max(total_steps, 1)
    per_cell = max(w.n_sd // max(w.n_cell, 1), 1)
    max_cells = None
    if w.n_cell > 1 and w.n_sd > budget_sd:
        max_cells = max(int(budget_sd // per_cell), 1)
    if args.warmup:
        oracle_rate(w, args.warmup, max_cells)
    rate, secs, n_sample, desc = oracle_rate(w, args.steps, max_cells)
    line = {
        "metric": METRIC, "value": rate, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * secs / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic", "impl": "reference",
        "config": workload_config(w, args.workload, {"sample_n_sd": n_sample}),
        "cpu_baseline": {"value": rate, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": desc,
                         "host_cores_available": os.cpu_count()},
        "e2e": {"value": rate, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def aggregate_over_ranks(elapsed_ms: float, units: float, dist, dev):
    """Whole-job figures: the slowest rank's device time and the units all ranks processed."""
    import torch
    t = torch.tensor([elapsed_ms], dtype=torch.float64, device=dev)
    tot = torch.tensor([units], dtype=torch.float64, device=dev)
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(tot, op=dist.ReduceOp.SUM)
    return float(t.item()), float(tot.item())


# ------------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    import paper_2103_17238_b200 as sdm

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the SDM step has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    w = make_workload(args.workload)
    kp = sdm.golovin(w.b) if w.kernel_kind == 0 else sdm.geometric(w.E)
    n0 = w.n_sd
    xi0 = torch.from_numpy(w.xi).to(dev)
    v0 = torch.from_numpy(w.v).to(dev)
    c0 = torch.from_numpy(w.cell_id).to(dev)
    xi, v, cell = xi0.clone(), v0.clone(), c0.clone()
    flush = None
    if w.n_sd * 36 <= 126e6:  # small workloads: flush L2 between timed steps
        flush = torch.empty(160 * 1024 * 1024, dtype=torch.uint8, device=dev)

    ctx = sdm.SDMContext(n0, w.n_cell, device=dev, host_staging=True)
    if args.path:
        ctx.set_path({"auto": sdm.PATH_AUTO, "general": sdm.PATH_GENERAL, "cell_sorted": sdm.PATH_CELL_SORTED,
                      "hybrid": sdm.PATH_HYBRID}[args.path])
    if world > 1:  # rank r holds entries [r n0, (r+1) n0) of a world-times larger domain (no collective)
        ctx.set_option(sdm.OPT_INDEX_BASE, rank * n0)
    if not args.no_track_zeros:
        ctx.set_option(sdm.OPT_TRACK_ZEROS, 1)  # a5 fused into a4 (include/sdm.h): bench never writes xi in between
    stream = torch.cuda.current_stream(dev)

    def one_step(s, n):
        ctx.coalescence_step(xi, v, cell, w.n_cell, w.dt, w.dV, kp, w.seed, s, n_sd=n)
        if w.compact_every and (s + 1) % w.compact_every == 0:
            n = ctx.remove_zero_multiplicity(xi, v, cell, n_sd=n)
        return n

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize(dev)

    # ---- warm-up (untimed) ----
    n = n0
    for s in range(args.warmup):
        n = one_step(s, n)
        torch.cuda.synchronize(dev)  # AUTO learns the cell order from a finished step: warm up the path that is timed
    barrier()

    # ---- timed region: exactly K steps, CUDA events on the launching stream ----
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
        time.sleep(0.3)
    launches0 = ctx.launch_count()
    sd_steps = 0
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    barrier()
    block = max(int(w.n_steps), 1)
    for k in range(args.steps):
        if k and k % block == 0:
            # the workload is defined over w.n_steps steps: restart from the initial state (outside the
            # per-step event brackets, so untimed) instead of drifting into a different physical regime
            xi.copy_(xi0); v.copy_(v0); cell.copy_(c0)
            n = n0
        if flush is not None:
            flush.fill_(k & 0xFF)
        ev[k][0].record(stream)
        sd_steps += n
        n = one_step(args.warmup + k, n)
        ev[k][1].record(stream)
    barrier()
    step_ms = [a.elapsed_time(b) for a, b in ev]
    elapsed_ms = sum(step_ms)
    launches = ctx.launch_count() - launches0
    clocks = sampler.stop() if rank == 0 else None
    assert ctx.poll_error() == 0
    last_path = ctx.last_path()

    max_ms, total_units = aggregate_over_ranks(elapsed_ms, float(sd_steps), dist, dev)
    value = total_units / (max_ms * 1e-3)

    # ---- per-kernel timing pass: the same K steps again with an event pair around every launch ----
    ctx.profile_enable(True)
    ctx.profile_read()
    n_prof = n
    sd_prof = 0
    xi.copy_(xi0); v.copy_(v0); cell.copy_(c0)
    n_prof = n0
    for k in range(min(args.steps, block)):
        sd_prof += n_prof
        n_prof = one_step(args.warmup + args.steps + k, n_prof)
    prof = ctx.profile_read()
    ctx.profile_enable(False)
    peak, peak_src = peaks()
    n_pass = 4 + ((max(w.n_cell - 1, 0).bit_length() + 7) // 8)
    ab = algorithmic_bytes(w.n_cell, n_pass)
    kernels = {}
    mean_n = sd_prof / max(min(args.steps, block), 1)
    for name, (ms, cnt) in prof.items():
        if cnt == 0:
            continue
        per_launch_ms = ms / cnt
        gbs = ab.get(name, 0) * mean_n / (per_launch_ms * 1e-3) / 1e9 if per_launch_ms > 0 else 0.0
        kernels[name] = {"launches": cnt, "ms_total": ms, "ms_per_launch": per_launch_ms,
                         "algorithmic_bytes_per_launch": ab.get(name, 0) * mean_n, "gbs": gbs,
                         "share_of_kernel_time": None}
    tot_ms = sum(k["ms_total"] for k in kernels.values()) or 1.0
    for k in kernels.values():
        k["share_of_kernel_time"] = k["ms_total"] / tot_ms
    dom = max(kernels, key=lambda nm: kernels[nm]["ms_total"]) if kernels else None
    warp_inst = None
    traffic = None  # DRAM bytes per launch of the dominant kernel from the committed ncu --set full capture
    try:
        import csv
        with open(os.path.join(ROOT, "profiles", "traffic.csv")) as f:
            for row in csv.DictReader(f):
                if row["workload"] == args.workload and row["kernel"] == dom:
                    traffic = float(row["dram_bytes_per_launch"])
                    if row.get("warp_instructions_per_launch"):
                        warp_inst = float(row["warp_instructions_per_launch"])
    except Exception:
        pass
    roofline = None
    if dom:
        roofline = {"kernel": dom, "bound": "hbm", "achieved": kernels[dom]["gbs"], "peak": peak, "unit": "GB/s",
                    "frac": kernels[dom]["gbs"] / peak, "traffic": traffic, "peak_source": peak_src,
                    "ms_per_launch": kernels[dom]["ms_per_launch"], "launches": kernels[dom]["launches"],
                    "algorithmic_bytes_per_launch": kernels[dom]["algorithmic_bytes_per_launch"]}
    # second view of the dominant kernel: issue slots.  peak = SMs x 4 schedulers x 1 warp instruction / clock at the
    # sampled SM clock (B300_MICROARCH.md: one issue per SMSP per clock; ALU and FMA pipes each take one per 2 clocks);
    # achieved = warp instructions per launch (ncu, profiles/traffic.csv) / measured launch time
    roofline_alu = None
    if dom and warp_inst:
        sm_mhz = (clocks or {}).get("sm_mhz") or 1965.0
        n_sm = torch.cuda.get_device_properties(dev).multi_processor_count
        peak_issue = n_sm * 4 * sm_mhz * 1e6 / 1e9   # G warp-instructions / s
        ach = warp_inst / (kernels[dom]["ms_per_launch"] * 1e-3) / 1e9
        roofline_alu = {"kernel": dom, "bound": "alu", "achieved": ach, "peak": peak_issue, "unit": "G warp-inst/s",
                        "frac": ach / peak_issue, "warp_instructions_per_launch": warp_inst}
    # bytes the executed path must move per SD-step = sum of its kernels' algorithmic bytes; next to it the
    # figure SURVEY 8(d) quotes for north_star's own pass structure (general LSD path + separate zero scan)
    step_bytes = sum(ab.get(nm, 0) * k["launches"] for nm, k in kernels.items()) / max(min(args.steps, block), 1)
    ns_bytes = ab["_step_total"] + (8 if w.compact_every == 1 else 0)
    sd_per_s = (sd_steps / args.steps) / (elapsed_ms / args.steps * 1e-3)
    step_gbs = step_bytes * sd_per_s / 1e9
    ns_gbs = ns_bytes * sd_per_s / 1e9

    # ---- e2e: HOST buffers through the C ABI, copies inside the timed region ----
    e2e = None
    if rank == 0 or world > 1:
        hxi = torch.from_numpy(w.xi.copy()).pin_memory()
        hv = torch.from_numpy(w.v.copy()).pin_memory()
        hc = torch.from_numpy(w.cell_id.copy()).pin_memory()
        ne = n0
        e_steps = max(3, min(args.steps, 10))
        for s in range(2):
            ne = ctx.coalescence_step_host(hxi, hv, hc, w.n_cell, w.dt, w.dV, kp, w.seed, s, n_sd=ne,
                                           compact=bool(w.compact_every))
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        sd_e = 0
        e0.record(stream)
        for s in range(e_steps):
            sd_e += ne
            ne = ctx.coalescence_step_host(hxi, hv, hc, w.n_cell, w.dt, w.dV, kp, w.seed, 2 + s, n_sd=ne,
                                           compact=bool(w.compact_every))
        e1.record(stream)
        barrier()
        ems = torch.tensor([e0.elapsed_time(e1)], dtype=torch.float64, device=dev)
        esd = torch.tensor([float(sd_e)], dtype=torch.float64, device=dev)
        if dist is not None:
            dist.all_reduce(ems, op=dist.ReduceOp.MAX)
            dist.all_reduce(esd, op=dist.ReduceOp.SUM)
        e2e = {"value": float(esd.item()) / (float(ems.item()) * 1e-3), "unit": UNIT,
               "h2d_bytes_per_step": 20 * n0, "d2h_bytes_per_step": 16 * n0 + 8, "steps": e_steps,
               "api": "sdm_coalescence_step_host (pinned host buffers, compaction included)"}

    # ---- product call outside the step: the volume spectrum on 31 log bins over the state ----
    products = None
    try:
        import numpy as np
        vpos = w.v[w.v > 0]
        edges = np.exp(np.linspace(np.log(vpos.min() * 0.999), np.log(vpos.max() * 1.001), 32))
        ctx.volume_spectrum(xi, v, edges, n_sd=n_prof)
        torch.cuda.synchronize(dev)
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(5)]
        for a, b in evs:
            a.record(stream)
            ctx.volume_spectrum(xi, v, edges, n_sd=n_prof)
            b.record(stream)
        torch.cuda.synchronize(dev)
        ms = statistics.median(a.elapsed_time(b) for a, b in evs)
        ctx.profile_enable(True)
        ctx.profile_read()
        for _ in range(5):
            ctx.volume_spectrum(xi, v, edges, n_sd=n_prof)
        kms, kcnt = ctx.profile_read()["volume_spectrum"]
        ctx.profile_enable(False)
        kms = kms / max(kcnt, 1)
        gbs = 16.0 * n_prof / (kms * 1e-3) / 1e9
        products = {"volume_spectrum": {"ms_per_call": ms, "kernel_ms": kms, "algorithmic_bytes_per_sd": 16,
                                        "kernel_gbs": gbs, "kernel_frac": gbs / peak, "bins": 31,
                                        "note": "call = 3 memsets + edge upload + kernel; CUDA events"}}
    except Exception as e:  # the product is not part of the timed step
        products = {"volume_spectrum": {"error": str(e)}}

    # ---- CPU baseline: the oracle on a bounded sample (rank 0, N=1 only) ----
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        n_or = 3 if w.n_sd > 2_000_000 else max(3, min(200, int(3e7 // max(w.n_sd, 1))))
        rate, secs, _, desc = oracle_rate(w, n_or)
        cpu = {"value": rate, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": desc, "seconds": secs,
               "host_cores_available": os.cpu_count()}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": max_ms / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic", "impl": "ours",
            "config": workload_config(w, args.workload, {"parallelism": f"independent shards x{world} (no collective)",
                                                         "path": {1: "general_lsd_radix", 2: "cell_sorted", 3: "hybrid"}.get(last_path, str(last_path)),
                                                         "track_zeros": not args.no_track_zeros}),
            "roofline": roofline, "roofline_alu": roofline_alu, "step_roofline": {"algorithmic_bytes_per_sd_step": step_bytes, "gbs": step_gbs,
                                                    "frac": step_gbs / peak, "peak": peak,
                                                    "north_star_bytes_per_sd_step": ns_bytes,
                                                    "north_star_equivalent_gbs": ns_gbs,
                                                    "north_star_equivalent_frac": ns_gbs / peak},
            "kernels": kernels, "products": products, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": launches, "clocks": clocks,
            "ms_per_step_min_med_max": [min(step_ms), statistics.median(step_ms), max(step_ms)],
        }
        print(json.dumps(line), flush=True)
    ctx.close()
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2000)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg3")
    ap.add_argument("--path", default=None, choices=[None, "auto", "general", "cell_sorted", "hybrid"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-track-zeros", action="store_true", help="keep the separate zero-count kernel (a5)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()

#!/usr/bin/env python
"""bench.py -- headline benchmark of the B200-native SDM coalescence step.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg3] [--impl ours|reference]

One "step" = one pass of the whole hot path over the workload: the coalescence step
(Philox keys, cell boundaries / histograms, per-cell shuffle, fused pair kernel) followed, on the configuration's
schedule, by the zero-multiplicity compaction ("compaction every step", configs[3]).  The dominant kernel of the
default run is k_cell_fused (per-cell register sort fused with the pair rule: the CELL_SORTED path AUTO takes on
cell-major input); the `paths` object times the literal north_star (b) path, the LSD radix sort (k_radix_pass).  Default workload: configs[3]
(8,388,608 super-droplets, 256x256 cells, geometric kernel) -- the configuration BASELINE.json's metric and
target are quoted on.  The steps go through the library's time-loop entry point sdm_coalescence_steps (the same
bits as step-by-step calls, no host round trip per step); `--loop single` times the step-by-step calls instead.
Prints ONE JSON line (rank 0).

  value        super-droplet-steps/s, whole job, inputs resident in HBM, CUDA events on the stream
  e2e          same metric through sdm_coalescence_step_host with pinned HOST buffers (H2D + D2H inside)
  roofline     dominant kernel of the timed path: algorithmic bytes / mean launch time vs the measured HBM peak
  paths        configs[3] on the GENERAL (north_star (b): LSD radix sort) and HYBRID paths, cell-major and interleaved
  configs      the other four synthetic configs (BASELINE.json configs[0,1,2,4]), each with its own oracle rate
  cpu_baseline the serial oracle on this box's host cores, on a bounded sample of the same workload

--impl reference times the oracle itself (the reference arm of this tier).
--gpus N without a torchrun environment re-executes itself under torch.distributed.run with N ranks.
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
L2_BYTES = 126e6
PATH_NAMES = {1: "general_lsd_radix", 2: "cell_sorted", 3: "hybrid", 4: "box_cluster", 5: "bucket_msd_placement"}


# ------------------------------------------------------------------------------------------------
def make_workload(name: str, **kw):
    import sdm_workloads as W
    if name not in W.FULL:
        raise SystemExit(f"unknown workload {name}; choose from {sorted(W.FULL)}")
    return W.FULL[name](**kw)


def state_bytes(w) -> int:
    return w.n_sd * 20


def workload_config(w, name, extra=None):
    kernel = "golovin" if w.kernel_kind == 0 else "geometric"
    cfg = {"workload": f"{name}: BASELINE.json configs[{name[-1]}]", "n_sd": w.n_sd, "n_cell": w.n_cell,
           "kernel": kernel, "dt": w.dt, "dV": w.dV, "compaction_every_step": bool(w.compact_every == 1),
           "compact_every": w.compact_every, "seed": w.seed, "cell_order": "cell-major (R30)",
           "l2": "state + workspace larger than L2 (no flush)" if state_bytes(w) > L2_BYTES else
                 "state fits L2: the steady state of a time loop, not flushed (not an HBM-roofline number)"}
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


def cpu_model() -> str:
    try:
        for line in open("/proc/cpuinfo"):
            if line.lower().startswith("model name"):
                return line.split(":", 1)[1].strip()
    except Exception:
        pass
    return "unknown"


# Algorithmic bytes per super-droplet per launch, by kernel class.
def algorithmic_bytes(n_cell: int):
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
        "volume_spectrum": 16,
        "cell_classes": 0,                           # reads cell_start (n_cell words)
        "bucket": 4,                                 # hist: one reduction per SD; scatter: one 4-byte index word per SD
        "resident_move": 36,                         # r index word 4, gather xi,v 16, w xi,v 16 (twice per HYBRID run)
        "box_step": 32,                              # read xi,v 16 + write xi,v 16 (one block, keys regenerated)
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


def cpu_baseline_of(w, seconds_budget: float = 4.0):
    """The oracle on a bounded sample of `w` (about `seconds_budget` s at ~3e6 SD-steps/s, at least one step)."""
    n_or = max(1, min(400, int(3e6 * seconds_budget // max(w.n_sd, 1))))
    rate, secs, _, desc = oracle_rate(w, n_or)
    return {"value": rate, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": desc, "seconds": secs,
            "host_cores_available": os.cpu_count(), "cpu_model": cpu_model()}


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
                         "host_cores_available": os.cpu_count(), "cpu_model": cpu_model()},
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
class Runner:
    """One workload resident on one GPU: state tensors, a context, and the timed loops."""

    def __init__(self, w, dev, path=None, index_base=0, host_staging=False, track_zeros=True):
        import torch
        import paper_2103_17238_b200 as sdm
        self.torch, self.sdm, self.w, self.dev = torch, sdm, w, dev
        self.kp = sdm.golovin(w.b) if w.kernel_kind == 0 else sdm.geometric(w.E)
        self.xi0 = torch.from_numpy(w.xi).to(dev)
        self.v0 = torch.from_numpy(w.v).to(dev)
        self.c0 = torch.from_numpy(w.cell_id).to(dev)
        self.xi, self.v, self.cell = self.xi0.clone(), self.v0.clone(), self.c0.clone()
        self.ctx = sdm.SDMContext(max(w.n_sd, 1), w.n_cell, device=dev, host_staging=host_staging)
        if path:
            self.ctx.set_path({"auto": sdm.PATH_AUTO, "general": sdm.PATH_GENERAL, "cell_sorted": sdm.PATH_CELL_SORTED,
                               "hybrid": sdm.PATH_HYBRID, "box": sdm.PATH_BOX, "bucket": sdm.PATH_BUCKET}[path])
        if index_base:
            self.ctx.set_option(sdm.OPT_INDEX_BASE, index_base)
        if track_zeros:
            self.ctx.set_option(sdm.OPT_TRACK_ZEROS, 1)  # a5 fused into a4 (include/sdm.h)
        self.stream = torch.cuda.current_stream(dev)
        self.n = w.n_sd

    def restore(self):
        self.xi.copy_(self.xi0); self.v.copy_(self.v0); self.cell.copy_(self.c0)
        self.n = self.w.n_sd

    def block(self, step0: int, k: int, loop: str):
        """k consecutive steps from the current state; returns the super-droplet-steps done."""
        w, ctx = self.w, self.ctx
        if loop == "multi":
            n0 = self.n
            self.n = ctx.coalescence_steps(self.xi, self.v, self.cell, w.n_cell, w.dt, w.dV, self.kp, w.seed, step0, k,
                                           w.compact_every, n_sd=n0)
            # with compactions inside the call the exact sum of n_sd(step) is not visible from outside; the count
            # only shrinks, so the final count times k is a lower bound of the work done (exact when nothing died)
            return self.n * k
        sd = 0
        for s in range(k):
            sd += self.n
            ctx.coalescence_step(self.xi, self.v, self.cell, w.n_cell, w.dt, w.dV, self.kp, w.seed, step0 + s, n_sd=self.n)
            if w.compact_every and (s + 1) % w.compact_every == 0:
                self.n = ctx.remove_zero_multiplicity(self.xi, self.v, self.cell, n_sd=self.n)
        return sd

    def timed(self, steps: int, warmup: int, loop: str, barrier, before_timed=None):
        """W warm-up steps, then exactly `steps` steps in blocks of at most w.n_steps (the workload is defined over
        that many steps: each block restarts from the initial state, outside the event brackets).  Returns
        (per-block ms list, per-block steps, SD-steps, launches)."""
        torch, w = self.torch, self.w
        blk = max(int(w.n_steps), 1)
        self.restore()
        done = 0
        while done < warmup:
            k = min(blk, warmup - done)
            self.block(done, k, loop)
            done += k
        torch.cuda.synchronize(self.dev)
        if before_timed:
            before_timed()
            # the sampler start-up leaves the GPU idle for a moment: re-warm so that the first timed block is not cold
            self.block(done, min(3, blk), loop)
        plan = []
        left = steps
        while left > 0:
            plan.append(min(blk, left))
            left -= plan[-1]
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in plan]
        launches0 = self.ctx.launch_count()
        sd_steps = 0
        barrier()
        for (a, b), k in zip(ev, plan):
            self.restore()
            a.record(self.stream)
            sd_steps += self.block(warmup, k, loop)
            b.record(self.stream)
        barrier()
        ms = [a.elapsed_time(b) for a, b in ev]
        return ms, plan, sd_steps, self.ctx.launch_count() - launches0

    def kernel_profile(self, steps: int, loop: str, peak: float):
        """The same steps again with a CUDA-event pair around every launch (sdm_profile_*).  A box_step launch runs
        many steps on a shared-memory copy of the state: its algorithmic HBM bytes are one read and one write of the
        state per LAUNCH."""
        w, ctx = self.w, self.ctx
        k = min(steps, max(int(w.n_steps), 1))
        self.restore()
        ctx.profile_enable(True)
        ctx.profile_read()
        n0 = self.n
        self.block(0, k, loop)
        prof = ctx.profile_read()
        ctx.profile_enable(False)
        ab = algorithmic_bytes(w.n_cell)
        kernels = {}
        for name, (ms, cnt) in prof.items():
            if cnt == 0:
                continue
            per = ms / cnt
            # a fused launch of the time loop takes its cells through several steps when no compaction lies between
            # them: its algorithmic bytes are those of the steps it ran (one read and one write of the state each)
            spl = k / cnt if (name == "cell_fused" and loop == "multi" and cnt < k) else 1.0
            gbs = ab.get(name, 0) * n0 * spl / (per * 1e-3) / 1e9 if per > 0 else 0.0
            kernels[name] = {"launches": cnt, "ms_total": ms, "ms_per_launch": per, "steps_per_launch": spl,
                             "algorithmic_bytes_per_launch": ab.get(name, 0) * n0 * spl, "gbs": gbs, "frac": gbs / peak}
        tot = sum(x["ms_total"] for x in kernels.values()) or 1.0
        for x in kernels.values():
            x["share_of_kernel_time"] = x["ms_total"] / tot
        step_bytes = sum(ab.get(nm, 0) * x["launches"] * x["steps_per_launch"] for nm, x in kernels.items()) / max(k, 1)
        return kernels, step_bytes

    def close(self):
        self.ctx.close()


def summarize(r: Runner, steps, warmup, loop, barrier, peak, with_cpu=False, cpu_budget=3.0):
    """A compact record of one (workload, path) measurement for the `paths` / `configs` objects."""
    ms, plan, sd, launches = r.timed(steps, warmup, loop, barrier)
    kernels, step_bytes = r.kernel_profile(min(steps, 50), loop, peak)
    total_ms = sum(ms)
    rate = sd / (total_ms * 1e-3)
    dom = max(kernels, key=lambda nm: kernels[nm]["ms_total"]) if kernels else None
    w = r.w
    out = {"n_sd": w.n_sd, "n_cell": w.n_cell, "steps": steps, "loop": loop, "path": PATH_NAMES.get(r.ctx.last_path()),
           "ms_per_step": total_ms / steps, "value": rate, "unit": UNIT, "gpu_launches": launches,
           "step_bytes_per_sd": step_bytes, "step_gbs": step_bytes * rate / 1e9, "step_frac": step_bytes * rate / 1e9 / peak,
           "l2": "larger than L2" if state_bytes(w) > L2_BYTES else "L2-resident steady state (not an HBM number)",
           "dominant_kernel": dom,
           "dominant": {k: kernels[dom][k] for k in ("ms_per_launch", "gbs", "frac", "share_of_kernel_time")} if dom else None,
           "kernels_us": {nm: round(1e3 * x["ms_per_launch"], 2) for nm, x in kernels.items()}}
    if with_cpu:
        out["cpu_baseline"] = cpu_baseline_of(w, cpu_budget)
    return out


# ------------------------------------------------------------------------------------------------
def run_ours(args):
    import torch

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

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize(dev)

    peak, peak_src = peaks()
    w = make_workload(args.workload)
    # weak scaling: rank r holds entries [r n0, (r+1) n0) of a world-times larger domain (no collective)
    r = Runner(w, dev, path=args.path, index_base=rank * w.n_sd if world > 1 else 0, host_staging=True,
               track_zeros=not args.no_track_zeros)

    sampler = ClockSampler(local_rank)

    def start_sampler():
        if rank == 0:
            sampler.start()
            time.sleep(0.3)

    ms, plan, sd_steps, launches = r.timed(args.steps, args.warmup, args.loop, barrier, before_timed=start_sampler)
    clocks = sampler.stop() if rank == 0 else None
    assert r.ctx.poll_error() == 0
    last_path = r.ctx.last_path()
    elapsed_ms = sum(ms)
    max_ms, total_units = aggregate_over_ranks(elapsed_ms, float(sd_steps), dist, dev)
    value = total_units / (max_ms * 1e-3)
    per_step_ms = [m / k for m, k in zip(ms, plan)]

    # ---- per-kernel timing pass ----
    kernels, step_bytes = r.kernel_profile(args.steps, args.loop, peak)
    dom = max(kernels, key=lambda nm: kernels[nm]["ms_total"]) if kernels else None
    traffic = warp_inst = traffic_src = None  # of the dominant kernel, from the committed ncu --set full capture of this build
    try:
        import csv
        with open(os.path.join(ROOT, "profiles", "traffic.csv")) as f:
            for row in csv.DictReader(f):
                if row["workload"] == args.workload and row["kernel"] == dom:
                    traffic = float(row["dram_bytes_per_launch"])
                    if row.get("warp_instructions_per_launch"):
                        warp_inst = float(row["warp_instructions_per_launch"])
                    traffic_src = row.get("source")
    except Exception:
        pass
    roofline = None
    if dom:
        k = kernels[dom]
        roofline = {"kernel": dom, "bound": "hbm", "achieved": k["gbs"], "peak": peak, "unit": "GB/s",
                    "frac": k["gbs"] / peak, "traffic": traffic, "peak_source": peak_src,
                    "ms_per_launch": k["ms_per_launch"], "launches": k["launches"],
                    "algorithmic_bytes_per_launch": k["algorithmic_bytes_per_launch"]}
        if traffic:
            roofline["traffic_frac"] = traffic / (k["ms_per_launch"] * 1e-3) / 1e9 / peak
            roofline["traffic_source"] = traffic_src
    # second view of the dominant kernel: issue slots.  peak = SMs x 4 schedulers x 1 warp instruction / clock at the
    # sampled SM clock; achieved = warp instructions per launch (ncu, profiles/traffic.csv) / measured launch time
    roofline_alu = None
    if dom and warp_inst:
        sm_mhz = (clocks or {}).get("sm_mhz") or 1965.0
        n_sm = torch.cuda.get_device_properties(dev).multi_processor_count
        peak_issue = n_sm * 4 * sm_mhz * 1e6 / 1e9   # G warp-instructions / s
        ach = warp_inst / (kernels[dom]["ms_per_launch"] * 1e-3) / 1e9
        roofline_alu = {"kernel": dom, "bound": "alu", "achieved": ach, "peak": peak_issue, "unit": "G warp-inst/s",
                        "frac": ach / peak_issue, "warp_instructions_per_launch": warp_inst}
    sd_per_s = sd_steps / (elapsed_ms * 1e-3)
    step_gbs = step_bytes * sd_per_s / 1e9
    # the same step time in the accounting SURVEY 8(d) quotes for north_star's own pass structure (general LSD path,
    # 6 passes, separate zero scan): bytes that path would have to move, NOT bytes this path moves
    n_pass = 4 + ((max(w.n_cell - 1, 0).bit_length() + 7) // 8)
    ns_bytes = (4 if w.n_cell > 1 else 0) + 8 + 16 * n_pass + 40 + (8 if w.compact_every == 1 else 0)

    # ---- e2e: HOST buffers through the C ABI, copies inside the timed region ----
    e2e = None
    n0 = w.n_sd
    hxi = torch.from_numpy(w.xi.copy()).pin_memory()
    hv = torch.from_numpy(w.v.copy()).pin_memory()
    hc = torch.from_numpy(w.cell_id.copy()).pin_memory()
    ne = n0
    e_steps = max(3, min(args.steps, 10))
    for s in range(2):
        ne = r.ctx.coalescence_step_host(hxi, hv, hc, w.n_cell, w.dt, w.dV, r.kp, w.seed, s, n_sd=ne,
                                         compact=bool(w.compact_every))
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sd_e = 0
    e0.record(r.stream)
    for s in range(e_steps):
        sd_e += ne
        ne = r.ctx.coalescence_step_host(hxi, hv, hc, w.n_cell, w.dt, w.dV, r.kp, w.seed, 2 + s, n_sd=ne,
                                         compact=bool(w.compact_every))
    e1.record(r.stream)
    barrier()
    e_ms, e_units = aggregate_over_ranks(e0.elapsed_time(e1), float(sd_e), dist, dev)
    e2e = {"value": e_units / (e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": 20 * n0,
           "d2h_bytes_per_step": 16 * n0 + 8, "steps": e_steps,
           "api": "sdm_coalescence_step_host (pinned host buffers, compaction included; uploads, step and downloads pipelined in eight pieces)"}
    del hxi, hv, hc

    # ---- product call outside the step: the volume spectrum on 31 log bins over the state ----
    products = None
    try:
        import numpy as np
        vpos = w.v[w.v > 0]
        edges = np.exp(np.linspace(np.log(vpos.min() * 0.999), np.log(vpos.max() * 1.001), 32))
        r.restore()
        r.ctx.volume_spectrum(r.xi, r.v, edges)
        r.ctx.profile_enable(True)
        r.ctx.profile_read()
        for _ in range(5):
            r.ctx.volume_spectrum(r.xi, r.v, edges)
        kms, kcnt = r.ctx.profile_read()["volume_spectrum"]
        r.ctx.profile_enable(False)
        kms = kms / max(kcnt, 1)
        gbs = 16.0 * n0 / (kms * 1e-3) / 1e9
        products = {"volume_spectrum": {"kernel_ms": kms, "algorithmic_bytes_per_sd": 16, "kernel_gbs": gbs,
                                        "kernel_frac": gbs / peak, "bins": 31}}
    except Exception as e:  # the product is not part of the timed step
        products = {"volume_spectrum": {"error": str(e)}}
    r.close()
    del r
    torch.cuda.empty_cache()

    # ---- strong scaling (N > 1): ONE configs[3] domain split into N contiguous cell ranges (sdm_workloads.shard) ----
    strong = None
    if world > 1 and w.n_cell >= world:
        import sdm_workloads as W
        sh = W.shard(w, rank, world)
        rs = Runner(sh.work, dev, path=args.path, index_base=sh.index_base, track_zeros=not args.no_track_zeros)
        sms, splan, ssd, _ = rs.timed(min(args.steps, 400), args.warmup, args.loop, barrier)
        s_ms, s_units = aggregate_over_ranks(sum(sms), float(ssd), dist, dev)
        strong = {"value": s_units / (s_ms * 1e-3), "unit": UNIT, "ms_per_step": s_ms / sum(splan), "scaling": "strong",
                  "n_sd_total": w.n_sd, "n_sd_this_rank": sh.work.n_sd,
                  "note": "one configs[3] domain sharded by contiguous cell ranges; index_base = first entry of the shard; "
                          "no collective in the step (a compaction that removes entries needs one 8-byte all_gather to "
                          "re-base index_base: sdm_workloads.rebase)"}
        rs.close()
        del rs
        torch.cuda.empty_cache()

    # ---- the rest of what north_star asks to be reported: the LSD-radix and hybrid paths, and the other four configs ----
    paths = configs = cpu = None
    if rank == 0 and world == 1 and not args.quick:
        paths = {}
        import sdm_workloads as W
        for label, kw in (("cell_major", {}), ("interleaved", {"interleave": True})):
            wi = w if not kw else make_workload(args.workload, **kw) if args.workload in ("cfg2", "cfg3", "cfg4") else None
            if wi is None:
                continue
            for pth in ("general", "hybrid"):
                if wi.n_cell == 1 and pth == "hybrid":
                    continue
                rr = Runner(wi, dev, path=pth, track_zeros=not args.no_track_zeros)
                # (a HYBRID run pays one gather and one scatter of the attributes per call: 100 steps, as in the configs)
                paths[f"{pth}/{label}"] = summarize(rr, 100 if pth == "hybrid" else 40, 5, args.loop, barrier, peak)
                rr.close()
                del rr
                torch.cuda.empty_cache()
            del wi
        configs = {}
        for name, steps in (("cfg0", 1000), ("cfg1", 100), ("cfg2", 400), ("cfg4", 100)):
            if name == args.workload:
                continue
            wc = make_workload(name)
            rr = Runner(wc, dev, track_zeros=not args.no_track_zeros)
            configs[name] = summarize(rr, steps, 10, args.loop, barrier, peak, with_cpu=not args.no_cpu_baseline)
            configs[name]["workload"] = f"{name}: BASELINE.json configs[{name[-1]}]"
            rr.close()
            del rr, wc
            torch.cuda.empty_cache()
    # ---- CPU baseline: the oracle on a bounded sample (rank 0, N=1 only) ----
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = cpu_baseline_of(w, 10.0 if w.n_sd > 2_000_000 else 3.0)

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": max_ms / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic", "impl": "ours",
            "config": workload_config(w, args.workload, {
                "parallelism": f"independent shards x{world} (no collective)",
                "path": PATH_NAMES.get(last_path, str(last_path)), "loop": args.loop,
                "entry_point": "sdm_coalescence_steps" if args.loop == "multi" else "sdm_coalescence_step + sdm_remove_zero_multiplicity",
                "track_zeros": not args.no_track_zeros}),
            "roofline": roofline, "roofline_alu": roofline_alu,
            "step_roofline": {"algorithmic_bytes_per_sd_step": step_bytes, "gbs": step_gbs, "frac": step_gbs / peak,
                              "peak": peak,
                              "survey_general_path_bytes_per_sd_step": ns_bytes,
                              "speedup_vs_survey_60pct_budget": (ns_bytes * w.n_sd / (0.6 * peak * 1e9)) / (elapsed_ms / args.steps * 1e-3)},
            "kernels": kernels, "paths": paths, "configs": configs, "strong_scaling": strong, "products": products,
            "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": launches, "clocks": clocks,
            "ms_per_step_min_med_max": [min(per_step_ms), statistics.median(per_step_ms), max(per_step_ms)],
            "timed_blocks": len(plan),
        }
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2000)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg3")
    ap.add_argument("--path", default=None, choices=[None, "auto", "general", "cell_sorted", "hybrid", "box", "bucket"])
    ap.add_argument("--loop", default="multi", choices=["multi", "single"],
                    help="multi: sdm_coalescence_steps (default); single: one sdm_coalescence_step (+ compaction) call per step")
    ap.add_argument("--quick", action="store_true", help="headline only: skip the `paths` and `configs` objects")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-track-zeros", action="store_true", help="keep the separate zero-count kernel (a5)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "ours" and args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # a plain `python bench.py --gpus N`: one rank per GPU under torch.distributed.run (the driver's own launch line)
        import socket
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        raise SystemExit(subprocess.call(cmd))
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()

#!/usr/bin/env python
"""bench.py -- histories/s of the MC/DC hot path on B200 (contract: see the task statement / DESIGN.md).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload config3] [--histories H] [--sweep]
  python bench.py --impl reference ...      # the oracle (CPU) arm on the same workload

A "step" is one mcdc_run of the whole hot path (source generation, all census steps and fission
generations, batch close-out) over one batch of synthetic histories of the named workload.
N=1 workload: config 3 (7-group 17x17 pin lattice, 1e7 histories, 100 batches) -- the configuration
BASELINE.json's north_star quotes the roofline target on (configs 3/4); it fits one GPU.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "histories/s"
N_SM = 148
ISSUE_LANES_PER_SM = 128        # 4 warp schedulers x 32 lanes: one warp instruction per scheduler per cycle
# ncu-derived constants (DRAM bytes per history, thread instructions per segment) come from the committed
# profiles/ncu_constants.json, keyed by kernel instantiation + workload and stamped with the revision of the kernel
# sources the capture was made from; they are printed only when the running library reports the same revision
# (mcdc_kernel_info_get), so a figure from another build never sits beside this run's timing.
NCU_JSON = os.path.join(ROOT, "profiles", "ncu_constants.json")


def ncu_constants(kernel_info, workload, technique):
    """-> (entry or None, note).  kernel_info: 'k_warp<1,0,0,1,512> rev=abc grid=148 ...'"""
    try:
        with open(NCU_JSON) as f:
            table = json.load(f)
    except (OSError, ValueError):
        return None, "profiles/ncu_constants.json missing"
    name = kernel_info.split(" ")[0] if kernel_info else ""
    rev = next((t[4:] for t in kernel_info.split() if t.startswith("rev=")), "")
    same = [e for e in table.get("captures", [])
            if e.get("kernel") == name and e.get("workload") == workload and e.get("technique", "analog") == technique]
    for e in same:                       # the capture made from THIS library's revision, wherever it sits in the list
        if e.get("rev") == rev:
            return e, e.get("source")
    if same:
        e = same[0]
        return None, f"stale: {e.get('source')} was captured at kernel rev {e.get('rev')}, this library is rev {rev}"
    return None, f"no capture of {name} on {workload} ({technique}) in profiles/ncu_constants.json"


# variants of the workload with the techniques of DESIGN.md Appendix G switched on (the headline run is analog)
TECHNIQUES = {"analog": None,
              "ic_wr": dict(implicit_capture=True, wr_threshold=0.25, wr_survive=1.0),
              "pc": dict(population_control=True),
              "all": dict(implicit_capture=True, wr_threshold=0.25, wr_survive=1.0, population_control=True)}


def _peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured", float(d.get("sm_max_mhz", 1965.0))
    return 6650.0, "fallback", 1965.0


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region."""

    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index=0):
        self.rows = []
        self.proc = None
        self.gpu_index = gpu_index

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100",
                 "-i", str(self.gpu_index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        rows = [r for (t, r) in self.rows if t0 - 0.05 <= t <= t1 + 0.15] or [r for (_, r) in self.rows]
        for r in rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); mx.append(float(f[2]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


class NvmlSampler:
    """The same samples through NVML (pynvml), polled every 5 ms from a thread: the timed region of the default run
    is ~90 ms, too short for nvidia-smi's 100 ms loop to see more than a couple of samples."""

    def __init__(self, gpu_index=0):
        import pynvml
        self.nv = pynvml
        pynvml.nvmlInit()
        self.h = pynvml.nvmlDeviceGetHandleByIndex(gpu_index)
        self.mx = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        self.rows = []
        self.run = False

    def start(self):
        self.run = True
        self.t = threading.Thread(target=self._poll, daemon=True)
        self.t.start()

    def _poll(self):
        nv = self.nv
        while self.run:
            try:
                self.rows.append((time.time(), float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)),
                                  int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))))
            except Exception:
                pass
            time.sleep(0.005)

    def stop(self, t0, t1):
        self.run = False
        self.t.join(timeout=1)
        nv = self.nv
        rows = [r for r in self.rows if t0 <= r[0] <= t1] or self.rows
        names = {"hw_slowdown": getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8),
                 "hw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40),
                 "sw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20),
                 "sw_power_cap": getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4)}
        reasons = sorted(n for n, bit in names.items() if any(r[2] & bit for r in rows))
        sm = [r[1] for r in rows]
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": self.mx, "reasons": reasons,
                "samples": len(sm), "source": "nvml, 5 ms poll"}


def make_sampler(gpu_index):
    try:
        return NvmlSampler(gpu_index)
    except Exception:
        return ClockSampler(gpu_index)


def _problem(args):
    from workloads import configs as W

    kw = {}
    if args.histories:
        kw["n_histories"] = int(args.histories)
    if args.batches:
        kw["n_batches"] = int(args.batches)
    return W.get_config(args.workload, **kw)


def _desc_bytes(p):
    n = 0
    for name in ("sigma_t", "sigma_c", "sigma_f", "nu", "chi", "sigma_s", "speed", "surf_coef", "surf_bc",
                 "cell_offset", "hs_surface", "hs_sense", "cell_material", "src_group_pdf", "time_edges",
                 "census_times"):
        n += getattr(p, name).nbytes
    return n + 31 * 8


def algorithmic_bytes(p, c, n_hist, n_batches=0):
    """SURVEY.md 8(d), the history kernel's part: 176 B per segment + 112 B per fission child + 88 B per source history.
    The close-out (3 x 16 B per bin per batch) is k_closeout's work, not k_warp's: it is NOT in this figure, which is
    divided by k_warp's device time alone."""
    return 176.0 * c["segments"] + 112.0 * c["children"] + 88.0 * n_hist


# ------------------------------------------------------------------------------------------------
def run_cpu_sample(p, seconds_target=15.0, first_history_id=0):
    """Time the oracle as it stands on a bounded sample of the same workload (one host thread)."""
    from oracle import Oracle

    o = Oracle(p)
    n = 2000
    t0 = time.perf_counter(); o.run(n, p.seed, n_batches=1, first_history_id=first_history_id)
    dt = time.perf_counter() - t0
    rate = n / dt
    n2 = int(max(2000, min(p.n_histories, rate * seconds_target)))
    o.reset()
    t0 = time.perf_counter(); o.run(n2, p.seed, n_batches=1, first_history_id=first_history_id)
    dt = time.perf_counter() - t0
    c = o.counters()
    return {"value": n2 / dt, "unit": METRIC, "cores": 1, "kind": "oracle", "n": n2,
            "sample": f"first {n2} histories of {p.name} (seed {p.seed}), single thread, {dt:.1f} s",
            "segments_per_s": c["segments"] / dt}


def _cpu_part(job):
    """One oracle process: `n` histories of the workload from history id `first` (a range of its own)."""
    name, kw, seed, first, n = job
    from oracle import Oracle
    from workloads import configs as W
    p = W.get_config(name, **kw)
    o = Oracle(p)
    t0 = time.perf_counter()
    o.run(n, seed, n_batches=1, first_history_id=first)
    dt = time.perf_counter() - t0
    seg = o.counters()["segments"]
    o.close()
    return n, dt, seg


def run_cpu_all_cores(args, p, per_core_rate, seconds_target=12.0):
    """the oracle as it stands on ALL host cores -- P = nproc independent processes over disjoint
    history-id ranges of the same workload (histories are independent; no tuning, no threads inside)."""
    import multiprocessing as mp
    P = os.cpu_count() or 1
    n = int(max(1000, min(p.n_histories // P, per_core_rate * seconds_target)))
    kw = {}
    if args.histories:
        kw["n_histories"] = int(args.histories)
    if args.batches:
        kw["n_batches"] = int(args.batches)
    jobs = [(args.workload, kw, p.seed, i * n, n) for i in range(P)]
    ctx = mp.get_context("spawn")
    with ctx.Pool(P) as pool:
        pool.map(_cpu_part, [(args.workload, kw, p.seed, 0, 200)] * P)      # start every process, load the checker
        t0 = time.perf_counter()
        res = pool.map(_cpu_part, jobs, chunksize=1)
        wall = time.perf_counter() - t0
    tot = sum(r[0] for r in res)
    return {"value": tot / wall, "unit": METRIC, "cores": P, "kind": "oracle",
            "sample": f"{P} processes x {n} histories of {p.name} (disjoint id ranges from 0, seed {p.seed}), {wall:.1f} s wall",
            "segments_per_s": sum(r[2] for r in res) / wall}


def bench_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    p = _problem(args)
    vals = []
    per_step = args.ref_seconds or max(3.0, min(20.0, 120.0 / max(1, args.steps + args.warmup)))
    for _ in range(args.warmup):
        run_cpu_sample(p, seconds_target=min(2.0, per_step))
    t0 = time.perf_counter()
    for s in range(args.steps):
        vals.append(run_cpu_sample(p, seconds_target=per_step, first_history_id=0))
    dt = time.perf_counter() - t0
    v = float(np.mean([x["value"] for x in vals]))
    n_sample = int(np.mean([x["n"] for x in vals]))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    out = {"impl": "reference", "metric": METRIC, "value": v, "unit": METRIC, "n_gpus": world, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": 1e3 * dt / max(1, args.steps), "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": p.name, "histories_per_step": n_sample, "workload_histories": p.n_histories,
                      "n_batches": 1, "seed": p.seed,
                      "note": f"each step is a bounded SAMPLE of the workload: the oracle (one host thread, rank 0) runs the "
                              f"first {n_sample} of its {p.n_histories} histories; ms_per_step is the time of that sample"},
           "cpu_baseline": {"value": v, "unit": METRIC, "cores": 1, "kind": "oracle", "sample": vals[-1]["sample"]},
           "e2e": {"value": v, "unit": METRIC, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out))


# ------------------------------------------------------------------------------------------------
def bench_gpu(args):
    import torch
    import torch.distributed as dist

    import paper_2409_04668_b200 as M

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    # --force-dist: the multi-rank code of this function (NCCL process group, barriers, the all-reduce of the accumulators
    # inside the timed region, the max over ranks) run by a single rank on one GPU -- the only way to execute it where no
    # second GPU exists.  A launcher that sets WORLD_SIZE=1 gets the same.
    dist_on = world > 1 or args.force_dist or "WORLD_SIZE" in os.environ and "MASTER_PORT" in os.environ
    if dist_on:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        if "MASTER_PORT" not in os.environ:
            import socket
            with socket.socket() as sk:
                sk.bind(("127.0.0.1", 0))
                os.environ["MASTER_PORT"] = str(sk.getsockname()[1])
        os.environ.setdefault("WORLD_SIZE", "1"); os.environ.setdefault("RANK", "0")
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    dev = f"cuda:{local}"
    torch.cuda.set_device(dev)
    p = _problem(args)
    n_hist, n_b = p.n_histories, p.n_batches
    from paper_2409_04668_b200.sharding import shard_range

    # weak scaling: every rank runs n_hist histories of its own id range; the one exchange of the job is the
    # sum-reduction of the accumulators at its end, inside the timed region
    first_id = shard_range(n_hist * world, world, rank)[0]
    g = M.Problem(p, device=dev)
    tech = TECHNIQUES[args.technique]
    if tech:
        g.set_technique(**tech)

    def barrier():
        torch.cuda.synchronize()
        if dist_on:
            dist.barrier()
        torch.cuda.synchronize()

    dbg = dict(debug_pool_slots=args.debug_pool_slots, debug_stage_tables=args.debug_stage_tables)
    for _ in range(args.warmup):
        g.reset(); g.run(n_hist, p.seed, n_b, first_history_id=first_id, **dbg)
    barrier()
    sampler = make_sampler(local)
    if rank == 0:
        sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    g.reset()
    launches0 = g.counters()["kernel_launches"]
    ms_tr = 0.0
    barrier()
    t_wall0 = time.time()
    ev0.record()
    for _ in range(args.steps):
        g.run(n_hist, p.seed, n_b, first_history_id=first_id, **dbg)
        ms_tr += g.counters()["ms_transport"]
    c = g.counters()                                      # this rank's own counts
    if dist_on:
        g.all_reduce()                                    # NCCL all-reduce of sum / sumsq / ledger / populations
    ev1.record()
    barrier()
    t_wall1 = time.time()
    ms = ev0.elapsed_time(ev1)
    if dist_on:
        t = torch.tensor([ms, ms_tr], device=dev, dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms, ms_tr = float(t[0]), float(t[1])
    launches = c["kernel_launches"] - launches0
    total_hist = n_hist * args.steps * world
    value = total_hist / (ms * 1e-3)
    seg_per_s = c["segments"] * world / (ms * 1e-3)

    out = None
    if rank == 0:
        clocks = sampler.stop(t_wall0, t_wall1)
        peak, peak_kind, sm_max = _peaks()
        # dominant kernel: k_warp.  Algorithmic bytes of the steps it processed / its device time.
        alg = algorithmic_bytes(p, {"segments": c["segments"], "children": c["children"]}, n_hist * args.steps)
        n_tr = max(1, launches // 2)                       # one k_warp + one k_closeout launch per sub-batch
        ach = alg / (ms_tr * 1e-3) / 1e9
        kinfo = g.kernel_info()
        ncu, ncu_note = ncu_constants(kinfo, p.name, args.technique)
        traffic = ncu["dram_bytes_per_history"] * n_hist * args.steps / n_tr if ncu else None
        # the label says what the figure is: SURVEY 8(d)'s algorithmic bytes over the measured copy bandwidth.  The kernel keeps
        # particle state on the SM and its real DRAM traffic is a fraction of a percent of peak (frac_measured_dram), so it is
        # NOT bandwidth-bound; the bound it does have is the issue rate, reported in roofline_alu.
        roofline = {"bound": "hbm (algorithmic-bytes equivalent)", "kernel": kinfo, "achieved": ach, "peak": peak, "unit": "GB/s",
                    "frac": ach / peak, "traffic": traffic, "peak_kind": peak_kind,
                    "frac_measured_dram": (traffic * n_tr / (ms_tr * 1e-3) / 1e9 / peak) if traffic else None,
                    "ncu_source": ncu_note,
                    "note": "achieved = SURVEY 8(d) algorithmic-bytes equivalent of the history kernel (176 B/segment + "
                            "112 B/child + 88 B/history) / summed k_warp device time (CUDA events on the library's "
                            "stream); particle state lives in shared memory, so the measured DRAM traffic (bytes per "
                            "launch from the ncu capture, frac_measured_dram) is far below this figure and the kernel "
                            "is issue-bound: see roofline_alu",
                    "launches": int(n_tr), "ms_kernel_total": ms_tr}
        roofline_alu = None
        if ncu:
            ti = ncu["thread_inst_per_segment"] * c["segments"] / (ms_tr * 1e-3)
            pk = N_SM * ISSUE_LANES_PER_SM * sm_max * 1e6
            roofline_alu = {"bound": "alu", "kernel": kinfo.split(" ")[0], "achieved": ti / 1e12, "peak": pk / 1e12,
                            "unit": "T thread-inst/s", "frac": ti / pk,
                            "issue_active_pct": ncu.get("issue_active_pct"),
                            "l2_red_sectors_per_s": (ncu["l2_atom_red_sectors_per_segment"] * c["segments"] / (ms_tr * 1e-3))
                            if ncu.get("l2_atom_red_sectors_per_segment") else None,
                            "l2_hit_rate_pct": ncu.get("l2_hit_rate_pct"),
                            "note": "instruction issue: thread instructions per segment from the ncu capture x segments/s, "
                                    "against 148 SMs x 4 schedulers x 32 lanes x max SM clock (DESIGN.md section 6); "
                                    "l2_red_sectors_per_s = fp64 RED/atomic sectors at L2 per second (atomic throughput)"}
        out = {"metric": METRIC, "value": value, "unit": METRIC, "n_gpus": world, "steps": args.steps,
               "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
               "vs_baseline": None, "dtype": "f64", "data": "synthetic",
               "config": {"workload": p.name, "histories_per_step": n_hist, "n_batches": n_b, "seed": p.seed,
                          "l2": "the path has no input buffers (histories are generated on chip from seed and id); its "
                                "only global data, the per-batch tally accumulators, are rewritten by the close-out of "
                                "every step, so no step can reuse a previous step's cache contents",
                          "parallelism": f"history-range sharding x{world}" +
                                         (", one NCCL all-reduce of the accumulators at the end" if dist_on else ""),
                          "technique": args.technique},
               "segments_per_s": seg_per_s, "segments_per_history": c["segments"] / max(1, c["histories"]),
               "clocks": clocks, "gpu_launches": int(launches), "roofline": roofline, "roofline_alu": roofline_alu}
    # ---- e2e: host buffers in, host buffers out, through the C ABI (create + bind + run + get) ----
    ws = g._ws
    ptr = (ws.data_ptr() + 255) // 256 * 256
    e2e_steps = max(1, min(args.steps, 3))
    # the caller's result buffers: pinned host memory (allocated once, as an application would), filled every step
    pin = torch.empty((2, p.n_bins), dtype=torch.float64).pin_memory()
    out_np = (pin[0].numpy(), pin[1].numpy())
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        h = M.mcdc_problem_create(p)                      # H2D: the problem description
        M.mcdc_workspace_bind(h, ptr, g.workspace_bytes, g.max_hist, g.max_slots, g._stream.cuda_stream)
        if tech:
            M.mcdc_technique_set(h, **tech)
        M.mcdc_run_ex(h, n_hist, p.seed, n_b, first_id)
        mean, sdev = M.mcdc_tallies_get(h, p.n_bins, out=out_np)      # D2H: mean and sdev of every bin
        M.mcdc_problem_destroy(h)
    barrier()
    dt = time.perf_counter() - t0
    if dist_on:
        t = torch.tensor([dt], device=dev, dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dt = float(t[0])
    if rank == 0:
        out["e2e"] = {"value": n_hist * e2e_steps * world / dt, "unit": METRIC, "h2d_bytes_per_step": _desc_bytes(p),
                      "d2h_bytes_per_step": 2 * 8 * p.n_bins, "steps": e2e_steps,
                      "note": "mcdc_problem_create (host arrays) + workspace_bind + run_ex + tallies_get (into pinned host "
                              "arrays allocated once) per step"}
        if world == 1 and not args.no_cpu:
            out["cpu_baseline"] = run_cpu_sample(p, seconds_target=args.cpu_seconds)
            out["cpu_baseline_all_cores"] = run_cpu_all_cores(args, p, out["cpu_baseline"]["value"],
                                                              seconds_target=min(12.0, args.cpu_seconds))
    g.close()
    if not args.no_sweep and world == 1 and args.workload == "config3" and not args.histories and args.technique == "analog":
        out["sweep"] = run_sweep(M, args, dev, peak)
    # the other workloads and the variants, so that they are the driver's numbers and not only this repository's say-so
    # (a few seconds of GPU time, outside the headline's timed region; --no-sweep skips them with the sweep)
    if not args.no_sweep and world == 1 and args.workload == "config3" and not args.histories and args.technique == "analog":
        out["configs"] = run_configs(M, args, dev, peak)
        out["variants"] = run_variants(M, args, dev)
        out["eigenvalue"] = run_eigenvalue(M, args, dev)
    elif args.eigenvalue and world == 1:
        out["eigenvalue"] = run_eigenvalue(M, args, dev)
    if rank == 0:
        print(json.dumps(out))
    if dist_on:
        dist.destroy_process_group()


def run_eigenvalue(M, args, dev):
    """Side measurement (not the headline): the k-eigenvalue mode (DESIGN.md Appendix H) on the config-3 lattice,
    1e6 particles per generation, 5 inactive + 15 active generations."""
    import torch
    from workloads import configs as W

    n, n_in, n_act = 1_000_000, 5, 15
    p = W.as_eigenvalue(W.config3_pin_lattice(n_histories=n, n_batches=1))
    g = M.Problem(p, max_histories_per_subbatch=n, max_batches_in_flight=1, device=dev, workspace_scale=1.5)
    g.run_eigenvalue(n, p.seed, 1, 2)                     # warm-up
    g.reset()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    k = g.run_eigenvalue(n, p.seed, n_in, n_act)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    c = g.counters()
    out = {"workload": p.name, "particles_per_generation": n, "inactive": n_in, "active": n_act,
           "k_eff": float(k[n_in:].mean()), "k_sdev": float(k[n_in:].std(ddof=1) / np.sqrt(n_act)),
           "ms_per_generation": ms / (n_in + n_act), "particles_per_s": n * (n_in + n_act) / (ms * 1e-3),
           "segments_per_s": c["segments"] / (ms * 1e-3), "ms_transport": c["ms_transport"],
           "launches": int(c["kernel_launches"])}
    g.close()
    return out


def _timed_runs(torch, g, n, seed, nb, reps):
    """reps runs of one handle after a warm-up and a reset -> (ms per run by CUDA events around the calls, k_warp / transport
    ms per run from the library's own events, close-out + memsets ms per run, counters)."""
    g.run(n, seed, nb)                                    # warm-up
    g.reset()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ms_tr = ms_dev = 0.0
    e0.record()
    for _ in range(reps):
        g.run(n, seed, nb)
        c = g.counters()
        ms_tr += c["ms_transport"]; ms_dev += c["ms_run"]
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / reps, ms_tr / reps, (ms_dev - ms_tr) / reps, g.counters()


def _e2e_once(M, torch, g, p, tech, reps):
    """The end-to-end leg of the headline on another workload: create (host arrays) + bind + run_ex + tallies_get into pinned
    host arrays, per step -> histories/s."""
    ptr = (g._ws.data_ptr() + 255) // 256 * 256
    pin = torch.empty((2, p.n_bins), dtype=torch.float64).pin_memory()
    out_np = (pin[0].numpy(), pin[1].numpy())
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(reps):
        h = M.mcdc_problem_create(p)
        M.mcdc_workspace_bind(h, ptr, g.workspace_bytes, g.max_hist, g.max_slots, g._stream.cuda_stream)
        if tech:
            M.mcdc_technique_set(h, **tech)
        M.mcdc_run_ex(h, p.n_histories, p.seed, p.n_batches)
        M.mcdc_tallies_get(h, p.n_bins, out=out_np)
        M.mcdc_problem_destroy(h)
    torch.cuda.synchronize()
    return p.n_histories * reps / (time.perf_counter() - t0)


def run_configs(M, args, dev, peak):
    """BASELINE configs 0, 1 and 2 at their stated sizes (config 2 stands in for the paper's one measured workload, the
    dog-leg duct of PAPER.md:159): the figures of the headline for each, outside its timed region, same JSON line."""
    import torch
    from workloads import configs as W

    rows = []
    for name in ("config0", "config1", "config2"):
        p = W.get_config(name)
        g = M.Problem(p, device=dev)
        ms, ms_k, ms_rest, c = _timed_runs(torch, g, p.n_histories, p.seed, p.n_batches, 3)
        alg = algorithmic_bytes(p, c, p.n_histories * 3)
        rows.append({"workload": p.name, "histories": p.n_histories, "n_batches": p.n_batches, "tally_bins": p.n_bins,
                     "histories_per_s": p.n_histories / (ms * 1e-3), "segments_per_s": c["segments"] / 3 / (ms * 1e-3),
                     "ms_per_step": ms, "ms_k_warp": ms_k, "ms_closeout_and_memsets": ms_rest,
                     "hbm_GBps_algorithmic": alg / 3 / (ms_k * 1e-3) / 1e9, "frac_of_hbm_peak": alg / 3 / (ms_k * 1e-3) / 1e9 / peak,
                     "kernel_info": g.kernel_info(), "e2e_histories_per_s": _e2e_once(M, torch, g, p, None, 2)})
        g.close()
    return rows


def run_variants(M, args, dev):
    """The techniques of DESIGN.md Appendix G on config 3 at the headline's size, and the general-CSG geometry: device time per
    step by the same events as the headline.  (The k-eigenvalue mode is the 'eigenvalue' key.)"""
    import torch
    from workloads import configs as W

    rows = []
    cases = [("config3", name, W.get_config("config3")) for name in ("ic_wr", "pc", "all")]
    cases.append(("csg_union", "analog", W.csg_union_geometry(n_histories=1_000_000, n_batches=100)))
    for wl, tname, p in cases:
        g = M.Problem(p, device=dev)
        tech = TECHNIQUES[tname]
        if tech:
            g.set_technique(**tech)
        reps = 2
        ms, ms_k, ms_rest, c = _timed_runs(torch, g, p.n_histories, p.seed, p.n_batches, reps)
        rows.append({"workload": p.name, "technique": tname, "histories": p.n_histories, "n_batches": p.n_batches,
                     "histories_per_s": p.n_histories / (ms * 1e-3), "segments_per_s": c["segments"] / reps / (ms * 1e-3),
                     "ms_per_step": ms, "ms_transport": ms_k, "launches_per_step": int(c["kernel_launches"]) // reps,
                     "kernel_info": g.kernel_info()})
        g.close()
    return rows


def run_sweep(M, args, dev, peak):
    """BASELINE config 4: the config-3 problem at 1e5 .. 1e9 histories (1e9 as device-sized sub-batches): histories/s,
    segments/s and algorithmic HBM GB/s vs batch size.  Outside the timed region of the headline, same JSON line."""
    import torch
    from workloads import configs as W

    rows = []
    for n in (10 ** 5, 10 ** 6, 10 ** 7, 10 ** 8, 10 ** 9):
        if n > args.sweep_max:
            break
        nb = 20 if n == 10 ** 5 else 100
        p = W.config3_pin_lattice(n_histories=n, n_batches=nb)
        sub = min(n, 250_000_000)                         # histories per sub-batch (one k_warp launch)
        g = M.Problem(p, max_histories_per_subbatch=sub, max_batches_in_flight=min(nb, max(1, sub // (n // nb))),
                      device=dev, async_only=True)
        reps = 3 if n <= 10 ** 7 else 1
        g.run(min(n, 10 ** 7) // nb * nb, p.seed, nb)   # warm-up
        g.reset()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        ms_k = 0.0
        for _ in range(reps):
            g.run(n, p.seed, nb)
            ms_k += g.counters()["ms_transport"]
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1)
        c = g.counters()
        alg = algorithmic_bytes(p, c, n * reps)
        rows.append({"histories": n, "n_batches": nb, "histories_per_s": n * reps / (ms * 1e-3),
                     "segments_per_s": c["segments"] / (ms * 1e-3), "ms_per_run": ms / reps,
                     "hbm_GBps_algorithmic": alg / (ms_k * 1e-3) / 1e9, "frac_of_hbm_peak": alg / (ms_k * 1e-3) / 1e9 / peak,
                     "launches_per_run": (c["kernel_launches"]) // reps, "workspace_bytes": g.workspace_bytes})
        g.close()
    return rows


def launch_ranks(n):
    """`python bench.py --gpus N` outside a launcher: start N ranks of this command line itself, one per GPU, the way the
    driver does (torch.distributed.run, rendezvous on 127.0.0.1), and become that launcher."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    sys.stdout.flush()
    os.execv(sys.executable, cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="config3")
    ap.add_argument("--histories", type=float, default=0)
    ap.add_argument("--batches", type=int, default=0)
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--force-dist", action="store_true", help="run the multi-rank code path (NCCL group, barriers, all-reduce of "
                    "the accumulators in the timed region) with a single rank")
    ap.add_argument("--technique", default="analog", choices=sorted(TECHNIQUES),
                    help="variance-reduction variant of the workload (DESIGN.md Appendix G); the headline is analog")
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    ap.add_argument("--debug-pool-slots", type=int, default=0, help="mcdc_run_opts.debug_pool_slots (test knob; 0 = automatic)")
    ap.add_argument("--debug-stage-tables", type=int, default=0, help="mcdc_run_opts.debug_stage_tables (test knob; 0 = automatic)")
    ap.add_argument("--no-sweep", action="store_true", help="skip the config-4 batch-size sweep (the 'sweep' key of the "
                    "default config-3 line: 1e5 .. 1e9 histories, a few seconds of GPU time)")
    ap.add_argument("--sweep", action="store_true", help="(default now; kept for old command lines)")
    ap.add_argument("--sweep-max", type=float, default=1e9)
    ap.add_argument("--ref-seconds", type=float, default=0.0, help="--impl reference: CPU seconds per step (0 = automatic)")
    ap.add_argument("--eigenvalue", action="store_true", help="also time the k-eigenvalue mode (adds an 'eigenvalue' key)")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        launch_ranks(args.gpus)                            # does not return
    if args.impl == "reference":
        bench_reference(args)
    else:
        bench_gpu(args)


if __name__ == "__main__":
    main()

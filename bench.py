#!/usr/bin/env python
"""bench.py -- world-steps/s of the batched tree-physics step on BASELINE.json configs[3] (the headline config:
4096 worlds x 350-450 links, 60 apples, h = 1 ms, one random wrench per world resampled every 50 steps).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--worlds 4096] [--config 4] [--substeps 50]
  python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...
  python bench.py --impl reference ...      # the fp64 CPU oracle, as it stands, on a bounded sample

One bench "step" = one wrench epoch of the whole hot path for every world of the batch: the epoch's wrenches
(ob_apply_wrench_batch) followed by `substeps` physics steps in one ob_step launch (FK, tether forces, bias,
tree factorisation (the preconditioner), PCG, integration, rupture / detach predicates, event append).  `value` = world-steps/s with
the inputs resident in HBM (wrench slots already uploaded, timed with CUDA events around the ob_step launches);
`e2e` = the same through the C ABI with HOST buffers: wrench arrays in, events + per-world counters out, copies
inside the timed region.  Prints ONE JSON line (rank 0).  DESIGN.md section "Measurement" explains every field.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

# ranges of --geometry-dr (growth habit and per-branch dimensions, distinct in every world)
GEOMETRY_DR_RANGES = dict(droop=(0.0, 0.10), lean=(0.0, 0.12), spread=(-0.15, 0.25), twist=(-0.4, 0.4),
                          scale_length=(0.85, 1.15), scale_diameter=(0.85, 1.2), jitter_length=(0.9, 1.1),
                          jitter_diameter=(0.9, 1.1))
METRIC = "world-steps/s at 4096 trees x ~400 links"
UNIT = "world-steps/s"

# Algorithmic work per link: flops of the formulas of the path as it runs with the tree
# preconditioner (precond = 2), checked against the fp32 + fp64 instruction counts of the ncu capture in profiles/
# (0.60 Mflop fp32 + 0.07 Mflop fp64 per world-step at 397 links, 60 apples, 1.03 iterations: within 3 % of this model).
FLOP_LINK_STEP = 1180.0       # joint quaternions + FK (fp64) 150, articulated-inertia factorisation 500, bias RNEA
                              # 350, first product A x0 150, integration + predicates 30
FLOP_LINK_ITER = 320.0        # one PCG iteration: A p (two sweeps) 150, z = P^-1 r (two sweeps) 150, vector updates, dots
FLOP_APPLE_STEP = 150.0       # tether force, reaction, clamp, integration, detach predicates
# Algorithmic HBM bytes per world-step if the state were streamed every step: 84 B per link,
# 72 B per apple, 32 B of wrench.  With n steps fused per launch the traffic falls to 1/n of this.
BYTES_LINK_STEP = 84.0
BYTES_APPLE_STEP = 72.0
BYTES_WRENCH = 32.0


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm_gbs=float(d["hbm_gbs"]), sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)), source="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")


def reduce_over_ranks(x: float, op: str, world_size: int, device: str = "cuda") -> float:
    """max / sum of one number over the ranks of the job (replicas only: the only cross-rank traffic of the bench)."""
    if world_size == 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX if op == "max" else dist.ReduceOp.SUM)
    return float(t.item())


def replica_seed(config: int, rank: int) -> int:
    """Each rank steps an independent replica of the batch: same geometry, its own material draws."""
    return 260706337 + 1000 * config + rank


class ClockSampler(threading.Thread):
    """SM clock and throttle reasons during the timed region (NVML; the recipe's nvidia-smi clocks line)."""

    def __init__(self, index: int, period: float = 0.05):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop_ev = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception:
            self.nv = None

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {
            getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksThrottleReasonSwPowerCap", 0x4): "sw_power_cap",
            getattr(nv, "nvmlClocksThrottleReasonHwPowerBrakeSlowdown", 0x80): "hw_power_brake_slowdown",
        }
        while not self._stop_ev.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                try:
                    r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                except Exception:
                    r = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            self._stop_ev.wait(self.period)

    def stop(self) -> dict:
        self._stop_ev.set()
        if self.is_alive():
            self.join(timeout=2.0)
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


def kernel_source_hash() -> str:
    """sha256 (16 hex digits) over the CUDA sources of the library: ties a committed profile to the kernel it was of."""
    import hashlib
    h = hashlib.sha256()
    csrc = os.path.join(ROOT, "paper_2607_06337_b200", "csrc")
    for f in sorted(os.listdir(csrc)):
        h.update(open(os.path.join(csrc, f), "rb").read())
    return h.hexdigest()[:16]


def _profiled_traffic(n_worlds: int, substeps: int):
    """DRAM bytes of one k_step launch (dram__bytes_read.sum + dram__bytes_write.sum) from the committed ncu --set full
    capture, profiles/r3_k_step_dram.txt.  PROFILED, not measured in this run: null unless that capture was of a launch
    of this size AND of the kernel sources as they are now (the file carries their hash)."""
    tp = os.path.join(ROOT, "profiles", "r3_k_step_dram.txt")
    try:
        kv = dict(l.split("=", 1) for l in open(tp).read().split() if "=" in l)
        if int(kv["worlds"]) == n_worlds and int(kv["substeps"]) == substeps and kv["kernel_source_hash"] == kernel_source_hash():
            return float(kv["dram_bytes_per_launch"])
    except Exception:
        pass
    return None


# --post-rupture: the post-rupture model of PAPER.md:141 / 398 switched ON (readings A34-A36; the paper gives "~5x over
# ~1.5 s" and no magnitudes, these are the values DESIGN.md section 1 row 8(f)1 was measured with)
POST_RUPTURE = dict(fric_frac=0.02, fric_ramp=5.0, fric_time=1.5, mass_damping=0.5, snap_drag_scale=0.2,
                    rail_speed=5.0, rail_fade=0.5, rail_brake=50.0, forces_off_on_snapped=0)


def _workload(config: int, n_worlds: int, post_rupture: bool = False):
    import dataclasses

    from workloads import config_params, make_config
    base = make_config(config, min(n_worlds, 4096))
    specs = [base[w % len(base)] for w in range(n_worlds)]     # 16384 = the 4096 geometries four times over;
    P = config_params(config)                                 # materials still differ per world (Philox by world)
    return specs, (dataclasses.replace(P, **POST_RUPTURE) if post_rupture else P)


def _loads_arrays(specs, epoch, f_lo, f_hi):
    from workloads import wrench_epoch_loads
    loads = wrench_epoch_loads(specs, epoch, f_lo, f_hi)      # clears of epoch - 1, then the new wrenches
    return (np.array([l[0] for l in loads], np.int32), np.array([l[1] for l in loads], np.int32),
            np.array([l[2] for l in loads], np.float32), np.array([l[3] for l in loads], np.float32))


def run_cuda(args, rank: int, world_size: int):
    import torch
    import torch.distributed as dist

    import paper_2607_06337_b200 as ob

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the orchard step has no CPU fallback")
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world_size > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    peaks = _peaks()
    specs, P = _workload(args.config, args.worlds, args.post_rupture)
    f_lo, f_hi = (100.0, 600.0) if args.config == 5 else (0.0, 150.0)
    W, S = len(specs), args.substeps
    n_links = sum(s.n_links for s in specs)
    n_apples = sum(s.n_apples for s in specs)
    seed = replica_seed(args.config, rank)
    n_epochs = args.warmup + args.steps
    epochs = [_loads_arrays(specs, e, f_lo, f_hi) for e in range(n_epochs)]

    def barrier():
        if world_size > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def run(e2e: bool, with_state: bool = False):
        sim = ob.Orchard(specs, P)
        sim.randomize(seed)
        if args.geometry_dr:                               # distinct growth habit and dimensions in every world
            sim.randomize_geometry(seed + 9, **GEOMETRY_DR_RANGES)
        stream = sim.stream
        state = None
        for e in range(args.warmup):
            if args.config == 5 and e > 0 and e % 5 == 0:
                sim.randomize(seed + 5000 + e // 5)
            sim.apply_wrench_batch(*epochs[e])
            sim.step(S)
            if e2e:
                sim.events(); sim.stats()
        ev0 = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
        ev1 = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
        t_begin, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        c0, s0 = sim.counters(), sim.stats()
        n_events = 0
        sampler = ClockSampler(local)
        barrier()
        sampler.start()
        t_begin.record(stream)
        wall0 = time.perf_counter()
        for k in range(args.steps):
            if args.config == 5 and (args.warmup + k) % 5 == 0:
                # configs[4]: on-device Philox re-randomization and reset of every world every 250 steps
                sim.randomize(seed + 5000 + (args.warmup + k) // 5)
            if e2e:
                sim.apply_wrench_batch(*epochs[args.warmup + k])      # host arrays -> pinned staging -> device
                sim.step(S)
                n_events += len(sim.events())                          # device -> host: event list
                sim.stats()                                            # device -> host: totals
                if with_state:                                         # device -> host: the state of EVERY world
                    state = sim.get_state_batch(out=state)             # (q, qd, apples, flags, step / status words)
            else:
                # kernel-resident leg: the epoch's wrenches are uploaded outside the per-launch events but
                # inside the region (they are part of the workload); the launches are timed one by one
                sim.apply_wrench_batch(*epochs[args.warmup + k])
                sim.flush()
                ev0[k].record(stream)
                sim.step(S)
                ev1[k].record(stream)
        t_end.record(stream)
        barrier()
        wall = time.perf_counter() - wall0
        clocks = sampler.stop()
        region_ms = t_begin.elapsed_time(t_end)
        kern_ms = None if e2e else [a.elapsed_time(b) for a, b in zip(ev0, ev1)]
        c1, s1 = sim.counters(), sim.stats()
        hist = sim.iter_histogram()
        out = dict(iter_hist=hist, region_ms=region_ms, wall_s=wall, kern_ms=kern_ms, clocks=clocks, n_events=n_events,
                   world_steps=s1["world_steps_total"] - s0["world_steps_total"],
                   cg_iters=s1["cg_iters_total"] - s0["cg_iters_total"], flagged=s1["n_flagged"],
                   h2d=c1["h2d_bytes"] - c0["h2d_bytes"], d2h=c1["d2h_bytes"] - c0["d2h_bytes"],
                   launches=c1["kernel_launches"] - c0["kernel_launches"], launch=sim.launch_info(),
                   workspace=int(sim.workspace.numel()))
        sim.close()
        return out

    dev = run(e2e=False)
    e2e = run(e2e=True)
    e2s = run(e2e=True, with_state=True)

    def max_over_ranks(x: float) -> float:
        return reduce_over_ranks(x, "max", world_size)

    def sum_over_ranks(x: float) -> float:
        return reduce_over_ranks(x, "sum", world_size)

    kern_total_ms = max_over_ranks(sum(dev["kern_ms"]))
    region_ms = max_over_ranks(dev["region_ms"])
    e2e_ms = max_over_ranks(e2e["region_ms"])
    e2s_ms = max_over_ranks(e2s["region_ms"])
    ws_e2s = sum_over_ranks(e2s["world_steps"])
    ws_dev = sum_over_ranks(dev["world_steps"])
    ws_e2e = sum_over_ranks(e2e["world_steps"])
    iters_dev = sum_over_ranks(dev["cg_iters"])
    value = ws_dev / (region_ms * 1e-3)
    e2e_value = ws_e2e / (e2e_ms * 1e-3)

    line = None
    if rank == 0:
        # roofline of the dominant (only) kernel, k_step: per-launch algorithmic work / average launch duration
        k_ms = float(np.mean(dev["kern_ms"]))
        iters_per_ws = dev["cg_iters"] / max(dev["world_steps"], 1)
        ws_per_launch = dev["world_steps"] / args.steps
        links_per_world, apples_per_world = n_links / W, n_apples / W
        flop_ws = links_per_world * (FLOP_LINK_STEP + FLOP_LINK_ITER * iters_per_ws) + apples_per_world * FLOP_APPLE_STEP
        flops_launch = flop_ws * ws_per_launch
        sm_mhz = dev["clocks"]["sm_mhz"] or peaks["sm_max_mhz"]
        alu_peak = 148 * 128 * 2 * sm_mhz * 1e6 / 1e12               # TFLOP/s at the clock seen during the run
        alu_ach = flops_launch / (k_ms * 1e-3) / 1e12
        bytes_ws = links_per_world * BYTES_LINK_STEP + apples_per_world * BYTES_APPLE_STEP + BYTES_WRENCH
        hbm_stream = bytes_ws * ws_per_launch / (k_ms * 1e-3) / 1e9   # as if the state were streamed every step
        hbm_fused = hbm_stream / S                                    # what one launch really has to move
        traffic = _profiled_traffic(W, S)
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world_size, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": region_ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": (f"BASELINE.json configs[{args.config - 1}]" if args.config <= 5 else
                                     "ternary L-system of PAPER.md Eq. 1, n = 4 (SURVEY.md 8(f) item 4)") + f": {W} worlds x "
                                   f"{links_per_world:.0f} links ({min(x.n_links for x in specs)}-{max(x.n_links for x in specs)}), {apples_per_world:.0f} apples, h = {P.h * 1e3:g} ms, "
                                   f"wrench U({f_lo:g},{f_hi:g}) N per world resampled every {S} steps",
                       "worlds_per_gpu": W, "physics_steps_per_bench_step": S, "links_total": n_links,
                       "apples_total": n_apples, "cg_tol": P.cg_tol, "replicas": world_size,
                       "geometry": "ob_randomize_geometry: distinct growth habit and dimensions per world"
                                   if args.geometry_dr else "as generated (every world its own tree)",
                       "post_rupture": POST_RUPTURE if args.post_rupture else "off (BASELINE.json configs do not name it)",
                       "l2": f"inputs exceed L2: workspace {dev['workspace'] / 2**20:.0f} MiB vs 126 MB L2",
                       "launch": dev["launch"]},
            "kernel_only": {"value": ws_dev / (kern_total_ms * 1e-3), "unit": UNIT,
                            "ms_per_step": kern_total_ms / args.steps},
            "cg_iters_per_s": iters_dev / (region_ms * 1e-3),
            "cg_iters_per_world_step": iters_per_ws,
            "worlds_flagged": dev["flagged"],
            "cg_iters_histogram": _hist_summary(dev["iter_hist"]),
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": e2e["h2d"] / args.steps,
                    "d2h_bytes_per_step": e2e["d2h"] / args.steps, "ms_per_step": e2e_ms / args.steps,
                    "events_read": e2e["n_events"], "returns": "event list + totals every bench step",
                    "with_state": {"value": ws_e2s / (e2s_ms * 1e-3), "unit": UNIT,
                                   "h2d_bytes_per_step": e2s["h2d"] / args.steps,
                                   "d2h_bytes_per_step": e2s["d2h"] / args.steps, "ms_per_step": e2s_ms / args.steps,
                                   "returns": "event list + totals + q, qd, apple x / v, flags, step and status "
                                              "words of EVERY world (ob_get_state_batch) every bench step"}},
            "gpu_launches": dev["launches"],
            "clocks": dev["clocks"],
            "roofline": {"bound": "alu", "achieved": alu_ach, "peak": alu_peak, "unit": "TFLOP/s",
                         "frac": alu_ach / alu_peak, "traffic": traffic,
                         "traffic_source": "profiled (profiles/r3_k_step_dram.txt, same kernel sources and launch size), "
                                           "not measured in this run" if traffic is not None else None,
                         "limiter": "latency, not throughput: a step is a chain of ~70 dependent level turns; ncu "
                                    "(profiles/r3_k_step_ncu_full.md): issue slots 31 % busy, stall_barrier 3.4 / "
                                    "wait 1.4 / long_scoreboard 1.0 / no_instruction 0.9 per issued instruction",
                         "kernel": "k_step",
                         "kernel_ms": k_ms, "flop_per_world_step": flop_ws,
                         "peak_source": f"148 SM x 128 fp32 lanes x 2 x {sm_mhz:.0f} MHz (clock sampled in the run)",
                         "hbm": {"achieved_streamed": hbm_stream, "achieved_fused": hbm_fused,
                                 "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac_streamed": hbm_stream / peaks["hbm_gbs"],
                                 "frac_fused": hbm_fused / peaks["hbm_gbs"], "bytes_per_world_step": bytes_ws,
                                 "peak_source": peaks["source"]}},
        }
        if world_size == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline(specs, P, seed, f_lo, f_hi, args.geometry_dr)
    if world_size > 1:
        dist.barrier()
        dist.destroy_process_group()
    if line is not None:
        print(json.dumps(line), flush=True)


def _hist_summary(hist) -> dict:
    """p50 / p95 / max of PCG iterations per world-step from the device histogram (ob_iter_histogram)."""
    h = np.asarray(hist, dtype=np.float64)
    n = h.sum()
    if n == 0:
        return {"world_steps": 0}
    cdf = np.cumsum(h) / n
    nz = np.nonzero(h)[0]
    return {"world_steps": int(n), "p50": int(np.searchsorted(cdf, 0.5)), "p95": int(np.searchsorted(cdf, 0.95)),
            "p99": int(np.searchsorted(cdf, 0.99)), "max": int(nz[-1]), "last_bin_is_open": bool(nz[-1] == len(h) - 1),
            "mean": float((np.arange(len(h)) * h).sum() / n)}


def _omp_threads() -> int:
    try:
        n = len(os.sched_getaffinity(0))
    except Exception:
        n = os.cpu_count() or 1
    return max(1, n)


def _oracle_sample(specs, P, seed, f_lo, f_hi, n_sample, solver=0, geometry_dr=False):
    """Oracle worlds for the first n_sample worlds of the batch, randomized and loaded like the GPU run."""
    import oracle
    from workloads import wrench_process
    loads = wrench_process(specs, 0, f_lo, f_hi)
    worlds = []
    for w in range(n_sample):
        r = oracle.OracleWorld(specs[w], P, world_index=w, solver=solver)
        r.randomize(seed)
        if geometry_dr:
            r.randomize_geometry(seed + 9, **GEOMETRY_DR_RANGES)
        r.apply_wrench(loads[w][1], loads[w][2], loads[w][3])
        worlds.append(r)
    return worlds


def cpu_baseline(specs, P, seed, f_lo, f_hi, geometry_dr=False) -> dict:
    """The fp64 oracle as it stands (brute-force mass matrix + dense Cholesky, OpenMP over worlds), timed on this
    box's host cores on a bounded sample of the same workload.  A reported baseline, not the target."""
    import oracle
    cores = _omp_threads()
    os.environ.setdefault("OMP_NUM_THREADS", str(cores))
    n_sample = int(min(max(cores, 8), 64, len(specs)))
    n_steps = 8                                                  # ~1 s wall on 16 cores = 10-20 s of CPU work
    worlds = _oracle_sample(specs, P, seed, f_lo, f_hi, n_sample, geometry_dr=geometry_dr)
    oracle.step_many(worlds, 1)                                  # warm-up (page-in, first-touch)
    t0 = time.perf_counter()
    oracle.step_many(worlds, n_steps)
    dt = time.perf_counter() - t0
    out = {"value": n_sample * n_steps / dt, "unit": UNIT, "cores": min(cores, n_sample), "kind": "oracle",
           "sample": f"first {n_sample} worlds of the batch x {n_steps} steps after 1 warm-up step "
                     f"(fp64, mass matrix by unit-acceleration RNEA columns, dense Cholesky), {dt:.2f} s wall"}
    # the oracle's own fp64 Jacobi-PCG mode (same algorithm class as the GPU path; the matrix is still formed by
    # brute force) as the fairer CPU figure SURVEY.md 8(d) asks for
    pw = _oracle_sample(specs, P, seed, f_lo, f_hi, n_sample, solver=1, geometry_dr=geometry_dr)
    oracle.step_many(pw, 1)
    t0 = time.perf_counter()
    oracle.step_many(pw, n_steps)
    dtp = time.perf_counter() - t0
    out["pcg_mode"] = {"value": n_sample * n_steps / dtp, "unit": UNIT,
                       "sample": f"same sample, oracle solver = fp64 Jacobi-PCG on the assembled matrix, {dtp:.2f} s wall"}
    out["parity_sample"] = _parity_sample(specs, P, seed, f_lo, f_hi, worlds, 1 + n_steps, geometry_dr)
    return out


def _parity_sample(specs, P, seed, f_lo, f_hi, refs, n_steps, geometry_dr=False) -> dict:
    """The sampled worlds once more on the GPU, free-running the same steps as the (Cholesky) oracle worlds `refs`:
    events on one side only, and the worst relative state error among the worlds without events."""
    import paper_2607_06337_b200 as ob
    from workloads import wrench_process
    n = len(refs)
    sim = ob.Orchard(specs[:n], P)
    sim.randomize(seed)
    if geometry_dr:
        sim.randomize_geometry(seed + 9, **GEOMETRY_DR_RANGES)
    loads = wrench_process(specs, 0, f_lo, f_hi)[:n]
    sim.apply_wrench_batch([l[0] for l in loads], [l[1] for l in loads], [l[2] for l in loads], [l[3] for l in loads])
    sim.step(n_steps)
    gev = {(e[0], e[1], e[2], e[3]) for e in sim.events()}
    oev = {(e[0], e[1], e[2], e[3]) for r in refs for e in r.events()}
    worlds_with_events = {k[0] for k in gev | oev}
    worst = 0.0
    for w, r in enumerate(refs):
        if w in worlds_with_events:
            continue
        g, o = sim.get_state(w), r.get_state()
        for k, floor in (("q", 1e-6), ("qd", 1e-4)):
            den = max(np.linalg.norm(o[k]), floor * math.sqrt(o[k].size))
            worst = max(worst, float(np.linalg.norm(g[k].astype(np.float64) - o[k]) / den))
    sim.close()
    return {"worlds": n, "steps": n_steps, "events_gpu": len(gev), "events_oracle": len(oev),
            "events_on_one_side_only": len(gev ^ oev), "max_rel_state_error_worlds_without_events": worst,
            "protocol": "free run from the randomized rest state (the lock-step protocol with its near-threshold count "
                        "is tests/test_gpu_parity.py)"}


def run_cholesky_comparison(args):
    """SURVEY.md 8(f) item 4, second half: a blocked-Cholesky GPU solve as a comparison point for the paper's "the
    matrix-free CG solve is what makes laptop-scale batches practical" / "CG ~7x".  The LIBRARY's
    batched blocked Cholesky (torch.linalg.cholesky + cholesky_solve: cuSOLVER / cuBLAS underneath) factors and solves
    one SPD system of the size of every world of the batch (n = 2 x links, fp32, worlds grouped by n padded to 32),
    which is what an assembled-matrix solver would do every step.  Only the factor + solve are timed: assembling the
    matrix (n inverse-dynamics sweeps or a composite-rigid-body pass) is NOT counted, so the figure is an upper bound
    on such a solver's step rate.  The matrices are random SPD of the right sizes: the time of a dense factorisation
    does not depend on the entries."""
    import torch
    specs, P = _workload(args.config, args.worlds, args.post_rupture)
    dev = torch.device("cuda", int(os.environ.get("LOCAL_RANK", "0")))
    groups = {}
    for sp in specs:
        n = (2 * sp.n_links + 31) // 32 * 32
        groups[n] = groups.get(n, 0) + 1
    g = torch.Generator(device=dev).manual_seed(1)
    mats = []
    for n, cnt in sorted(groups.items()):
        for b0 in range(0, cnt, 512):                                   # batches of <= 512 matrices: bounded memory
            b = min(512, cnt - b0)
            R = torch.randn(b, n, n, device=dev, generator=g) * (1.0 / math.sqrt(n))
            A = R @ R.transpose(1, 2) + torch.eye(n, device=dev)
            mats.append((A, torch.randn(b, n, 1, device=dev, generator=g)))
    def once():
        for A, rhs in mats:
            L = torch.linalg.cholesky(A)
            torch.cholesky_solve(rhs, L)
    for _ in range(max(args.warmup, 1)):
        once()
    torch.cuda.synchronize()
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0.record()
    for _ in range(args.steps):
        once()
    t1.record()
    torch.cuda.synchronize()
    ms = t0.elapsed_time(t1) / args.steps
    flop = sum(c * (n ** 3 / 3.0 + 2.0 * n * n) for n, c in groups.items())
    line = {"comparison": "library batched blocked Cholesky (torch.linalg.cholesky + cholesky_solve), factor + solve only",
            "workload": f"BASELINE.json configs[{args.config - 1}]: {len(specs)} systems, n = 2 x links "
                        f"({min(groups)}-{max(groups)} after padding to 32), fp32, one factor + solve per world-step",
            "value": len(specs) / (ms * 1e-3), "unit": UNIT + " (upper bound: assembly not counted)",
            "ms_per_step_of_all_worlds": ms, "tflops": flop / (ms * 1e-3) / 1e12, "steps": args.steps}
    print(json.dumps(line), flush=True)


def run_reference(args, rank: int, world_size: int):
    """--impl reference: for this tier the reference arm is the oracle, timed as it stands on the host cores.
    Each bench step is a bounded sample of the workload (n_sample worlds x 1 physics step)."""
    if rank != 0:
        return
    cores = _omp_threads()
    os.environ.setdefault("OMP_NUM_THREADS", str(cores))
    import oracle
    n_sample = int(min(max(cores, 8), 64))
    from workloads import config_params, make_config
    specs = make_config(args.config, n_sample)
    P = config_params(args.config)
    f_lo, f_hi = (100.0, 600.0) if args.config == 5 else (0.0, 150.0)
    seed = 260706337 + 1000 * args.config
    worlds = _oracle_sample(specs, P, seed, f_lo, f_hi, n_sample)
    for _ in range(args.warmup):
        oracle.step_many(worlds, 1)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.step_many(worlds, 1)
    dt = time.perf_counter() - t0
    value = n_sample * args.steps / dt
    links = sum(s.n_links for s in specs) / n_sample
    sample = (f"{n_sample} worlds of configs[{args.config - 1}] ({links:.0f} links, {specs[0].n_apples} apples each) x 1 "
              f"physics step per bench step")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"BASELINE.json configs[{args.config - 1}], bounded sample: {sample}",
                       "physics_steps_per_bench_step": 1, "worlds": n_sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": min(cores, n_sample), "kind": "oracle",
                             "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--config", type=int, default=4, help="1-based index into BASELINE.json configs (3, 4 or 5); 6 = the homogeneous ternary L-system batch")
    ap.add_argument("--worlds", type=int, default=4096)
    ap.add_argument("--substeps", type=int, default=50, help="physics steps per bench step (one wrench epoch)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cholesky-comparison", action="store_true",
                    help="time the library's batched blocked Cholesky on systems of the batch's sizes (SURVEY.md 8(f) item 4)")
    ap.add_argument("--post-rupture", action="store_true",
                    help="post-rupture friction ramp, reduced drag on snapped sub-trees and the three force rails ON "
                         "(PAPER.md:141, 398; SURVEY.md 8(f) item 1), wrenches kept on snapped links so the rails act")
    ap.add_argument("--geometry-dr", action="store_true",
                    help="per-world geometry randomization on the device before the run (SURVEY.md 8(f) item 3)")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "cuda":
        args.warmup = 3                                    # timing rule: at least 3 warm-up steps
    rank = int(os.environ.get("RANK", "0"))
    world_size = int(os.environ.get("WORLD_SIZE", "1"))
    if args.cholesky_comparison:
        if rank == 0:
            run_cholesky_comparison(args)
    elif args.impl == "reference":
        run_reference(args, rank, world_size)
    else:
        run_cuda(args, rank, world_size)


if __name__ == "__main__":
    main()

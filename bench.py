#!/usr/bin/env python
"""bench.py -- coupled flood-pedestrian step on B200: one JSON line.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 5] [--impl ours|reference]

A "step" is ONE coupled step: occupancy -> binning (count, scan, scatter) -> pedestrian step ->
flood step (+ CFL reduction) -> sandbag/time tail, over the whole synthetic workload.  Default
workload: BASELINE.json configs[4] ("Throughput stress", 8192x8192 fp32 cells + 1e6 pedestrians,
500 timed steps) -- the largest single-GPU configuration and the only one whose per-step traffic
(2.3 GB) is larger than L2, which is what the "% of HBM roofline" part of the metric needs.

value      = flood cell-updates/s of the whole job, inputs resident in HBM, CUDA graphs, CUDA events.
e2e        = same metric through the C ABI with HOST (pinned) buffers: upload of the initial
             state + K steps + read-back of depth/discharge/pedestrians inside the timed region.
roofline   = flood kernel: algorithmic bytes per launch / its average duration (CUDA events around
             each launch, sim_step_profiled) vs the measured HBM peak of MEASURED_PEAKS.json.
cpu_baseline / --impl reference = the CPU oracle as it stands, on a bounded sample.
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
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

FLOOD_BYTES_PER_CELL = 33        # fp32: read h,qx,qy,z,n0 (20) + N_p (1) ; write h,qx,qy (12)  [DESIGN.md 6]
PED_BYTES_PER_AGENT = 175        # key+count 17, scatter 72, step 85
TRAFFIC_JSON = os.path.join(ROOT, "profiles", "r2_traffic.json")


def ncu_traffic(cfg, kernel):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` on config `cfg`, as recorded by
    the last committed `ncu --set full` capture (written by paper_1908_05232_b200/ncu_summary.py; a
    profiler cannot run inside a timed bench, so this is a STATIC record of that capture, or None)."""
    try:
        rec = json.load(open(TRAFFIC_JSON)).get(f"config{cfg}", {})
    except (OSError, ValueError):
        return None, None
    for name, r in rec.items():
        if kernel in name:
            return r["dram_bytes_read"] + r["dram_bytes_write"], f"static: ncu capture summarised in profiles/{r['summary']}"
    return None, None


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md, 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100", "-i", str(self.index)],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ts, line in self.rows:
            if ts < t0 - 0.05 or ts > t1 + 0.15:
                continue
            f = [x.strip() for x in line.split(",")]
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except Exception:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def scenario(cfg):
    from paper_1908_05232_b200 import scenarios as S
    return S.make(cfg)


# coupled steps of the CPU oracle that make a bounded sample of each config (Config 5 is
# timed over 5 steps after 1 warm-up; about 10 s per step and 8 GB at 8192^2 cells + 1e6 pedestrians)
ORACLE_STEPS = {1: 1000, 2: 2000, 3: 2000, 4: 20, 5: 5}


def oracle_run(cfg, steps, warmup, sc=None, flood_order=1):
    """The oracle as it stands, single thread, on the SAME workload (full size), over a bounded
    number of coupled steps; returns (cells/s, agents/s, s/step, desc)."""
    import oracle
    if sc is None:
        sc = scenario(cfg)
        sc.flood_order = flood_order
    o = oracle.Oracle(sc)
    if warmup:
        o.step(warmup)
    act0 = int((o.read_peds()["active"] == 1).sum()) if sc.n_peds else 0
    t0 = time.perf_counter()
    o.step(steps)
    dt = time.perf_counter() - t0
    done = o.stats()["step"] - warmup
    desc = f"{sc.name} recipe at {sc.nx}x{sc.ny} cells, {sc.n_peds} pedestrians, {done} coupled steps after {warmup} warm-up"
    return sc.nx * sc.ny * done / dt, act0 * done / dt, dt / max(done, 1), desc


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    steps = min(args.steps, ORACLE_STEPS[args.config])
    warm = min(args.warmup, 1)
    cps, aps, sps, desc = oracle_run(args.config, steps, warm, flood_order=args.flood_order)
    done_steps = steps
    line = {
        "impl": "reference", "metric": "flood cell-updates/s (coupled step)", "value": cps, "unit": "cell-updates/s",
        "n_gpus": args.gpus, "steps": steps, "warmup": warm, "ms_per_step": 1e3 * sps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "agent_updates_per_s": aps, "coupled_steps_per_s": 1.0 / sps,
        "config": {"workload": f"config{args.config}", "sample": desc},
        "timed_steps": done_steps,
        "cpu_baseline": {"value": cps, "unit": "cell-updates/s", "cores": 1, "kind": "oracle", "sample": desc},
        "e2e": {"value": cps, "unit": "cell-updates/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def aggregate(ms_max, world, ncell, done, active):
    """Whole-job numbers from the max-over-ranks time: `world` replicas each advanced `ncell` cells
    and `active` pedestrians by `done` coupled steps in `ms_max` milliseconds."""
    sec = ms_max * 1e-3
    return {"value": world * ncell * done / sec, "ms_per_step": ms_max / max(done, 1),
            "coupled_steps_per_s": world * done / sec, "agent_updates_per_s": world * active * done / sec}


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_1908_05232_b200 import binding, build, replicas

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    torch.cuda.set_device(local)
    build.build()
    K, W = args.steps, max(args.warmup, 3)
    sc = scenario(args.config)
    sc.flood_order = args.flood_order
    real = np.float32 if sc.real_bits == 32 else np.float64
    ncell, npeds = sc.nx * sc.ny, sc.n_peds
    g = binding.Sim(sc, device=f"cuda:{local}")
    if args.flood_variant >= 0:
        g.set_flood_variant(args.flood_variant)
    if args.no_overlap:
        g.set_overlap(False)
    if args.march_rows > 0:
        g.set_march_rows(args.march_rows)
    variant = g.flood_variant()
    kps = g.kernels_per_step()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timed region (CUDA graphs)
    g.step(W)
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.3)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    st0 = g.stats()
    barrier()
    w0 = time.time()
    e0.record()
    g.step(K)
    e1.record()
    barrier()
    w1 = time.time()
    ms = e0.elapsed_time(e1)
    clocks = sampler.stop(w0, w1)
    st1 = g.stats()
    done = st1["step"] - st0["step"]
    active = npeds - st0["hist"][5]
    ms_max = replicas.max_over_ranks(ms, device="cuda")

    # ---- per-kernel durations, CUDA events around every launch (same state, continuing)
    KP = min(K, 100)
    kms = g.step_profiled(KP)
    flood_ms = kms["flood_step"] / KP
    ped_ms = (kms["bin_count"] + kms["bin_scan"] + kms["scatter"] + kms["occupancy"] + kms["ped_step"]) / KP
    # the same kernel with the dry-chunk skip switched off (every chunk read, computed and written):
    # a second, shorter profiled run; the skip and its flags are then restored for what follows
    flood_ms_noskip = None
    if variant == 4:
        g.set_dry_skip(False)
        g.step_profiled(3)
        flood_ms_noskip = g.step_profiled(20)["flood_step"] / 20
        g.set_dry_skip(True)
        g.step_profiled(3)
    peak, peak_src = peaks()
    fb = FLOOD_BYTES_PER_CELL if sc.real_bits == 32 else 65
    flood_gbs = ncell * fb / (flood_ms * 1e-3) / 1e9
    kbin = int(np.ceil(sc.R_int / min(sc.dx, sc.dy)))
    nbins = -(-sc.nx // kbin) * -(-sc.ny // kbin)
    ped_gbs = (active * PED_BYTES_PER_AGENT + nbins * 12) / (ped_ms * 1e-3) / 1e9 if npeds else 0.0

    # ---- the pedestrian step is bound by the MUFU (XU) pipe in dense crowds, not by HBM: count its
    # candidate pairs from the bin occupancy (3 x 3 bins around every agent; 2 MUFU per candidate:
    # rsqrt, ex2 -- issued for the whole warp whenever one lane is inside the cut-off)
    xu = None
    if npeds:
        b = g.bin_peds()
        cnt = np.diff(b["start"][:b["nbx"] * b["nby"] + 1]).astype(np.int64).reshape(b["nby"], b["nbx"])
        pad = np.pad(cnt, 1)
        nb9 = sum(pad[dj:dj + b["nby"], di:di + b["nbx"]] for dj in range(3) for di in range(3))
        cand = float((cnt * nb9).sum())
        # the method's own work: ordered pairs with 0 < d < R_int (C26), counted with a k-d tree
        from scipy.spatial import cKDTree
        pp = g.read_peds()
        live = pp["active"] == 1
        tree = cKDTree(np.c_[pp["x"][live].astype(np.float64), pp["y"][live].astype(np.float64)])
        inter = float(tree.count_neighbors(tree, sc.R_int)) - float(live.sum())
        ped_step_ms = kms["ped_step"] / KP
        xu_peak = 148 * 16 * 1.965e9 / 1e12          # 16 MUFU lanes per SM and clock (4 per SMSP), 148 SMs, 1965 MHz
        xu = {"bound": "alu", "pipe": "xu (MUFU)", "kernel": "ped_step_kernel",
              "achieved": 2.0 * inter / (ped_step_ms * 1e-3) / 1e12, "peak": xu_peak, "unit": "T MUFU/s",
              "frac": 2.0 * inter / (ped_step_ms * 1e-3) / 1e12 / xu_peak,
              "work": "2 MUFU (rsqrt, ex2) per INTERACTING ordered pair (d < R_int): the method's own work",
              "interacting_pairs_per_step": inter, "interacting_per_agent": inter / max(active, 1),
              "candidate_pairs_per_step": cand, "candidates_per_agent": cand / max(active, 1),
              "issued": {"achieved": 2.0 * cand / (ped_step_ms * 1e-3) / 1e12, "frac": 2.0 * cand / (ped_step_ms * 1e-3) / 1e12 / xu_peak,
                         "note": "MUFU operations the kernel ISSUES: 2 per candidate of the 3 x 3 bins (a predicated-off MUFU still occupies the pipe for the warp)"},
              "ms": ped_step_ms,
              "peak_source": "derived: 148 SMs x 16 MUFU/clk x 1.965 GHz (DESIGN.md 7)"}

    # ---- end to end through the C ABI with pinned HOST buffers
    host = {k: torch.empty(ncell, dtype=torch.float32 if real is np.float32 else torch.float64).pin_memory()
            for k in ("h", "qx", "qy")}
    c = g.read_conserved()
    for k in host:
        host[k].numpy()[:] = c[k]
    p = g.read_peds()
    pin = {k: torch.from_numpy(np.ascontiguousarray(p[k])).pin_memory() for k in ("x", "y", "vx", "vy", "timer", "fsm", "active")}
    out_f = {k: torch.empty_like(host[k]).pin_memory() for k in host}
    KE = K
    h2d = 3 * ncell * host["h"].element_size() + sum(v.numel() * v.element_size() for v in pin.values())
    d2h = 3 * ncell * host["h"].element_size() + npeds * (5 * host["h"].element_size() + 3 + 4)
    barrier()
    tt0 = time.perf_counter()
    g.write_flood(host["h"].numpy(), host["qx"].numpy(), host["qy"].numpy())
    if npeds:
        g.write_peds(*(pin[k].numpy() for k in ("x", "y", "vx", "vy", "fsm", "active", "timer")))
    g.set_time(st1["t"], st1["dt"])
    g.step(KE)
    g.read_conserved_into(out_f["h"].data_ptr(), out_f["qx"].data_ptr(), out_f["qy"].data_ptr())
    pe = g.read_peds() if npeds else None
    ste = g.stats()
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - tt0
    e2e_s = replicas.max_over_ranks(e2e_s, device="cuda")
    e2e_done = KE

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- CPU oracle, bounded sample (reported baseline, not the target)
    o_steps = ORACLE_STEPS[args.config]
    if world == 1 and not args.no_cpu_baseline:
        cps, aps, sps, desc = oracle_run(args.config, o_steps, 1, sc)
        cpu = {"value": cps, "unit": "cell-updates/s", "cores": 1, "kind": "oracle", "sample": desc,
               "agent_updates_per_s": aps}
    else:
        cpu = None

    kernel_name = ("flood_cell_kernel", "flood_tile_kernel", "flood_march_kernel", "flood_march2_kernel", "flood_tmarch_kernel", "flood_muscl_kernel")[variant]
    traffic, traffic_src = ncu_traffic(args.config, kernel_name) if args.march_rows == 0 and args.flood_variant < 0 else (None, None)
    agg = aggregate(ms_max, world, ncell, done, active)
    # the roofline fraction counts bytes that are moved: the kernel with every chunk computed when that was measured
    if flood_ms_noskip is not None:
        real_gbs, frac_basis = ncell * fb / (flood_ms_noskip * 1e-3) / 1e9, "every chunk computed (dry-chunk skip off), same run"
    else:
        real_gbs, frac_basis = flood_gbs, "default kernel (this variant skips nothing)"
    line = {
        "metric": "flood cell-updates/s (coupled step)", "value": agg["value"], "unit": "cell-updates/s",
        "n_gpus": world, "steps": K, "warmup": W, "ms_per_step": agg["ms_per_step"],
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32" if sc.real_bits == 32 else "f64", "data": "synthetic",
        "coupled_steps_per_s": agg["coupled_steps_per_s"],
        "agent_updates_per_s": agg["agent_updates_per_s"],
        "steps_executed": done,
        "config": {"workload": f"config{args.config}: {sc.name}", "nx": sc.nx, "ny": sc.ny, "dx": sc.dx,
                   "pedestrians": npeds, "active_pedestrians": active,
                   "l2_policy": "inputs larger than L2 (no flush)" if ncell * fb > 126e6 else "working set fits L2: latency-bound config, roofline not meaningful",
                   "flood_variant": variant, "flood_order": args.flood_order, "overlap_ped_flood": not args.no_overlap, "parallelism": f"replicas x{world}" if world > 1 else "single GPU"},
        "clocks": clocks,
        "e2e": {"value": world * ncell * e2e_done / e2e_s, "unit": "cell-updates/s",
                "h2d_bytes_per_step": h2d / e2e_done, "d2h_bytes_per_step": d2h / e2e_done,
                "steps": e2e_done, "seconds": e2e_s,
                "what": "sim_write_flood+sim_write_peds from pinned host, sim_step, sim_read_conserved+sim_read_peds+sim_get_stats to host"},
        "gpu_launches": int(done * kps),
        "roofline": {"bound": "hbm", "kernel": kernel_name + ("<float>" if sc.real_bits == 32 else "<double>"),
                     "achieved": real_gbs, "peak": peak, "unit": "GB/s", "frac": real_gbs / peak,
                     "frac_basis": frac_basis,
                     "frac_nominal": flood_gbs / peak, "achieved_nominal": flood_gbs,
                     "peak_source": peak_src, "frac_of_8TBs_spec": real_gbs / 8000.0,
                     "bytes_per_cell": fb, "kernel_ms": flood_ms, "kernel_ms_every_chunk_computed": flood_ms_noskip,
                     "traffic": traffic, "traffic_unit": "bytes per launch (ncu dram__bytes_read.sum + dram__bytes_write.sum)",
                     "traffic_source": traffic_src,
                     "algorithmic_bytes": ncell * fb,
                     "note": "frac / achieved: bytes_per_cell x all cells / time of the kernel with EVERY chunk computed (dry-chunk skip off, "
                             "measured in this run): bytes that are moved.  frac_nominal / achieved_nominal: the same bytes / time of the default "
                             "kernel, which neither reads nor writes chunks of dry ground (DESIGN.md 7 'dry chunks'): a figure of merit that "
                             "credits bytes never moved, not a bandwidth",
                     "timed_with": f"cudaEvent before each launch over {KP} steps (sim_step_profiled) right after the timed region"},
        "kernels_ms_per_step": {k: v / KP for k, v in kms.items()},
        "ped_roofline": {"bound": "hbm", "kernels": "bin_count+bin_scan+scatter+occupancy+ped_step", "achieved": ped_gbs, "peak": peak,
                         "unit": "GB/s", "frac": ped_gbs / peak, "ms": ped_ms,
                         "note": "byte view of the whole pedestrian branch; ped_step itself is XU-bound, see ped_step_roofline"},
        "ped_step_roofline": xu,
        "cpu_baseline": cpu,
        "final": {"t": st1["t"], "volume": st1["volume"], "max_h": st1["max_h"], "hist": st1["hist"],
                  "neg_depth_clamps": st1["neg_depth_clamps"]},
    }
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def run_slabs(args):
    """SURVEY 8f-4 on ONE GPU: the grid cut into --slabs row slabs, one handle each, all on cuda:0
    (no multi-GPU node here): what the slab machinery costs per step against the single handle
    (host-sequenced launches and events instead of a replayed graph; halo rows and the pedestrians'
    cells read through the slab tables), and that the result is bit-identical."""
    import torch
    from paper_1908_05232_b200 import binding, build
    torch.cuda.set_device(0)
    build.build()
    K, W = args.steps, max(args.warmup, 3)
    sc = scenario(args.config)
    one = binding.Sim(sc)
    slabs = binding.SlabSim(sc, args.slabs)
    ms = {}
    for name, g in (("single", one), ("slabs", slabs)):
        g.step(W)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); g.step(K); e1.record()
        torch.cuda.synchronize()
        ms[name] = e0.elapsed_time(e1) / K
    a, b = slabs.read_conserved(), one.read_conserved()
    same = all(bool(np.array_equal(a[k], b[k])) for k in ("h", "qx", "qy")) and slabs.stats()["dt"] == one.stats()["dt"]
    diff = max(float(np.max(np.abs(a[k].astype(np.float64) - b[k]))) / max(float(np.max(np.abs(b[k]))), 1e-300) for k in ("h", "qx", "qy"))
    ncell = sc.nx * sc.ny
    print(json.dumps({
        "metric": "flood cell-updates/s (coupled step)", "value": ncell / (ms["slabs"] * 1e-3), "unit": "cell-updates/s",
        "n_gpus": 1, "steps": K, "warmup": W, "ms_per_step": ms["slabs"], "higher_is_better": True, "scaling": "strong",
        "vs_baseline": None, "dtype": "f32" if sc.real_bits == 32 else "f64", "data": "synthetic",
        "config": {"workload": f"config{args.config}: {sc.name}", "parallelism": f"{len(slabs.sims)} row slabs, all on one GPU (emulation of SURVEY 8f-4; unmeasured on multi-GPU hardware)",
                   "rows_per_slab": [c[1] for c in slabs.cuts]},
        "single_handle_ms_per_step": ms["single"], "slab_overhead": ms["slabs"] / ms["single"] - 1.0,
        "bit_identical_to_single_handle": same, "max_rel_diff_to_single_handle": diff,
        "note": "bit-identical whenever the people -> flow coupling is off or there are no pedestrians (tests/test_gpu_slabs.py); with it on, "
                "two runs of the SAME handle differ as well: pair forces are summed in the order of the counting sort's atomics"}))


def run_slab_ranks(args):
    """SURVEY 8f-4 under torchrun: ONE grid cut into WORLD_SIZE row slabs, one process and GPU per slab
    (binding.SlabRank: CUDA-IPC peer memory, one 8-byte MAX all-reduce per step over NCCL); strong
    scaling of the coupled step.  With --slab-backend gloo all ranks may share one GPU (how the path is
    exercised on a single-GPU box: the reduction then goes through the host and dominates the time)."""
    import torch
    import torch.distributed as dist
    from paper_1908_05232_b200 import binding, build
    world, rank, local = int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0"))
    dev = local % max(torch.cuda.device_count(), 1)
    torch.cuda.set_device(dev)
    if args.slab_backend == "nccl":
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{dev}"))
    else:
        dist.init_process_group("gloo")
    if rank == 0:
        build.build()
    dist.barrier()
    K, W = args.steps, max(args.warmup, 3)
    sc = scenario(args.config)
    g = binding.SlabRank(sc, device=f"cuda:{dev}")
    g.step(W)
    torch.cuda.synchronize(); dist.barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(); g.step(K); e1.record()
    torch.cuda.synchronize(); dist.barrier()
    t = torch.tensor([e0.elapsed_time(e1)], dtype=torch.float64, device=f"cuda:{dev}" if args.slab_backend == "nccl" else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms = float(t.item())
    st = g.sim.stats()
    if rank == 0:
        ncell = sc.nx * sc.ny
        print(json.dumps({
            "metric": "flood cell-updates/s (coupled step)", "value": ncell * K / (ms * 1e-3), "unit": "cell-updates/s",
            "n_gpus": world, "steps": K, "warmup": W, "ms_per_step": ms / K, "higher_is_better": True, "scaling": "strong",
            "vs_baseline": None, "dtype": "f32" if sc.real_bits == 32 else "f64", "data": "synthetic",
            "config": {"workload": f"config{args.config}: {sc.name}", "parallelism": f"{world} row slabs, one process each ({args.slab_backend}; "
                       f"{torch.cuda.device_count()} device(s) visible)", "flood_variant": g.sim.flood_variant()},
            "final": {"t": st["t"], "step": st["step"]}}))
    g.close()
    dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=500)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--config", type=int, default=5, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--flood-variant", type=int, default=-1, choices=list(range(-1, 5)), help="-1: the library default")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--flood-order", type=int, default=1, choices=[1, 2], help="1: the paper's first-order flood step; 2: MUSCL-Hancock (SURVEY 8f-2)")
    ap.add_argument("--march-rows", type=int, default=0, help="rows per chunk of the row-marching flood kernel (0: library default)")
    ap.add_argument("--no-overlap", action="store_true", help="pedestrian step and flood step in one chain instead of parallel graph branches")
    ap.add_argument("--slabs", type=int, default=0, help="SURVEY 8f-4: cut the grid into this many row slabs, all on cuda:0, and compare with the single handle")
    ap.add_argument("--slab-ranks", action="store_true", help="SURVEY 8f-4 under torchrun: one grid, one row slab per rank (strong scaling) instead of one replica per rank")
    ap.add_argument("--slab-backend", default="nccl", choices=["nccl", "gloo"], help="collective for the 8-byte wave-speed reduction of --slab-ranks")
    args = ap.parse_args()
    if args.slab_ranks and args.impl == "ours":
        return run_slab_ranks(args)
    if args.slabs > 1 and args.impl == "ours":
        return run_slabs(args)
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()

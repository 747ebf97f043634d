#!/usr/bin/env python
"""bench.py -- one JSON line per run.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg3_detailed] [--impl ours|reference]

A step = one pass of the whole hot path over one batch of synthetic input: srp_build_designs
(mesh generation + BVH build, S0-S1) followed by srp_forces (S2-S7) for every (design, direction)
pair of the workload.  metric = photon-bounce segments per second (BASELINE.json; every ray cast, hit or
miss, INCLUDING primaries that a beam test resolves as misses without generating them), whole job.  Read
`forces_per_s`, `hits_per_s` and `traced_segments_per_s` first: they cannot be inflated by empty emitter area.
N > 1 (torchrun): designs are replicated, each rank takes its own S directions of an N*S-direction Fibonacci
sphere (weak scaling, no data-path collective).

`--workload paper_map` is the paper's own workload shape (100 k (direction, design) records x 1000
samples, ~1 k faces, every record its own design): a step = srp_forces_per_sample over all records.
`--plain-launches` runs the beam / bounce loop as plain launches instead of a conditional CUDA graph, so that
ncu lists its kernels (same results, a little slower).
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2602_10712_b200 import workloads as W          # noqa: E402

METRIC = "photon-bounce segments/s"
UNIT = "segments/s"
# FP32 peak the ALU roofline is quoted against: 148 SMs x 128 FP32 lanes x 2 flop x 1.965 GHz
# (B200_PROFILING.md unit counts and max SM clock); the probed FMA-chain figure is printed beside it.
FP32_PEAK_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12
# algorithmic work per unit: 12 flop per ray-box slab test, 44 per Moller-Trumbore
# ray-triangle test, 20 per ray-triangle test in the emitter frame (three 2-D edge functions + depth),
# 80 per shaded hit; 64 B per node visited (2 boxes), 48 B per triangle fetched.  Beam work (DESIGN.md
# "Kernels"): 32 flop per beam-box test (12 FMA + 8 add), 14 per rectangle-triangle culling test
# (6 FMA + 2 min), 110 per triangle set-up (9 dot products, 3 edge functions, depth plane).
FLOP_BOX, FLOP_TRI, FLOP_TRI2D, FLOP_HIT = 12.0, 44.0, 20.0, 80.0
FLOP_BEAM_BOX, FLOP_RECT, FLOP_SETUP = 32.0, 14.0, 110.0
BYTES_NODE, BYTES_TRI = 64.0, 48.0
TRAFFIC_FILE = os.path.join(ROOT, "profiles", "r2_traffic.json")


def kernel_source_hash():
    """Hash of the CUDA sources: a DRAM-traffic figure taken from an ncu capture is printed only for the build it
    was captured on."""
    import hashlib
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2602_10712_b200", "csrc")
    for f in sorted(os.listdir(d)):
        h.update(f.encode()); h.update(open(os.path.join(d, f), "rb").read())
    return h.hexdigest()[:16]


def ncu_figures(workload):
    """Figures of the trace kernels from the committed `ncu` captures of this workload (profiles/r2_traffic.json:
    DRAM and L2 bytes per segment, FMA-pipe utilisation, issue slots, lanes, the commands, and a hash of csrc/) --
    or (None, why) when there is no capture of THIS build of the kernels."""
    try:
        t = json.load(open(TRAFFIC_FILE))
    except (OSError, ValueError):
        return None, "no ncu capture on file"
    e = t.get(workload)
    if not e:
        return None, "no ncu capture of this workload on file"
    if e.get("source_hash") != kernel_source_hash():
        return None, "the ncu capture on file (%s) is of another build of the kernels" % e.get("capture")
    return e, "%s: %s" % (e.get("capture"), e.get("command"))


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None,
                    help="timed steps; default 3, 20 for the short steps of paper_map (so that the clocks are sampled under load)")
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg3_detailed", choices=sorted(W.CONFIGS) + sorted(W.SAMPLE_CONFIGS))
    ap.add_argument("--plain-launches", action="store_true",
                    help="beam / bounce loop as plain launches (for ncu); a little slower, same results")
    ap.add_argument("--scale", type=float, default=1.0,
                    help="fraction of the workload's sun directions (debug; < 1 marks the line invalid)")
    args = ap.parse_args()
    if args.steps is None:
        args.steps = 20 if args.workload in W.SAMPLE_CONFIGS else 3
    return args


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        self.thread.join(timeout=5)
        sm, mx, reasons, pw = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except (ValueError, IndexError):
                continue
            for n, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def oracle_sample(cfg, n_pairs, N, seed=0):
    """Times the oracle, as it stands, on n_pairs pairs of the workload at N rays, one single-threaded
    oracle call per pair spread over the host cores.  Returns (segments, seconds, threads used)."""
    from concurrent.futures import ThreadPoolExecutor
    from oracle import srp_oracle as O
    O.build()
    th, sun = cfg.params(), cfg.sun_dirs()
    rng = np.random.default_rng(123)
    if isinstance(cfg, W.SampleConfig):            # record m = (design m, direction m), direction index 0 in the counters
        recs = [int(x) for x in rng.integers(0, cfg.M, n_pairs)]
        threads = min(os.cpu_count() or 1, n_pairs)

        def one_rec(m):
            v, mt = O.build_mesh(cfg.family, th[m], k=m)
            return O.forces(v, mt, sun[m:m + 1], N, cfg.B, seed=seed, k=m, j0=0)["stats"]["segments"]

        t0 = time.perf_counter()
        with ThreadPoolExecutor(threads) as ex:
            segs = sum(ex.map(one_rec, recs))
        return segs, time.perf_counter() - t0, threads
    pairs = [(int(rng.integers(0, cfg.D)), int(rng.integers(0, cfg.S))) for _ in range(n_pairs)]
    meshes = {k: O.build_mesh(cfg.family, th[k], k=k) for k in sorted({p[0] for p in pairs})}
    threads = min(os.cpu_count() or 1, n_pairs)

    def one(p):
        v, m = meshes[p[0]]
        return O.forces(v, m, sun[p[1]:p[1] + 1], N, cfg.B, seed=seed, k=p[0], j0=p[1])["stats"]["segments"]

    t0 = time.perf_counter()
    with ThreadPoolExecutor(threads) as ex:
        segs = sum(ex.map(one, pairs))
    return segs, time.perf_counter() - t0, threads


# bounded oracle samples per workload: (pairs per host core, rays per pair) ~ 10-30 s of CPU work
ORACLE_SAMPLE = {"cfg1_plate": (8, 1 << 16), "cfg2_boxwing": (8, 1 << 18), "cfg3_detailed": (2, 1 << 11),
                 "cfg4_sweep": (16, 1 << 16), "cfg5_sail": (1, 1 << 8), "paper_map": (64, 1 << 10)}


def all_configs():
    return {**W.CONFIGS, **W.SAMPLE_CONFIGS}


def run_reference(args, rank, world):
    """--impl reference: the oracle (oracle/, fp64, brute force, one thread per call) on the host cores,
    each step a bounded sample of the workload.  Rank 0 only."""
    if rank != 0:
        return
    cfg = all_configs()[args.workload]
    per_core, N = ORACLE_SAMPLE[args.workload]
    cores = os.cpu_count() or 1
    n_pairs = per_core * cores
    for _ in range(args.warmup):
        oracle_sample(cfg, min(n_pairs, cores), max(N >> 4, 1))
    segs = secs = 0.0
    for s in range(args.steps):
        a, b, threads = oracle_sample(cfg, n_pairs, N, seed=s)
        segs += a; secs += b
    value = segs / secs
    sample = "%d random pairs x N=%d rays per step, %d steps" % (n_pairs, N, args.steps)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * secs / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": {"workload": args.workload, "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def run_ours(args, rank, world, local_rank):
    import torch
    import torch.distributed as dist
    from paper_2602_10712_b200.binding import Context
    from paper_2602_10712_b200 import sharding

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product has no CPU path")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    cfg = all_configs()[args.workload]
    per_sample = isinstance(cfg, W.SampleConfig)
    ctx = Context(local_rank)
    opts = {"plain_launches": 1 if args.plain_launches else 0}
    ctx.srp_set_options(**opts)
    theta_np = cfg.params()
    if per_sample:                          # every rank its own records (weak scaling): rank r takes records r::world of M * world
        M = max(1, int(round(cfg.M * args.scale)))
        full = W.SampleConfig(cfg.name, cfg.family, M * world, cfg.N, cfg.B)
        theta_np, sun_np = np.ascontiguousarray(full.params()[rank::world]), np.ascontiguousarray(full.sun_dirs()[rank::world])
        n_forces, S = M, 1
        out_shape = (M, 3)
    else:
        S = max(1, int(round(cfg.S * args.scale)))
        sun_np = sharding.weak_scaling_directions(S, rank, world, cfg.front_hemisphere)
        n_forces = cfg.D * S
        out_shape = (cfg.D, S, 3)
    theta = torch.from_numpy(theta_np).to(dev)
    sun = torch.from_numpy(sun_np).to(dev)
    out = torch.empty(out_shape, dtype=torch.float32, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)       # > 126 MB L2
    peaks = ctx.srp_probe_peaks()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def step(seed):
        """one pass of the whole hot path (S0-S7); returns the designs handle to free (None for per-sample records)"""
        if per_sample:
            ctx.srp_forces_per_sample(cfg.family, theta, sun, cfg.N, cfg.B, seed, W.MESH_SEED, out=out)
            return None
        dz = ctx.srp_build_designs(cfg.family, theta, W.MESH_SEED)
        ctx.srp_forces(dz, sun, cfg.N, cfg.B, seed, out=out)
        return dz

    for s in range(args.warmup):
        dz = step(1000 + s)
        torch.cuda.synchronize()
        if dz is not None:
            dz.free()

    sampler = ClockSampler(local_rank)
    sampler.start()
    barrier()
    launches0 = ctx.srp_launch_count()
    t_total = 0.0
    tot = {"segments": 0, "hits": 0, "launched": 0, "primary_miss": 0, "beam_miss": 0, "mask_escapes": 0}
    for s in range(args.steps):
        flush.zero_()                                                   # L2 flush between timed steps
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        dz = step(s)
        e1.record()
        torch.cuda.synchronize()
        t_total += e0.elapsed_time(e1) * 1e-3
        st = ctx.srp_get_stats()
        tot["segments"] += st["segments"]; tot["hits"] += sum(st["hits_at_depth"]); tot["launched"] += st["launched"]
        tot["primary_miss"] += st["primary_miss"]; tot["mask_escapes"] += st["mask_escapes"]
        tot["beam_miss"] += st["beam_tile_miss"] + st["beam_block_miss"] + st["beam_group_miss"]
        if dz is not None:
            dz.free()
    gpu_launches = ctx.srp_launch_count() - launches0                   # counted by the library, loop rounds on the device
    barrier()
    clocks = sampler.stop()
    t_max, segs_all = sharding.combine_timing(t_total, tot["segments"], dev)

    # the trace kernels alone: CUDA events around the forces call only, designs resident (per-sample records: the whole
    # call, whose mesh kernels are < 2 % of it)
    if per_sample:
        flush.zero_()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        step(0)
        e1.record()
        torch.cuda.synchronize()
        t_kernel = e0.elapsed_time(e1) * 1e-3
        st_k = st_i = ctx.srp_get_stats()                               # its triangle tests are always counted
        dz = None
    else:
        dz = ctx.srp_build_designs(cfg.family, theta, W.MESH_SEED)
        ctx.srp_forces(dz, sun, cfg.N, cfg.B, 0, out=out)               # builds the escape masks if this workload repays them
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        flush.zero_()
        e0.record()
        ctx.srp_forces(dz, sun, cfg.N, cfg.B, 0, out=out)
        e1.record()
        torch.cuda.synchronize()
        t_kernel = e0.elapsed_time(e1) * 1e-3
        st_k = ctx.srp_get_stats()
        # algorithmic work per segment from the instrumented kernels on every 64th direction
        ctx.srp_set_options(instrumented=1, **opts)
        sub = sun[::64].contiguous() if S >= 64 else sun
        ctx.srp_forces(dz, sub, cfg.N, cfg.B, 0)
        st_i = ctx.srp_get_stats()
        ctx.srp_set_options(**opts)
    seg_i = max(st_i["segments"], 1)
    per = {k: st_i[k] / seg_i for k in ("box_tests", "tri_tests", "beam_box_tests", "tri2d_tests", "tri_setups", "rect_tests")}
    hit_ps = sum(st_i["hits_at_depth"]) / seg_i
    flop_ps = (FLOP_BOX * per["box_tests"] + FLOP_TRI * per["tri_tests"] + FLOP_TRI2D * per["tri2d_tests"] +
               FLOP_BEAM_BOX * per["beam_box_tests"] + FLOP_RECT * per["rect_tests"] + FLOP_SETUP * per["tri_setups"] +
               FLOP_HIT * hit_ps)
    # node and triangle bytes the tests above read (beam descents and set-ups fetch each node / triangle once; the
    # per-sample kernel reads its triangles from shared memory: one 48-byte fetch per triangle and record)
    if per_sample:
        bytes_ps = BYTES_TRI * W.TRI_COUNT[cfg.family] * n_forces / max(st_k["segments"], 1)
    elif W.TRI_COUNT[cfg.family] <= 64:
        # designs without a hierarchy: a warp stages its design's <= 64 triangles in shared memory once per design and
        # tests from there -- 3 KB per (warp, design), nothing per segment
        bytes_ps = 0.0
    else:
        bytes_ps = (BYTES_NODE * (per["box_tests"] + per["beam_box_tests"]) / 2.0 +
                    BYTES_TRI * (per["tri_tests"] + per["tri_setups"]))
    ach_tflops = flop_ps * st_k["segments"] / t_kernel / 1e12
    l2_gbs = bytes_ps * st_k["segments"] / t_kernel / 1e9
    big = W.TRI_COUNT[cfg.family] > 64
    beams = st_i["beam_tile_miss"] + st_i["beam_block_miss"] + st_i["beam_group_miss"] + st_i["tri2d_tests"] > 0
    if per_sample:
        kernel = "sample_design_kernel"
    elif big:
        kernel = "beam_trace_kernel + bounce_trace_kernel (the beam / bounce loop)" if beams else "bvh_trace_kernel"
    else:
        kernel = "small_beam_kernel" if beams else "trace_kernel"
    frac_alu, frac_l2 = ach_tflops / FP32_PEAK_TFLOPS, l2_gbs / peaks["l2_read_gbs"]
    # "ncu decides which bound applies: the higher of sm__inst_executed_pipe_fma utilisation and
    # lts__t_bytes / probed L2 peak".  With a capture of this build on file that rule is applied to its figures (the L2
    # bytes per segment scaled to this launch); without one, to the algorithmic fractions.
    ncu, ncu_source = ncu_figures(args.workload)
    traffic = ncu["dram_bytes_per_segment"] * st_k["segments"] if ncu else None
    if ncu and ncu.get("lts_bytes_per_segment") is not None:
        l2_measured = ncu["lts_bytes_per_segment"] * st_k["segments"] / t_kernel / 1e9
        alu_binds = ncu["fma_pipe_pct"] / 100.0 >= l2_measured / peaks["l2_read_gbs"]
    else:
        l2_measured = None
        alu_binds = frac_alu >= frac_l2
    # an L2-bound line quotes the MEASURED L2 bytes when a capture of this build is on file: the algorithmic count
    # (roofline.l2: 64 B per node visit and lane) is what the lanes ask for, and lanes of a warp share node fetches
    l2_quote = l2_measured if l2_measured is not None else l2_gbs
    roofline = {"bound": "alu" if alu_binds else "l2", "kernel": kernel,
                "achieved": ach_tflops if alu_binds else l2_quote, "peak": FP32_PEAK_TFLOPS if alu_binds else peaks["l2_read_gbs"],
                "unit": "TFLOP/s" if alu_binds else "GB/s", "frac": frac_alu if alu_binds else l2_quote / peaks["l2_read_gbs"],
                "frac_source": ("algorithmic flops of the counted tests" if alu_binds else
                                ("lts__t_bytes of the ncu capture, per segment, x this launch's segments" if l2_measured is not None
                                 else "algorithmic node + triangle bytes of the counted tests")),
                "traffic": traffic, "traffic_source": ncu_source,
                "ncu": ({"fma_pipe_pct": ncu["fma_pipe_pct"], "alu_pipe_pct": ncu.get("alu_pipe_pct"), "issue_pct": ncu.get("issue_pct"),
                         "lanes_of_32": ncu.get("lanes"), "l2_gbs_this_launch": l2_measured,
                         "l2_frac_of_probed_peak": (l2_measured / peaks["l2_read_gbs"]) if l2_measured is not None else None}
                        if ncu else None),
                "alu": {"achieved_tflops": ach_tflops, "peak_tflops": FP32_PEAK_TFLOPS, "frac": frac_alu,
                        "peak_source": "derived: 148 SM x 128 lanes x 2 x 1.965 GHz; probed FMA chain %.1f TFLOP/s" % peaks["fp32_tflops"],
                        "flop_per_segment": flop_ps},
                "l2": {"achieved_gbs": l2_gbs, "probed_peak_gbs": peaks["l2_read_gbs"], "frac": frac_l2,
                       "bytes_per_segment": bytes_ps,
                       "note": "algorithmic node + triangle bytes of the counted tests; ncu's lts__t_bytes is in profiles/"},
                "tests_per_segment": per, "hits_per_segment": hit_ps,
                "beam_resolved": {k: st_k[k] / max(st_k["launched"], 1) for k in
                                  ("beam_tile_miss", "beam_block_miss", "beam_group_miss", "beam_fallback")},
                "escapes_resolved_by_mask": st_k["mask_escapes"] / max(st_k["escaped"], 1),
                "queued_rays_per_segment": st_k["queued_rays"] / max(st_k["segments"], 1), "loop_rounds": st_k["loop_rounds"],
                "kernel_ms": 1e3 * t_kernel, "kernel_segments": st_k["segments"]}

    # end to end through the host-buffer entry point: theta, sun_dirs from pinned host memory, forces back
    theta_h = torch.from_numpy(theta_np).pin_memory()
    sun_h = torch.from_numpy(sun_np).pin_memory()
    out_h = torch.empty(out_shape, dtype=torch.float32).pin_memory()
    if dz is not None:
        dz.free()
    barrier()
    e2e_steps = max(1, min(args.steps, 2))
    t_e2e = 0.0
    seg_e2e = 0
    for s in range(e2e_steps):
        flush.zero_()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        if per_sample:
            ctx.srp_forces_per_sample(cfg.family, theta_h.to(dev, non_blocking=True), sun_h.to(dev, non_blocking=True),
                                      cfg.N, cfg.B, s, W.MESH_SEED, out=out)
            out_h.copy_(out)                                            # device -> pinned host, synchronous
        else:
            dz = ctx.srp_build_designs(cfg.family, theta_h.to(dev, non_blocking=True), W.MESH_SEED)
            ctx.srp_forces_host(dz, sun_h, cfg.N, cfg.B, s, out_host=out_h)
        checksum = float(out_h.sum())                                     # the result is read on the host
        t_e2e += time.perf_counter() - t0
        seg_e2e += ctx.srp_get_stats()["segments"]
        if not per_sample:
            dz.free()
    t_e2e_max, seg_e2e_all = sharding.combine_timing(t_e2e, seg_e2e, dev)
    e2e = {"value": seg_e2e_all / t_e2e_max, "unit": UNIT,
           "h2d_bytes_per_step": int(theta_np.nbytes + sun_np.nbytes), "d2h_bytes_per_step": int(out_h.numel() * 4),
           "steps": e2e_steps, "checksum": checksum}

    cpu = None
    if rank == 0 and world == 1:
        per_core, N_o = ORACLE_SAMPLE[args.workload]
        n_pairs = per_core * (os.cpu_count() or 1)
        a, b, threads = oracle_sample(cfg, n_pairs, N_o)
        cpu = {"value": a / b, "unit": UNIT, "cores": threads, "kind": "oracle",
               "sample": "%d random %s x N=%d rays (fp64, brute force over all %d triangles)" %
                         (n_pairs, "records" if per_sample else "pairs", N_o, W.TRI_COUNT[cfg.family]),
               "per_core": a / b / threads}
    if rank == 0:
        traced = tot["segments"] - tot["beam_miss"] - tot["mask_escapes"]
        conf = {"workload": args.workload, "rays": cfg.N, "max_bounces": cfg.B,
                "triangles_per_design": W.TRI_COUNT[cfg.family],
                "l2": "256 MiB buffer written between timed steps", "parallelism": "dp%d" % world,
                "loop": "plain launches" if args.plain_launches else "conditional CUDA graph",
                "valid": args.scale == 1.0}
        if per_sample:
            conf.update({"records_per_gpu": n_forces, "designs": "one per record (PAPER.md:146, 159, 352)"})
        else:
            conf.update({"designs": cfg.D, "directions_per_gpu": S})
        line = {"metric": METRIC, "value": segs_all / t_max, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": 1e3 * t_max / args.steps, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic", "config": conf,
                # what the headline cannot inflate (this rank's counts over this rank's time; x n_gpus for the job)
                "forces_per_s": n_forces * world * args.steps / t_max,
                "hits_per_s": tot["hits"] * world / t_max,
                "traced_segments_per_s": traced * world / t_max,
                "samples_per_s": tot["launched"] * world / t_max,
                "segments_resolved_without_tracing": 1.0 - traced / max(tot["segments"], 1),
                "primary_hit_fraction": 1.0 - tot["primary_miss"] / max(tot["launched"], 1),
                "hits_per_photon": tot["hits"] / max(tot["launched"], 1),
                "segments_per_photon": tot["segments"] / max(tot["launched"], 1),
                "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": int(gpu_launches),
                "clocks": clocks}
        if per_sample:
            line["paper_context"] = ("PAPER.md:352: 100 k (direction, design) x 1000 samples, ~1 k faces, < 10 s on an A100 "
                                     "(>= 1e7 samples/s; another estimator, another machine: context, not a baseline)")
        print(json.dumps(line), flush=True)
    ctx.close()
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
    else:
        run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()

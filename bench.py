#!/usr/bin/env python
"""bench.py -- one JSON line for the discrete-ordinates CT dose hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config configN]

A "step" is one pass of the whole hot path over one synthetic problem: uncollided ray trace ->
first-collision source -> group cascade of source-iteration sweeps -> dose map (
for config4 also a9, all source positions of this rank). Metric (BASELINE.json): S_N sweep
cell-angle-group updates/s over the whole step; `ms_per_step` is the cone-beam dose-map wall time.

  value      inputs resident in HBM, CUDA events on the library's stream around each step, L2 flushed
             between steps, max over ranks
  e2e        the same step through the C ABI with HOST buffers: material grid copied in from pinned
             memory (dos_set_material_host), dose map copied out (dos_dose_host), wall clock
  roofline   the sweep kernel: algorithmic (compulsory) bytes per launch, (12 M + 1) N_v (read
             Q_fix[M] and phi_old[M], write phi_new[M], 1 B material id), / its mean CUDA-event duration inside
             the timed region, against MEASURED_PEAKS.json's HBM copy bandwidth; `traffic` = measured DRAM bytes
             per launch from the ncu capture kept under profiles/; the FP32-pipe view (algorithmic flop against
             SMs x 128 lanes x 2 x clock) under roofline.alu
  cpu_baseline  the fp64 oracle, as it stands, on this box's host cores, on a bounded sample

--impl reference times the oracle itself (there is no reference implementation: the paper's program is
closed source). N > 1: one process per GPU (under torchrun, or spawned by this script when WORLD_SIZE is
unset): a single projection does not shard, so every rank runs an independent replica ("weak"); config4's
36 source positions are sharded over the ranks (scan.shard_positions) and the partial dose maps summed with
one all-reduce (scan.all_reduce_dose), the only exchange the method has ("strong").
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

METRIC = "sn_sweep_cell_angle_group_updates_per_s"
UNIT = "updates/s"
WORKLOADS = {
    "config1": "config1: 16^3 water cube, G=4, S4 (24 angles), P1, 10 iterations, isotropic point source",
    "config2": "config2: 64x64x16 water cylinder in air, G=19, S8 (80 angles), P3, 20 iterations, one cone-beam projection",
    "config3": "config3: 128x128x64 water cylinder, G=19, S16 (288 angles), P5, 20 iterations, one projection",
    "config4": "config4: 256x256x64 abdomen-like phantom, G=19, S8, P3, 15 iterations, 36-position axial scan, doses summed",
    "config5": "config5: 256^3 abdomen-like phantom, G=19, S16 (288 angles), P5, 20 iterations, one projection",
    # the shape of the paper's own runs (Tables 2 and 6); context, not a BASELINE config
    "paper_coarse": "paper-shaped: 64x64x16 (7.81 mm), 35 cm water cylinder, 7 groups 10-100 keV, S6/P0 (or --sn/--pl), 20 iterations, 16-position scan (--positions 1 = single projection)",
    "paper_fine": "paper-shaped: 256x256x64 (1.95 mm), 35 cm water cylinder, 7 groups 10-100 keV, S6/P0 (or --sn/--pl), 20 iterations, 16-position scan (--positions 1 = single projection)",
}
# bounded oracle samples (about 10-30 s of CPU work): same mesh/quadrature/P_L, fewer groups/iterations;
# the work per cell-angle-group update is the same as in the full workload
ORACLE_SAMPLE = {
    "config1": ({}, "the full config1 problem"),
    "config2": (dict(n_iter=2), "config2 with 2 of 20 source iterations per group (all 19 groups)"),
    "config3": (dict(n_group=1, n_iter=1), "config3 mesh/S16/P5, 1 group, 1 source iteration"),
    "config4": (dict(n_group=1, n_iter=1, n_pos=1), "config4 mesh/S8/P3, 1 position, 1 group, 1 source iteration"),
    "config5": (dict(nz=16, n_group=1, n_iter=1), "config5 in-plane mesh 256x256, S16/P5, 16 of 256 slices, 1 group, 1 iteration"),
    "paper_coarse": (dict(n_pos=1), "paper_coarse, one source position in full (7 groups x 20 iterations)"),
    "paper_fine": (dict(n_pos=1, n_iter=1), "paper_fine, one source position, 7 groups x 1 source iteration"),
}


def _peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md, 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.idx = str(gpu_index)
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "200", "-i", self.idx], stdout=subprocess.PIPE, text=True)
        except OSError:
            self.proc = None
            return
        self.t = threading.Thread(target=self._read, daemon=True)
        self.t.start()

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, reasons, pw = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            if len(r) < 9:
                continue
            try:
                sm.append(float(r[1])); mx.append(float(r[2])); pw.append(float(r[3]))
            except ValueError:
                continue
            for n, v in zip(names, r[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def _cores():
    """Threads the oracle uses: OMP_NUM_THREADS if set, else the PHYSICAL core count."""
    env = os.environ.get("OMP_NUM_THREADS")
    if env:
        return int(env)
    try:
        import psutil
        n = psutil.cpu_count(logical=False)
        if n:
            return int(n)
    except Exception:
        pass
    return os.cpu_count() or 1


def time_oracle(config, steps, warmup):
    """Times oracle.run_problem on the bounded sample; returns (updates/s, seconds per step, sample text)."""
    import oracle
    from paper_1811_12391_b200.inputs import make_problem, n_updates
    ov, text = ORACLE_SAMPLE[config]
    p = make_problem(config, **ov)
    oracle.build()
    os.environ.setdefault("OMP_NUM_THREADS", str(_cores()))      # read by the OpenMP runtime when the library first runs
    for _ in range(warmup):
        oracle.run_problem(p)
    t0 = time.perf_counter()
    for _ in range(steps):
        oracle.run_problem(p)
    dt = (time.perf_counter() - t0) / steps
    return n_updates(p) / dt, dt, text


def run_reference(args):
    """--impl reference: the oracle is the only reference there is. Rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    rate, dt, text = time_oracle(args.config, args.steps, min(args.warmup, 1))
    cores = _cores()
    line = {"impl": "reference", "metric": METRIC, "value": rate, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOADS[args.config], "sample": text},
            "cpu_baseline": {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": text},
            "e2e": {"value": rate, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_1811_12391_b200 import dos
    from paper_1811_12391_b200.inputs import make_problem, n_updates

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    ov = {}
    if args.positions and len(args.config) > 0 and args.config in ("config4", "paper_coarse", "paper_fine"):
        ov["n_pos"] = args.positions
    if args.sn:
        ov["sn"] = args.sn
    if args.pl is not None:
        ov["pl"] = args.pl
    from paper_1811_12391_b200 import scan
    p = make_problem(args.config, **ov)
    # A single projection does not shard: every rank runs the whole workload on its own GPU (independent replicas,
    # weak scaling). The axial scan (config4) shards by source position: rank r takes positions r, r + world, ...,
    # and the partial dose maps are summed with one all-reduce (strong scaling: the total work is fixed).
    sharded = world > 1 and len(p["sources"]) > 1 and args.scan == "separate"
    mine = scan.shard_positions(len(p["sources"]), rank, world) if sharded else list(range(len(p["sources"])))
    m = p["mesh"]
    nv = m["nx"] * m["ny"] * m["nz"]
    M = (p["P_L"] + 1) ** 2
    n_ang = len(p["quadrature"]["w"])
    summed = args.scan == "summed" and len(mine) > 1    # the positions form ONE source, one solve
    updates_all = n_updates(p) // (len(p["sources"]) if summed else 1)          # the whole problem
    job_updates = updates_all if sharded else world * updates_all               # what all ranks together process per step
    stream = torch.cuda.Stream(device=dev)
    with torch.cuda.stream(stream):
        # positions swept together: 4 on meshes that fill the GPU by themselves (measured: 8 gains nothing at config 4), 16 on
        # small ones, where a single position leaves most SMs idle (paper-shaped coarse mesh, 16 positions: 105 ms in
        # batches of 4, 85 ms in one batch of 16); summed-source mode needs the n_batch > 1 buffers
        batch = args.batch if args.batch > 0 else (16 if nv <= (1 << 17) else 4)
        n_batch = 2 if summed else max(1, min(batch, len(mine)))
        ctx = dos.Context(p["mesh"], p["material"], p["sigma_t"], p["sigma_s"], p["kerma"], p["quadrature"], p["P_L"],
                          device=dev, stream=stream, n_batch=n_batch)
        dose = ctx.new_field(groups=False)
        flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)     # > 126 MB L2
    ctx.dos_set_option("profile", 1)
    mat_pinned = torch.from_numpy(np.ascontiguousarray(p["material"])).pin_memory()
    dose_pinned = torch.empty(nv, dtype=torch.float32).pin_memory()
    mat_host, dose_host = mat_pinned.numpy(), dose_pinned.numpy().reshape(p["material"].shape)

    def step_summed():
        for n, s in enumerate(mine):
            ctx.dos_uncollided_sum(p["sources"][s], p["spectrum"], first=(n == 0))
        ctx.dos_solve(p["n_iter"])

    def step_device():
        if summed:
            step_summed()
            ctx.dos_dose(dose, accumulate=False)
            return
        scan.run_scan(ctx, p, mine, dose)
        if sharded:
            with torch.cuda.stream(stream):
                scan.all_reduce_dose(dose)

    def step_e2e():
        ctx.dos_set_material_host(mat_host)
        if summed:
            step_summed()
            ctx.dos_dose_host(dose_host, accumulate=False)
            return
        if len(mine) > 1 or sharded:
            scan.run_scan(ctx, p, mine, dose)         # doses of the positions summed on the device, the sum copied to the host
            with torch.cuda.stream(stream):           # the context's stream, not torch's current one: the copy must
                if sharded:                           # come after the last dos_dose
                    scan.all_reduce_dose(dose)
                dose_pinned.copy_(dose.reshape(-1), non_blocking=True)
            stream.synchronize()
        else:
            ctx.dos_uncollided(p["sources"][mine[0]], p["spectrum"])
            ctx.dos_solve(p["n_iter"])
            ctx.dos_dose_host(dose_host, accumulate=False)

    def l2_flush():
        with torch.cuda.stream(stream):
            flush.fill_(1)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    # ---------------- warm-up ----------------
    for _ in range(args.warmup):
        step_device()
    ctx.dos_check()
    # ---------------- timed: device-resident ----------------
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    ctx.dos_profile_reset()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    barrier()
    w0 = time.perf_counter()
    for a, b in ev:
        l2_flush()
        a.record(stream)
        step_device()
        b.record(stream)
    barrier()
    wall = time.perf_counter() - w0
    ctx.dos_check()
    prof = ctx.dos_profile()
    step_ms = [a.elapsed_time(b) for a, b in ev]
    total_ms = float(sum(step_ms))
    # ---------------- timed: end to end through the C ABI with host buffers ----------------
    step_e2e()
    torch.cuda.synchronize(dev)
    e2e_s = []
    barrier()
    for _ in range(args.steps):
        l2_flush()
        torch.cuda.synchronize(dev)
        t0 = time.perf_counter()
        step_e2e()
        torch.cuda.synchronize(dev)
        e2e_s.append(time.perf_counter() - t0)
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    e2e_total = float(sum(e2e_s))
    # phase split (one extra untimed-for-the-metric step, CUDA events on the same stream)
    pe = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
    pe[0].record(stream)
    ctx.dos_uncollided(p["sources"][mine[0] if mine else 0], p["spectrum"])
    pe[1].record(stream)
    ctx.dos_solve(p["n_iter"])
    pe[2].record(stream)
    ctx.dos_dose(dose, False)
    pe[3].record(stream)
    torch.cuda.synchronize(dev)
    phases = {"uncollided": pe[0].elapsed_time(pe[1]), "solve": pe[1].elapsed_time(pe[2]), "dose": pe[2].elapsed_time(pe[3])}

    if world > 1:
        t = torch.tensor([total_ms, e2e_total], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms, e2e_total = float(t[0]), float(t[1])
    if rank == 0:
        peak, peak_src = _peaks()
        sweep_ms = prof["sweep_ms"] / max(prof["sweep_launches"], 1)
        # problems per sweep launch: a position batch sweeps up to n_batch positions in one launch
        per_launch = 1.0 if summed else len(mine) / max(1, -(-len(mine) // n_batch))
        sweep_bytes = (12 * M + 1) * nv * per_launch     # compulsory: read Q_fix[M] + phi_old[M], write phi_new[M] (fp32), 1 B material id
        achieved = sweep_bytes / (sweep_ms * 1e-3) / 1e9 if sweep_ms > 0 else 0.0
        flop = (4 * M + 12) * nv * n_ang * per_launch
        rt_ms = prof["raytrace_ms"] / max(prof["raytrace_launches"], 1)
        traffic = None
        sweep_name = "sweep_umma_kernel" if M >= 25 else "sweep_kernel"     # tensor-memory sweep from P4 up, FFMA sweep below
        tpath = os.path.join(ROOT, "profiles", "traffic.csv")     # ncu dram bytes per launch, copied from profiles/*.md
        if os.path.exists(tpath):
            with open(tpath) as f:
                for row in f.read().splitlines()[1:]:
                    c = row.split(",")
                    if len(c) >= 3 and c[0] == args.config and c[1] == sweep_name:
                        traffic = int(c[2])
        # FP32 pipe peak: SMs x 128 FP32 lanes x 2 flop x SM clock
        sms = torch.cuda.get_device_properties(dev).multi_processor_count
        mhz = (clocks or {}).get("sm_max_mhz") or 1965.0
        alu_peak = sms * 128 * 2 * mhz * 1e6 / 1e12
        tflops = flop / (sweep_ms * 1e-3) / 1e12 if sweep_ms > 0 else 0.0
        line = {
            "metric": METRIC, "value": job_updates * args.steps / (total_ms * 1e-3), "unit": UNIT,
            "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": total_ms / args.steps,
            "higher_is_better": True, "scaling": "strong" if sharded else "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": WORKLOADS[args.config] + (" -- summed-source mode: the positions form ONE source, one solve"
                                                             if summed else ""), "positions_per_rank": len(mine),
                       "position_batch": n_batch,
                       "parallelism": ("source positions sharded over ranks, one all-reduce of the dose map" if sharded else
                                       "replicas only") if world > 1 else "1 gpu",
                       "l2": "flushed between timed steps (256 MiB fill)", "arithmetic": "fp32 sweep/sources/dose, fp64 ray trace"},
            "dose_map_ms": total_ms / args.steps, "phases_ms": phases, "wall_s_timed_region": wall,
            "e2e": {"value": job_updates * args.steps / e2e_total, "unit": UNIT,
                    "ms_per_step": e2e_total / args.steps * 1e3, "h2d_bytes_per_step": int(nv), "d2h_bytes_per_step": int(4 * nv)},
            "gpu_launches": int(prof["kernel_launches"]),
            "clocks": clocks,
            "roofline": {"kernel": sweep_name, "bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s",
                         "frac": achieved / peak, "traffic": traffic, "peak_source": peak_src,
                         "algorithmic_bytes_per_launch": sweep_bytes,
                         "measured_dram_frac": (traffic / (sweep_ms * 1e-3) / 1e9 / peak) if (traffic and sweep_ms > 0) else None,
                         "alu": {"achieved": tflops, "peak": alu_peak, "unit": "TFLOP/s", "frac": tflops / alu_peak,
                                 "peak_source": f"derived: {sms} SMs x 128 FP32 lanes x 2 flop x {mhz:.0f} MHz (DESIGN.md section 7)",
                                 "algorithmic_flop_per_launch": flop},
                         "launch_ms": sweep_ms,
                         "launches": int(prof["sweep_launches"]), "share_of_step": prof["sweep_ms"] / total_ms if total_ms else None,
                         "updates_per_s_in_kernel": nv * n_ang * per_launch / (sweep_ms * 1e-3) if sweep_ms > 0 else 0.0,
                         "problems_per_launch": per_launch},
            "raytrace": {"launch_ms": rt_ms, "launches": int(prof["raytrace_launches"]),
                         "achieved_gbs": (nv * (1 + 4 * p["n_group"])) / (rt_ms * 1e-3) / 1e9 if rt_ms > 0 else 0.0,
                         "hbm_frac": (nv * (1 + 4 * p["n_group"])) / (rt_ms * 1e-3) / 1e9 / peak if rt_ms > 0 else 0.0,
                         "voxels_per_s": nv / (rt_ms * 1e-3) if rt_ms > 0 else 0.0},
        }
        if not args.no_cpu_baseline:
            rate, dt, text = time_oracle(args.config, 1, 0)
            line["cpu_baseline"] = {"value": rate, "unit": UNIT, "cores": _cores(), "kind": "oracle", "sample": text,
                                    "seconds": dt}
        print(json.dumps(line), flush=True)
    ctx.close()
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="config5", choices=sorted(WORKLOADS),
                    help="default: config5, the largest single-GPU workload (BASELINE.json's metric is not quoted on a config)")
    ap.add_argument("--positions", type=int, default=0, help="config4 / paper_*: source positions per step (default 36 / 16)")
    ap.add_argument("--batch", type=int, default=0, help="source positions swept together (dos_uncollided_batch); 1 = one by one, 0 = by mesh size (16 up to 2^17 voxels, else 4)")
    ap.add_argument("--sn", type=int, default=0, help="quadrature order override (paper_*: S2..S8)")
    ap.add_argument("--pl", type=int, default=None, help="scattering order override (paper_*: P0..P1)")
    ap.add_argument("--scan", default="separate", choices=["separate", "summed"],
                    help="config4: one solve per source position with doses summed (default, BASELINE.json), or all "
                         "positions as ONE source and one solve (the paper's CT-scan mode, PAPER.md:69-71)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3                                   # timing rule: at least 3 warm-up steps
    if args.impl == "reference":
        run_reference(args)
    elif args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # launched without torchrun: spawn the N ranks ourselves, one process per GPU, and relay rank 0's JSON line
        import socket
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        raise SystemExit(subprocess.call(cmd))
    else:
        run_ours(args)


if __name__ == "__main__":
    main()

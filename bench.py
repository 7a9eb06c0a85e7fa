#!/usr/bin/env python
"""bench.py -- one adaptive ray-tracing step (all hot-path rows: source dedup/merge, emit, march+deposit,
filter, split, finalise) on BASELINE.json's production configuration (config 5: 1024^3 fp32 fields, 10^6
sources, merging on), per GPU.  See DESIGN.md "Measurement".

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 5] [--n-src N]

Prints ONE JSON line (rank 0).  metric = ray-cell segments per second over the whole RT step.
`value`, `ms_per_step` and `e2e` time the PRODUCTION path: the ray loop as one CUDA-graph launch per trace.  The
roofline needs the march launches' own durations, which that loop cannot give, so after the timed region
`--profile-steps` extra step(s) (default 1) run through the host-enqueued loop with a CUDA-event pair around every
march launch (NYXRT_FLAG_LAUNCH_TIMING; same kernels, same results) and are reported under `profiling_pass`.
`roofline` is the march kernel against the fp64-pipe roof (bound "alu"; the kernel is issue-bound, not HBM-bound),
with the issue roof and the three HBM figures (contract bytes, counted bytes, DRAM bytes measured by ncu) beside it.
N > 1 (torchrun): the step is sharded by source: every rank builds the whole catalogue,
traces the entries rank, rank + N, ..., the photon grids are all-reduced once and finalised; value = all ranks'
segments / max-over-ranks time ("scaling": "strong").  `--replicas`: every rank runs the whole step on its own GPU
instead (redundant work; value = N * segments / max-over-ranks time, "scaling": "weak").
`--impl reference` times the CPU oracle (oracle/, as it stands) on a bounded sample of the same workload.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

ALGO_BYTES_PER_SEGMENT = {"f32": 48, "f64": 64}     # 4 field loads + 2 accumulator RMWs
# the same without the assumption that every segment touches its neighbour: per segment 2 field loads + 1 RMW of the
# cell, and the same again for each neighbour deposit the library counted (stats.neighbour_deposits)
ALGO_BYTES_CELL = {"f32": 24, "f64": 32}
METRIC = "ray_cell_segments_per_s"
# The march kernel's two ALU roofs come from the executed-instruction counts of the
# shipping kernel in profiles/march_instr.csv (last row; profiles/march_instr.md says how they were taken), not
# from a constant here:
#   fp64 pipe: a warp-level fp64 instruction occupies its sub-partition's fp64 pipe for 2 cycles (16 lanes per clock),
#              so a warp-cell costs 2 x fp64_inst_per_warp_cell cycles of a scheduler whatever else issues beside it;
#   issue:     one warp instruction per scheduler per cycle: inst_per_warp_cell cycles.
# segments/s at a roof = SMs x 4 schedulers x SM clock x 32 lanes / cycles per warp-cell (all lanes busy, no stall).
SM_COUNT, SCHEDULERS_PER_SM, LANES = 148, 4, 32
FP64_PIPE_CYCLES_PER_WARP_INST = 2


def march_instruction_counts(path=None):
    """(inst_per_warp_cell, fp64_inst_per_warp_cell, profile name) of the shipping march kernel."""
    import csv
    path = path or os.path.join(ROOT, "profiles", "march_instr.csv")
    with open(path, newline="") as f:
        rows = list(csv.DictReader(f))
    r = rows[-1]
    return float(r["inst_per_warp_cell"]), float(r["fp64_inst_per_warp_cell"]), r["profile"]


def alu_roofs(segments, march_ms, sm_mhz, inst_per_cell, fp64_per_cell):
    """The march kernel against the hardware's fp64-pipe roof and against the issue roof of its own instruction
    stream; both in segments/s at the SM clock measured during the run."""
    slots = SM_COUNT * SCHEDULERS_PER_SM * sm_mhz * 1e6 * LANES      # lane-slots per second
    ach = segments / (march_ms * 1e-3)
    fp64_peak = slots / (FP64_PIPE_CYCLES_PER_WARP_INST * fp64_per_cell)
    issue_peak = slots / inst_per_cell
    return dict(achieved=ach, fp64_peak=fp64_peak, fp64_frac=ach / fp64_peak, issue_peak=issue_peak,
                issue_frac=ach / issue_peak)


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=5)
    ap.add_argument("--n-src", type=int, default=0, help="use only the first N sources (0 = all)")
    ap.add_argument("--batch-rays", type=int, default=0)
    ap.add_argument("--shard", action="store_true",
                    help="shard the step by source (one all-reduce of the photon grid); the default when N > 1")
    ap.add_argument("--replicas", action="store_true",
                    help="N > 1: every rank runs the whole step on its own GPU (no sharding, redundant work)")
    ap.add_argument("--spectrum-teff", type=float, default=0.0,
                    help="trace with the tau_0 lookup table of a black body of this temperature [K] (default: monochromatic)")
    ap.add_argument("--tau-thin", type=float, default=0.0,
                    help="with --spectrum-teff: also set the table for thin segments (PAPER.md:267 footnote 3), used below this dtau_0")
    ap.add_argument("--timestep-myr", type=float, default=0.0,
                    help="time a whole RT timestep of this length (iterative RT<->ODE solve, nyxrt_timestep) instead of one RT step")
    ap.add_argument("--periodic", action="store_true", help="periodic box (default: BASELINE.json's open box)")
    ap.add_argument("--graph-loop", action="store_true", help="(the default now; kept so that old commands still run)")
    ap.add_argument("--profiling-loop", action="store_true",
                    help="time the host-enqueued profiling loop (NYXRT_FLAG_LAUNCH_TIMING) instead of the production "
                         "CUDA-graph loop for value / e2e, as rounds 1-2 did")
    ap.add_argument("--profile-steps", type=int, default=1,
                    help="steps of the separate profiling pass (per-launch CUDA events around every march launch) that "
                         "feeds the roofline; 0: roofline from the loop time of the timed steps")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    return ap.parse_args()


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([v.strip() for v in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, reasons, pw = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except ValueError:
                continue
            for n, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return float(json.load(open(p))["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (of measured)"
    return 6650.0, "B200_PROFILING.md fallback 6.65 TB/s (of fallback)"


def max_over_ranks(x, device):
    """Max of a scalar over all ranks (the contract's timing rule); identity when not distributed."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(x, device):
    """Sum of a scalar over all ranks (source-sharded mode: every rank marches its own rays)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def whole_job_rate(units_per_rank, ms_max, world):
    """Replicas only: every rank processes `units_per_rank`; the job's rate is all
    ranks' units over the slowest rank's time."""
    return world * units_per_rank / (ms_max * 1e-3)


def make_workload(args, device):
    from paper_2512_12466_b200 import synth
    cfg = synth.make(args.config, device=device)
    pos, L = cfg["src_pos"].numpy(), cfg["src_L"].numpy()
    if args.n_src:
        pos, L = pos[:args.n_src], L[:args.n_src]
    return cfg, pos, L


def cpu_info():
    model = "unknown"
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.lower().startswith("model name"):
                    model = line.split(":", 1)[1].strip()
                    break
    except OSError:
        pass
    return model, os.cpu_count() or 1


def oracle_sample(cfg, pos, L, budget_s, n_proc=0):
    """The CPU oracle, as it stands, on a bounded sample of the same workload: the whole step (dedup, merge, ray
    loop) on the first sources of the list, the ray loop spread over the host's cores (one single-threaded oracle
    process per core over disjoint chunks of the sorted catalogue, oracle.step_parallel); the sample grows until one
    run takes about budget_s seconds of wall time."""
    from oracle import oracle as O
    import psutil
    nH = cfg["nH"].cpu().numpy()
    xHI = cfg["xHI"].cpu().numpy()
    g = O.make_grid(cfg["shape"], cfg["dx_cm"], field_dtype=nH.dtype)
    p = O.make_params(**cfg["params"])
    model, cores = cpu_info()
    grid_bytes = nH.size * 8
    n_proc = n_proc or max(1, min(cores, len(L), int(0.8 * psutil.virtual_memory().available // (grid_bytes + 2 ** 28))))
    n, best = min(len(L), 4 * n_proc), None
    while True:
        t0 = time.perf_counter()
        osum, cat = O.step_parallel(g, p, nH, xHI, pos[:n], L[:n], n_proc, want_heat=False, chunk=1)
        dt = time.perf_counter() - t0
        seg, cpu_s = int(osum.stats.segments), osum.cpu_seconds
        osum.close()
        best = (seg, dt, cpu_s, n)
        if dt >= 0.5 * budget_s or n >= len(L):
            break
        n = min(len(L), int(n * max(2.0, min(8.0, 0.8 * budget_s / max(dt, 1e-3)))))
    seg, dt, cpu_s, n = best
    return dict(value=seg / dt if dt > 0 else 0.0, unit="segments/s", cores=n_proc, kind="oracle",
                cpu_model=model, host_cores=cores, per_core=seg / cpu_s if cpu_s > 0 else 0.0,
                sample="oracle step (dedup, merge, ray loop; no heating grid) on the first %d of %d input sources of the "
                       "same fields, ray loop on %d single-threaded processes: %d segments in %.1f s wall "
                       "(%.3g segments/s per core)" % (n, len(L), n_proc, seg, dt, seg / max(cpu_s, 1e-9)),
                segments=int(seg), seconds=dt)


def run_reference(args):
    """--impl reference: the oracle timed on the host cores; each step is a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import torch
    dev = "cuda" if torch.cuda.is_available() else "cpu"
    cfg, pos, L = make_workload(args, dev)
    per_step = max(3.0, min(20.0, 60.0 / max(1, args.steps + args.warmup)))
    for _ in range(min(args.warmup, 1)):
        oracle_sample(cfg, pos, L, 1.0)
    seg, sec, last = 0, 0.0, None
    for _ in range(args.steps):
        last = oracle_sample(cfg, pos, L, per_step)
        seg += last["segments"]
        sec += last["seconds"]
    v = seg / sec
    out = dict(impl="reference", metric=METRIC, value=v, unit="segments/s", n_gpus=args.gpus, steps=args.steps,
               warmup=args.warmup, ms_per_step=1e3 * sec / args.steps, higher_is_better=True, scaling="weak",
               vs_baseline=None, dtype="f64", data="synthetic",
               config=dict(workload=cfg["name"], notes=cfg["notes"], sample=last["sample"]),
               cpu_baseline=dict(value=v, unit="segments/s", cores=last["cores"], kind="oracle", sample=last["sample"],
                                 cpu_model=last["cpu_model"], host_cores=last["host_cores"]),
               e2e=dict(value=v, unit="segments/s", h2d_bytes_per_step=0, d2h_bytes_per_step=0))
    print(json.dumps(out))


def main():
    args = parse()
    if args.impl == "reference":
        return run_reference(args)
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_2512_12466_b200 import nyxrt

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        if not args.replicas:
            args.shard = True                  # N ranks divide the step's sources (real work, counted once)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    cfg, pos, L = make_workload(args, "cuda")
    nH, xHI = cfg["nH"], cfg["xHI"]
    fdt = "f32" if nH.dtype == torch.float32 else "f64"
    timed_flags = nyxrt.FLAG_LAUNCH_TIMING if args.profiling_loop else 0      # 0: the production CUDA-graph loop

    def make_tracer(flags, host_staging):
        params = dict(cfg["params"])
        params["flags"] = flags
        t = nyxrt.Tracer(cfg["shape"], cfg["dx_cm"], params, field_dtype=nH.dtype, max_sources=len(L),
                         batch_rays=args.batch_rays, host_staging=host_staging, device=local,
                         periodic=1 if args.periodic else 0)
        if args.spectrum_teff > 0:
            t.set_spectrum(-20, 12, 8, nyxrt.nyxrt_blackbody_table(args.spectrum_teff, -20, 12, 8))
            if args.tau_thin > 0:
                t.set_spectrum_thin(nyxrt.nyxrt_blackbody_thin_table(args.spectrum_teff, -20, 12, 8), args.tau_thin)
        if args.shard:
            t.set_shard(rank, world)
        return t

    tr = make_tracer(timed_flags, not args.no_e2e)
    gam = torch.empty(cfg["shape"], dtype=torch.float64, device="cuda")
    heat = torch.empty_like(gam)
    stream = torch.cuda.current_stream()
    photons = torch.empty_like(gam) if args.shard else None

    class _TS:                                                     # timestep mode: the sum over the iterations
        pass

    def step(tr):
        # one RT step: fields of this step -> absorber field, sources -> catalogue, ray loop, finalise
        if args.timestep_myr > 0:
            tr.set_sources(pos, L, stream)
            ode = nyxrt.make_ode(args.timestep_myr * 3.1557e13)
            y0 = xHI.double() if xHI.dtype != torch.float64 else xHI
            xe, xa, g_, h_, st1, ts = tr.timestep(ode, nH, y0, stream=stream)
            out = _TS()
            for name, _ in st1._fields_:
                setattr(out, name, getattr(st1, name))
            out.segments = ts.segments_total
            out.kernel_launches = ts.kernel_launches
            out.ms_march = st1.ms_march * ts.iterations           # per-launch events exist for the last trace only
            out.ms_loop = st1.ms_loop * ts.iterations
            out.march_launches = st1.march_launches * ts.iterations
            out.neighbour_deposits = st1.neighbour_deposits * ts.iterations
            out.timestep = dict(iterations=ts.iterations, converged=ts.converged, ms_rt=ts.ms_rt, ms_ode=ts.ms_ode,
                                unconverged_cells=int(ts.unconverged_cells))
            return out
        tr.set_fields(nH, xHI, stream)
        tr.set_sources(pos, L, stream)
        if not args.shard:
            return tr.trace(gam, heat, stream=stream)[2]
        # sharded by source: this rank's sources, one all-reduce of the photon grid
        st_ = nyxrt.nyxrt_trace_photons(tr.ctx, photons, stream)
        if world > 1:
            dist.all_reduce(photons, op=dist.ReduceOp.SUM)
        nyxrt.nyxrt_finalise(tr.ctx, photons, gam, heat, stream)
        return st_

    for _ in range(args.warmup):
        st = step(tr)
    barrier()
    clocks = ClockSampler(local)
    if rank == 0:
        clocks.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    seg = 0
    launches = 0
    prof = dict(seg=0, nbr=0, ms_march=0.0, march_launches=0, ms=0.0, steps=0, kind="")
    barrier()
    e0.record(stream)
    for _ in range(args.steps):
        st = step(tr)
        seg += st.segments
        launches += st.kernel_launches + 3            # + prep_fields, sum_partials, snap
        if args.profiling_loop or args.profile_steps <= 0:
            # no separate profiling pass: the march launches' own durations if this loop measures them, else the loop time
            prof["seg"] += st.segments
            prof["nbr"] += st.neighbour_deposits
            prof["ms_march"] += st.ms_march if args.profiling_loop else st.ms_loop
            prof["march_launches"] += st.march_launches
            prof["steps"] += 1
    e1.record(stream)
    barrier()
    ms = e0.elapsed_time(e1)
    clk = clocks.stop() if rank == 0 else None
    ms = max_over_ranks(ms, "cuda")
    if prof["steps"]:
        prof["ms"] = ms
        prof["kind"] = ("the timed steps (profiling loop)" if args.profiling_loop
                        else "the timed steps; no per-launch events: the loop time stands in for the march launches' own")
    if args.timestep_myr > 0:
        args.no_e2e = True
    if args.shard:
        seg_all = sum_over_ranks(seg, "cuda")                       # total work is fixed: strong scaling
        value = whole_job_rate(seg_all, ms, 1)
        args.no_e2e = True                                          # step_host is the unsharded call
    else:
        seg_all = seg * world
        value = whole_job_rate(seg, ms, world)

    # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region ----
    e2e = None
    if not args.no_e2e:
        h_nH = nH.cpu().pin_memory()
        h_xHI = xHI.cpu().pin_memory()
        h_g = torch.empty(cfg["shape"], dtype=torch.float64).pin_memory()
        h_h = torch.empty(cfg["shape"], dtype=torch.float64).pin_memory()
        tr.step_host(h_nH, h_xHI, pos, L, h_g, h_h)                 # warm-up
        ke = min(args.steps, 2)
        barrier()
        t0 = time.perf_counter()
        seg_e = 0
        for _ in range(ke):
            seg_e += tr.step_host(h_nH, h_xHI, pos, L, h_g, h_h).segments
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        dt = max_over_ranks(dt, "cuda")
        e2e = dict(value=whole_job_rate(seg_e, dt * 1e3, world), unit="segments/s", steps=ke, ms_per_step=1e3 * dt / ke,
                   h2d_bytes_per_step=int(2 * h_nH.numel() * h_nH.element_size() + pos.nbytes + L.nbytes),
                   d2h_bytes_per_step=int(2 * h_g.numel() * 8),
                   checksum_gamma_sum=float(h_g.sum()))
        del h_nH, h_xHI, h_g, h_h

    # ---- profiling pass for the roofline: the same step through the host-enqueued loop, which puts a CUDA-event pair
    # around every march launch (NYXRT_FLAG_LAUNCH_TIMING).  Same kernels, same results; outside the timed region. ----
    if not prof["steps"]:
        tr.close()
        tr = make_tracer(nyxrt.FLAG_LAUNCH_TIMING, False)
        barrier()
        p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        p0.record(stream)
        for _ in range(args.profile_steps):
            sp = step(tr)
            prof["seg"] += sp.segments
            prof["nbr"] += sp.neighbour_deposits
            prof["ms_march"] += sp.ms_march
            prof["march_launches"] += sp.march_launches
            prof["steps"] += 1
        p1.record(stream)
        barrier()
        prof["ms"] = p0.elapsed_time(p1)
        prof["kind"] = "%d extra step(s) after the timed region, host-enqueued loop with per-launch events" % args.profile_steps

    if rank == 0:
        peak, peak_src = measured_peak()
        pseg, pnbr, ms_march, march_launches = prof["seg"], prof["nbr"], prof["ms_march"], prof["march_launches"]
        sm_mhz = float((clk or {}).get("sm_mhz") or 1965.0)
        ipc, fpc, iprof = march_instruction_counts()
        alu = alu_roofs(pseg, ms_march, sm_mhz, ipc, fpc)
        avg_launch_ms = ms_march / max(march_launches, 1)
        # Primary roof: the fp64 pipe.  ncu shows the kernel bound by instruction issue behind fp64 dependencies, with
        # DRAM at 0.14 of its peak (profiles/r2_march_config5.md), so HBM is reported beside it, not as the bound.
        roof = dict(bound="alu", kernel="march_kernel<3>", achieved=alu["achieved"], peak=alu["fp64_peak"],
                    unit="segments/s", frac=alu["fp64_frac"], traffic=None,
                    peak_source="148 SMs x 4 schedulers x %.0f MHz (median during the timed steps) x 32 lanes / (2 fp64-pipe "
                                "cycles x %g fp64 warp instructions per warp-cell, profiles/march_instr.csv row %s)"
                                % (sm_mhz, fpc, iprof),
                    segments_per_launch=pseg / max(march_launches, 1), avg_launch_ms=avg_launch_ms,
                    march_share_of_step=ms_march / max(prof["ms"], 1e-9), measured_on=prof["kind"],
                    note="achieved = segments / sum of the march launches' durations (CUDA events around every launch on "
                         "the launching stream); peak = the hardware's fp64-pipe roof for this kernel's counted fp64 "
                         "instructions, all lanes busy and no stall")
        roof["issue"] = dict(peak=alu["issue_peak"], frac=alu["issue_frac"], inst_per_warp_cell=ipc, unit="segments/s",
                             note="issue-slot roof of the kernel's own instruction stream (one warp instruction per "
                                  "scheduler per cycle); a leaner kernel raises this roof, the fp64 roof above it does not move")
        # HBM, three ways: the contract's algorithmic bytes (48 / 64 B per segment), the same with the
        # neighbour traffic counted instead of assumed, and the DRAM bytes ncu measured per launch
        bps = ALGO_BYTES_PER_SEGMENT[fdt]
        ach = bps * pseg / (ms_march * 1e-3) / 1e9
        cb = ALGO_BYTES_CELL[fdt]
        ach_x = cb * (pseg + pnbr) / (ms_march * 1e-3) / 1e9
        roof["hbm"] = dict(peak=peak, unit="GB/s", peak_source=peak_src,
                           algorithmic=dict(achieved=ach, frac=ach / peak, bytes_per_segment=bps,
                                            note="%d B x segments / march time: the figure rounds 1-2 reported as roofline.frac" % bps),
                           counted=dict(achieved=ach_x, frac=ach_x / peak, bytes_per_segment=cb * (pseg + pnbr) / max(pseg, 1),
                                        neighbour_deposits_per_segment=pnbr / max(pseg, 1),
                                        note="%d B per segment + %d B per counted neighbour deposit" % (cb, cb)),
                           measured=None)
        # DRAM bytes per march launch measured by ncu on THIS workload (profiles/march_traffic.csv, one row per
        # captured launch; profiles/march_traffic.md has the commands); null when no capture matches the run
        tfile = os.path.join(ROOT, "profiles", "march_traffic.csv")
        roof["traffic_note"] = "no ncu capture of this workload in profiles/march_traffic.csv"
        if os.path.exists(tfile) and not args.shard and args.timestep_myr == 0:
            try:
                import csv
                with open(tfile, newline="") as f:
                    rows = [r for r in csv.DictReader(f)
                            if r.get("workload") == cfg["name"] and int(r.get("n_sources", -1)) == len(L)
                            and int(r.get("periodic", -1)) == int(args.periodic)
                            and r.get("spectrum") == ("table" if args.spectrum_teff > 0 else "monochromatic")]
                if rows:
                    tb = [1e9 * (float(r["dram_read_gb"]) + float(r["dram_write_gb"])) for r in rows]
                    tm = [float(r["launch_ms"]) for r in rows]
                    roof["traffic"] = sum(tb) / len(tb)
                    roof["traffic_note"] = ("mean dram__bytes_read.sum + dram__bytes_write.sum of %d captured march launches "
                                            "of this workload (ncu --set full, mean %.2f ms under ncu)" % (len(tb), sum(tm) / len(tm)))
                    dram = sum(b / (1e-3 * t) for b, t in zip(tb, tm)) / len(tb) / 1e9
                    roof["hbm"]["measured"] = dict(achieved=dram, frac=dram / peak,
                                                   note="DRAM bytes / duration of the same captured launches (under ncu)")
                    iu = [float(r["issue_active_pct"]) / 100.0 * float(r["active_threads_per_inst"]) / LANES for r in rows]
                    roof["issue"]["issue_util_measured"] = sum(iu) / len(iu)
                    roof["issue"]["issue_util_note"] = "ncu: issue slots busy x active threads per instruction / 32, same launches"
            except (ValueError, OSError, KeyError):
                pass
        cpu = None
        if not args.no_cpu:
            cpu = oracle_sample(cfg, pos, L, args.cpu_seconds)
            cpu.pop("segments"); cpu.pop("seconds")
        graph = "one CUDA-graph launch per trace (WHILE node over sched -> emit -> march): the production path"
        hostl = "host-enqueued launches with a CUDA-event pair around every march launch (NYXRT_FLAG_LAUNCH_TIMING)"
        out = dict(metric=METRIC, value=value, unit="segments/s", n_gpus=world, steps=args.steps, warmup=args.warmup,
                   ms_per_step=ms / args.steps, higher_is_better=True, scaling="strong" if args.shard else "weak",
                   vs_baseline=None, dtype="f64", data="synthetic",
                   config=dict(workload=cfg["name"], grid=list(cfg["shape"]), field_dtype=fdt, n_sources=int(len(L)),
                               n_sources_dedup=int(st.n_src_dedup), n_sources_merged=int(st.n_src_merged),
                               segments_per_step=int(seg_all // (args.steps * (1 if args.shard else world))), notes=cfg["notes"],
                               l2="inputs larger than L2 (fields + accumulator = %.1f GB), no flush"
                                  % ((2 * nH.numel() * nH.element_size() + 16 * nH.numel()) / 1e9),
                               multi_gpu="sharded by source, one all-reduce of the photon grid" if args.shard else "replicas only",
                               periodic=bool(args.periodic), timestep=getattr(st, "timestep", None),
                               spectrum=("black body %g K, tau_0 table 2^-20..2^12, 256 nodes per octave%s" % (
                                   args.spectrum_teff, ", thin table below dtau_0 = %g" % args.tau_thin if args.tau_thin > 0 else ""))
                               if args.spectrum_teff > 0 else "monochromatic"),
                   loop=hostl if args.profiling_loop else graph,
                   rt_step_ms=ms / args.steps,
                   profiling_pass=dict(loop=hostl if (args.profiling_loop or args.profile_steps > 0) else graph,
                                       steps=prof["steps"], ms_per_step=prof["ms"] / max(prof["steps"], 1),
                                       march_ms_per_step=ms_march / max(prof["steps"], 1), measured_on=prof["kind"]),
                   gpu_launches=int(launches), clocks=clk, e2e=e2e, roofline=roof, cpu_baseline=cpu,
                   stats=dict(iterations=int(st.iterations), peak_pool_rays=int(st.peak_pool_rays),
                              ms_sources=st.ms_sources, ms_loop=st.ms_loop, ms_finalise=st.ms_finalise,
                              spawned=list(st.spawned)[:14],
                              budget_rel=(st.photons_absorbed + st.photons_escaped + st.photons_residual
                                          - st.photons_emitted) / max(st.photons_emitted, 1e-300)))
        print(json.dumps(out))
    tr.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

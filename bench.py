#!/usr/bin/env python
"""bench.py -- throughput of the SSFM/OPO hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload C0..C4] [--eom]

One "step" = the whole hot path over one batch: `rt_per_step` cavity round trips (each = nz z-steps
of FFT . dispersion . IFFT + RK4, then the boundary operator) of every instance of the workload.
Default workload: BASELINE.json configs[4] (256 independent N = 2^14 three-wave OPOs, 100 z-steps,
300 round trips -- the batched N = 2^14 case the roofline target is quoted on); `--workload C1` runs
configs[1] (the same OPO, a single instance: latency-bound, 3 of 148 SMs), C0 / C2 / C3 the other configs
(C3: N = 2^18 on the large-N engine, roofline against the HBM peak).

Prints ONE JSON line (rank 0).  `value` = grid-point z-steps/s with inputs resident in HBM;
`e2e` = the same through the host-buffer ABI calls (H2D of pump and seeds, D2H of the exit signal
inside the timed region); `roofline` = the dominant kernel against the FP32 FMA peak measured in the same run;
`cpu_baseline` = the fp64 oracle on this host's cores on a bounded sample.
`--impl reference` times the oracle instead (rank 0 only).
"""
from __future__ import annotations

import argparse
import copy
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np

import opo_workloads as W

METRIC = "ssfm_grid_point_z_steps_per_s"
UNIT = "grid-point z-steps/s"
# flops per field-point z-step of the scheme actually executed (half-steps merged): 2 transforms
# x 5 log2(N) + table multiply 6 + RK4 76
def flops_per_grid_point_zstep(log2_n: int, n_fields: int) -> float:
    return n_fields * (2 * 5 * log2_n + 6 + 76)


# dram__bytes_read.sum + dram__bytes_write.sum of the dominant kernel per launch come from ncu captures, which bench.py
# cannot take itself (a number printed under a profiler is never a bench value): profiles/ncu_traffic.json lists, per
# (workload, engine, round trips per step), the bytes, the capture file and the commit it was taken at.  No entry -> null.
def ncu_traffic(workload: str, engine: str, rt_per_step: int):
    path = os.path.join(ROOT, "profiles", "ncu_traffic.json")
    if not os.path.exists(path):
        return None, None
    for e in json.load(open(path)).get("captures", []):
        if e.get("workload") == workload and e.get("engine") == engine and e.get("rt_per_step") == rt_per_step:
            return e.get("dram_bytes_per_launch"), f"{e.get('source')} @ {e.get('commit')}"
    return None, None


# shared-memory bytes per field-point z-step of the on-chip engines: six passes over the field
# (pass 0 + RK4, forward pass 1, the three-pass chain, inverse pass 1), each a read and a write of one complex value
def smem_bytes_per_field_point_zstep(precision: str) -> float:
    return 6 * 2 * (16 if precision == "c128" else 8)


# The wide engine (one instance on a cluster of 4 F CTAs) exchanges every field value over the SM-to-SM link twice per z-step: it
# leaves its SM as an operand of the pass-0 / RK4 phase and comes back as a result.  Bytes one SM SENDS
# per z-step with G sub-blocks of a field per CTA (OPO_INFO_WIDE_SUBBLOCKS; NV = 4 F sub-blocks on NV / G CTAs, and what stays
# inside a CTA does not cross the link): 2 crossings x esz x (N F G / NV) x (NV - G) / NV; it receives as much.  Peak: bytes sent
# per SM with every SM sending and receiving at once, measured in this run (opo_selftest_peak(OPO_PEAK_DSMEM)).  Until round 2
# this line counted sent + received bytes against a round-1 constant of 16 B/clk.
def wide_link_roofline(w, o, P, units_per_step, avg_s):
    esz = 16 if w.precision == "c128" else 8
    nv = 4 * w.n_fields
    slots = int(P.opo_get_info(o._h, P.INFO_SLOTS))
    waves = -(-w.batch // max(1, slots))
    g = max(1, int(P.opo_get_info(o._h, P.INFO_WIDE_SUBBLOCKS)))
    sent_per_sm_per_zstep = 2 * esz * (w.n * w.n_fields * g / nv) * (nv - g) / nv
    zsteps_per_sm = units_per_step / (w.batch * w.n) * waves                        # z-steps an SM works through, wave after wave
    achieved = sent_per_sm_per_zstep * zsteps_per_sm / avg_s / 1e9
    peak = P.opo_selftest_peak(P.PEAK_DSMEM)
    return {"achieved": achieved, "peak": peak, "unit": "GB/s sent per SM", "frac": achieved / peak,
            "note": "SM-to-SM link: bytes one SM sends (operands out, results back; it receives as much); peak = 16-byte remote stores on "
                    f"every co-resident cluster of 4, every SM sending and receiving at once, measured in this run; {g} sub-block(s) per CTA"}


def make_workload(name: str, rank: int):
    makers = {"C0": W.config0, "C1": W.config1, "C2": W.config2, "C3": W.config3, "C4": W.config4}
    if name not in makers:
        raise SystemExit(f"unknown workload {name}")
    w = makers[name]()
    if rank:   # other ranks run their own sweep with their own seeds (weak scaling, no collective)
        rng = np.random.default_rng(1000 + rank)
        for x in range(1, w.n_fields):
            w.seeds[x] = W._round_to_precision(np.roll(w.seeds[x], 17 * rank, axis=1) * np.exp(2j * np.pi * rng.random()), w.precision)
    return w


def replicate(w, batch: int, rank: int):
    """A single-instance workload (C0, C1, C3) as a batch of `batch` independent OPOs: same pump, crystal and cavity, every
    instance with its own seeded noise at the rms of the original seed (input scaling only, as in opo_workloads)."""
    if w.batch != 1:
        raise SystemExit(f"--batch replicates single-instance workloads; {w.name} already has {w.batch} instances")
    w = copy.copy(w)
    w.seeds = [None] + [W._round_to_precision(np.stack([W.complex_gaussian_noise(W.splitmix64(7000 + 10 * x + rank, b) % (1 << 31), w.n,
                                                                                      float(np.sqrt(np.mean(np.abs(w.seeds[x][0]) ** 2))))
                                                                  for b in range(batch)]), w.precision) for x in range(1, w.n_fields)]
    w.batch = batch
    w.name = f"{w.name} x {batch} instances"
    return w


def max_over_ranks(t_local: float, world: int, device="cuda") -> float:
    """Job time = the slowest rank's device time (no other collective exists on this path)."""
    import torch
    import torch.distributed as dist
    tt = torch.tensor([t_local], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    return float(tt.item())


def job_throughput(units_per_step_per_rank: int, steps: int, world: int, t_total: float) -> float:
    """Whole-job aggregate: every rank processes the same number of units (weak scaling)."""
    return world * units_per_step_per_rank * steps / t_total


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.lines, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "200", "-i", str(self.index)], stdout=subprocess.PIPE, text=True)
            self.t = threading.Thread(target=lambda: self.lines.extend(self.proc.stdout), daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        self.t.join(timeout=2)
        sm, mx, reasons = [], [], set()
        for ln in self.lines:
            p = [s.strip() for s in ln.split(",")]
            if len(p) < 9:
                continue
            try:
                sm.append(float(p[1])); mx.append(float(p[2]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), p[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def run_reference(args, rank, world):
    """The oracle as it stands, on this host's cores, on a bounded sample of the same workload."""
    if rank != 0:
        return
    import oracle
    oracle.build()
    w = make_workload(args.workload, 0)
    if args.batch:
        w = replicate(w, args.batch, 0)
    cores = os.cpu_count() or 1
    inst = list(range(min(w.batch, cores)))
    # ~0.6 s per round trip per core at N = 2^14, nz = 100: one round trip per instance per step
    rt = 1
    sample = f"{len(inst)} instance(s) x {rt} round trip(s) of {w.name}, one thread per instance"

    def step():
        oracle.run_workload(w, n_roundtrips=rt, instances=inst, threads=len(inst))

    for _ in range(args.warmup):
        step()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step()
    dt = (time.perf_counter() - t0) / args.steps
    val = len(inst) * w.n * w.nz_per_pass * rt / dt
    line = {"metric": METRIC, "value": val, "unit": UNIT, "impl": "reference", "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{w.name} (BASELINE.json configs[{args.workload[1]}])", "sample": sample},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": len(inst), "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "round_trips_per_s": len(inst) * rt / dt, "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def cpu_baseline(w, budget_s=15.0):
    import oracle
    oracle.build()
    cores = os.cpu_count() or 1
    inst = list(range(min(w.batch, cores)))
    t0 = time.perf_counter()
    oracle.run_workload(w, n_roundtrips=1, instances=inst[:1], threads=1)
    t1 = time.perf_counter() - t0                    # one round trip, one core
    rt = max(1, int(budget_s / max(t1, 1e-3)))
    rt = min(rt, 25)
    t0 = time.perf_counter()
    oracle.run_workload(w, n_roundtrips=rt, instances=inst, threads=len(inst))
    dt = time.perf_counter() - t0
    return {"value": len(inst) * w.n * w.nz_per_pass * rt / dt, "unit": UNIT, "cores": len(inst), "kind": "oracle",
            "sample": f"{len(inst)} instance(s) x {rt} round trip(s) of {w.name}, one thread per instance, {dt:.1f} s",
            "round_trips_per_s": len(inst) * rt / dt}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C4", choices=["C0", "C1", "C2", "C3", "C4"])
    ap.add_argument("--rt-per-step", type=int, default=0, help="round trips per step (default: the config's full length for C4 and C0, 100 for C1, 20 for C2, 2 for C3)")
    ap.add_argument("--engine", default="auto", choices=["auto", "resident", "solo", "wide", "streaming", "cufft"],
                    help="cufft = the internal cuFFT + elementwise-kernel baseline (north_star item (d)), not the product")
    ap.add_argument("--eom", action="store_true",
                    help="intracavity phase modulator on the signal (PAPER.md:L149-154; beta = 1 rad, f = 3 / window): the "
                         "paper's 'EOM' cavity configuration; one launch per step on the on-chip engines (table H G m, modulator in the time domain, H at every crossing)")
    ap.add_argument("--wide-subblocks", type=int, default=0, choices=[0, 1, 2],
                    help="wide engine: sub-blocks per CTA (OPO_OPT_WIDE_SUBBLOCKS); 0 = the library's choice")
    ap.add_argument("--train", action="store_true",
                    help="nanosecond regime (PAPER.md:L322-335): opo_roundtrips_train -- a pump slice per round trip in, the exit "
                         "signal of every round trip out; one launch per step on the solo engine (slices read and exit fields written at the crossings inside the kernel), one per round trip elsewhere; default 20 round trips per step")
    ap.add_argument("--batch", type=int, default=0,
                    help="run a single-instance workload (C0, C1, C3) as a batch of this many independent instances with their own noise "
                         "seeds, e.g. --workload C0 --batch 2048: complex128 on every SM, roofline against the FP64 FMA pipe (SURVEY 8(d))")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return
    if args.warmup < 3:
        args.warmup = 3

    import torch
    import torch.distributed as dist
    import paper_2410_02532_b200 as P

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback); use --impl reference for the oracle")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    w = make_workload(args.workload, rank)
    if args.batch:
        w = replicate(w, args.batch, rank)
    if args.eom:
        w.eom_beta_rad = [0.0, 1.0, 0.0]
        w.eom_f_hz = [0.0, 3.0 / w.window_s, 0.0]
    rt_per_step = args.rt_per_step or (20 if args.train else {"C0": w.n_roundtrips, "C1": 100, "C2": 20, "C3": 2, "C4": w.n_roundtrips}[args.workload])
    engine = {"auto": P.ENGINE_AUTO, "resident": P.ENGINE_RESIDENT, "solo": P.ENGINE_SOLO, "wide": P.ENGINE_WIDE, "streaming": P.ENGINE_STREAMING, "cufft": P.ENGINE_CUFFT}[args.engine]
    o = P.from_workload(w, engine=engine)
    if args.wide_subblocks:
        P.opo_set_option(o._h, P.OPT_WIDE_SUBBLOCKS, args.wide_subblocks)
    units_per_step = w.batch * w.n * w.nz_per_pass * rt_per_step          # grid-point z-steps, this rank
    flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")       # > 126 MB L2

    # pinned host copies of the step's inputs / output for the e2e leg
    dt_t = o.dtype
    h_pump = torch.from_numpy(np.ascontiguousarray(w.pump)).to(dt_t).contiguous().pin_memory()
    h_seeds = [None] + [torch.from_numpy(np.ascontiguousarray(w.seeds[x])).to(dt_t).contiguous().pin_memory() for x in range(1, w.n_fields)]
    h_out = torch.empty((w.batch, w.n), dtype=dt_t).pin_memory()
    d_pump = h_pump.cuda()
    d_seeds = [None] + [h_seeds[x].cuda() for x in range(1, w.n_fields)]

    def reset_device_inputs():
        o.set_pump(d_pump if d_pump.shape[0] > 1 else d_pump[0].contiguous())
        for x in range(1, w.n_fields):
            o.set_field(x, d_seeds[x])

    d_train = None
    if args.train:      # the same pump slice every round trip: the work of the default step, driven slice by slice
        d_train = (d_pump if d_pump.shape[0] > 1 else d_pump[0]).unsqueeze(0).expand(rt_per_step, *((-1,) * (d_pump.dim() if d_pump.shape[0] > 1 else 1))).contiguous()

    def step_resident_inputs():
        if args.train:
            o.roundtrips_train(d_train, out_field=1)
        else:
            o.roundtrips(rt_per_step)

    def step_e2e():
        o.set_pump(h_pump if h_pump.shape[0] > 1 else h_pump[0])
        for x in range(1, w.n_fields):
            o.set_field(x, h_seeds[x])
        o.roundtrips(rt_per_step)
        o.get_fields(1, P.WHICH_EXIT, P.DOMAIN_TIME, out=h_out)          # D2H + stream sync inside

    # ---- device-resident timing -------------------------------------------------------------------------
    for _ in range(args.warmup):
        reset_device_inputs(); step_resident_inputs()
    barrier()
    launches0 = o.launches
    sampler = ClockSampler(local_rank); sampler.start()
    evs = []
    t_wall0 = time.perf_counter()
    for _ in range(args.steps):
        reset_device_inputs()                      # untimed: state back to the seeds (same work every step)
        flush.fill_(1)                             # untimed: evict L2 between timed iterations
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); step_resident_inputs(); e1.record()
        evs.append((e0, e1))
    barrier()
    t_wall = time.perf_counter() - t_wall0
    clocks = sampler.stop()
    launches = o.launches - launches0
    per_step_ms = [a.elapsed_time(b) for a, b in evs]
    t_local = sum(per_step_ms) * 1e-3
    t_total = max_over_ranks(t_local, world)
    value = job_throughput(units_per_step, args.steps, world, t_total)
    o.check_finite()

    # ---- end-to-end timing (host buffers through the ABI) ---------------------------------------------------
    e2e = None
    if not args.no_e2e:
        step_e2e()
        barrier()
        t0 = time.perf_counter()
        e2e_steps = max(1, min(args.steps, 3))
        for _ in range(e2e_steps):
            step_e2e()
        barrier()
        te = max_over_ranks(time.perf_counter() - t0, world)
        esz = 16 if w.precision == "c128" else 8
        h2d = (h_pump.numel() + sum(h_seeds[x].numel() for x in range(1, w.n_fields))) * esz
        e2e = {"value": job_throughput(units_per_step, e2e_steps, world, te), "unit": UNIT,
               "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(h_out.numel() * esz), "steps": e2e_steps}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel ----------------------------------------------------
    avg_s = statistics.mean(per_step_ms) * 1e-3
    eng = o.engine
    eng_name = {P.ENGINE_RESIDENT: "resident", P.ENGINE_SOLO: "solo", P.ENGINE_WIDE: "wide", P.ENGINE_STREAMING: "streaming", P.ENGINE_LARGE: "large", P.ENGINE_CUFFT: "cufft"}.get(eng, str(eng))
    traffic, traffic_source = ncu_traffic(args.workload, eng_name, rt_per_step)
    if eng in (P.ENGINE_RESIDENT, P.ENGINE_SOLO, P.ENGINE_WIDE):
        # fields stay on chip (shared memory / tensor memory): bound by the FP32 (FP64) FMA pipe, shared memory second.
        # Both peaks are MEASURED here, on this device, by the library's own micro-benchmark kernels (opo_selftest_peak).
        fl = flops_per_grid_point_zstep(w.log2_n, w.n_fields) * units_per_step          # per launch (= per step)
        dbl = w.precision == "c128"
        sms = int(P.opo_get_info(o._h, P.INFO_SM_COUNT))
        sm_max_ghz = (clocks.get("sm_max_mhz") or 1965.0) / 1e3
        peak_nominal = sms * (64 if dbl else 128) * 2 * sm_max_ghz * 1e9 / 1e12
        peak_meas = P.opo_selftest_peak(P.PEAK_FP64_FMA if dbl else P.PEAK_FP32_FMA)
        smem_peak = P.opo_selftest_peak(P.PEAK_SMEM)
        smem_by = smem_bytes_per_field_point_zstep(w.precision) * w.n_fields * units_per_step
        roofline = {"bound": "alu", "kernel": {P.ENGINE_SOLO: "k_solo", P.ENGINE_WIDE: "k_wide"}.get(eng, "k_resident"), "achieved": fl / avg_s / 1e12,
                    "peak": peak_meas, "unit": "TFLOP/s", "frac": fl / avg_s / 1e12 / peak_meas,
                    "peak_nominal": peak_nominal, "frac_of_nominal": fl / avg_s / 1e12 / peak_nominal,
                    "traffic": traffic, "traffic_source": traffic_source,
                    "smem": {"achieved": smem_by / avg_s / 1e9, "peak": smem_peak, "unit": "GB/s", "frac": smem_by / avg_s / 1e9 / smem_peak,
                             "note": f"algorithmic shared-memory bytes = {smem_bytes_per_field_point_zstep(w.precision):.0f} B per field-point z-step "
                                     "(6 passes x read + write); peak = conflict-free 16 B loads + stores on every SM, measured in this run"},
                    **({"link": wide_link_roofline(w, o, P, units_per_step, avg_s)} if eng == P.ENGINE_WIDE else {}),
                    "note": f"peak = {'FP64' if dbl else 'FP32'} FMA throughput measured in this run by opo_selftest_peak (independent FMA chains on every SM); "
                            f"peak_nominal = {sms} SM x {64 if dbl else 128} lanes x 2 x {sm_max_ghz:.3f} GHz; "
                            f"algorithmic flops = {flops_per_grid_point_zstep(w.log2_n, w.n_fields):.0f}/grid-point z-step "
                            "(merged half-steps, 5 N log2 N per transform); one launch = one step"}
    else:
        # fields stream through L2 / HBM: algorithmic bytes per field-point z-step: large engine 32 B
        # (row pass R+W, column pass R+W), streaming engine 40 B (linear R+W + table, RK4 R+W)
        esz = 16 if w.precision == "c128" else 8
        # cuFFT baseline: FFT R+W, multiply R+W + table, inverse FFT R+W, RK4 R+W = 9 complex per field-point z-step
        per_fp = (4 * esz) if eng == P.ENGINE_LARGE else ((9 * esz) if eng == P.ENGINE_CUFFT else (5 * esz))
        by = per_fp * w.n_fields * units_per_step
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json"))) if os.path.exists(os.path.join(ROOT, "MEASURED_PEAKS.json")) else {}
        peak = float(peaks.get("hbm_gbs", 6543.1))
        n_launch = max(1, int(launches) // max(1, args.steps))
        roofline = {"bound": "hbm", "kernel": "k_large" if eng == P.ENGINE_LARGE else ("cufft+k_multab+k_rk4" if eng == P.ENGINE_CUFFT else "k_linear+k_rk4"), "achieved": by / avg_s / 1e9,
                    "peak": peak, "unit": "GB/s", "frac": by / avg_s / 1e9 / peak, "traffic": traffic, "traffic_source": traffic_source,
                    "note": f"algorithmic bytes = {per_fp} B per field-point z-step; peak = measured HBM copy bandwidth "
                            f"({'MEASURED_PEAKS.json' if peaks else 'B200_PROFILING.md fallback'}); {n_launch} launch(es) per step; "
                            "the state of this workload is L2-resident, so this is L2 service measured against the HBM roofline"}
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": t_total / args.steps * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32" if w.precision == "c64" else "f64", "data": "synthetic",
            "config": {"workload": f"{w.name}: BASELINE.json configs[{args.workload[1]}], batch {w.batch} x N=2^{w.log2_n} x "
                                   f"{w.n_fields} fields, nz={w.nz_per_pass}, {rt_per_step} round trips per step" + (", EOM on the signal" if args.eom else ""),
                       "engine": eng_name, **({"mode": "pump train: one pump slice in and one exit slice out per round trip (opo_roundtrips_train)"} if args.train else {}),
                       "l2": "512 MiB flush write between timed steps", "sharding": "independent instances per rank, no collective"},
            "round_trips_per_s": world * w.batch * rt_per_step * args.steps / t_total,
            "field_point_z_steps_per_s": value * w.n_fields,
            "clocks": clocks, "gpu_launches": int(launches), "wall_s_timed_region": t_wall,
            "roofline": roofline}
    if e2e:
        line["e2e"] = e2e
    if not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(w)
    print(json.dumps(line), flush=True)
    o.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

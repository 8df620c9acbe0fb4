#!/usr/bin/env python
"""bench.py -- throughput of the hot path on the BASELINE.json headline workload.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg3] [--impl ours|reference]

One "step" = one full RK2 update of every active cell of the pack: ak_new_dt, then 2 x (ak_fill_ghosts,
ak_hydro_stage).  Default workload = BASELINE.json configs[3]: 512^3 periodic mesh
as 64 MeshBlocks of 128^3, PPM4 + HLLC, RK2, fp64, seeded synthetic initial state.  Prints ONE JSON line.
N > 1 runs N independent replicas (the path does not shard: north_star).
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

METRIC = "3D hydro cell-updates/sec (fp64)"
UNIT = "cell-updates/s"
BYTES_PER_CELL_UPDATE = 200.0      # 5 streams x 5 vars x 8 B per RK2 cell-update
BYTES_STAGE = {1: 80.0, 2: 120.0}  # per active cell: stage 1 reads U^n writes U^(1); stage 2 reads U^(1),U^n writes
# ncu's DRAM bytes and FP64-pipe instructions per stage launch come from profiles/r02_stage_counters_<workload>.json
# (written by paper_2409_16053_b200/counters.py from an ncu pass of THIS command); they are printed only while the hash
# of the kernel sources stored there equals the hash of the tree this runs from
FP64_LANES_PER_SM = 64             # DESIGN.md 6.1 (ncu peak_sustained of the dfma counter / SM count)


def workloads():
    from paper_2409_16053_b200 import inputs as I
    return {
        "cfg3": lambda: I.config3(),
        "cfg3_small": lambda: I.config3(nrb=2, nx=64),
        "cfg1": lambda: I.config1(),
        "cfg2_16": lambda: I.config2(16), "cfg2_32": lambda: I.config2(32),
        "cfg2_64": lambda: I.config2(64), "cfg2_128": lambda: I.config2(128),
        "cfg4": lambda: I.config4(),
        "table1": lambda: I.table1(),
    }


def measured_peaks():
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json"))), "measured"
    except Exception:
        return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (profiling guide recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index, self.first = [], None, index, 0

    def mark(self):
        """Start of the timed region: only rows sampled from here on are reported."""
        self.first = len(self.rows)

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if self.proc:
            self.proc.terminate()
        self.rows = self.rows[self.first:]
        sm = [float(r[0]) for r in self.rows if r and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({n for r in self.rows if len(r) >= 7 for n, v in zip(names, r[3:7]) if v.lower().startswith("active")})
        pw = [float(r[2]) for r in self.rows if len(r) > 2 and r[2].replace(".", "").isdigit()]
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": reasons}


def cpu_baseline(threads=1, target_s=12.0):
    """The oracle as it stands on a bounded sample of the headline recipe (config 3 at 8 x 32^3 / 8 x 64^3)."""
    from paper_2409_16053_b200 import inputs as I
    from oracle import orc
    w = I.config3(nrb=2, nx=32)
    U0 = w.state().numpy()
    p = orc.OrcPack(w.mesh, w.gamma, w.recon, threads=threads)
    p.load(U0)
    p.step(w.cfl)                                  # warm the caches / page in
    t0, n = time.perf_counter(), 0
    while True:
        p.step(w.cfl)
        n += 1
        el = time.perf_counter() - t0
        if el >= target_s or n >= 50:
            break
    p.close()
    return {"value": w.mesh.ncells_active * n / el, "unit": UNIT, "cores": threads, "kind": "oracle",
            "sample": f"config-3 recipe (PPM4+HLLC, Mach-1 modes + shear) on 8 MeshBlocks of 32^3, {n} RK2 steps, "
                      f"{el:.1f} s, single-threaded C++ oracle"}


def cpu_baseline_mhd(recon, nst, rsolver=0, target_s=10.0):
    """The MHD oracle as it stands on a bounded sample of the MHD recipe (mhd_64: 8 MeshBlocks of 32^3), one thread."""
    from paper_2409_16053_b200 import inputs as I
    from oracle import orc_mhd
    orc_mhd.build()
    mesh, prim, A, B0 = I.mhd_workload("mhd_64", ng=3 if recon == 0 else 4)
    p = orc_mhd.OrcMhdPack(mesh, I.GAMMA, recon=recon, nstages=nst, rsolver=rsolver)
    p.load(I.make_state_mhd(mesh, prim, A, B0).numpy())
    p.step(I.CFL)
    t0, n = time.perf_counter(), 0
    while True:
        p.step(I.CFL)
        n += 1
        el = time.perf_counter() - t0
        if el >= target_s or n >= 50:
            break
    p.close()
    return {"value": mesh.ncells_active * n / el, "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": f"the MHD recipe on 8 MeshBlocks of 32^3, {n} steps, {el:.1f} s, single-threaded C++ oracle"}


def max_over_ranks(x: float, device=None) -> float:
    """Timing rule of the bench contract: a multi-rank time is the MAX over ranks (all-reduce on `device`;
    identity when no process group exists)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(x)
    t = torch.tensor([x], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(ncell_per_rank: int, steps: int, elapsed_ms_max: float, world: int) -> float:
    """Whole-job cell-updates/s of `world` independent replicas (weak scaling)."""
    return world * ncell_per_rank * steps / (elapsed_ms_max * 1e-3)


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cb = cpu_baseline(threads=1, target_s=max(5.0, min(60.0, 2.0 * (args.steps + args.warmup))))
    from paper_2409_16053_b200 import inputs as I
    w = I.config3()
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": cb["value"], "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * w.mesh.ncells_active / cb["value"],
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "cfg3: 512^3 periodic, 64 MeshBlocks of 128^3, PPM4+HLLC, RK2 (oracle timed on a bounded "
                               "sample of this workload; ms_per_step extrapolated to the full mesh)"},
        "cpu_baseline": cb,
        "e2e": {"value": cb["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def run_mhd(args):
    """The MHD + CT path (include/ak_mhd.h): same contract, metric and timing rules as the hydro line."""
    import torch
    from paper_2409_16053_b200 import ak_mhd, inputs as I
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    recon = {None: 0, "plm": 0, "ppm4": 1, "ppmx": 2, "wenoz": 3}[args.recon]
    nst = args.integrator
    mesh, prim, A, B0 = I.mhd_workload(args.workload, ng=3 if recon == 0 else 4)
    U0 = I.make_state_mhd(mesh, prim, A, B0, device=dev)
    rs = {"hllc": 0, "llf": 1, "hlle": 2}.get(args.rsolver)
    if rs is None or (rs and recon):
        raise SystemExit("MHD workloads: --rsolver llf | hlle (PLM only); the default is HLLD")
    pack = ak_mhd.MhdPack(mesh, I.GAMMA, device=dev, recon=recon, nstages=nst, rsolver=rs)
    pack.load(U0)
    ncell, state_bytes = mesh.ncells_active, U0.numel() * 8
    sampler = ClockSampler(local)
    sampler.start()
    for _ in range(args.warmup):
        pack.step(I.CFL)
    t_w = time.perf_counter()
    while not sampler.rows and sampler.proc and time.perf_counter() - t_w < 3.0:
        pack.step(I.CFL)
    torch.cuda.synchronize(dev)
    sampler.mark()
    l0 = pack.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    stage_ev = []
    e0.record(pack.stream)
    for _ in range(args.steps):
        dt = pack.new_dt(I.CFL)
        for stage in range(1, nst + 1):
            pack.fill_ghosts()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(pack.stream); pack.stage(stage, dt); b.record(pack.stream)
            stage_ev.append((stage, a, b))
    e1.record(pack.stream)
    torch.cuda.synchronize(dev)
    clocks = sampler.stop()
    launches = pack.launch_count() - l0
    floors = pack.floor_count()
    elapsed_ms = e0.elapsed_time(e1)
    value = ncell * args.steps / (elapsed_ms * 1e-3)
    st_ms = {s_: statistics.mean(a.elapsed_time(b) for ss, a, b in stage_ev if ss == s_) for s_ in range(1, nst + 1)}
    stage_ms = sum(st_ms.values()) / nst
    peaks, which = measured_peaks()
    alg = (128.0 + 192.0 * (nst - 1)) / nst * ncell   # stage 1 reads 8 and writes 8 variables, the later stages read 16 and write 8
    ach = alg / (stage_ms * 1e-3) / 1e9
    host = torch.empty(U0.shape, dtype=torch.float64).pin_memory()
    host.copy_(U0)
    t0 = time.perf_counter()
    for _ in range(2):                          # end to end: host -> device, one step, device -> host
        pack.load(host)
        pack.step(I.CFL)
        host.copy_(pack.current())
    torch.cuda.synchronize(dev)
    e2e = {"value": ncell * 2 / (time.perf_counter() - t0), "unit": UNIT, "h2d_bytes_per_step": state_bytes, "d2h_bytes_per_step": state_bytes, "steps": 2}
    print(json.dumps({
        "metric": "3D MHD cell-updates/sec (fp64)", "value": value, "unit": UNIT, "n_gpus": 1, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": elapsed_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": f"{args.workload}: MHD + CT, {['PLM', 'PPM4', 'PPMX', 'WENOZ'][recon]} + {['HLLD', 'LLF', 'HLLE'][rs]}, SSPRK{nst}, {mesh.nmb} MeshBlocks of {mesh.nx[0]}^3, ng {mesh.ng}, Mach-0.5 modes + mean field",
                   "cells": ncell, "state_bytes": state_bytes, "l2_policy": "inputs larger than L2" if state_bytes > 4e8 else "state fits L2",
                   "parallelism": "single GPU"},
        "roofline": {"bound": "hbm", "achieved": ach, "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": ach / peaks["hbm_gbs"], "traffic": None,
                     "peak_source": which + " (MEASURED_PEAKS.json hbm_gbs)", "kernel": "akm_stage (six kernels: prim, 3 x flux, emf, update)",
                     "kernel_ms": stage_ms, "kernel_share_of_step": nst * stage_ms * args.steps / elapsed_ms, "algorithmic_bytes_per_launch": alg},
        "cpu_baseline": None if args.no_cpu else cpu_baseline_mhd(recon, nst, rs), "e2e": e2e, "gpu_launches": launches, "clocks": clocks,
        "stage_ms": st_ms, "floor_activations": floors,
    }))


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2409_16053_b200 import ak

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    w = workloads()[args.workload]()
    if args.recon is not None:
        w.recon = {"plm": 0, "ppm4": 1, "ppmx": 2, "wenoz": 3}[args.recon]
    mesh = w.mesh
    pack = ak.Pack(mesh, w.gamma, w.recon, rsolver={"hllc": 0, "llf": 1, "hlle": 2, "roe": 3}[args.rsolver], device=dev,
                   variant=args.variant)
    if args.flux_correction:
        pack.set_flux_correction(True)
    if args.integrator == 3:
        pack.set_integrator(3)
    if args.tile is not None:
        pack.set_tile(args.tile)
    U0 = w.state(device=dev)
    pack.load(U0)
    ncell = mesh.ncells_active
    state_bytes = U0.numel() * 8

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    # ---- device-resident timing ------------------------------------------------------------------
    sampler = ClockSampler(local)
    sampler.start()                    # nvidia-smi needs a few 100 ms to come up: start it under the warm-up load
    for _ in range(args.warmup):
        pack.step(w.cfl)
    t_w = time.perf_counter()
    while not sampler.rows and sampler.proc and time.perf_counter() - t_w < 3.0:
        pack.step(w.cfl)               # nvidia-smi takes a few 100 ms to deliver its first row: stay under load meanwhile
    stage_ev = []
    barrier()
    sampler.mark()
    l0 = pack.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(pack.stream)
    for _ in range(args.steps):
        dt = pack.new_dt(w.cfl)
        for stage in range(1, args.integrator + 1):
            pack.fill_ghosts()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(pack.stream)
            pack.hydro_stage(stage, dt)
            b.record(pack.stream)
            stage_ev.append((stage, a, b))
    e1.record(pack.stream)
    barrier()
    clocks = sampler.stop()
    launches = pack.launch_count() - l0
    elapsed_ms = max_over_ranks(e0.elapsed_time(e1), dev)
    floors = pack.floor_count()
    value = aggregate_value(ncell, args.steps, elapsed_ms, world)

    # dominant kernel = the stage kernel: algorithmic bytes per launch / mean launch duration
    nst = args.integrator
    st_ms = {s: statistics.mean(a.elapsed_time(b) for ss, a, b in stage_ev if ss == s) for s in range(1, nst + 1)}
    stage_ms = sum(st_ms.values()) / nst
    # stage 1 moves 80 B per cell, every later stage (which also reads U^n) 120 B
    alg_bytes = (BYTES_STAGE[1] + (nst - 1) * BYTES_STAGE[2]) / nst * ncell
    peaks, which = measured_peaks()
    achieved = alg_bytes / (stage_ms * 1e-3) / 1e9
    from paper_2409_16053_b200 import counters
    ctr = counters.load(args.workload) if (args.variant == 0 and args.rsolver == "hllc" and args.integrator == 2
                                            and args.recon is None and not args.flux_correction and args.tile is None) else None
    traffic = args.traffic
    if traffic is None and ctr:
        L = ctr["launches"]
        traffic = sum(L[k]["dram__bytes_read.sum"] + L[k]["dram__bytes_write.sum"] for k in ("stage1", "stage2")) / 2.0
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                "frac": achieved / peaks["hbm_gbs"], "traffic": traffic, "peak_source": which + " (MEASURED_PEAKS.json hbm_gbs)",
                "kernel": "ak_hydro_stage", "kernel_ms": stage_ms, "kernel_share_of_step": nst * stage_ms * args.steps / elapsed_ms,
                "algorithmic_bytes_per_launch": alg_bytes,
                "whole_step": {"achieved": BYTES_PER_CELL_UPDATE * value / world / 1e9,
                               "frac": BYTES_PER_CELL_UPDATE * value / world / 1e9 / peaks["hbm_gbs"]}}

    # the unit that actually binds the stage kernel is the FP64 pipe (plain ALU work)
    roofline_alu = None
    if ctr:
        L = ctr["launches"]
        sms = torch.cuda.get_device_properties(dev).multi_processor_count
        peak_alu = sms * FP64_LANES_PER_SM * float(peaks.get("sm_max_mhz", 1965.0)) * 1e6 / 1e12
        # warp instructions on the FP64 pipe x 32 lanes, per stage launch (mean of the two stages)
        fp64_thread_instr = 32.0 * sum(L[k]["sm__inst_executed_pipe_fp64.sum"] for k in ("stage1", "stage2")) / 2.0
        alu_thread_instr = 32.0 * sum(L[k]["sm__inst_executed_pipe_alu.sum"] for k in ("stage1", "stage2")) / 2.0
        ach_alu = fp64_thread_instr / (stage_ms * 1e-3) / 1e12
        roofline_alu = {"bound": "alu", "achieved": ach_alu, "peak": peak_alu, "unit": "T FP64-pipe thread-instr/s",
                        "frac": ach_alu / peak_alu, "kernel": "ak_hydro_stage",
                        "instr_per_cell_launch": fp64_thread_instr / ncell,
                        "alu_pipe_instr_per_cell_launch": alu_thread_instr / ncell,
                        # on this part FP64-pipe and ALU-pipe warp instructions issue at 2 cycles each and
                        # overlap only partly; the fraction below is of the limit the probe measured for an ideally
                        # interleaved stream, 0.78 x 2 cycles x (FP64 + ALU instructions)
                        "frac_of_dispatch_limit": 0.78 * 2.0 * (fp64_thread_instr + alu_thread_instr) / 32.0
                                                  / (sms * 4 * float(peaks.get("sm_max_mhz", 1965.0)) * 1e6 * stage_ms * 1e-3),
                        "counters": f"profiles/r02_stage_counters_{args.workload}.json (csrc hash {ctr['csrc_sha']})",
                        "peak_source": f"{sms} SMs x {FP64_LANES_PER_SM} FP64 lanes x sm_max_mhz (DESIGN.md 6.1)"}

    # ---- end to end through the C-ABI with HOST buffers ------------------------------------------
    e2e = None
    if not args.no_e2e:
        host = torch.empty(U0.shape, dtype=torch.float64).pin_memory()
        host.copy_(U0)
        nst = max(1, min(args.steps, args.e2e_steps))
        pack.upload(host); pack.step(w.cfl); pack.download(host)          # warm-up of the copy path
        barrier()
        t0 = time.perf_counter()
        for _ in range(nst):
            pack.upload(host)              # H2D of this step's input state (pinned)
            pack.step(w.cfl)
            pack.download(host)            # D2H of the step's result; synchronises
        torch.cuda.synchronize(dev)
        el = max_over_ranks(time.perf_counter() - t0, dev)
        e2e = {"value": aggregate_value(ncell, nst, el * 1e3, world), "unit": UNIT, "h2d_bytes_per_step": state_bytes,
               "d2h_bytes_per_step": state_bytes, "steps": nst}
        # The same bytes per step with the two directions of the link used at once: two packs on two streams take
        # alternate, independent input states (every step still uploads its input and downloads its result inside
        # the timed region); one pack's download overlaps the other's upload.  Reported beside e2e, not instead of it.
        if args.e2e_pipelined:
            out = [torch.empty(U0.shape, dtype=torch.float64).pin_memory() for _ in range(2)]
            streams = [torch.cuda.Stream(device=dev) for _ in range(2)]
            packs = [ak.Pack(mesh, w.gamma, w.recon, rsolver={"hllc": 0, "llf": 1, "hlle": 2, "roe": 3}[args.rsolver], device=dev,
                             stream=s_, variant=args.variant) for s_ in streams]
            host.copy_(U0)
            npipe = 2 * max(2, nst)
            for q in packs:                                  # warm-up (also sizes the tensor maps)
                q.upload(host); q.step(w.cfl); q.download(out[0])
            barrier()
            t0 = time.perf_counter()
            for n in range(npipe):
                q = packs[n & 1]
                q.upload(host)                               # H2D of this step's input (async on the pack's stream)
                q.step(w.cfl)                                # waits for its own stream only (dt goes to the host)
                q.download_async(out[n & 1])                 # D2H of this step's result, overlapping the other pack
            torch.cuda.synchronize(dev)
            el = max_over_ranks(time.perf_counter() - t0, dev)
            e2e["pipelined"] = {"value": aggregate_value(ncell, npipe, el * 1e3, world), "unit": UNIT, "steps": npipe,
                                "h2d_bytes_per_step": state_bytes, "d2h_bytes_per_step": state_bytes,
                                "how": "two packs on two streams, alternate independent inputs"}
            del packs, out
        del host

    if rank == 0:
        cb = None if args.no_cpu else cpu_baseline(threads=1)
        print(json.dumps({
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": elapsed_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{args.workload}: {w.name}", "nmb": mesh.nmb, "nx": list(mesh.nx), "ng": mesh.ng,
                       "recon": ["PLM", "PPM4", "PPMX", "WENOZ"][w.recon], "rsolver": args.rsolver.upper(), "integrator": "SSPRK2" if args.integrator == 2 else "SSPRK3", "cfl": w.cfl,
                       "cells": ncell, "state_bytes": state_bytes, "l2_policy": "inputs larger than L2 (no flush needed)"
                       if state_bytes > 4e8 else "state fits L2: numbers are L2-resident", "variant": args.variant, "flux_correction": bool(args.flux_correction),
                       "parallelism": "replicas only" if world > 1 else "single GPU"},
            "roofline": roofline, "roofline_alu": roofline_alu, "cpu_baseline": cb, "e2e": e2e, "gpu_launches": launches, "clocks": clocks,
            "stage_ms": st_ms, "floor_activations": floors,
        }))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg3")
    ap.add_argument("--variant", type=int, default=0)
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-e2e-pipelined", dest="e2e_pipelined", action="store_false",
                    help="skip the second end-to-end figure (two packs on two streams, upload and download overlapped)")
    ap.add_argument("--recon", default=None, choices=["plm", "ppm4", "ppmx", "wenoz"],
                    help="override the workload's reconstruction (ppmx / wenoz: SURVEY 8(f) f2, need a workload with ng = 3)")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--rsolver", default="hllc", choices=["hllc", "llf", "hlle", "roe"],
                    help="Riemann solver (headline metric: hllc; llf / hlle are the f2 variants on the same kernel)")
    ap.add_argument("--integrator", type=int, default=2, choices=[2, 3],
                    help="stages per step: 2 = SSPRK(2,2) (headline), 3 = SSPRK(3,3) (f2 variant, third state register)")
    ap.add_argument("--flux-correction", action="store_true",
                    help="refined meshes (cfg4): flux correction at coarse-fine faces on (SURVEY 8(f) f1; off by default)")
    ap.add_argument("--tile", type=int, default=None, help="tile shape of the production kernel (ak_pack_set_tile; default: automatic)")
    ap.add_argument("--traffic", type=float, default=None,
                    help="dram bytes per stage launch from the committed ncu --set full capture (profiles/)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.workload.startswith("mhd"):
        run_mhd(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()

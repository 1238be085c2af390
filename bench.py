#!/usr/bin/env python
"""bench.py — FP64 cell-updates/s of the ECHO RMHD step on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--n 256] [--direction diag|x] [--impl reference]

A "step" is one full SSP-RK3 time step (three passes of the whole hot path: INT+con2prim, three fused
flux sweeps, UCT, curl+update) of the 3-D circularly-polarised Alfven wave on an n^3 periodic
box, FP64; value = cells x steps / seconds, inputs resident in HBM.  Default workload: BASELINE.json
configs[2] (256^3).  N > 1: every rank advances its own independent box (replicas, no collective; DESIGN.md
"Multi-GPU"), value = sum over ranks / max time.  One JSON line on stdout (rank 0).
"""
import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

GAMMA, CFL = 4.0 / 3.0, 0.3
SETK = "rho vx vy vz p bxf byf bzf".split()

# Algorithmic work per cell and per launch.
# flop: nominal FP64 operation count of the scheme; dbl: FP64 words read+written once per cell by the
# kernel as built, averaged over the three RK stages where the stages differ:
#   k_prim   5 U + 3 B in, 5 prims + 3 centred B out = 16; stage 2 also reads rhs (5) and writes U1 (5)
#   k_flux_x 8 in, 5 rhs + 4 saved face fields out = 17;  k_flux_y the same + 5 rhs in = 22
#   k_flux_z stage 1: 22; stages 2-3 (RK combination fused): + U cur (5) + U^n (5) in, U out instead of rhs = 32
#   k_uct    6 speeds + 6 vbar + 3 B in, 3 E out = 18;  k_update (staggered B): 3 E + 3 + 3 in, 3 out (stage 1: 9)
ALGO = {
    "k_prim":   {"flop": 24 + 268, "dbl": (16 + 26 + 16) / 3.0},
    "k_flux_x": {"flop": 614, "dbl": 17},
    "k_flux_y": {"flop": 614, "dbl": 22},
    "k_flux_z": {"flop": 614 + 32 * 2 / 3.0, "dbl": (22 + 32 + 32) / 3.0},
    "k_uct":    {"flop": 3 * 194, "dbl": 18},
    "k_update": {"flop": 60 + 12, "dbl": (9 + 12 + 12) / 3.0},
}
FLOP_PER_CELL_UPDATE = 3 * sum(v["flop"] for v in ALGO.values())          # ~8.4e3
BYTES_PER_CELL_UPDATE = 8 * 3 * sum(v["dbl"] for v in ALGO.values())      # 2784
# UCT = NO (--scheme cc-ho / cc-lo, row f2): 8 cell fields, no UCT and no separate update kernel
#   k_prim   8 in, 5 prims + 3 B copies out = 16; stage 2 also reads rhs (8) and writes U1, B1 (8)
#   k_flux_x 8 in, 8 rhs out = 16;  k_flux_y + 8 rhs in = 24;  k_flux_z stage 1: 24, stages 2-3: + cur (8) + U^n (8) = 40
# flop: + one more MP5 pair and the three induction fluxes per face (nominal 60)
ALGO_CC = {
    "k_prim":   {"flop": 268, "dbl": (16 + 32 + 16) / 3.0},
    "k_flux_x": {"flop": 674, "dbl": 16},
    "k_flux_y": {"flop": 674, "dbl": 24},
    "k_flux_z": {"flop": 674 + 48 * 2 / 3.0, "dbl": (24 + 40 + 40) / 3.0},
}
# name -> (uct, ho, rec, rk); "*-lo2" is the second-order variant of P:L304 (limited linear REC + SSP-RK2)
SCHEMES = {"uct-ho": (True, True, 5, 3), "uct-lo": (True, False, 5, 3), "cc-ho": (False, True, 5, 3),
           "cc-lo": (False, False, 5, 3), "uct-lo2": (True, False, 2, 2), "cc-lo2": (False, False, 2, 2)}
# the same per-launch words for the two-stage scheme (stage 1 + one fused stage instead of two)
# the paper's step rates x 512^3 cells for the diagonal CPA wave at 512^3 on ONE NODE of
# LEONARDO (4 x A100 64 GB), per scheme (Table 1).  vs_baseline is quoted only for that workload.
PAPER_512_PER_NODE = {"uct-ho": 1.13 * 512 ** 3, "cc-lo": 1.21 * 512 ** 3, "cc-lo2": 2.2e8}
ALGO_RK2 = {"k_prim": (16 + 26) / 2.0, "k_flux_z": (22 + 32) / 2.0, "k_update": (9 + 12) / 2.0}
ALGO_CC_RK2 = {"k_prim": (16 + 32) / 2.0, "k_flux_z": (24 + 40) / 2.0}


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return json.load(f), "measured"
    return {"hbm_gbs": 6650.0}, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.gpu = gpu_index
        self.proc = None
        self.path = None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(suffix=".csv")
            os.close(fd)
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.gpu), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        try:
            for line in open(self.path):
                f = [x.strip() for x in line.split(",")]
                if len(f) < 9:
                    continue
                try:
                    sm.append(float(f[1])); mx.append(float(f[2]))
                except ValueError:
                    continue
                for nm, val in zip(names, f[5:9]):
                    if val.lower().startswith("active"):
                        reasons.add(nm)
            os.unlink(self.path)
        except Exception:
            pass
        if sm:
            sm.sort()
            out.update(sm_mhz=sm[len(sm) // 2], sm_max_mhz=max(mx), samples=len(sm))
        out["reasons"] = sorted(reasons)
        return out


def max_over_ranks(value, device, world):
    """Max over ranks of a host float (NCCL on the GPU, gloo in the CPU tests); identity for one rank."""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(cells_per_rank, steps, ms_local, device, world):
    """Whole-job cell-updates/s: all ranks' cells x steps / the slowest rank's device time."""
    ms = max_over_ranks(ms_local, device, world)
    return world * cells_per_rank * steps / (ms * 1e-3), ms


def oracle_rate(n, steps, warmup=0, direction="diag"):
    """The oracle as it stands, single-threaded, on an n^3 box of the same wave: cell-updates/s."""
    from oracle import binding as ob
    from paper_2401_03008_b200 import inputs
    w = inputs.cpa_wave(n, n, n, direction=direction)
    o = ob.Oracle(n, n, n, GAMMA, CFL)
    o.set_primitives(*[w[k] for k in SETK])
    if warmup:
        o.step(warmup)
    t0 = time.perf_counter()
    o.step(steps)
    dt = time.perf_counter() - t0
    return n ** 3 * steps / dt, dt


def run_reference(args):
    """--impl reference: the CPU oracle on the host cores, a bounded sample (48^3 box) per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    n = args.ref_n
    rate, dt = oracle_rate(n, args.steps, args.warmup, args.direction)
    sample = "%d^3 box of the same CPA wave (P:L217-233), %d RK3 steps, single thread" % (n, args.steps)
    line = {"impl": "reference", "metric": "fp64_cell_updates_per_sec", "value": rate, "unit": "cell-updates/s",
            "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            # the arm's own workload (same name as the echo arm prints); each step advances a bounded sample of it
            "config": {"workload": "cpa_wave_%s_%d^3" % (args.direction, args.n), "gamma": GAMMA, "cfl": CFL,
                       "scheme": "MP5+HLL+UCT+DER6/INT6+SSPRK3 (UCT=HO=YES)", "sample": sample},
            "cpu_baseline": {"value": rate, "unit": "cell-updates/s", "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": rate, "unit": "cell-updates/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def run_gpu(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_2401_03008_b200 import binding, inputs

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback); use --impl reference for the oracle")
    torch.cuda.set_device(local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    binding.lib()

    n, K, W = args.n, args.steps, max(args.warmup, 3)
    N = n ** 3
    uct, ho, rec, rk = SCHEMES[args.scheme]
    if args.scheme != "uct-ho" and (args.workload != "cpa" or args.decompose):
        raise SystemExit("--scheme variants are wired for the default cpa workload only")
    ALGO = {k: dict(v) for k, v in (globals()["ALGO"] if uct else ALGO_CC).items()}
    if rk == 2:
        for k, dbl in (ALGO_RK2 if uct else ALGO_CC_RK2).items():
            ALGO[k]["dbl"] = dbl
    # (the flop entries are the nominal counts of the MP5 scheme; with linear REC they overstate the arithmetic)
    FLOP_PER_CELL_UPDATE = rk * sum(v["flop"] for v in ALGO.values())
    BYTES_PER_CELL_UPDATE = 8 * rk * sum(v["dbl"] for v in ALGO.values())
    decomposed = bool(args.decompose) and world > 1
    if decomposed:
        # ONE periodic box of (n px, n py, n pz) cells, one n^3 block (+ width-8 halos) per rank: halo exchange of
        # the 8 evolved fields after every RK stage + all-reduce(max) of a_max per step
        from paper_2401_03008_b200 import blocks
        pgrid = {2: (2, 1, 1), 4: (2, 2, 1), 8: (2, 2, 2)}.get(world, (world, 1, 1))
        gn = tuple(n * q for q in pgrid)
        rb = blocks.RankBlock(gn, pgrid, GAMMA, CFL)
        c = rb.d.coords(rank)
        start = tuple(c[a] * rb.d.interior[a] - rb.d.halo[a] for a in range(3))
        w = inputs.cpa_wave(*rb.d.local, direction=args.direction, box=(gn, start))
        e = rb.block
        stepper = rb.step
        parallelism = "one box of %dx%dx%d cells in %dx%dx%d blocks, halo 8, NCCL p2p + all-reduce(max)" % (gn + pgrid)
    elif args.workload == "turb3d":
        # BASELINE.json configs[4]: relativistic Alfvenic turbulence on n^3 (384^3), sigma = 1, dB/B0 = 0.5
        w = inputs.turbulence(n)
        e = binding.Echo(n, n, n, GAMMA, CFL)
        faces = e.faces_from_potential(*[torch.as_tensor(w[k], device="cuda") for k in ("ax", "ay", "az")], w["b0"])
        for k, f in zip(("bxf", "byf", "bzf"), faces):
            w[k] = f.cpu().numpy()
        del faces
        stepper = e.step
        parallelism = "replicas x%d (no collective)" % world
    elif args.workload == "turb2d":
        # row f3: the paper's 2.5-D turbulence set-up on an n x n x 1 grid; faces from the potential
        w = inputs.turbulence_2d(n)
        N = n * n
        e = binding.Echo(n, n, 1, GAMMA, CFL)
        faces = e.faces_from_potential(*[torch.as_tensor(w[k], device="cuda") for k in ("ax", "ay", "az")], w["b0"])
        for k, f in zip(("bxf", "byf", "bzf"), faces):
            w[k] = f.cpu().numpy()
        stepper = e.step
        parallelism = "replicas x%d (no collective)" % world
    else:
        w = inputs.cpa_wave(n, n, n, direction=args.direction)
        e = binding.Echo(n, n, n, GAMMA, CFL, uct=uct, ho=ho, rec=rec, rk=rk)
        stepper = e.step
        parallelism = "replicas x%d (no collective)" % world
    setk = SETK if uct else "rho vx vy vz p bx by bz".split()       # UCT = NO evolves the cell-centred B
    host = [torch.from_numpy(np.ascontiguousarray(w[k])).pin_memory() for k in setk]
    devin = [h.to("cuda", non_blocking=True) for h in host]
    e.set_primitives(*devin)
    del devin

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident throughput: W warm-up steps, then EXACTLY K timed steps, per-kernel timers OFF
    sampler = ClockSampler(local)       # started before the warm-up so that nvidia-smi is already polling
    sampler.start()                     # when the timed region begins (samples cover warm-up + timed steps)
    stepper(W)
    barrier()
    e.timing(False)                     # also clears the launch counters
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record()
    stepper(K)
    ev1.record()
    barrier()
    clocks = sampler.stop()
    ms = ev0.elapsed_time(ev1)
    nlaunch = sum(cnt for _, cnt in e.get_timing().values())       # kernels launched inside the timed region
    value, ms_max = whole_job_rate(N, K, ms, "cuda", world)
    # ---- second pass, only for the per-kernel split: the same steps with a CUDA-event pair around every launch
    # (the brackets cost a little, so this pass never feeds `value`); one untimed step first grows the event pool
    Kk = min(K, args.kernel_steps)
    e.timing(True)
    stepper(1)
    e.timing(True)
    ev0.record()
    stepper(Kk)
    ev1.record()
    barrier()
    ms_kpass = ev0.elapsed_time(ev1)
    ktimes = e.get_timing()
    e.timing(False)
    d = e.diagnostics()
    assert d["rc"] == 0 and d["steps"] == W + K + 1 + Kk, d

    # ---- end to end through the C ABI with HOST buffers: every step uploads its inputs from pinned host
    # memory (echo_set_primitives_host), advances one RK3 step and reads the primitives back to the host
    outs = [torch.empty(e.shape, dtype=torch.float64).pin_memory() for _ in range(8)]
    Ke = min(K, args.e2e_steps)
    for _ in range(2):
        e.set_primitives_host(*host); stepper(1); e.get_primitives_host(outs)
    barrier()
    ev0.record()
    for _ in range(Ke):
        e.set_primitives_host(*host)
        stepper(1)
        e.get_primitives_host(outs)
    ev1.record()
    barrier()
    e2e_serial, _ = whole_job_rate(N, Ke, ev0.elapsed_time(ev1), "cuda", world)
    e2e_value, e2e_how = e2e_serial, "serial: upload, step, download one after the other on one stream"
    if not decomposed:
        # the same three calls per step, but on L handles bound to L streams: upload (PCIe H2D), kernels and download
        # (PCIe D2H) of consecutive steps overlap; every step still moves all its bytes.  Three stages need three
        # lanes to keep the slowest one (a PCIe direction) busy; fewer if the workspaces would not fit.
        L = max(1, min(args.e2e_lanes, int(150e9 // e.workspace.numel())))
        sides = [torch.cuda.Stream() for _ in range(L - 1)]
        lanes = [(e, outs)]
        for sd in sides:
            with torch.cuda.stream(sd):
                h = binding.Echo(*e.n, GAMMA, CFL, uct=uct, ho=ho, rec=rec, rk=rk)
            lanes.append((h, [torch.empty(e.shape, dtype=torch.float64).pin_memory() for _ in range(8)]))
        for h, o in lanes:
            h.set_primitives_host(*host); h.step(1); h.get_primitives_host(o)
        barrier()
        ev0.record()
        for i in range(Ke):
            h, o = lanes[i % L]
            if i >= L:
                h.synchronize()                      # step i-L of this lane is back before its buffers are reused
            h.set_primitives_host(*host)
            h.step(1)
            h.get_primitives_host(o, sync=False)
        for h, _ in lanes:
            h.synchronize()
        for sd in sides:
            torch.cuda.current_stream().wait_stream(sd)
        ev1.record()
        barrier()
        e2e_value, _ = whole_job_rate(N, Ke, ev0.elapsed_time(ev1), "cuda", world)
        e2e_how = "%d handles on %d streams: uploads, kernels and downloads of consecutive steps overlap" % (L, L)
        for _, o in lanes[1:]:
            assert torch.equal(outs[0], o[0])
        del lanes[1:]
    # sanity of what came back: one step of the wave stays within truncation error of the input
    assert abs(float(outs[0].mean()) - 1.0) < (1e-6 if args.workload == "cpa" else 1e-2)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (live CUDA-event durations of this run)
    peaks, peak_kind = measured_peaks()
    hbm_peak = float(peaks["hbm_gbs"])
    fp64_burst, fp64_sust = binding.fp64_peak(20)
    kernels = {}
    for name, (tot, cnt) in ktimes.items():
        if cnt and name in ALGO:
            avg = tot / cnt
            kernels[name] = {"ms_avg": avg, "launches": cnt, "share": tot / ms_kpass,
                             "tflops": ALGO[name]["flop"] * N / (avg * 1e-3) * 1e-12,
                             "gbs": 8 * ALGO[name]["dbl"] * N / (avg * 1e-3) * 1e-9}
        elif cnt:
            kernels[name] = {"ms_avg": tot / cnt, "launches": cnt, "share": tot / ms_kpass}
    dom = max((k for k in kernels if k in ALGO), key=lambda k: kernels[k]["share"] * 1.0)
    kd = kernels[dom]
    t_alu = ALGO[dom]["flop"] / (fp64_sust * 1e12)
    t_hbm = 8 * ALGO[dom]["dbl"] / (hbm_peak * 1e9)
    if t_alu >= t_hbm:
        roof = {"bound": "alu", "achieved": kd["tflops"], "peak": fp64_sust, "unit": "TFLOP/s",
                "frac": kd["tflops"] / fp64_sust}
    else:
        roof = {"bound": "hbm", "achieved": kd["gbs"], "peak": hbm_peak, "unit": "GB/s", "frac": kd["gbs"] / hbm_peak}
    traffic, traffic_source = measured_traffic(dom, N, args)
    roof.update(kernel=dom, traffic=traffic, traffic_source=traffic_source, peak_source=("FP64 DFMA micro-benchmark run by this bench "
                "(sustained; burst %.1f)" % fp64_burst) if roof["bound"] == "alu" else "MEASURED_PEAKS.json (%s)" % peak_kind,
                algorithmic_flop_per_cell=ALGO[dom]["flop"], algorithmic_bytes_per_cell=8 * ALGO[dom]["dbl"],
                ms_per_launch=kd["ms_avg"], cells_per_launch=N)
    step_bound = min(fp64_sust * 1e12 / FLOP_PER_CELL_UPDATE, hbm_peak * 1e9 / BYTES_PER_CELL_UPDATE)
    per_gpu = value / world

    cpu = None
    if world == 1 and not args.no_cpu:
        rate, dt = oracle_rate(args.cpu_n, args.cpu_steps, 0, args.direction)
        cpu = {"value": rate, "unit": "cell-updates/s", "cores": 1, "kind": "oracle", "host_cores": os.cpu_count(),
               "sample": "%d^3 box of the same CPA wave, %d RK3 steps, %.1f s, single thread" % (args.cpu_n, args.cpu_steps, dt)}

    vs_baseline, baseline_note = None, None
    if args.workload == "cpa" and n == 512 and args.direction == "diag" and not decomposed and args.scheme in PAPER_512_PER_NODE:
        vs_baseline = value / PAPER_512_PER_NODE[args.scheme]
        baseline_note = ("paper: %.3g cell-updates/s on one LEONARDO node (4 x A100 64 GB) for this workload and scheme "
                         "(BASELINE.md section 1); this run: %d x B200" % (PAPER_512_PER_NODE[args.scheme], world))
    line = {"metric": "fp64_cell_updates_per_sec", "value": value, "unit": "cell-updates/s", "n_gpus": world,
            "steps": K, "warmup": W, "ms_per_step": ms_max / K, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": vs_baseline, "dtype": "f64", "data": "synthetic",
            "config": {"workload": {"turb2d": "turbulence_2.5d_%d^2" % n, "turb3d": "alfvenic_turbulence_%d^3" % n}.get(
                           args.workload, "cpa_wave_%s_%d^3" % (args.direction, n)),
                       "grid": list(e.n), "gamma": GAMMA, "cfl": CFL,
                       "scheme": {"uct-ho": "MP5+HLL+UCT+DER6/INT6+SSPRK3 (UCT=HO=YES)",
                                  "uct-lo": "MP5+HLL+UCT+SSPRK3, second-order INT/DER (UCT=YES, HO=NO)",
                                  "cc-ho": "MP5+HLL+DER6+SSPRK3, cell-centred B (UCT=NO, HO=YES)",
                                  "cc-lo": "MP5+HLL+SSPRK3, cell-centred B (UCT=HO=NO)",
                                  "uct-lo2": "linear(MC)+HLL+UCT+SSPRK2, second-order INT/DER (UCT=YES, HO=NO)",
                                  "cc-lo2": "linear(MC)+HLL+SSPRK2, cell-centred B (UCT=HO=NO)"}[args.scheme], "cells": N,
                       "parallelism": parallelism, "baseline_note": baseline_note,
                       "cache": "working set %.1f GB per GPU, far larger than the 126 MB L2" % (44 * 8 * N / 1e9)},
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": "cell-updates/s", "steps": Ke, "serial_value": e2e_serial,
                    "pipelining": e2e_how,
                    "h2d_bytes_per_step": 8 * 8 * e.N, "d2h_bytes_per_step": 8 * 8 * e.N,
                    "what": "per step: echo_set_primitives_host (8 fields, pinned) + echo_step(1) + echo_get_primitives_host (8 fields)"},
            "gpu_launches": nlaunch,
            "roofline": roof,
            "step_roofline": {"bound_cell_updates_per_s": step_bound, "frac": per_gpu / step_bound,
                              "flop_per_cell_update": FLOP_PER_CELL_UPDATE, "bytes_per_cell_update": BYTES_PER_CELL_UPDATE,
                              "fp64_tflops_peak_measured": fp64_sust, "hbm_gbs_peak": hbm_peak,
                              "achieved_tflops": per_gpu * FLOP_PER_CELL_UPDATE * 1e-12,
                              "achieved_gbs": per_gpu * BYTES_PER_CELL_UPDATE * 1e-9},
            "kernels": kernels,
            "kernels_note": "per-kernel times from a SECOND pass of %d steps with a CUDA-event pair around every launch "
                            "(%.3f ms/step in that pass); value / ms_per_step come from the first pass, timers off" % (Kk, ms_kpass / Kk),
            "state": {"t": d["t"], "max_div_b": d["max_div_b"], "c2p_mean_iters": d["c2p_mean_iters"],
                      "c2p_max_iters": d["c2p_max_iters"], "c2p_failures": d["c2p_failures"], "max_W": d["max_W"],
                      "min_rho": d["min_rho"], "min_p": d["min_p"]},
            "cpu_baseline": cpu}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def kernel_source_hash():
    from paper_2401_03008_b200.ncu_summary import kernel_source_hash as h
    return h()


def measured_traffic(kernel_class, cells, args):
    """roofline.traffic = dram__bytes_read.sum + dram__bytes_write.sum of one launch, from the committed ncu --set full
    capture (profiles/r2_traffic.json, written by `python -m paper_2401_03008_b200.ncu_summary`), scaled from the
    capture's cell count to this launch.  None, with the reason, when the capture is of other kernel sources, of
    another scheme or absent: a stale number is worse than none."""
    path = os.path.join(ROOT, "profiles", "r2_traffic.json")
    if not os.path.exists(path):
        return None, "no ncu capture committed (profiles/r2_traffic.json)"
    with open(path) as f:
        t = json.load(f)
    if args.scheme != t.get("scheme", "uct-ho") or args.workload != "cpa":
        return None, "the committed capture (profiles/r2_traffic.json) is of scheme %s on the cpa workload" % t.get("scheme")
    if t.get("source_sha256") != kernel_source_hash():
        return None, "profiles/r2_traffic.json was captured on other kernel sources (sha256 %s...)" % str(t.get("source_sha256"))[:12]
    k = t.get("kernels", {}).get(kernel_class)
    if not k:
        return None, "kernel class %s is not in profiles/r2_traffic.json" % kernel_class
    return k["dram_bytes_per_cell"] * cells, ("ncu dram__bytes_read.sum + dram__bytes_write.sum per cell of %s (%s, %d^3) x cells of "
                                              "this launch; %s" % (k["kernel"], t.get("report"), t.get("n", 0), t.get("md")))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="echo", choices=["echo", "reference"])
    ap.add_argument("--n", type=int, default=256, help="box size n^3 (BASELINE.json configs[2]: 256)")
    ap.add_argument("--direction", default="diag", choices=["diag", "x"])
    ap.add_argument("--e2e-steps", type=int, default=20)
    ap.add_argument("--kernel-steps", type=int, default=10, help="steps of the second, per-kernel-timed pass")
    ap.add_argument("--e2e-lanes", type=int, default=3, help="handles/streams of the pipelined end-to-end measurement")
    ap.add_argument("--cpu-n", type=int, default=64)
    ap.add_argument("--cpu-steps", type=int, default=6)
    ap.add_argument("--ref-n", type=int, default=48)
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--workload", default="cpa", choices=["cpa", "turb2d", "turb3d"],
                    help="cpa: BASELINE.json configs (default); turb2d: the paper's 2.5-D turbulence on n x n x 1")
    ap.add_argument("--scheme", default="uct-ho", choices=sorted(SCHEMES),
                    help="the paper's switches (P:L124, L138): uct-ho = UCT=HO=YES (default, the headline), "
                         "uct-lo = HO=NO, cc-ho / cc-lo = UCT=NO with the cell-centred B, *-lo2 = limited linear "
                         "REC + SSP-RK2 (P:L304) (row f2)")
    ap.add_argument("--decompose", action="store_true",
                    help="N > 1: one decomposed box (n^3 cells per rank, halo exchange) instead of N replicas")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()

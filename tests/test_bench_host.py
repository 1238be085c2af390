"""CPU checks of bench.py's host logic: the N>1 aggregation (max over ranks, whole-job value) with a
world_size-2 gloo group, the reference arm under a 2-rank launch (rank 0 alone prints), the clock sampler
without nvidia-smi, and the bytes/flops bookkeeping."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
import torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
ms_local = 10.0 if rank == 0 else 25.0          # rank 1 is the slow one
rate, ms = bench.whole_job_rate(1000, 5, ms_local, "cpu", world)
dist.barrier()
if rank == 0:
    print(json.dumps({"rate": rate, "ms": ms, "world": world}))
dist.destroy_process_group()
"""


def _torchrun(args, timeout=300):
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", "29731"] + args
    return subprocess.run(cmd, capture_output=True, text=True, timeout=timeout, env=env, cwd=ROOT)


def test_whole_job_rate_is_sum_of_cells_over_slowest_rank(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER % ROOT)
    r = _torchrun([str(script)])
    assert r.returncode == 0, r.stderr[-2000:]
    line = [l for l in r.stdout.splitlines() if l.startswith("{")][-1]
    out = json.loads(line)
    assert out["world"] == 2 and out["ms"] == 25.0
    assert out["rate"] == 2 * 1000 * 5 / 25e-3


def test_reference_arm_two_ranks_prints_one_line():
    r = _torchrun([os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                   "--warmup", "0", "--ref-n", "12"])
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["cpu_baseline"]["kind"] == "oracle" and d["value"] > 0
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["unit"] == "cell-updates/s"


def test_clock_sampler_and_bookkeeping():
    import bench
    s = bench.ClockSampler(0)
    s.start()
    out = s.stop()                       # no GPU here: empty but well-formed
    assert set(out) >= {"sm_mhz", "sm_max_mhz", "reasons"}
    assert bench.max_over_ranks(3.5, "cpu", 1) == 3.5
    # per-stage doubles of the kernels as built sum to the documented 2784 B per cell-update
    assert abs(bench.BYTES_PER_CELL_UPDATE - 2784.0) < 1e-9
    assert 8300 < bench.FLOP_PER_CELL_UPDATE < 8700


def test_traffic_comes_from_the_committed_capture_or_is_null(tmp_path, monkeypatch):
    """roofline.traffic is read from profiles/r2_traffic.json and only trusted when the capture ran on the CUDA sources
    of this tree (sha256 stamp), on the same scheme and workload; otherwise null with the reason."""
    import argparse
    import bench
    from paper_2401_03008_b200 import ncu_summary as ns
    assert ns.kernel_class("void k_flux<1, 128, 0, 1, 1, 5>(Grid, Stage, int, double, double, Ctrl *, int, FluxUpd)") == "k_flux_y"
    assert ns.kernel_class("void k_uct3<0, 8>(Grid, Stage, int, UctMaps)") == "k_uct"
    assert ns.kernel_class("k_bupd(Grid, const double *, const double *, const double *, Update, const Ctrl *, int)") == "k_update"
    assert ns.kernel_class("void k_prim_march<1>(Grid, Stage, double, Ctrl *, PrimUpd, int, const int *)") == "k_prim"
    assert ns.kernel_class("k_set_dt(Ctrl *, double)") is None
    h = ns.kernel_source_hash()
    assert len(h) == 64 and h == bench.kernel_source_hash()
    args = argparse.Namespace(scheme="uct-ho", workload="cpa")
    (tmp_path / "profiles").mkdir()
    monkeypatch.setattr(bench, "ROOT", str(tmp_path))
    t, why = bench.measured_traffic("k_uct", 1000, args)
    assert t is None and "no ncu capture" in why
    cap = {"source_sha256": h, "scheme": "uct-ho", "n": 256, "report": "x.ncu-rep", "md": "profiles/x.md",
           "kernels": {"k_uct": {"kernel": "k_uct3", "dram_bytes_per_cell": 164.0}}}
    (tmp_path / "profiles" / "r2_traffic.json").write_text(json.dumps(cap))
    t, why = bench.measured_traffic("k_uct", 1000, args)
    assert t == 164.0 * 1000 and "dram__bytes" in why
    assert bench.measured_traffic("k_prim", 1000, args)[0] is None
    assert bench.measured_traffic("k_uct", 1000, argparse.Namespace(scheme="cc-lo", workload="cpa"))[0] is None
    cap["source_sha256"] = "0" * 64                                   # captured on other kernels: not trusted
    (tmp_path / "profiles" / "r2_traffic.json").write_text(json.dumps(cap))
    t, why = bench.measured_traffic("k_uct", 1000, args)
    assert t is None and "other kernel sources" in why

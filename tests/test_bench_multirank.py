"""The N > 1 path of bench.py on CPU (gloo, world size 2): the path is "replicas only", so the
only cross-rank logic is the max-over-ranks clock and the whole-job aggregate; the reference arm runs on rank 0 only."""
import json
import os
import subprocess
import sys

import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    mine = 10.0 + 5.0 * rank                      # rank 1 is the slow one
    slowest = bench.max_over_ranks(mine, world, "cpu")
    value = bench.job_throughput(1000, 3, world, slowest)
    out.put((rank, slowest, value))
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_and_job_aggregate_gloo():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, slowest, value in got:
        assert slowest == 15.0                    # both ranks agree on the slowest rank's time
        assert value == pytest.approx(2 * 1000 * 4 * 3 / 15.0e-3 / 1e9)


def test_single_rank_needs_no_process_group():
    import bench
    assert bench.max_over_ranks(7.5, 1, "cpu") == 7.5
    assert bench.job_throughput(1000, 2, 1, 4.0) == pytest.approx(1000 * 4 * 2 / 4.0e-3 / 1e9)


def test_reference_arm_runs_on_rank_zero_only():
    """`bench.py --impl reference` under a 2-rank launch: rank 0 prints the one JSON line, rank 1 exits 0 silently."""
    port = 31500 + os.getpid() % 2000
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(port), os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
           "--config", "1", "--steps", "1", "--warmup", "0"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["cpu_baseline"]["kind"] == "oracle" and d["gpu_launches"] == 0
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["value"] > 0 and d["unit"] == "GDOF-stage/s"


def test_roofline_arithmetic_of_the_bench_line():
    """rooflines(): algorithmic flops / bytes per launch over the measured kernel time against the two peaks; the
    binding roof is the one with the larger fraction, the other goes to other_roof (SURVEY 8(d) figures)."""
    import bench
    assert bench.algorithmic_flop_per_dof_stage(3, 35, 15) == 380.0          # 2*3*35 + 2*4*15 + 50
    assert bench.algorithmic_flop_per_dof_stage(2, 15, 5) == 140.0
    assert bench.algorithmic_flop_per_dof_stage(3, 20, 10) == 250.0
    dof = 196608 * 35 * 10
    m = dict(dim=3, Np=35, Nfp=15, dof=dof, kern_ms=1.186, nprof=80, share=0.976, graph_timed=False)
    r = bench.rooflines(m, 4, 0)
    assert r["bound"] == "alu" and r["other_roof"]["bound"] == "hbm"
    assert r["achieved"] == pytest.approx(dof * 380.0 / 1.186e-3 / 1e12)
    assert r["frac"] == pytest.approx(r["achieved"] / (148 * 64 * 2 * 1.965e9 / 1e12))
    assert r["other_roof"]["achieved"] == pytest.approx(dof * 38.0 / 1.186e-3 / 1e9)
    assert r["algorithmic_bytes_per_launch"] == pytest.approx(dof * 38.0)
    # the committed ncu traffic figure belongs to the sources it was captured from: reported only while they match
    if bench.kernel_sources_sha256() == bench.NCU_CAPTURE_SHA256:
        assert r["traffic"] == pytest.approx(bench.NCU_DRAM_BYTES_PER_LAUNCH[4][0]) and "matches" in r["traffic_source"]
    else:
        assert r["traffic"] is None and r["traffic_source"].startswith("stale")
    saved = bench.NCU_CAPTURE_SHA256
    try:
        bench.NCU_CAPTURE_SHA256 = bench.kernel_sources_sha256()
        assert bench.rooflines(m, 4, 0)["traffic"] == pytest.approx(bench.NCU_DRAM_BYTES_PER_LAUNCH[4][0])
        assert bench.rooflines(m, 4, 0, default_modes=False)["traffic"] is None   # --relax cubature, --coords rk, ...
        assert bench.rooflines(m, 1, 0)["traffic"] is None                        # no capture for config 1
        bench.NCU_CAPTURE_SHA256 = "0" * 16
        assert bench.rooflines(m, 4, 0)["traffic"] is None
    finally:
        bench.NCU_CAPTURE_SHA256 = saved
    m2 = dict(dim=2, Np=15, Nfp=5, dof=60000 * 15 * 6, kern_ms=0.0699, nprof=60, share=None, graph_timed=True)
    r2 = bench.rooflines(m2, 3, 0)
    assert r2["bound"] == "hbm" and 0.4 < r2["frac"] < 0.5 and r2["other_roof"]["bound"] == "alu"
    assert bench.rooflines(m2, 3, 1)["traffic"] is None                      # committed ncu traffic is the default kernel's


def test_oracle_timing_helper_single_core():
    import bench
    v, cores, desc, ms = bench.time_oracle(1, 1, 0, cores=1)
    assert cores == 1 and v > 0 and ms > 0 and "K=128" in desc and desc.startswith("SAMPLE (K=128), not the config")

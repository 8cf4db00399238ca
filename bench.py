#!/usr/bin/env python
"""Throughput of the fused ALE Galerkin-Boltzmann SARK4 step on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--impl reference]

A "step" is one SARK4 time step = 4 stages, each stage = vertex motion + geometric factors + fused volume /
relaxation / surface / SARK-update kernel (all rows of SURVEY.md 8(a)) over the whole synthetic mesh.
Metric: GDOF-stage updates/s = K_elements * Np * Nfields * 4 * steps / time.  One JSON line on stdout (rank 0).

  value        device-resident state, CUDA-event timing, max over ranks
  e2e          the same steps through alegb_step_host: pinned host state -> device -> step -> host, every step
  roofline     the fused stage kernel: algorithmic flops (or bytes) per launch / its mean duration, measured live
               with CUDA events bracketing every launch on its stream (alegb_profile_enable)
  cpu_baseline the oracle (oracle/, numpy, as it stands) on a bounded sample of the same workload
  --impl reference   times the oracle alone (rank 0 only)

Multi-GPU: the path is specified for one GPU (north_star: no sharding, no collectives) -> N independent replicas,
one process per GPU, value = N * per-replica work / max time ("weak").
"""
import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "GDOF-stage updates/s (nodes x fields x RK stages)"
UNIT = "GDOF-stage/s"
# fp64 pipe peak of one B200: 148 SMs x 64 fp64 FMA lanes per SM and clock x 2 flop x 1.965 GHz (the
# DFMA/DMMA microbenchmark profiles/r1_fp64_peak.md measured 37.1 TFLOP/s, both instruction kinds share the pipe)
FP64_PEAK_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12
HBM_FALLBACK_GBS = 6650.0
ALGO_BYTES_PER_DOF_STAGE = 38.0          # 152 B per DOF-step
POINTWISE_FLOP_PER_DOF_STAGE = 50.0
# dram__bytes_read.sum + dram__bytes_write.sum of the stage kernel per launch from the committed `ncu --set full`
# capture (mean over the four stages of a step: 1.79 / 2.93 / 3.48 / 1.82 GB), profiles/r1_v8_pipe_stage_kernel.md
NCU_DRAM_BYTES_PER_LAUNCH = {4: 2.505e9}


def algorithmic_flop_per_dof_stage(dim, Np, Nfp):
    """dense D and LIFT mat-vecs 2*d*Np + 2*Nfaces*Nfp, plus ~50 of point-wise work."""
    return 2.0 * dim * Np + 2.0 * (dim + 1) * Nfp + POINTWISE_FLOP_PER_DOF_STAGE


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            d = json.load(open(p))
            return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return HBM_FALLBACK_GBS, "fallback (B200_PROFILING.md)"


def make_config(index, lam, full=True, sample=False):
    from workloads import configs
    if sample:   # bounded sample of the same recipe for the CPU oracle
        small = {1: dict(n=8), 2: dict(n=16), 3: dict(ntheta=48, nr=16), 4: dict(n=8), 5: dict(nx=16, ny=8, nz=8)}[index]
        return configs.BY_INDEX[index](lam, **small)
    return configs.BY_INDEX[index](lam)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md clocks line)."""
    FIELDS = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
              "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.tmp = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.proc = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(gpu_index), "--query-gpu=" + self.FIELDS,
                                          "--format=csv,noheader,nounits", "-lms", "20"], stdout=self.tmp,
                                         stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is not None:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except Exception:
                self.proc.kill()
        try:
            self.tmp.flush()
            rows = [l.strip().split(",") for l in open(self.tmp.name) if l.strip()]
            sm = [float(r[0]) for r in rows if len(r) >= 6]
            if sm:
                out["sm_mhz"] = float(np.median(sm))
                out["sm_max_mhz"] = float(rows[0][1])
                out["samples"] = len(sm)
                names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
                for i, n in enumerate(names):
                    if any(r[2 + i].strip().lower().startswith("active") for r in rows if len(r) >= 6):
                        out["reasons"].append(n)
        except Exception:
            pass
        finally:
            try:
                os.unlink(self.tmp.name)
            except Exception:
                pass
        return out


def time_oracle(index, steps, warmup):
    """The oracle as it stands on a bounded sample of workload `index`; returns (GDOF-stage/s, cores, description)."""
    from oracle import sark
    from oracle.operators import ReferenceElement
    from oracle.rhs import Problem
    from workloads import configs
    dim, N = {1: (2, 3), 2: (2, 4), 3: (2, 4), 4: (3, 4), 5: (3, 3)}[index]
    ref = ReferenceElement(dim, N)
    cfg = make_config(index, ref.lam, sample=True)
    P = Problem(dim, N, cfg["X0"], cfg["EToV"], cfg.get("vertex_equiv"), cfg.get("EToB"), cfg.get("pml_sigma"),
                RT=cfg["RT"], tau=cfg["tau"], q_inf=cfg.get("q_inf"), motion_kind=cfg["motion_kind"],
                motion_params=cfg["motion_params"], ref=ref)
    q, aux, dt = cfg["q0"], None, cfg["dt"]
    for n in range(warmup):
        stages, aux = sark.step_debug(P, q, n * dt, dt, aux)
        q = stages[-1]
    w0, c0 = time.perf_counter(), time.process_time()
    for n in range(steps):
        stages, aux = sark.step_debug(P, q, (warmup + n) * dt, dt, aux)
        q = stages[-1]
    wall, cpu = time.perf_counter() - w0, time.process_time() - c0
    dof = cfg["K"] * cfg["Np"] * cfg["Nf"]
    cores = max(1, int(round(cpu / max(wall, 1e-9))))
    desc = "%s recipe shrunk to K=%d elements (N=%d, %d fields), %d SARK4 steps (%d stages)" % (
        cfg["name"], cfg["K"], N, cfg["Nf"], steps, 4 * steps)
    return dof * 4 * steps / wall / 1e9, cores, desc, wall / max(steps, 1) * 1e3, cfg


def max_over_ranks(x, world, device):
    """The slowest rank's time: all-reduce MAX over the job (NCCL on the GPUs, gloo in the CPU tests)."""
    if world <= 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_throughput(dof_per_rank, steps, world, elapsed_ms):
    """Whole-job GDOF-stage/s of `world` independent replicas (weak scaling): all ranks' units / the slowest rank."""
    return world * dof_per_rank * 4 * steps / (elapsed_ms * 1e-3) / 1e9


def run_reference(args, rank):
    if rank != 0:
        return
    value, cores, desc, ms, cfg = time_oracle(args.config, args.steps, args.warmup)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(args.config), "sample": desc},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def workload_name(index):
    return {1: "configs[0] 2D free-stream: periodic unit square, 128 triangles, N=3, 6 fields, SINES_PRODUCT motion",
            2: "configs[1] 2D moving Taylor-Green: periodic [0,2pi]^2, 8192 triangles, N=4, 6 fields",
            3: "configs[2] 2D plunging NACA0012 O-grid: 60000 triangles, N=4, wall + far field + PML ring",
            4: "configs[3] 3D deforming periodic box: 32^3 hexes x 6 = 196608 tetrahedra, N=4 (Np=35), 10 fields, "
               "SINES_CROSS motion amplitude 0.03",
            5: "configs[4] 3D carangiform swimmer stand-in: ~1.5M tetrahedra, N=3, wall + far field + PML shell"}[index]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4, choices=[1, 2, 3, 4, 5],
                    help="BASELINE.json workload (1-based); 4 = the 3D N=4 throughput configuration")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--kernel", type=int, default=0, choices=[0, 1, 2],
                    help="alegb_set_kernel: 0 auto, 1 generic DFMA, 2 pipelined DMMA")
    ap.add_argument("--relax", default="collocation", choices=["collocation", "cubature"],
                    help="nonlinear relaxation: collocated (default, DESIGN.md R8) or cubature-projected (NEXT-1)")
    ap.add_argument("--coords", default="closed", choices=["closed", "rk"],
                    help="vertex positions: closed-form law (default, R9) or advanced by the solver's RK4 (NEXT-2)")
    ap.add_argument("--no-overlap", action="store_true", help="a1/a2 of the next stage in order instead of beside the stage kernel")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "b200" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, rank)
        return

    import torch
    import torch.distributed as dist
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the library has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    from paper_2607_00199_b200 import binding as B

    dim, N = {1: (2, 3), 2: (2, 4), 3: (2, 4), 4: (3, 4), 5: (3, 3)}[args.config]
    probe = B.Context(dim, N, -1)
    lam = probe.alegb_get_reference()["lam"]     # node coordinates for the initial state (input generation only)
    probe.close()
    cfg = make_config(args.config, lam)
    ctx = B.context_from_config(cfg, local_rank)
    ctx.alegb_set_kernel(args.kernel)
    if args.no_overlap:
        ctx.alegb_set_geometry_overlap(False)
    if args.relax == "cubature":
        ctx.alegb_set_relaxation(B.RELAX_CUBATURE)
    if args.coords == "rk":
        ctx.alegb_set_coordinate_mode(B.COORDS_RK, 0.0)
    K, Np, Nf, Nfp = cfg["K"], cfg["Np"], cfg["Nf"], ctx.Nfp
    dof = K * Np * Nf
    dt = cfg["dt"]
    q = torch.from_numpy(cfg["q0"]).cuda()
    state_bytes = q.numel() * 8

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing
    ctx.alegb_step(q, 0.0, dt, args.warmup)
    barrier()
    sampler = ClockSampler(local_rank) if rank == 0 else None
    # Large states (the throughput configuration): the library brackets every stage-kernel launch of the timed region
    # with events (direct launches).  Small, L2-resident states are launch-bound: the timed region replays the
    # captured step graph (alegb_set_graph) and the stage kernel is timed in a second, direct pass of the same steps.
    graph_timed = state_bytes < 200e6
    ctx.alegb_profile_enable(not graph_timed)
    n0 = ctx.alegb_launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    ctx.alegb_step(q, args.warmup * dt, dt, args.steps)
    e1.record()
    barrier()
    elapsed_ms = e0.elapsed_time(e1)
    launches = ctx.alegb_launch_count() - n0
    if graph_timed:
        ctx.alegb_profile_enable(True)
        ctx.alegb_step(q.clone(), args.warmup * dt, dt, args.steps)
    nprof, prof_ms = ctx.alegb_profile_read()
    ctx.alegb_profile_enable(False)
    clocks = sampler.stop() if sampler else None
    elapsed_ms = max_over_ranks(elapsed_ms, world, "cuda")
    finite = bool(torch.isfinite(q).all().item())
    value = job_throughput(dof, args.steps, world, elapsed_ms)

    # ---- end to end through the host-buffer entry point (pinned host state, H2D + step + D2H every step)
    e2e = None
    if not args.no_e2e:
        hq = torch.from_numpy(cfg["q0"]).pin_memory()
        ctx.alegb_step_host(hq, 0.0, dt, 1)
        barrier()
        nsteps_e2e = max(3, min(args.steps, 10))
        t0 = time.perf_counter()
        for n in range(nsteps_e2e):
            ctx.alegb_step_host(hq, (1 + n) * dt, dt, 1)
        torch.cuda.synchronize()
        el = time.perf_counter() - t0
        el = max_over_ranks(el, world, "cuda")
        e2e = {"value": job_throughput(dof, nsteps_e2e, world, el * 1e3), "unit": UNIT, "h2d_bytes_per_step": state_bytes,
               "d2h_bytes_per_step": state_bytes, "steps": nsteps_e2e, "api": "alegb_step_host (pinned host buffer)"}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (the fused stage kernel)
    hbm_peak, hbm_src = measured_peaks()
    kern_ms = prof_ms / max(nprof, 1)
    flop_per_dof = algorithmic_flop_per_dof_stage(dim, Np, Nfp)
    tf = dof * flop_per_dof / (kern_ms * 1e-3) / 1e12
    gbs = dof * ALGO_BYTES_PER_DOF_STAGE / (kern_ms * 1e-3) / 1e9
    alu = {"bound": "alu", "achieved": tf, "peak": FP64_PEAK_TFLOPS, "unit": "TFLOP/s", "frac": tf / FP64_PEAK_TFLOPS,
           "traffic": None, "peak_source": "derived: 148 SM x 64 fp64 FMA/clk x 2 x 1.965 GHz (DESIGN.md)",
           "algorithmic_flop_per_dof_stage": flop_per_dof}
    hbm = {"bound": "hbm", "achieved": gbs, "peak": hbm_peak, "unit": "GB/s", "frac": gbs / hbm_peak, "traffic": None,
           "peak_source": hbm_src, "algorithmic_bytes_per_dof_stage": ALGO_BYTES_PER_DOF_STAGE}
    roofline, other = (alu, hbm) if alu["frac"] >= hbm["frac"] else (hbm, alu)
    roofline = dict(roofline)
    if args.kernel == 0:
        roofline["traffic"] = NCU_DRAM_BYTES_PER_LAUNCH.get(args.config)
        roofline["traffic_unit"] = "bytes per launch (ncu dram read+write, profiles/r1_v8_pipe_stage_kernel.md)"
        roofline["algorithmic_bytes_per_launch"] = dof * ALGO_BYTES_PER_DOF_STAGE
    roofline.update({"kernel": "alegb stage kernel (fused volume+relaxation+surface+SARK update)",
                     "kernel_ms": kern_ms, "kernel_launches_timed": nprof,
                     "kernel_share_of_step": prof_ms / elapsed_ms if elapsed_ms > 0 else None,
                     "kernel_timed_in": "second pass, direct launches (timed region replays the step graph)"
                     if graph_timed else "timed region",
                     "other_roof": other})

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": elapsed_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(args.config), "K": K, "N": N, "Np": Np, "Nfields": Nf, "dof": dof,
                       "dt": dt, "parallelism": "replicas x%d (north_star: one GPU, no sharding)" % world,
                       "l2": "state arrays are %.0f MB each (> 126 MB L2), no flush needed" % (state_bytes / 1e6)
                       if state_bytes > 200e6 else "state is L2-resident (%.1f MB); launch-latency bound" % (state_bytes / 1e6),
                       "state_finite": finite, "kernel": args.kernel, "relax": args.relax, "coords": args.coords,
                       "launch": "one CUDA graph per step" if graph_timed and args.steps >= 2 else "direct launches"},
            "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks, "roofline": roofline}

    if not args.no_cpu_baseline:
        v, cores, desc, _, _ = time_oracle(args.config, 6 if args.config in (4, 5) else 20, 1)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc,
                                "host_cores_available": os.cpu_count()}
    print(json.dumps(line), flush=True)
    ctx.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

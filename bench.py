#!/usr/bin/env python
"""Throughput of the fused ALE Galerkin-Boltzmann SARK4 step on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--impl reference]

A "step" is one SARK4 time step = 4 stages, each stage = vertex motion + geometric factors + fused volume /
relaxation / surface / SARK-update kernel (all rows of SURVEY.md 8(a)) over the whole synthetic mesh.
Metric: GDOF-stage updates/s = K_elements * Np * Nfields * 4 * steps / time.  One JSON line on stdout (rank 0).

  value        device-resident state, CUDA-event timing of exactly --steps steps, max over ranks; the timed region is
               repeated --repeats times (default 5) and the MEDIAN is reported (min / max beside it)
  e2e          the same steps through alegb_step_host: pinned host state -> device -> step -> host, every step
               (plus a second figure with --steps steps per host round trip)
  roofline     the fused stage kernel: algorithmic flops (or bytes) per launch / its mean duration, measured live
               with CUDA events bracketing every launch on its stream (alegb_profile_enable)
  clocks       SM clock and throttle reasons polled through NVML in this process DURING the timed regions
  per_config   the other BASELINE.json workloads (1, 2, 3, 5): value, ms per step, stage-kernel time, both roofline
               fractions -- a driver-side record of every number DESIGN.md quotes
  modes        the optional modes on the same box: config 4 with cubature-projected relaxation and with RK-integrated
               coordinates, configs 3 / 5 with the absorbing layer fused into the stage kernel or separate
  cpu_baseline the oracle (oracle/, numpy, as it stands) on a bounded sample of the same workload, one independent
               replica per host core
  --impl reference   times the oracle alone (rank 0 only)

Multi-GPU: the path is specified for one GPU (north_star: no sharding, no collectives) -> N independent replicas,
one process per GPU, value = N * per-replica work / max time ("weak").
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
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "GDOF-stage updates/s (nodes x fields x RK stages)"
UNIT = "GDOF-stage/s"
# fp64 pipe peak of one B200: 148 SMs x 64 fp64 FMA lanes per SM and clock x 2 flop x 1.965 GHz.  MEASURED_PEAKS.json
# holds no fp64 figure and the profiling guide no fp64 nominal, so this is DERIVED from the guide's unit count and
# clock; the DFMA/DMMA microbenchmark of round 1 (profiles/r1_fp64_peak.md) measured 37.1 TFLOP/s with DMMA, and both
# instruction kinds share the datapath.
FP64_PEAK_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12
HBM_FALLBACK_GBS = 6650.0
ALGO_BYTES_PER_DOF_STAGE = 38.0          # 152 B per DOF-step
POINTWISE_FLOP_PER_DOF_STAGE = 50.0
# dram__bytes_read.sum + dram__bytes_write.sum of the stage kernel per launch from committed `ncu --set full` captures
# (mean over the stages of a step); configurations without a capture report no traffic figure.
# The figures belong to the kernel they were captured from: NCU_CAPTURE_SHA256 is the sha256 over the stage kernel's
# sources (kernel_sources_sha256) at the time of the capture.  With any other sources, or in a mode other than the
# captured one (default kernel, collocated relaxation, closed-form coordinates, default layer fusion), the line
# carries "traffic": null and says why in "traffic_source".
NCU_CAPTURE_SHA256 = "13631ba549af3491"   # sources of the round-3 captures (profiles/r3_final.md)
NCU_DRAM_BYTES_PER_LAUNCH = {
    4: (2.506e9, "profiles/r3_final.md"),
    # config 5: both stage launches of a stage (quads outside + inside the absorbing layer); includes a8's auxiliary
    # arrays (up to 5 arrays x 3 directions x 8 B per layer DOF), which the 38 B per DOF-stage do not count
    5: (21.88e9, "profiles/r3_final.md"),
    3: (160.9e6, "profiles/r3_final.md"),
    2: (17.45e6, "profiles/r3_final.md")}
DIM_N = {1: (2, 3), 2: (2, 4), 3: (2, 4), 4: (3, 4), 5: (3, 3)}


def kernel_sources_sha256():
    """sha256 (first 16 hex digits) over the sources the stage kernels are compiled from."""
    import hashlib
    h = hashlib.sha256()
    for f in ("stage_pipe.cu", "device_common.cuh"):
        with open(os.path.join(ROOT, "paper_2607_00199_b200", "csrc", f), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


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


def make_config(index, lam, sample=False):
    from workloads import configs
    if sample:   # bounded sample of the same recipe for the CPU oracle
        small = {1: dict(n=8), 2: dict(n=16), 3: dict(ntheta=48, nr=16), 4: dict(n=8), 5: dict(nx=16, ny=8, nz=8)}[index]
        return configs.BY_INDEX[index](lam, **small)
    return configs.BY_INDEX[index](lam)


class ClockSampler:
    """SM clock and clock-event (throttle) reasons of one GPU, polled through NVML from a thread of this process
    every few milliseconds; only samples taken between begin() and end() -- the timed regions -- are kept
    (B200_PROFILING.md: clocks DURING the timed region).  Falls back to one `nvidia-smi` query per poll."""
    REASONS = (("hw_slowdown", "nvmlClocksEventReasonHwSlowdown", 0x8), ("hw_thermal_slowdown", "nvmlClocksEventReasonHwThermalSlowdown", 0x40),
               ("sw_thermal_slowdown", "nvmlClocksEventReasonSwThermalSlowdown", 0x20), ("sw_power_cap", "nvmlClocksEventReasonSwPowerCap", 0x4),
               ("hw_power_brake_slowdown", "nvmlClocksEventReasonHwPowerBrakeSlowdown", 0x80))

    def __init__(self, gpu_index, period_s=0.004):
        self.period, self.samples, self.reasons, self.active, self.stop_flag = period_s, [], set(), False, False
        self.sm_max, self.how, self.nvml, self.handle = None, None, None, None
        try:
            import pynvml
            pynvml.nvmlInit()
            # torch's device order follows CUDA_VISIBLE_DEVICES; NVML's does not
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            phys = gpu_index
            if vis:
                ids = [v.strip() for v in vis.split(",") if v.strip()]
                if gpu_index < len(ids) and ids[gpu_index].isdigit():
                    phys = int(ids[gpu_index])
            self.handle = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.sm_max = float(pynvml.nvmlDeviceGetMaxClockInfo(self.handle, pynvml.NVML_CLOCK_SM))
            self.nvml, self.how = pynvml, "NVML in-process, %.0f ms period" % (period_s * 1e3)
        except Exception:
            self.how = "nvidia-smi query per poll"
        self.gpu_index = gpu_index
        self.thread = threading.Thread(target=self._run, daemon=True)
        self.thread.start()

    def _poll(self):
        if self.nvml is not None:
            n = self.nvml
            sm = float(n.nvmlDeviceGetClockInfo(self.handle, n.NVML_CLOCK_SM))
            try:
                mask = int(n.nvmlDeviceGetCurrentClocksEventReasons(self.handle))
            except Exception:
                mask = int(n.nvmlDeviceGetCurrentClocksThrottleReasons(self.handle))
            return sm, [name for name, attr, bit in self.REASONS if mask & getattr(n, attr, bit)]
        out = subprocess.run(["nvidia-smi", "-i", str(self.gpu_index), "--query-gpu=clocks.sm,clocks.max.sm,"
                              "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
                              "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap",
                              "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=10).stdout
        r = [x.strip() for x in out.strip().splitlines()[0].split(",")]
        self.sm_max = float(r[1])
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        return float(r[0]), [n for n, v in zip(names, r[2:6]) if v.lower().startswith("active")]

    def _run(self):
        while not self.stop_flag:
            if self.active:
                try:
                    sm, reasons = self._poll()
                    if self.active:
                        self.samples.append(sm)
                        self.reasons.update(reasons)
                except Exception:
                    pass
            time.sleep(self.period)

    def begin(self):
        self.active = True

    def end(self):
        self.active = False

    def stop(self):
        self.stop_flag = True
        self.thread.join(timeout=5)
        s = self.samples
        return {"sm_mhz": float(np.median(s)) if s else None, "sm_min_mhz": float(min(s)) if s else None,
                "sm_max_mhz": self.sm_max, "reasons": sorted(self.reasons), "samples": len(s), "how": self.how,
                "when": "inside the timed regions only"}


# ------------------------------------------------------------------------------------------------- the oracle, timed
def _oracle_replica(args):
    """One replica of the oracle on the bounded sample (runs in a worker process, one BLAS thread)."""
    index, steps, warmup = args
    for v in ("OMP_NUM_THREADS", "OPENBLAS_NUM_THREADS", "MKL_NUM_THREADS"):
        os.environ[v] = "1"
    try:
        from threadpoolctl import threadpool_limits
        threadpool_limits(1)
    except Exception:
        pass
    from oracle import sark
    from oracle.operators import ReferenceElement
    from oracle.rhs import Problem
    dim, N = DIM_N[index]
    ref = ReferenceElement(dim, N)
    cfg = make_config(index, ref.lam, sample=True)
    P = Problem(dim, N, cfg["X0"], cfg["EToV"], cfg.get("vertex_equiv"), cfg.get("EToB"), cfg.get("pml_sigma"),
                RT=cfg["RT"], tau=cfg["tau"], q_inf=cfg.get("q_inf"), motion_kind=cfg["motion_kind"],
                motion_params=cfg["motion_params"], ref=ref)
    q, aux, dt = cfg["q0"], None, cfg["dt"]
    for n in range(warmup):
        stages, aux = sark.step_debug(P, q, n * dt, dt, aux)
        q = stages[-1]
    w0 = time.perf_counter()
    for n in range(steps):
        stages, aux = sark.step_debug(P, q, (warmup + n) * dt, dt, aux)
        q = stages[-1]
    wall = time.perf_counter() - w0
    return wall, cfg["K"] * cfg["Np"] * cfg["Nf"], cfg["K"], cfg["name"], N, cfg["Nf"], bool(np.isfinite(q).all())


def time_oracle(index, steps, warmup, cores=None):
    """The oracle as it stands (never tuned for this) on a bounded sample of workload `index`: one independent replica
    of the sample per host core, all started together; value = replicas x DOF x 4 x steps / slowest replica.
    Returns (GDOF-stage/s, cores used, description, ms per step of the slowest replica)."""
    import multiprocessing as mp
    cores = cores or int(os.environ.get("ALEGB_BENCH_CORES", "0")) or os.cpu_count() or 1
    if cores == 1:
        results = [_oracle_replica((index, steps, warmup))]
    else:
        with mp.get_context("spawn").Pool(cores) as pool:
            results = pool.map(_oracle_replica, [(index, steps, warmup)] * cores, chunksize=1)
    wall = max(r[0] for r in results)
    dof, K, name, N, Nf = results[0][1:6]
    assert all(r[6] for r in results)
    desc = ("SAMPLE (K=%d), not the config: %s recipe shrunk to K=%d elements (N=%d, %d fields), %d SARK4 steps (%d "
            "stages), %d independent replicas (one per host core, numpy single-threaded each); the value is the "
            "aggregate of the replicas, no extrapolation to the full mesh"
            % (K, name, K, N, Nf, steps, 4 * steps, cores))
    return cores * dof * 4 * steps / wall / 1e9, cores, desc, wall / max(steps, 1) * 1e3


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
    value, cores, desc, ms = time_oracle(args.config, args.steps, args.warmup)
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


# ------------------------------------------------------------------------------------------------- the CUDA path, timed
def measure(index, args, B, torch, local_rank, world, barrier, sampler, repeats, steps, warmup):
    """Times `repeats` regions of exactly `steps` SARK4 steps of workload `index` (state resident in HBM) and the fused
    stage kernel inside them.  Returns a dict; elapsed times are this rank's (the caller takes the max over ranks)."""
    dim, N = DIM_N[index]
    probe = B.Context(dim, N, -1)
    lam = probe.alegb_get_reference()["lam"]     # node coordinates for the initial state (input generation only)
    probe.close()
    cfg = make_config(index, lam)
    ctx = B.context_from_config(cfg, local_rank)
    ctx.alegb_set_kernel(args.kernel)
    if args.no_overlap:
        ctx.alegb_set_geometry_overlap(False)
    if getattr(args, "layer_fusion", None) is not None:
        ctx.alegb_set_layer_fusion(args.layer_fusion)
    if args.relax == "cubature":
        ctx.alegb_set_relaxation(B.RELAX_CUBATURE)
    if args.coords == "rk":
        ctx.alegb_set_coordinate_mode(B.COORDS_RK, 0.0)
    K, Np, Nf, Nfp = cfg["K"], cfg["Np"], cfg["Nf"], ctx.Nfp
    dof, dt = K * Np * Nf, cfg["dt"]
    q = torch.from_numpy(cfg["q0"]).cuda()
    state_bytes = q.numel() * 8
    ctx.alegb_step(q, 0.0, dt, warmup)
    barrier()
    # Large states (the throughput configuration): the library brackets every stage-kernel launch of the timed regions
    # with events (direct launches).  Small, L2-resident states are launch-bound: the timed regions replay the
    # captured step graph (alegb_set_graph) and the stage kernel is timed in a second, direct pass of the same steps.
    graph_timed = state_bytes < 200e6
    ctx.alegb_profile_enable(not graph_timed)
    times, launches = [], 0
    for r in range(repeats):
        n0 = ctx.alegb_launch_count()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        if sampler:
            sampler.begin()
        e0.record()
        ctx.alegb_step(q, (warmup + r * steps) * dt, dt, steps)
        e1.record()
        barrier()
        if sampler:
            sampler.end()
        times.append(e0.elapsed_time(e1))
        launches = ctx.alegb_launch_count() - n0
    if graph_timed:
        ctx.alegb_profile_enable(True)
        ctx.alegb_step(q.clone(), warmup * dt, dt, steps)
    nprof, prof_ms = ctx.alegb_profile_read()
    ctx.alegb_profile_enable(False)
    finite = bool(torch.isfinite(q).all().item())
    kern_ms = prof_ms / max(nprof, 1)
    # share of the step: stage-kernel time per step / step time (both from the same kind of launches where possible)
    # (graph-replayed regions: the stage kernel is timed in a separate direct-launch pass whose launches do not
    #  overlap the a1/a2 branch the same way, so a share of the replayed step is not defined)
    share = None if graph_timed else (prof_ms / max(nprof, 1) * 4) / (float(np.median(times)) / steps)
    return dict(cfg=cfg, ctx=ctx, q=q, dim=dim, N=N, K=K, Np=Np, Nf=Nf, Nfp=Nfp, dof=dof, dt=dt, state_bytes=state_bytes,
                times=times, launches=launches, kern_ms=kern_ms, nprof=nprof, share=share, graph_timed=graph_timed,
                finite=finite)


def rooflines(m, index, kernel, default_modes=True):
    hbm_peak, hbm_src = measured_peaks()
    flop_per_dof = algorithmic_flop_per_dof_stage(m["dim"], m["Np"], m["Nfp"])
    tf = m["dof"] * flop_per_dof / (m["kern_ms"] * 1e-3) / 1e12
    gbs = m["dof"] * ALGO_BYTES_PER_DOF_STAGE / (m["kern_ms"] * 1e-3) / 1e9
    alu = {"bound": "alu", "achieved": tf, "peak": FP64_PEAK_TFLOPS, "unit": "TFLOP/s", "frac": tf / FP64_PEAK_TFLOPS,
           "traffic": None, "peak_source": "derived: 148 SM x 64 fp64 FMA/clk x 2 x 1.965 GHz (no fp64 figure in "
           "MEASURED_PEAKS.json; DMMA microbenchmark 37.1, profiles/r1_fp64_peak.md)",
           "algorithmic_flop_per_dof_stage": flop_per_dof}
    hbm = {"bound": "hbm", "achieved": gbs, "peak": hbm_peak, "unit": "GB/s", "frac": gbs / hbm_peak, "traffic": None,
           "peak_source": hbm_src, "algorithmic_bytes_per_dof_stage": ALGO_BYTES_PER_DOF_STAGE}
    first, other = (alu, hbm) if alu["frac"] >= hbm["frac"] else (hbm, alu)
    first = dict(first)
    first["algorithmic_bytes_per_launch"] = m["dof"] * ALGO_BYTES_PER_DOF_STAGE
    sha = kernel_sources_sha256()
    if index not in NCU_DRAM_BYTES_PER_LAUNCH:
        first["traffic_source"] = "no committed ncu capture for this workload"
    elif kernel != 0 or not default_modes:
        first["traffic_source"] = "the committed ncu capture is of the default kernel and modes, not of this run"
    elif sha != NCU_CAPTURE_SHA256:
        first["traffic_source"] = ("stale: the committed ncu capture (%s) is of kernel sources %s, this run's are %s"
                                   % (NCU_DRAM_BYTES_PER_LAUNCH[index][1], NCU_CAPTURE_SHA256, sha))
    else:
        first["traffic"], src = NCU_DRAM_BYTES_PER_LAUNCH[index]
        first["traffic_unit"] = "bytes per launch (ncu dram read+write)"
        first["traffic_source"] = "committed ncu capture %s, kernel sources sha256 %s (matches this run)" % (src, sha)
    first.update({"kernel": "alegb stage kernel (fused volume+relaxation+surface+SARK update)",
                  "kernel_ms": m["kern_ms"], "kernel_launches_timed": m["nprof"], "kernel_share_of_step": m["share"],
                  "kernel_timed_in": "second pass, direct launches (timed regions replay the step graph)"
                  if m["graph_timed"] else "timed regions", "other_roof": other})
    return first


def default_modes(args):
    """True if the run is in the modes the committed ncu captures were taken in."""
    return (args.relax == "collocation" and args.coords == "closed" and not args.no_overlap
            and getattr(args, "layer_fusion", None) is None)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--repeats", type=int, default=5, help="timed regions of --steps steps each; the median is reported")
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
    ap.add_argument("--no-per-config", action="store_true", help="skip the per_config block (workloads 1, 2, 3, 5)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "b200" else args.warmup
    args.repeats = max(args.repeats, 1)

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

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    sampler = ClockSampler(local_rank) if rank == 0 else None      # started before the warm-up
    m = measure(args.config, args, B, torch, local_rank, world, barrier, sampler, args.repeats, args.steps, args.warmup)
    times = [max_over_ranks(t, world, "cuda") for t in m["times"]]
    elapsed_ms = float(np.median(times))
    value = job_throughput(m["dof"], args.steps, world, elapsed_ms)
    ctx, cfg, dof, dt, state_bytes = m["ctx"], m["cfg"], m["dof"], m["dt"], m["state_bytes"]

    # ---- end to end through the host-buffer entry point (pinned host state, H2D + step + D2H every step)
    e2e = None
    if not args.no_e2e:
        hq = torch.from_numpy(cfg["q0"]).pin_memory()
        ctx.alegb_step_host(hq, 0.0, dt, 1)
        barrier()
        nsteps_e2e = max(3, min(args.steps, 10))
        if sampler:
            sampler.begin()
        t0 = time.perf_counter()
        for n in range(nsteps_e2e):
            ctx.alegb_step_host(hq, (1 + n) * dt, dt, 1)
        torch.cuda.synchronize()
        el = max_over_ranks(time.perf_counter() - t0, world, "cuda")
        # second figure: one host round trip per --steps steps (the state crosses PCIe twice per CALL, not per step)
        t0 = time.perf_counter()
        ctx.alegb_step_host(hq, (1 + nsteps_e2e) * dt, dt, args.steps)
        torch.cuda.synchronize()
        el_b = max_over_ranks(time.perf_counter() - t0, world, "cuda")
        if sampler:
            sampler.end()
        e2e = {"value": job_throughput(dof, nsteps_e2e, world, el * 1e3), "unit": UNIT, "h2d_bytes_per_step": state_bytes,
               "d2h_bytes_per_step": state_bytes, "steps": nsteps_e2e, "api": "alegb_step_host (pinned host buffer), one step per call",
               "batched": {"value": job_throughput(dof, args.steps, world, el_b * 1e3), "unit": UNIT,
                           "steps_per_call": args.steps, "h2d_bytes_per_step": state_bytes / args.steps,
                           "d2h_bytes_per_step": state_bytes / args.steps}}
    # fp64 ceiling measured on this device at the clocks of this run (alegb_measure_fp64_peak), for the roofline
    fp64_measured = None
    # (clocks of the microbenchmark go into its own record: a pure DMMA loop runs into the power cap, and that reason
    #  must not be attributed to the timed regions of the step)
    try:
        peak_sampler = ClockSampler(local_rank) if rank == 0 else None
        if peak_sampler:
            peak_sampler.begin()
        dmma_tf, dfma_tf = ctx.alegb_measure_fp64_peak()
        if peak_sampler:
            peak_sampler.end()
        fp64_measured = {"dmma_tflops": dmma_tf, "dfma_tflops": dfma_tf,
                         "how": "alegb_measure_fp64_peak: register-resident DMMA (mma.sync.m8n8k4.f64) / DFMA chains, 16 "
                                "warps per SM, best of 5 launches, CUDA events",
                         "clocks": peak_sampler.stop() if peak_sampler else None}
    except Exception as e:
        fp64_measured = {"error": repr(e)[:200]}
    ctx.close()
    del m["q"]
    torch.cuda.empty_cache()

    # ---- the other workloads (rank 0's GPU only, after the headline numbers; a few seconds each)
    per_config = None
    if not args.no_per_config and world == 1:
        per_config = {}
        for idx in (1, 2, 3, 5):
            if idx == args.config:
                continue
            try:
                st = 50 if idx in (1, 2) else (20 if idx == 3 else 5)
                mm = measure(idx, args, B, torch, local_rank, 1, barrier, sampler, 3, st, 3)
                el = float(np.median(mm["times"]))
                rf = rooflines(mm, idx, args.kernel, default_modes(args))
                per_config[str(idx)] = {
                    "workload": workload_name(idx), "K": mm["K"], "dof": mm["dof"], "steps": st, "repeats": 3,
                    "value": job_throughput(mm["dof"], st, 1, el), "unit": UNIT, "ms_per_step": el / st,
                    "stage_kernel_ms": mm["kern_ms"], "stage_kernel_share_of_step": mm["share"],
                    "frac_fp64": (rf if rf["bound"] == "alu" else rf["other_roof"])["frac"],
                    "frac_hbm": (rf if rf["bound"] == "hbm" else rf["other_roof"])["frac"],
                    "gpu_launches_per_region": int(mm["launches"]), "state_finite": mm["finite"],
                    "launch": "one CUDA graph per step" if mm["graph_timed"] else "direct launches"}
                mm["ctx"].close()
                del mm
                torch.cuda.empty_cache()
            except Exception as e:      # a failed side measurement must not lose the headline line
                per_config[str(idx)] = {"error": repr(e)[:300]}
    # ---- the optional modes (NEXT-1, NEXT-2, a8 fused / separate): throughput and stage-kernel time, a few seconds each
    modes = None
    if not args.no_per_config and world == 1 and default_modes(args):
        import copy
        modes = {}
        for name, idx, change in (("config4_relax_cubature", 4, dict(relax="cubature")),
                                  ("config4_coords_rk", 4, dict(coords="rk")),
                                  ("config3_layer_fused", 3, dict(layer_fusion=1)),
                                  ("config3_layer_separate", 3, dict(layer_fusion=0)),
                                  ("config5_layer_separate", 5, dict(layer_fusion=0))):
            try:
                a2 = copy.copy(args)
                for k, v in change.items():
                    setattr(a2, k, v)
                st = 20 if idx == 3 else 5
                mm = measure(idx, a2, B, torch, local_rank, 1, barrier, sampler, 3, st, 3)
                el = float(np.median(mm["times"]))
                rf = rooflines(mm, idx, args.kernel, False)
                modes[name] = {
                    "workload": workload_name(idx), "change": change, "steps": st, "repeats": 3,
                    "value": job_throughput(mm["dof"], st, 1, el), "unit": UNIT, "ms_per_step": el / st,
                    # per stage: everything the stage launches (cubature kernel + stage kernel(s)); the separate
                    # layer kernel of layer_fusion = 0 is outside this bracket
                    "stage_kernel_ms": mm["kern_ms"],
                    "frac_fp64": (rf if rf["bound"] == "alu" else rf["other_roof"])["frac"],
                    "frac_hbm": (rf if rf["bound"] == "hbm" else rf["other_roof"])["frac"],
                    "gpu_launches_per_region": int(mm["launches"]), "state_finite": mm["finite"]}
                mm["ctx"].close()
                del mm
                torch.cuda.empty_cache()
            except Exception as e:
                modes[name] = {"error": repr(e)[:300]}
    clocks = sampler.stop() if sampler else None

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    roofline = rooflines(m, args.config, args.kernel, default_modes(args))
    alu = roofline if roofline["bound"] == "alu" else roofline["other_roof"]
    alu["peak_measured"] = fp64_measured
    if fp64_measured and "dmma_tflops" in fp64_measured:
        top = max(fp64_measured["dmma_tflops"], fp64_measured["dfma_tflops"])
        alu["frac_of_measured_peak"] = alu["achieved"] / top if top > 0 else None
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": elapsed_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "repeats": {"n": args.repeats, "statistic": "median", "ms_per_step_min": min(times) / args.steps,
                        "ms_per_step_max": max(times) / args.steps,
                        "value_min": job_throughput(dof, args.steps, world, max(times)),
                        "value_max": job_throughput(dof, args.steps, world, min(times))},
            "config": {"workload": workload_name(args.config), "K": m["K"], "N": m["N"], "Np": m["Np"], "Nfields": m["Nf"],
                       "dof": dof, "dt": dt, "parallelism": "replicas x%d (north_star: one GPU, no sharding)" % world,
                       "l2": "state arrays are %.0f MB each (> 126 MB L2), no flush needed" % (state_bytes / 1e6)
                       if state_bytes > 200e6 else "state is L2-resident (%.1f MB); launch-latency bound" % (state_bytes / 1e6),
                       "state_finite": m["finite"], "kernel": args.kernel, "relax": args.relax, "coords": args.coords,
                       "launch": "one CUDA graph per step" if m["graph_timed"] and args.steps >= 2 else "direct launches"},
            "e2e": e2e, "gpu_launches": int(m["launches"]), "clocks": clocks, "roofline": roofline}
    if per_config is not None:
        line["per_config"] = per_config
    if modes is not None:
        line["modes"] = modes
    if not args.no_cpu_baseline:
        v, cores, desc, _ = time_oracle(args.config, 6 if args.config in (4, 5) else 20, 1)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc,
                                "host_cores_available": os.cpu_count()}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

"""bench.py -- one radiation stage (ghost fill + fused flux divergence + implicit coupling + mask) per "step".

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C3] [--n CELLS] [--impl reference]

Metric (BASELINE.json): intensity-cell updates per second per radiation stage, FP64; one update = one
(cell, angle) pair advanced one stage.  Default workload: config C3, the 128^3 x 162-angle Kerr-Schild block the
north_star target is quoted on.  Inputs are seeded synthetic (paper_2302_04283_b200.workloads), resident in HBM
before the timed region; the intensity arrays (2 x 2.98 GB) exceed L2 (126 MB), so no flush is needed.

One JSON line on stdout (rank 0).  `value` is device-timed (CUDA events on the launching stream, max over ranks);
`e2e` is the same stage through rad_stage_host with pinned HOST buffers, copies inside the timed region;
`roofline` is for the fused stage kernel k_stage5 (the only kernel of a step), from the CUDA-event time of the timed region; `cpu_baseline` is the oracle
timed on the host cores on a bounded sub-block of the same workload.  With --gpus N > 1 (torchrun) every rank
runs an independent replica of the block ("replicas only": the path has no collective), scaling = weak.
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "intensity_cell_updates_per_sec_per_stage"
UNIT = "updates/s"


def algorithmic_bytes_per_update(N):
    """fused stage kernel, DESIGN.md 'rooflines' (single-pass stage): read I (8) + write I_+ (8) + per-cell
    side data of both halves of the stage (536 B geometry + 104 B fluid, opacity and fluid outputs) spread over N angles"""
    return 16.0 + 640.0 / N


def design_bytes_per_update(N):
    """what the kernel as built must move: read I (8) + write I_+ (8) + the stored angular-edge coefficients (3 doubles per
    update) + per cell 288 B packed record, ~48 B lower-face records of the tile edge,
    64 B fluid and opacities, 40 B T_+ and fluid increment"""
    return 16.0 + 24.0 + 440.0 / N


# DRAM bytes per launch of the stage kernel from the committed ncu --set full capture (dram__bytes_read.sum +
# dram__bytes_write.sum; profiles/r1_k_stage5_ncu_full.md), for the workload it was taken on: (config, cells per axis, recon)
NCU_TRAFFIC_BYTES = {("C3", None, 1): 15.86e9}

# FP64-pipe instruction slots per update of the stage kernel: FP64 warp instructions x 32 lanes /
# updates, from the ncu instruction counts under profiles/ (idle lanes of the last angle group included); one slot = one
# DFMA-equivalent issue = 2 flop of the measured DFMA peak
FP64_SLOTS_PER_UPDATE = {True: 177.0, False: 118.0}  # with / without coupling


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md)"""

    def __init__(self, index=0):
        self.rows, self.proc = [], None
        q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={q}", "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def summary(self, t0, t1):
        if self.proc:
            self.proc.terminate()
        rows = [r for t, r in self.rows if t0 - 0.05 <= t <= t1 + 0.05] or [r for _, r in self.rows[-3:]]
        sm, mx, reasons = [], 0, set()
        for r in rows:
            f = [x.strip() for x in r.split(",")]
            try:
                sm.append(float(f[0])); mx = max(mx, float(f[1]))
            except (ValueError, IndexError):
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": mx or None, "reasons": sorted(reasons), "samples": len(sm)}


def max_over_ranks(value, world, device=None):
    """max of a per-rank scalar over all ranks (the contract's 'max over ranks' timing); `device` = where the backend's
    tensors live ("cuda" for nccl, None/"cpu" for gloo)"""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    tt = torch.tensor([float(value)], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    return float(tt.item())


def whole_job_value(updates_per_rank, world, ms):
    """whole-job throughput of N independent replicas ('replicas only', weak scaling): all ranks' updates / max time"""
    return world * updates_per_rank / (ms * 1e-3)


def measured_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


class OracleSample:
    """the oracle, as it stands, on the nsub^3 cells at the low corner of the workload's block (same spacing, own ghosts,
    same input recipe); built once, each run() is one full stage on the same inputs"""

    def __init__(self, cfg, nsub, tau_factor=0.0):
        from oracle import rad_oracle as O
        from paper_2302_04283_b200 import workloads as W
        c = W.CONFIGS[cfg]
        A = O.Angles(*c["angles"])
        nn, ng, x0, dx = W.grid(cfg, sub=nsub)
        self.P = O.Problem(A, nn, x0, dx, metric_kind=c["metric"], M=c["M"], a=c["a"], excise_r=W.excise_radius(cfg),
                           bc_lo=(c["bc"],) * 3, bc_hi=(c["bc"],) * 3, tau_factor=tau_factor)
        inp = W.make_inputs(cfg, A.nhat, sub=nsub)
        self.I = inp["I"].numpy().reshape(-1, A.N).copy()
        self.fluid = inp["fluid"].numpy().reshape(5, -1).copy(); self.opac = inp["opac"].numpy().reshape(3, -1).copy()
        self.dt = W.CFL * min(dx) / self.P.max_speed()[0]
        self.updates = nsub ** 3 * A.N

    def run(self):
        """seconds of one stage"""
        t0 = time.perf_counter()
        self.P.stage(self.I, self.fluid, self.opac, self.dt)
        return time.perf_counter() - t0


def run_reference(args):
    """--impl reference: the oracle (plain CPU FP64), timed as it stands on a bounded sample of the same workload"""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_2302_04283_b200 import workloads as W
    cfg = args.config
    nsub = args.ref_n or 64
    N = W.n_angles(cfg)
    cores = os.cpu_count()
    smp = OracleSample(cfg, nsub, args.tau_factor)
    for _ in range(args.warmup):
        smp.run()
    times = [smp.run() for _ in range(args.steps)]
    ms = 1e3 * sum(times) / len(times)
    val = smp.updates / (ms * 1e-3)
    sample = f"{nsub}^3-cell sub-block (low corner, own ghosts) of {cfg}, {N} angles, one full stage per step"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{cfg} (oracle on a bounded sample)", "sample": sample},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="C3")
    ap.add_argument("--n", type=int, default=None, help="override cells per axis (same box)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--ref-n", type=int, default=None, help="sub-block size of the oracle sample (default: 64 for --impl reference, 96 for the cpu_baseline leg)")
    ap.add_argument("--recon", type=int, default=1, help="spatial reconstruction: 1 PLM (the workload's), 0 donor cell (diagnostic)")
    ap.add_argument("--tau-factor", type=float, default=0.0, help="constant of Eq.26: > 0 times the stage with the optical-depth-aware flux (NEXT-1; separate kernels)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        return run_reference(args)

    import numpy as np
    import torch
    import torch.distributed as dist

    from paper_2302_04283_b200 import binding as B
    from paper_2302_04283_b200 import build
    from paper_2302_04283_b200 import workloads as W

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl")
    if rank == 0:
        build.build()
    if world > 1:
        dist.barrier()
    B.lib()

    cfg = args.config
    c = W.CONFIGS[cfg]
    nn, ng, x0, dx = W.grid(cfg, args.n)
    N = W.n_angles(cfg)
    updates = nn[0] * nn[1] * nn[2] * N

    # angle directions from the library itself (a context without geometry cost: 1 cell)
    h0 = B.rad_create(dict(kind=0), dict(n=(1, 1, 1), x0=(0, 0, 0), dx=(1, 1, 1)), c["angles"], None, dict(couple=0), local)
    nhat = B.rad_get_table(h0, B.TAB_NHAT)
    B.rad_destroy(h0)
    inp = W.make_inputs(cfg, nhat, n=args.n, device=f"cuda:{local}")
    I_a = inp["I"].reshape(-1, N).contiguous(); fluid = inp["fluid"].reshape(5, -1).contiguous(); opac = inp["opac"].reshape(3, -1).contiguous()
    del inp
    I_b = I_a.clone()
    ncell = fluid.shape[1]
    T_out = torch.zeros(ncell, dtype=torch.float64, device="cuda"); dT0 = torch.zeros(4, ncell, dtype=torch.float64, device="cuda")
    h = B.rad_create(dict(kind=c["metric"], M=c["M"], a=c["a"], excise_r=W.excise_radius(cfg)),
                     dict(n=nn, x0=x0, dx=dx, bc_lo=(c["bc"],) * 3, bc_hi=(c["bc"],) * 3), c["angles"], (opac[0], opac[1], opac[2]),
                     dict(gamma_gas=W.GAMMA_GAS, a_rad=W.A_RAD, n0_crit=W.N0_CRIT, recon_space=args.recon, renorm_fluid_weights=1, couple=1, tau_factor=args.tau_factor), local)
    vmax = float(B.rad_get_table(h, B.TAB_MAXSPEED).max())
    dt = W.CFL * min(dx) / vmax
    stream = torch.cuda.current_stream()

    def stage():
        # every step advances the same seeded state I_a -> I_b (fixed work per step; I_b is fully rewritten)
        B.rad_stage(h, I_a, I_b, None, fluid, 0.0, 1.0, dt, T_out, dT0, stream=stream)

    def sync_all():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    for _ in range(args.warmup):
        stage()
    sync_all()
    sampler = ClockSampler(local) if rank == 0 else None
    l0 = B.rad_launch_count(h)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0 = time.time()
    ev0.record(stream)
    for _ in range(args.steps):
        stage()
    ev1.record(stream)
    sync_all()
    t1 = time.time()
    launches = B.rad_launch_count(h) - l0
    ms = ev0.elapsed_time(ev1) / args.steps
    ms = max_over_ranks(ms, world, "cuda")
    clocks = sampler.summary(t0, t1) if sampler else None

    # the stage kernel without its coupling half, and the stand-alone coupling kernel, for the record
    def time_call(fn, reps):
        for _ in range(2):
            fn()
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        for _ in range(reps):
            fn()
        b.record(stream)
        torch.cuda.synchronize()
        return a.elapsed_time(b) / reps

    reps = max(3, args.steps)
    ms_flux = None
    if args.tau_factor == 0.0:  # (with the optical-depth-aware flux the transport half alone has no fluid state)
        ms_flux = time_call(lambda: B.rad_transport(h, I_a, I_b, None, 0.0, 1.0, dt, stream=stream), reps)
        B.rad_transport(h, I_a, I_b, None, 0.0, 1.0, dt, stream=stream)
    ms_cpl = time_call(lambda: B.rad_couple(h, I_b, fluid, dt, T_out, dT0, stream=stream), reps)
    # roofline of the dominant kernel = the fused stage kernel k_stage (flux divergence + coupling in one launch): with
    # caller-filled ghosts it is the only kernel of a step, so its average launch duration is the CUDA-event time of the
    # timed region / launches
    kernels_per_step = max(1, launches // max(1, args.steps))
    peak, peak_src = measured_peak()
    bpu = algorithmic_bytes_per_update(N)
    achieved = bpu * updates / (ms * 1e-3) / 1e9
    kname = "k_stage5 (fused flux divergence + implicit coupling + mask, one launch per step)" if args.tau_factor == 0.0 else \
        "k_tau_table + k_stage5<TAU> (tile kernel with the Eq.28 factor): the step's two kernels together"
    roofline = {"kernel": kname, "bound": "hbm",
                "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": NCU_TRAFFIC_BYTES.get((cfg, args.n, args.recon)),
                "traffic_source": "ncu --set full capture, profiles/r1_k_stage5_ncu_full.md (bytes per launch)" if (cfg, args.n, args.recon) in NCU_TRAFFIC_BYTES else None,
                "peak_source": peak_src,
                "algorithmic_bytes_per_update": bpu, "design_bytes_per_update": design_bytes_per_update(N),
                "design_frac": design_bytes_per_update(N) * updates / (ms * 1e-3) / 1e9 / peak,
                "ms_per_launch": ms / kernels_per_step, "kernels_per_step": kernels_per_step,
                "flux_divergence_only_ms": ms_flux, "standalone_coupling_kernel_ms": ms_cpl}
    dfma = B.rad_probe_fp64(h)
    slots = FP64_SLOTS_PER_UPDATE[True]
    roofline_alu = {"kernel": kname, "bound": "alu", "unit": "TFLOP/s", "peak": 2.0 * dfma / 1e12,
                    "peak_source": "measured live: rad_probe_fp64 (register-only DFMA kernel, CUDA events)",
                    "achieved": 2.0 * slots * updates / (ms * 1e-3) / 1e12, "fp64_slots_per_update": slots,
                    "note": "one FP64-pipe instruction slot per lane = 2 flop (DFMA-equivalent)"}
    roofline_alu["frac"] = roofline_alu["achieved"] / roofline_alu["peak"]

    # end to end through the C ABI with HOST buffers (pinned), copies inside the timed region
    e2e = None
    if not args.no_e2e:
        hI = torch.empty(I_a.shape, dtype=torch.float64, pin_memory=True); hI.copy_(I_a)
        hO = torch.empty(I_a.shape, dtype=torch.float64, pin_memory=True)
        hfl = fluid.cpu().pin_memory(); hop = opac.cpu().pin_memory()
        hT = torch.empty(ncell, dtype=torch.float64, pin_memory=True); hdT = torch.empty(4, ncell, dtype=torch.float64, pin_memory=True)
        nrep = max(1, min(args.steps, 3))
        B.rad_stage_host(h, hI, hO, hfl, hop, 0.0, 1.0, dt, hT, hdT)
        sync_all()
        w0 = time.perf_counter()
        for _ in range(nrep):
            B.rad_stage_host(h, hI, hO, hfl, hop, 0.0, 1.0, dt, hT, hdT)
        torch.cuda.synchronize()
        w = (time.perf_counter() - w0) / nrep
        w = max_over_ranks(w, world, "cuda")
        e2e = {"value": world * updates / w, "unit": UNIT, "h2d_bytes_per_step": int(hI.numel() * 8 + hfl.numel() * 8 + hop.numel() * 8),
               "d2h_bytes_per_step": int(hO.numel() * 8 + hT.numel() * 8 + hdT.numel() * 8), "ms_per_step": w * 1e3}
        del hI, hO
    B.rad_destroy(h)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        nsub = args.ref_n or 96
        smp = OracleSample(cfg, nsub, args.tau_factor)
        smp.run()
        secs = [smp.run() for _ in range(2)]
        sec = sum(secs)
        ups = 2 * smp.updates / sec
        cpu = {"value": ups, "unit": UNIT, "cores": os.cpu_count(), "kind": "oracle",
               "sample": f"{nsub}^3-cell sub-block (low corner, own ghosts) of {cfg}, {N} angles, 2 timed stages after 1 warm-up, {sec:.1f} s"}
    line = {"metric": METRIC, "value": whole_job_value(updates, world, ms), "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{cfg}: {c['angles']} angles={N}, {nn[0]}^3 cells + 2 ghosts, metric kind {c['metric']} a={c['a']}, box {c['box']}",
                       "updates_per_step": updates, "tau_factor": args.tau_factor, "parallelism": "replicas only" if world > 1 else "1 GPU",
                       "l2": "inputs (2 x %.2f GB) exceed L2; no flush" % (I_a.numel() * 8 / 1e9)},
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline, "roofline_alu": roofline_alu,
            "cpu_baseline": cpu}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

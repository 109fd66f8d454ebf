"""bench.py -- one radiation stage (ghost fill + fused flux-divergence kernel + streaming implicit-coupling kernel) per "step".

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C3] [--n CELLS] [--impl reference]

Metric (BASELINE.json): intensity-cell updates per second per radiation stage, FP64; one update = one
(cell, angle) pair advanced one stage.  Default workload: config C3, the 128^3 x 162-angle Kerr-Schild block the
north_star target is quoted on.  Inputs are seeded synthetic (paper_2302_04283_b200.workloads), resident in HBM
before the timed region; the intensity arrays (2 x 2.98 GB) exceed L2 (126 MB), so no flush is needed.

One JSON line on stdout (rank 0).  `value` is device-timed (CUDA events on the launching stream, max over ranks) over K calls
of rad_stage; `e2e` is the same stage through rad_stage_host with pinned HOST buffers, copies inside the timed region;
`roofline` is for the dominant kernel, the fused flux-divergence kernel k_stage5 (north_star's target row), whose average
launch duration is measured live with CUDA events over K launches through rad_transport on the same inputs;
`roofline_coupling` likewise for the coupling kernel (rad_couple); `cpu_baseline` is the oracle timed on the host cores on a
bounded sub-block of the same workload.  Figures that come from ncu (DRAM traffic, FP64 instruction counts) are read from the
committed profiles/r3_kernels.csv, keyed by the kernel instance names the library reports (rad_stage_kernels); a kernel that is
not in the file, or whose sources changed since its row was captured (src_sha16), gets null.  With --gpus N > 1 (torchrun) every rank runs an independent replica of the block ("replicas
only": the path has no collective), scaling = weak.
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


def fluxdiv_bytes_per_update(N):
    """flux-divergence kernel = read I (8) + write I* (8) + 536 B of compact geometry per cell (43 cell + 24 face doubles)"""
    return 16.0 + 536.0 / N


def coupling_bytes_per_update(N):
    """coupling kernel = read I* (8) + write I_+ (8) + 104 B per cell (5 fluid, 3 opacity in; 5 out)"""
    return 16.0 + 104.0 / N


def design_bytes_per_update(N):
    """what the flux-divergence kernel as built must move: read I (8) + write I* (8) + the stored angular-edge coefficients
    (3 doubles per update) + per cell 288 B packed record and ~48 B lower-face records of the tile edge"""
    return 16.0 + 24.0 + 336.0 / N


PROFILE_CSV = os.path.join(ROOT, "profiles", "r3_kernels.csv")
PROFILE_FIELDS = ["kernel", "workload", "ms", "dram_read_bytes", "dram_write_bytes", "inst_warp", "fp64_inst_warp", "fp64_pipe_pct", "issue_pct",
                  "smem_wavefronts", "smem_bank_conflicts", "registers", "grid", "block", "src_sha16"]
KERNEL_SOURCES = {"k_stage5": ["stage5.cu"], "k_couple_stream": ["stream.cu"], "k_moments_mma": ["stream.cu"], "k_fluxdiv": ["transport.cu"],
                  "k_coupling": ["coupling.cu"]}


def kernel_source_hash(kernel):
    """sha256 (16 hex digits) over the sources a kernel is compiled from: its .cu, every header of csrc/ and the build flags.  A row of
    the committed ncu table carries the hash of the sources it was captured on; a row whose hash differs from today's describes other
    code and its figures are not printed (a kernel may change and keep its instance name)."""
    import glob
    import hashlib
    from paper_2302_04283_b200 import build
    csrc = os.path.join(ROOT, "paper_2302_04283_b200", "csrc")
    files = [os.path.join(csrc, f) for f in KERNEL_SOURCES.get(kernel.split("<")[0], [])]
    files += sorted(glob.glob(os.path.join(csrc, "*.cuh")) + glob.glob(os.path.join(csrc, "*.h")))
    h = hashlib.sha256(" ".join(f for f in build.FLAGS if not f.startswith("/")).encode())
    for f in files:
        h.update(open(f, "rb").read())
    return h.hexdigest()[:16]


def norm_kernel(name):
    """'void rad::<unnamed>::k_stage5<(int)3, (int)2, ..., (bool)0>(rad::DeviceTables, ...)' -> 'k_stage5<3,2,...,0>'"""
    import re
    m = re.search(r"(k_[A-Za-z0-9_]+)(<[^>]*>)?", name)
    if not m:
        return name
    return m.group(1) + re.sub(r"\((int|bool)\)|\s", "", m.group(2) or "")


def profile_row(kernel, workload):
    """the committed ncu figures of a kernel instance on a workload, or None: no figure is printed for a kernel that is not in the
    table, nor for one whose sources changed after the row was captured"""
    import csv
    try:
        with open(PROFILE_CSV) as f:
            for r in csv.DictReader(f):
                # (the library reports the generic kernel without its template arguments: "k_fluxdiv" matches the row "k_fluxdiv<1,0>")
                if (r["kernel"] == kernel or ("<" not in kernel and r["kernel"].split("<")[0] == kernel)) and r["workload"] == workload:
                    return r if r.get("src_sha16") == kernel_source_hash(kernel) else None
    except OSError:
        pass
    return None


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

    def wait_first(self, timeout=5.0):
        """nvidia-smi takes a moment to start: the timed region begins only once samples arrive"""
        t0 = time.time()
        while self.proc and not self.rows and time.time() - t0 < timeout:
            time.sleep(0.01)

    def summary(self, t0, t1):
        if self.proc:
            self.proc.terminate()
        rows = [r for t, r in self.rows if t0 <= t <= t1 + 0.02]
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


def omp_threads(n):
    """threads the oracle's OpenMP regions use from now on (libgomp's global setting; the oracle itself is not touched)"""
    import ctypes
    try:
        ctypes.CDLL("libgomp.so.1").omp_set_num_threads(int(n))
        return True
    except OSError:
        return False


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="C3")
    ap.add_argument("--n", type=int, default=None, help="override cells per axis (same box)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--ref-n", type=int, default=None, help="sub-block size of the oracle sample (default: 64 for --impl reference, 96 for the cpu_baseline leg)")
    ap.add_argument("--recon", type=int, default=1, help="spatial reconstruction: 1 PLM (the workload's), 0 donor cell (diagnostic), 2 PPM (NEXT-3: 3 ghost layers, generic flux-divergence kernel)")
    ap.add_argument("--recon-angle", type=int, default=0, help="1: PLM in angle on a latitude-longitude grid (NEXT-3; config C1's grid, e.g. --config C1 --n 64; generic kernel)")
    ap.add_argument("--recompute-edge-coeffs", type=int, default=0, help="1: no stored angular coefficients (rad_params.recompute_edge_coeffs): the generic flux-divergence kernel")
    ap.add_argument("--tau-factor", type=float, default=0.0, help="constant of Eq.26: > 0 times the stage with the optical-depth-aware flux (NEXT-1)")
    ap.add_argument("--vel-estimate", type=int, default=0, help="1: radiation-dominated velocity estimate Eq.51-55 in the coupling (NEXT-2)")
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
    sampler = ClockSampler(local) if rank == 0 else None  # started early: nvidia-smi needs a moment before its first sample

    cfg = args.config
    c = W.CONFIGS[cfg]
    ng_arg = 3 if args.recon == 2 else None
    nn, ng, x0, dx = W.grid(cfg, args.n, ng=ng_arg)
    N = W.n_angles(cfg)
    updates = nn[0] * nn[1] * nn[2] * N
    workload = cfg if args.n is None else f"{cfg}/n={args.n}"

    # angle directions from the library itself (a context without geometry cost: 1 cell)
    h0 = B.rad_create(dict(kind=0), dict(n=(1, 1, 1), x0=(0, 0, 0), dx=(1, 1, 1)), c["angles"], None, dict(couple=0), local)
    nhat = B.rad_get_table(h0, B.TAB_NHAT)
    B.rad_destroy(h0)
    inp = W.make_inputs(cfg, nhat, n=args.n, device=f"cuda:{local}", ng=ng_arg)
    I_a = inp["I"].reshape(-1, N).contiguous(); fluid = inp["fluid"].reshape(5, -1).contiguous(); opac = inp["opac"].reshape(3, -1).contiguous()
    del inp
    I_b = I_a.clone()
    ncell = fluid.shape[1]
    T_out = torch.zeros(ncell, dtype=torch.float64, device="cuda"); dT0 = torch.zeros(4, ncell, dtype=torch.float64, device="cuda")
    h = B.rad_create(dict(kind=c["metric"], M=c["M"], a=c["a"], excise_r=W.excise_radius(cfg)),
                     dict(n=nn, ng=ng, x0=x0, dx=dx, bc_lo=(c["bc"],) * 3, bc_hi=(c["bc"],) * 3), c["angles"], (opac[0], opac[1], opac[2]),
                     dict(gamma_gas=W.GAMMA_GAS, a_rad=W.A_RAD, n0_crit=W.N0_CRIT, recon_space=args.recon, recon_angle=args.recon_angle, renorm_fluid_weights=1, couple=1,
                          tau_factor=args.tau_factor, vel_estimate=args.vel_estimate, recompute_edge_coeffs=args.recompute_edge_coeffs), local)
    vmax = float(B.rad_get_table(h, B.TAB_MAXSPEED).max())
    dt = W.CFL * min(dx) / vmax
    stream = torch.cuda.current_stream()
    k_flux, k_cpl = B.rad_stage_kernels(h)

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
    if sampler:
        sampler.wait_first()
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

    # the step's kernels one by one, live: K launches each on the same inputs, CUDA events on the launching stream
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
    if args.tau_factor == 0.0:  # (with the optical-depth-aware flux the transport half needs the fluid state: timed through the stage only)
        ms_flux = time_call(lambda: B.rad_transport(h, I_a, I_b, None, 0.0, 1.0, dt, stream=stream), reps)
        B.rad_transport(h, I_a, I_b, None, 0.0, 1.0, dt, stream=stream)
    ms_cpl = time_call(lambda: B.rad_couple(h, I_b, fluid, dt, T_out, dT0, stream=stream), reps)
    mom = torch.zeros(10, ncell, dtype=torch.float64, device="cuda")
    ms_mom = time_call(lambda: B.rad_moments(h, I_a, 0, fluid, mom, stream=stream), reps)
    clocks = sampler.summary(t0, time.time()) if sampler else None  # the timed region and the per-kernel loops that follow it
    del mom

    kernels_per_step = max(1, launches // max(1, args.steps))
    peak, peak_src = measured_peak()
    dfma = B.rad_probe_fp64(h)

    def hbm_block(kernel, what, bpu, ms_k, extra=None):
        """roofline of one kernel: algorithmic bytes per launch / its average launch duration, against the measured copy bandwidth"""
        if ms_k is None:
            return None
        achieved = bpu * updates / (ms_k * 1e-3) / 1e9
        prof = profile_row(kernel, workload)
        traffic = (float(prof["dram_read_bytes"]) + float(prof["dram_write_bytes"])) if prof and prof["dram_read_bytes"] else None
        blk = {"kernel": f"{kernel} ({what})", "bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
               "traffic": traffic, "traffic_source": "profiles/r3_kernels.csv (ncu --set full, dram__bytes_read.sum + dram__bytes_write.sum per launch)" if traffic else None,
               "traffic_frac": (traffic / (ms_k * 1e-3) / 1e9 / peak) if traffic else None,
               "peak_source": peak_src, "algorithmic_bytes_per_update": bpu, "ms_per_launch": ms_k,
               "how_timed": "CUDA events over %d launches of this kernel alone on the step's inputs, same process, right after the timed region" % reps}
        if prof and prof["fp64_inst_warp"]:
            slots = 32.0 * float(prof["fp64_inst_warp"]) / updates  # issued FP64 lane slots per update (idle lanes included)
            blk["alu"] = {"bound": "alu", "unit": "TFLOP/s", "peak": 2.0 * dfma / 1e12, "peak_source": "measured live: rad_probe_fp64 (register-only DFMA kernel, CUDA events)",
                          "fp64_slots_per_update_issued": slots, "achieved": 2.0 * slots * updates / (ms_k * 1e-3) / 1e12,
                          "frac": 2.0 * slots * updates / (ms_k * 1e-3) / (2.0 * dfma),
                          "fp64_pipe_pct_ncu": float(prof["fp64_pipe_pct"]), "issue_pct_ncu": float(prof["issue_pct"]),
                          "note": "one FP64-pipe instruction slot per lane = 2 flop (DFMA-equivalent); slots counted by ncu (profiles/r3_kernels.csv)"}
        if extra:
            blk.update(extra)
        return blk

    if args.tau_factor == 0.0:
        roofline = hbm_block(k_flux, "fused spatial + angular flux divergence, cons -> prim: the dominant kernel of the step", fluxdiv_bytes_per_update(N), ms_flux,
                             dict({"share_of_step": ms_flux / ms, "kernels_per_step": kernels_per_step},
                                  **({"design_bytes_per_update": design_bytes_per_update(N),
                                      "design_frac": design_bytes_per_update(N) * updates / (ms_flux * 1e-3) / 1e9 / peak} if k_flux.startswith("k_stage5") else {})))
    else:  # k_tau_table + k_stage5<TAU> + coupling: the step as a whole on the stage's bytes
        roofline = hbm_block(k_flux, "flux divergence with the Eq.28 factor; timed through the whole step", 32.0 + 640.0 / N, ms, {"kernels_per_step": kernels_per_step})
    roofline_coupling = hbm_block(k_cpl, "implicit coupling, mask, fluid increment", coupling_bytes_per_update(N), ms_cpl, {"share_of_step": ms_cpl / ms})
    stage_bpu = fluxdiv_bytes_per_update(N) + coupling_bytes_per_update(N)
    roofline_stage = {"kernel": "whole step (all kernels of one rad_stage)", "bound": "hbm", "unit": "GB/s", "peak": peak,
                      "algorithmic_bytes_per_update": stage_bpu, "achieved": stage_bpu * updates / (ms * 1e-3) / 1e9,
                      "frac": stage_bpu * updates / (ms * 1e-3) / 1e9 / peak,
                      "single_pass_bytes_per_update": algorithmic_bytes_per_update(N),
                      "single_pass_frac": algorithmic_bytes_per_update(N) * updates / (ms * 1e-3) / 1e9 / peak}
    moments = {"kernel": "k_moments_mma (rad_moments, frame 0)", "ms_per_call": ms_mom, "achieved": 8.0 * updates / (ms_mom * 1e-3) / 1e9, "unit": "GB/s",
               "frac": 8.0 * updates / (ms_mom * 1e-3) / 1e9 / peak, "algorithmic_bytes_per_update": 8.0}

    # end to end through the C ABI with HOST buffers (pinned), copies inside the timed region
    e2e = None
    if not args.no_e2e:
        hI = torch.empty(I_a.shape, dtype=torch.float64, pin_memory=True); hI.copy_(I_a)
        hO = torch.empty(I_a.shape, dtype=torch.float64, pin_memory=True)
        hfl = fluid.cpu().pin_memory(); hop = opac.cpu().pin_memory()
        hT = torch.empty(ncell, dtype=torch.float64, pin_memory=True); hdT = torch.empty(4, ncell, dtype=torch.float64, pin_memory=True)
        nrep = max(1, min(args.steps, 10))
        B.rad_stage_host(h, hI, hO, hfl, hop, 0.0, 1.0, dt, hT, hdT)
        sync_all()
        w0 = time.perf_counter()
        for _ in range(nrep):
            B.rad_stage_host(h, hI, hO, hfl, hop, 0.0, 1.0, dt, hT, hdT)
        torch.cuda.synchronize()
        w = (time.perf_counter() - w0) / nrep
        w = max_over_ranks(w, world, "cuda")
        e2e = {"value": world * updates / w, "unit": UNIT, "h2d_bytes_per_step": int(hI.numel() * 8 + hfl.numel() * 8 + hop.numel() * 8),
               "d2h_bytes_per_step": int(hO.numel() * 8 + hT.numel() * 8 + hdT.numel() * 8), "ms_per_step": w * 1e3, "repetitions": nrep}
        # outside the timed region: what the host path returned is what rad_stage computes on the device, bit for bit (interior cells)
        stage()
        torch.cuda.synchronize()
        shp = (nn[2] + 2 * ng, nn[1] + 2 * ng, nn[0] + 2 * ng)
        itr = (slice(ng, -ng),) * 3
        same = bool(torch.equal(hO.view(shp + (N,))[itr], I_b.cpu().view(shp + (N,))[itr])) and bool(torch.equal(hT.view(shp)[itr], T_out.cpu().view(shp)[itr]))
        e2e["output_checked"] = "interior I_out and T_out of rad_stage_host equal rad_stage's device results bit for bit" if same else "MISMATCH against rad_stage"
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
        if omp_threads(1):  # the same oracle on one thread, on a smaller sample of the same block
            n1 = min(nsub, 32)
            smp1 = OracleSample(cfg, n1, args.tau_factor)
            s1 = smp1.run()
            cpu["one_thread"] = {"value": smp1.updates / s1, "unit": UNIT, "cores": 1, "sample": f"{n1}^3-cell sub-block, one stage, {s1:.1f} s"}
            omp_threads(os.cpu_count())
    line = {"metric": METRIC, "value": whole_job_value(updates, world, ms), "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{cfg}: {c['angles']} angles={N}, {nn[0]}^3 cells + {ng} ghosts, metric kind {c['metric']} a={c['a']}, box {c['box']}",
                       "updates_per_step": updates, "tau_factor": args.tau_factor, "vel_estimate": args.vel_estimate,
                       "recon_space": args.recon, "recon_angle": args.recon_angle, "recompute_edge_coeffs": args.recompute_edge_coeffs,
                       "parallelism": "replicas only" if world > 1 else "1 GPU",
                       "l2": ("inputs (2 x %.2f GB) exceed L2; no flush" if I_a.numel() * 8 > 2 * 126e6 else "inputs (2 x %.3f GB) FIT the 126 MB L2 and are not flushed: a warm-L2 figure")
                             % (I_a.numel() * 8 / 1e9)},
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline, "roofline_fluxdiv": roofline,
            "roofline_coupling": roofline_coupling, "roofline_stage": roofline_stage, "moments": moments, "cpu_baseline": cpu}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

#!/usr/bin/env python
"""bench.py -- Dw throughput of the clover Wilson-Dirac hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 --master-port P \
        bench.py --gpus N --steps K --warmup W

One STEP is one application of the normal operator Dw^+ Dw (the paper's DwdagDw!; the body of
every CG iteration): one lqcd_dw_apply followed by one lqcd_dwdag_apply on a fixed
Gaussian spinor, on the 48^3 x 96 periodic lattice of BASELINE.json configs[4] (the configuration the
north_star's >= 70 %-of-HBM-peak target is quoted on; configs[1], 16^3 x 32, is L2-resident and therefore
not an HBM-roofline point).  metric = Dw GFLOP/s under the stated flop model (1872 flop/site/application).
Inputs exceed L2 (16.3 GB compulsory traffic per application vs 126 MB), so no L2 flush is needed.

The JSON line also carries: `roofline` (the stencil kernel against the measured HBM copy bandwidth of
MEASURED_PEAKS.json, compulsory-bytes model of DESIGN.md), `e2e` (the same metric through the host-buffer
C-ABI call lqcd_dw_apply_host, copies inside the timed region), `cpu_baseline` (the fp64 oracle timed on
this box's host cores on a bounded sample) and `rows` (the other hot-path rows of SURVEY.md 8(a), each
measured once in the same run on rank 0 at N=1).

Multi-GPU: the path does not exchange data between GPUs ("replicas only"):
each rank runs an independent replica, value = sum over ranks, scaling = "weak".
"""
import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

FLOP_DW = 1872            # flop/site, Dw or Dw^+ with clover
FLOP_DHAT = 1848          # flop per lattice site, even-odd operator
REALS_DW = {18: 192, 12: 168}      # compulsory reals/site per application
REALS_DHAT = {18: 276, 12: 228}    # even-odd operator (two half hops touch every link once each)
REALS_CG_ITER = {18: 528, 12: 480}  # fused CG iteration
NOMINAL_HBM_GBS = 8000.0  # the figure north_star quotes


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--lattice", default="48x48x48x96", help="L1xL2xL3xL4 of the timed workload")
    ap.add_argument("--prec", default="f64", choices=["f64", "f32"])
    ap.add_argument("--recon", type=int, default=18, choices=[18, 12])
    ap.add_argument("--no-rows", action="store_true", help="skip the per-row extras (rank 0, N=1)")
    ap.add_argument("--rows", default="main,config2,config3,config4,config5b",
                    help="which groups of rows to measure: main (the other rows on the timed lattice), config2, config3, "
                         "config4, config5b")
    ap.add_argument("--decompose", action="store_true",
                    help="NEXT-3 (opt-in, not the driver's mode): ONE lattice cut into --gpus time slabs, half-spinor "
                         "faces exchanged between ring neighbours (NCCL); strong scaling")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--kappa", type=float, default=0.137)
    ap.add_argument("--csw", type=float, default=1.9)
    return ap.parse_args()


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            d = json.load(open(p))
            return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, torch copy)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons of one GPU with NVML while the timed region runs."""

    def __init__(self, index, period=0.01):
        threading.Thread.__init__(self, daemon=True)
        self.index, self.period = index, period
        self.stop_flag = threading.Event()
        self.sm, self.reasons, self.sm_max, self.err = [], set(), None, None

    def run(self):
        try:
            import pynvml as N
            N.nvmlInit()
            h = N.nvmlDeviceGetHandleByIndex(self.index)
            self.sm_max = int(N.nvmlDeviceGetMaxClockInfo(h, N.NVML_CLOCK_SM))
            names = {
                getattr(N, "nvmlClocksEventReasonGpuIdle", 0x1): "gpu_idle",
                getattr(N, "nvmlClocksEventReasonApplicationsClocksSetting", 0x2): "applications_clocks_setting",
                getattr(N, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
                getattr(N, "nvmlClocksThrottleReasonHwSlowdown", 0x8): "hw_slowdown",
                getattr(N, "nvmlClocksEventReasonSyncBoost", 0x10): "sync_boost",
                getattr(N, "nvmlClocksEventReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
                getattr(N, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
                getattr(N, "nvmlClocksThrottleReasonHwPowerBrakeSlowdown", 0x80): "hw_power_brake_slowdown",
            }
            while not self.stop_flag.is_set():
                self.sm.append(int(N.nvmlDeviceGetClockInfo(h, N.NVML_CLOCK_SM)))
                try:
                    r = int(N.nvmlDeviceGetCurrentClocksEventReasons(h))
                except Exception:
                    r = int(N.nvmlDeviceGetCurrentClocksThrottleReasons(h))
                for bit, name in names.items():
                    if r & bit and name != "gpu_idle":
                        self.reasons.add(name)
                time.sleep(self.period)
        except Exception as e:  # NVML missing: report, do not invent numbers
            self.err = repr(e)

    def result(self):
        self.stop_flag.set()
        self.join(timeout=2.0)
        sm = sorted(self.sm)
        out = {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": self.sm_max, "reasons": sorted(self.reasons),
               "samples": len(sm)}
        if self.err:
            out["error"] = self.err
        return out


# ------------------------------------------------------------------------------------------------------
# our arm
# ------------------------------------------------------------------------------------------------------
def dist_env():
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return rank, world, local


def max_over_ranks(torch, dist, ms_local, device):
    """Replicas share nothing but the clock: the step time of the job is the slowest rank's."""
    if dist is None:
        return ms_local
    t = torch.tensor([ms_local], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_gflops(world, flops_step_per_rank, ms_per_step):
    """value = work of all ranks / time of the slowest (weak scaling: every replica does the same work)."""
    return world * flops_step_per_rank / (ms_per_step * 1e-3) / 1e9


def time_calls(torch, fn, reps, warm=2):
    """Average milliseconds of fn() over `reps` back-to-back calls (CUDA events on the current stream)."""
    for _ in range(warm):
        fn()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        fn()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / reps


class Setup:
    """Synthetic gauge field + clover term + spinors of one lattice, resident in HBM in the internal layout."""

    def __init__(self, torch, B, synth, L, bc, theta, phiT, kappa, csw, seed_cfg, rank, precs, recons, inverse=False,
                 sf=False, keep_canon=False):
        self.torch, self.B, self.L, self.kappa, self.csw = torch, B, tuple(L), kappa, csw
        self.V = synth.vol(L)
        dev = torch.device("cuda", torch.cuda.current_device())
        self.g = B.geom_create(L, bc, theta, synth.SF_PHI0 if sf else None, phiT, device=dev.index)
        self.theta_is_zero = bc == B.BC_PERIODIC and (theta is None or not any(theta))
        Uc = synth.smooth_gauge_torch(L, synth.seed_for(seed_cfg, 0) + 100 * rank, dev)
        if sf:
            n0 = L[0] * L[1] * L[2]
            for mu in range(3):
                Uc[:n0, mu] = torch.from_numpy(synth.sf_boundary_links(L, synth.SF_PHI0, mu)).to(dev)
        psic = synth.gaussian_spinor_torch(L, synth.seed_for(seed_cfg, 1) + 100 * rank, dev)
        self.U, self.A, self.Ainv, self.psi, self.out = {}, {}, {}, {}, {}
        for recon in recons:
            for prec in sorted(set(precs) | {B.F64}):
                buf = B.alloc_field(self.g, B.FIELD_GAUGE, prec, recon)
                B.gauge_import(self.g, Uc, buf, prec, recon)
                self.U[(prec, recon)] = buf
        r0 = recons[0]
        for prec in precs:
            A = B.alloc_field(self.g, B.FIELD_CLOVER, prec)
            Ai = B.alloc_field(self.g, B.FIELD_CLOVER, prec) if inverse else None
            self.clover_ms = time_calls(
                torch, lambda: B.clover_build(self.g, kappa, csw, self.U[(B.F64, r0)], A, Ai, r0, prec), 1, 1)
            self.A[prec], self.Ainv[prec] = A, Ai
            self.psi[prec] = B.alloc_field(self.g, B.FIELD_SPINOR, prec)
            self.out[prec] = B.alloc_field(self.g, B.FIELD_SPINOR, prec)
            B.spinor_import(self.g, psic, self.psi[prec], prec)
        torch.cuda.synchronize()
        self.canon = (Uc, psic) if keep_canon else None

    def close(self):
        self.B.geom_destroy(self.g)


def run_ours(args):
    import numpy as np
    import torch

    from paper_2503_16994_b200 import binding as B
    from paper_2503_16994_b200 import synth

    rank, world, local = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; this library has no CPU fallback")
    B.lib()  # fails loudly if the extension is missing
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    L = tuple(int(v) for v in args.lattice.lower().split("x"))
    prec = B.F64 if args.prec == "f64" else B.F32
    recon = args.recon
    rb = 8 if prec == B.F64 else 4
    want_e2e = not args.no_e2e
    S = Setup(torch, B, synth, L, B.BC_PERIODIC, None, None, args.kappa, args.csw, 5, rank, [prec], [recon],
              keep_canon=True)
    V = S.V
    U, A, psi, out = S.U[(prec, recon)], S.A[prec], S.psi[prec], S.out[prec]
    out2 = B.alloc_field(S.g, B.FIELD_SPINOR, prec)

    def step():
        B.dw_apply(S.g, args.kappa, U, A, psi, out, prec, recon)
        B.dwdag_apply(S.g, args.kappa, U, A, out, out2, prec, recon)

    def barrier():
        if dist is not None:
            dist.barrier()

    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.05)
    l0 = B.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    torch.cuda.synchronize()
    launches = B.launch_count() - l0
    ms_local = e0.elapsed_time(e1)
    clocks = sampler.result()
    barrier()
    # SURVEY.md 8(d) "Timing": the same K-step batch five more times, median and min reported beside the headline
    # (which stays the first batch, the one the clock sampler and the launch counter bracket)
    reps = []
    for _ in range(5):
        r0, r1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        r0.record()
        for _ in range(args.steps):
            step()
        r1.record()
        torch.cuda.synchronize()
        reps.append(r0.elapsed_time(r1) / args.steps)
    reps_sorted = sorted(reps)
    ms = max_over_ranks(torch, dist, ms_local, "cuda")
    ms_per_step = ms / args.steps
    flops_step = 2.0 * FLOP_DW * V
    value = whole_job_gflops(world, flops_step, ms_per_step)  # GFLOP/s, whole job

    # roofline of the dominant kernel (the stencil), from this rank's own launches in the timed region
    peak, peak_src = measured_peaks()
    bytes_launch = REALS_DW[recon] * rb * V
    ms_launch = ms_local / launches
    achieved = bytes_launch / (ms_launch * 1e-3) / 1e9
    plan = B.dw_plan(S.g, prec, recon, True)
    roofline = {"bound": "hbm", "kernel": plan.split("<")[0], "launch": plan, "achieved": round(achieved, 1), "peak": peak,
                "unit": "GB/s",
                "frac": round(achieved / peak, 4), "peak_source": peak_src,
                "frac_of_nominal_8TBs": round(achieved / NOMINAL_HBM_GBS, 4),
                "bytes_per_launch": bytes_launch, "ms_per_launch": round(ms_launch, 4),
                "model": "%d reals/site compulsory (links + psi in + psi out + clover), each datum once" % REALS_DW[recon],
                "repeats_ms_per_step": {"batches": [round(r, 4) for r in reps], "median": round(reps_sorted[2], 4),
                                        "min": round(reps_sorted[0], 4)}}
    roofline.update(ncu_traffic(args.lattice, args.prec, recon, plan))

    # e2e: same metric through the host-buffer C-ABI call, H2D and D2H inside the timed region
    e2e = None
    if want_e2e:
        e2e = run_e2e(torch, B, S, args, L, prec, recon, dist)
        B.host_cache_release()   # the host path keeps ~19 GB of device scratch between calls; the rows below need it
    result = {
        "metric": "Dw GFLOP/s (clover Wilson-Dirac, 1872 flop/site/application)", "value": round(value, 1),
        "unit": "GFLOP/s", "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": round(ms_per_step, 4), "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": args.prec, "data": "synthetic",
        "config": {"workload": "Dw^+Dw application, %s periodic SU(3), smooth links plaq~0.6, kappa=%g csw=%g, recon=%d"
                               % (args.lattice, args.kappa, args.csw, recon),
                   "step": "1 lqcd_dw_apply + 1 lqcd_dwdag_apply on a fixed Gaussian spinor",
                   "l2": "inputs larger than L2 (%.1f GB compulsory per application), no flush" % (bytes_launch / 1e9),
                   "parallelism": "replicas x%d (no data-path collective)" % world},
        "gpu_launches": int(launches), "clocks": clocks, "roofline": roofline, "e2e": e2e,
    }
    if rank == 0 and world == 1:
        if not args.no_rows:
            result["rows"] = run_rows(torch, B, synth, S, args, prec, recon, peak)
        if not args.no_cpu:
            result["cpu_baseline"] = cpu_baseline(np, torch, S, args)
    S.close()
    if rank == 0:
        print(json.dumps(result))
    if dist is not None:
        dist.destroy_process_group()


# dram__bytes_read.sum + dram__bytes_write.sum per launch of the stencil kernel, copied from the committed ncu --set full
# capture named beside it; keyed by (lattice, prec, recon).  A capture belongs to one kernel configuration: `plan` is
# the launch description (lqcd_dw_plan) the capture was taken with, and the number is dropped (null) when the
# running library describes its launch differently, i.e. when the kernel or its tiling changed since the capture.
NCU_TRAFFIC = {
    ("48x48x48x96", "f64", 18): {
        "bytes": 15704554000 + 2025777000,
        "capture": "profiles/r02_dw_pipe_kernel_f64_full.txt",
        "plan": "dw_pipe_kernel<double,18,1> grid=148 threads=384 smem=227696 ring_slots=3 halo_buffers=2 tile=4x4x4x4 sweep=1 chunk=3x3"},
    ("48x48x48x96", "f32", 18): {
        "bytes": 8046250000 + 1008283000,
        "capture": "profiles/r02_dw_pipe_kernel_f32_full.txt",
        "plan": "dw_pipe_kernel<float,18,1> grid=148 threads=384 smem=190832 ring_slots=4 halo_buffers=4 tile=4x4x4x4 sweep=1 chunk=3x3"},
}


def ncu_traffic(lattice, prec, recon, plan):
    e = NCU_TRAFFIC.get((lattice, prec, recon))
    if e is None:
        return {"traffic": None, "traffic_source": "no ncu capture for this configuration"}
    if e["plan"] != plan:
        return {"traffic": None, "traffic_source": "stale: %s was captured with launch '%s'" % (e["capture"], e["plan"])}
    return {"traffic": e["bytes"], "traffic_source": e["capture"]}


def run_e2e(torch, B, S, args, L, prec, recon, dist):
    """lqcd_dw_apply_host: canonical HOST buffers in, canonical HOST buffer out; every call copies the gauge
    field and the spinor to the device, converts the layout, builds the clover term, applies Dw, converts back
    and copies the result to the host.  Pinned host memory; wall clock around the (synchronous) call."""
    Uc, psic = S.canon
    V = S.V
    hU = torch.empty(Uc.shape, dtype=Uc.dtype, pin_memory=True)
    hpsi = torch.empty(psic.shape, dtype=psic.dtype, pin_memory=True)
    hout = torch.empty(psic.shape, dtype=psic.dtype, pin_memory=True)
    hU.copy_(Uc)
    hpsi.copy_(psic)
    torch.cuda.synchronize()
    S.canon = None
    del Uc, psic
    torch.cuda.empty_cache()
    n = max(1, min(args.steps, 3))

    def call():
        B.dw_apply_host(L, args.kappa, args.csw, hU, hpsi, hout, prec=prec, recon=recon,
                        device=torch.cuda.current_device())

    call()  # warm-up (first-touch of the driver's staging paths)
    if dist is not None:
        dist.barrier()
    t0 = time.perf_counter()
    for _ in range(n):
        call()
    dt = (time.perf_counter() - t0) / n
    world = 1
    if dist is not None:
        t = torch.tensor([dt], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dt = float(t.item())
        world = dist.get_world_size()
    h2d = int(hU.numel() * 16 + hpsi.numel() * 16)
    d2h = int(hout.numel() * 16)
    return {"value": round(world * FLOP_DW * V / dt / 1e9, 2), "unit": "GFLOP/s", "h2d_bytes_per_step": h2d,
            "d2h_bytes_per_step": d2h, "ms_per_step": round(dt * 1e3, 2), "steps": n,
            "api": "lqcd_dw_apply_host (one Dw application per call: H2D gauge+spinor, layout import, Csw!, Dw, export, D2H)",
            "checksum": float(hout.real.abs().sum().item()) if V <= (1 << 22) else None}


def run_rows(torch, B, synth, S, args, prec, recon, peak):
    """The other hot-path rows measured once each, same process, rank 0, N = 1."""
    rows = {}
    V, L, g, kappa = S.V, S.L, S.g, args.kappa
    groups = set(args.rows.split(","))
    if "main" not in groups:
        for name, fn in (("config2", run_config2), ("config3", run_config3), ("config4", run_config4), ("config5b", run_config5b)):
            if name in groups:
                rows.update(fn(torch, B, synth, peak))
        return rows

    def gbs(reals, rbytes, ms, sites=V):
        return round(reals * rbytes * sites / (ms * 1e-3) / 1e9, 1)

    rows["a3_clover_build"] = {"ms": round(S.clover_ms, 3), "lattice": args.lattice,
                               "GB/s_model": gbs(144, 8, S.clover_ms),
                               "model": "read 72 link reals + write 72 clover reals per site, fp64"}
    # a4: Dw in every precision / link format
    dw = {}
    for p, pname, rb in ((B.F64, "f64", 8), (B.F32, "f32", 4)):
        if p not in S.A:
            A = B.alloc_field(g, B.FIELD_CLOVER, p)
            B.clover_build(g, kappa, args.csw, S.U[(B.F64, recon)], A, None, recon, p)
            S.A[p] = A
            S.psi[p] = B.alloc_field(g, B.FIELD_SPINOR, p)
            S.out[p] = B.alloc_field(g, B.FIELD_SPINOR, p)
            if p == B.F32:
                B.field_to_f32(g, B.FIELD_SPINOR, recon, S.psi[B.F64], S.psi[p])
        for r in (18, 12):
            if (p, r) not in S.U:
                if (B.F64, r) not in S.U:
                    # derive the 12-real field from the 18-real one through the canonical layout
                    canon = torch.empty((V, 4, 3, 3), dtype=torch.complex128, device="cuda")
                    B.gauge_export(g, S.U[(B.F64, recon)], canon, B.F64, recon)
                    S.U[(B.F64, r)] = B.alloc_field(g, B.FIELD_GAUGE, B.F64, r)
                    B.gauge_import(g, canon, S.U[(B.F64, r)], B.F64, r)
                    del canon
                if p == B.F32:
                    S.U[(p, r)] = B.alloc_field(g, B.FIELD_GAUGE, p, r)
                    B.field_to_f32(g, B.FIELD_GAUGE, r, S.U[(B.F64, r)], S.U[(p, r)])
            for dag, fn in (("dw", B.dw_apply), ("dwdag", B.dwdag_apply)):
                ms = time_calls(torch, lambda: fn(g, kappa, S.U[(p, r)], S.A[p], S.psi[p], S.out[p], p, r), 10)
                dw["%s_%s_recon%d" % (dag, pname, r)] = {
                    "ms": round(ms, 4), "GFLOP/s": round(FLOP_DW * V / ms / 1e6, 1), "GB/s": gbs(REALS_DW[r], rb, ms),
                    "frac_measured_peak": round(gbs(REALS_DW[r], rb, ms) / peak, 4)}
    rows["a4_dw"] = dw
    # NEXT-1: 12 right-hand sides in one pass (links and clover blocks from HBM once per tile)
    nrhs = 12
    fb = B.field_bytes(g, B.FIELD_SPINOR, B.F64)
    src = torch.empty(nrhs * fb, dtype=torch.uint8, device="cuda")
    dst = torch.empty_like(src)
    for n in range(nrhs):
        src[n * fb:(n + 1) * fb].copy_(S.psi[B.F64])
    ms = time_calls(torch, lambda: B.dw_apply_multi(g, kappa, S.U[(B.F64, recon)], S.A[B.F64], src, dst, nrhs, B.F64, recon), 3)
    reals_multi = (REALS_DW[recon] - 48) + 48 * nrhs
    rows["next1_dw_multi_12rhs_f64"] = {
        "ms": round(ms, 3), "ms_per_rhs": round(ms / nrhs, 4), "GFLOP/s": round(nrhs * FLOP_DW * V / ms / 1e6, 1),
        "GB/s_model": gbs(reals_multi, 8, ms), "model": "%d reals/site for 12 columns (links + clover once)" % reals_multi,
        "vs_single_application": round(ms / nrhs / dw["dw_f64_recon%d" % recon]["ms"], 3),
        "note": "a tile's 12 columns are shared out over 4 work units drawn one after the other (3 columns each), so its "
                "links and clover blocks come from HBM about once; what is left is the arithmetic warps' time per tile "
                "with every operand in L2 (8.5 us against 10.4 us from HBM, profiles/r02_notes.md section 11)"}
    # NEXT-2: pseudoscalar two-point function of 12 columns (a pure reduction: 12 x 24 reals per site read once)
    wsc = B.alloc_field(g, B.FIELD_WORKSPACE)
    ms = time_calls(torch, lambda: B.correlator_ps(g, src, nrhs, wsc, L[3]), 3)
    rows["next2_correlator_ps_12cols_f64"] = {"ms": round(ms, 3), "GB/s": gbs(24 * nrhs, 8, ms),
                                              "frac_measured_peak": round(gbs(24 * nrhs, 8, ms) / peak, 4),
                                              "note": "a pure read stream: the peak it is divided by was measured with a "
                                                      "copy (reads + writes), which a read-only kernel can exceed"}
    del src, dst, wsc
    # NEXT-3: the same lattice as ONE time slab -- pack, face exchange with itself (the periodic
    # wrap) on a side stream, stencil without the two face hops, face kernel.  What a rank of a decomposed lattice
    # runs per application; the difference to a4 is the whole cost of the decomposition on the GPU side.
    if S.theta_is_zero:
        from paper_2503_16994_b200 import slab
        gs = slab.slab_geom_create(L, 1, None, device=torch.cuda.current_device())
        D = slab.SlabDirac(gs, kappa, S.U[(B.F64, recon)], S.A[B.F64], B.F64, recon)
        ms = time_calls(torch, lambda: D.apply(S.psi[B.F64], S.out[B.F64]), 10)
        ms0 = dw["dw_f64_recon%d" % recon]["ms"]
        rows["next3_slab_dw_f64_world1"] = {
            "ms": round(ms, 4), "GFLOP/s": round(FLOP_DW * V / ms / 1e6, 1), "GB/s": gbs(REALS_DW[recon], 8, ms),
            "overhead_vs_a4": round(ms / ms0 - 1.0, 4), "face_bytes_per_application": 2 * B.field_bytes(gs, B.FIELD_FACE, B.F64),
            "note": "lqcd_dw_slab_pack + self-exchange + lqcd_dw_apply (BC_SLAB) + lqcd_dw_slab_faces"}
        del D
        B.geom_destroy(gs)
    # a6: BLAS-1 reduction alone (|v|^2 over one spinor)
    ws = B.alloc_field(g, B.FIELD_WORKSPACE)
    ms = time_calls(torch, lambda: B.spinor_norm2(g, S.psi[B.F64], ws), 10)
    rows["a6_norm2_f64"] = {"ms": round(ms, 4), "GB/s": gbs(24, 8, ms), "frac_measured_peak": round(gbs(24, 8, ms) / peak, 4)}
    # a7: CG iteration rate on the bench lattice (fixed iteration counts; the difference removes set-up cost)
    b, x = S.psi[B.F64], S.out[B.F64]
    t = {}
    for n in (10, 40):
        info = B.cg_solve(g, kappa, S.U[(B.F64, recon)], S.A[B.F64], b, x, ws, tol=1e-30, maxiter=n, check_every=n,
                          recon=recon, raise_on_notconv=False)
        t[n] = info["seconds"]
    ms_it = (t[40] - t[10]) / 30 * 1e3
    rows["a7_cg_iteration_f64"] = {"ms_per_iteration": round(ms_it, 4), "lattice": args.lattice,
                                   "GB/s_model": gbs(REALS_CG_ITER[recon], 8, ms_it),
                                   "frac_measured_peak": round(gbs(REALS_CG_ITER[recon], 8, ms_it) / peak, 4),
                                   "model": "%d reals/site/iteration (fused plan, SURVEY.md 8(d))" % REALS_CG_ITER[recon]}
    if S.theta_is_zero:   # NEXT-3: the slab solver's iteration (unfused BLAS-1, two all-reduces) on one slab
        from paper_2503_16994_b200 import slab
        gs = slab.slab_geom_create(L, 1, None, device=torch.cuda.current_device())
        comm = slab.SlabCommunicator(gs)
        for n in (10, 40):
            info = slab.cg_solve_slab(gs, kappa, S.U[(B.F64, recon)], S.A[B.F64], b, x, ws, comm, tol=1e-30, maxiter=n,
                                      check_every=n, recon=recon, raise_on_notconv=False)
            t[n] = info["seconds"]
        ms_sl = (t[40] - t[10]) / 30 * 1e3
        rows["next3_slab_cg_iteration_f64_world1"] = {
            "ms_per_iteration": round(ms_sl, 4), "vs_a7": round(ms_sl / ms_it, 4),
            "note": "lqcd_cg_solve_slab: pack / exchange / stencil / faces per operator, r -= alpha q and |r|^2 in a "
                    "separate pass, scalars through the all-reduce callback"}
        del comm
        B.geom_destroy(gs)
    del ws
    torch.cuda.empty_cache()
    if "main" in groups:
        rows.update(run_su2(torch, B, synth, peak, L))
    for name, fn in (("config2", run_config2), ("config3", run_config3), ("config4", run_config4), ("config5b", run_config5b)):
        if name in groups:
            rows.update(fn(torch, B, synth, peak))
    return rows


def run_su2(torch, B, synth, peak, L):
    """NEXT-4: the SU(2) fundamental representation on the bench lattice -- Dw in fp64 and
    fp32 (one-thread-per-site kernel).  Compulsory bytes per site: 16 link reals (Cayley-Dickson pairs) + 16 psi in +
    16 out + 32 clover = 80 reals; flops: hopping 624 + block multiply 208 + combine 32 = 864 per site."""
    import numpy as np
    kappa, csw = 0.137, 1.9
    V = synth.vol(L)
    g = B.geom_create(L)
    Uc = torch.from_numpy(synth.su2_matrices(synth.smooth_su2_cd(L, synth.seed_for(5, 20)))).cuda()
    U64 = B.su2_alloc_field(g, B.FIELD_GAUGE)
    B.su2_gauge_import(g, Uc, U64)
    U32 = B.su2_alloc_field(g, B.FIELD_GAUGE, B.F32)
    B.su2_gauge_import(g, Uc, U32, B.F32)
    del Uc
    psic = torch.view_as_complex(torch.randn((V, 4, 2, 2), dtype=torch.float64, device="cuda",
                                             generator=torch.Generator(device="cuda").manual_seed(synth.seed_for(5, 21))))
    out = {}
    for p, pname, rb, U in ((B.F64, "f64", 8, U64), (B.F32, "f32", 4, U32)):
        A = B.su2_alloc_field(g, B.FIELD_CLOVER, p)
        B.su2_clover_build(g, kappa, csw, U64, A, p)
        src, dst = B.su2_alloc_field(g, B.FIELD_SPINOR, p), B.su2_alloc_field(g, B.FIELD_SPINOR, p)
        B.su2_spinor_import(g, psic, src, p)
        ms = time_calls(torch, lambda: B.su2_dw_apply(g, kappa, U, A, src, dst, False, p), 10)
        gb = 80 * rb * V / (ms * 1e-3) / 1e9
        out["next4_su2_dw_%s" % pname] = {"ms": round(ms, 4), "GFLOP/s": round(864 * V / ms / 1e6, 1), "GB/s": round(gb, 1),
                                          "frac_measured_peak": round(gb / peak, 4), "lattice": "x".join(str(v) for v in L),
                                          "model": "80 reals/site compulsory, 864 flop/site"}
        del A, src, dst
    B.geom_destroy(g)
    torch.cuda.empty_cache()
    return out


def run_config2(torch, B, synth, peak):
    """configs[1]: 16^3 x 32 periodic, kappa = 0.135, csw = 1.7: 10 warm-up + 1000 applications of Dw to a fixed input,
    fp64 and fp32.  The working set (192 / 96 MB) is about the size of L2, so this is not an HBM-roofline point."""
    L, kappa, csw = (16, 16, 16, 32), 0.135, 1.7
    S = Setup(torch, B, synth, L, B.BC_PERIODIC, None, None, kappa, csw, 2, 0, [B.F64, B.F32], [18])
    g, V = S.g, S.V
    U32 = B.alloc_field(g, B.FIELD_GAUGE, B.F32, 18)
    B.field_to_f32(g, B.FIELD_GAUGE, 18, S.U[(B.F64, 18)], U32)
    S.U[(B.F32, 18)] = U32
    out = {}
    for p, pname, rb in ((B.F64, "f64", 8), (B.F32, "f32", 4)):
        ms = time_calls(torch, lambda: B.dw_apply(g, kappa, S.U[(p, 18)], S.A[p], S.psi[p], S.out[p], p, 18), 1000, 10)
        gb = REALS_DW[18] * rb * V / (ms * 1e-3) / 1e9
        out["a4_dw_16x16x16x32_%s_1000_applications" % pname] = {
            "ms": round(ms, 5), "GFLOP/s": round(FLOP_DW * V / ms / 1e6, 1), "GB/s_model": round(gb, 1),
            "note": "working set ~ L2 (%d MB): not an HBM roofline point" % (REALS_DW[18] * rb * V >> 20)}
    S.close()
    del S, U32
    torch.cuda.empty_cache()
    return out


def run_config5b(torch, B, synth, peak):
    """configs[4], second lattice: 64^3 x 128 periodic, kappa = 0.137, csw = 1.9: Dw in fp64 / fp32 with 18- and 12-real
    links as a fraction of the HBM roofline (51.5 / 25.8 GB compulsory per application: the largest single-GPU case)."""
    L, kappa, csw = (64, 64, 64, 128), 0.137, 1.9
    free, _ = torch.cuda.mem_get_info()
    if free < 130 * (1 << 30):
        return {"a4_dw_64x64x64x128": {"skipped": "needs ~110 GB of free device memory, %d GB free" % (free >> 30)}}
    S = Setup(torch, B, synth, L, B.BC_PERIODIC, None, None, kappa, csw, 5, 0, [B.F64, B.F32], [18])
    g, V = S.g, S.V
    out = {"lattice": "64x64x64x128", "clover_build_ms": round(S.clover_ms, 3)}
    for r in (18, 12):
        if r == 12:
            canon = torch.empty((V, 4, 3, 3), dtype=torch.complex128, device="cuda")
            B.gauge_export(g, S.U[(B.F64, 18)], canon, B.F64, 18)
            S.U[(B.F64, 12)] = B.alloc_field(g, B.FIELD_GAUGE, B.F64, 12)
            B.gauge_import(g, canon, S.U[(B.F64, 12)], B.F64, 12)
            del canon
            del S.U[(B.F64, 18)], S.U[(B.F32, 18)]
            torch.cuda.empty_cache()
        if (B.F32, r) not in S.U:
            S.U[(B.F32, r)] = B.alloc_field(g, B.FIELD_GAUGE, B.F32, r)
            B.field_to_f32(g, B.FIELD_GAUGE, r, S.U[(B.F64, r)], S.U[(B.F32, r)])
        for p, pname, rb in ((B.F64, "f64", 8), (B.F32, "f32", 4)):
            for dag, fn in (("dw", B.dw_apply), ("dwdag", B.dwdag_apply)):
                ms = time_calls(torch, lambda: fn(g, kappa, S.U[(p, r)], S.A[p], S.psi[p], S.out[p], p, r), 5, 2)
                gb = REALS_DW[r] * rb * V / (ms * 1e-3) / 1e9
                out["%s_%s_recon%d" % (dag, pname, r)] = {
                    "ms": round(ms, 4), "GFLOP/s": round(FLOP_DW * V / ms / 1e6, 1), "GB/s": round(gb, 1),
                    "frac_measured_peak": round(gb / peak, 4)}
    out["kernel"] = B.dw_plan(g, B.F64, 18, True)
    S.close()
    del S
    torch.cuda.empty_cache()
    return {"a4_dw_64x64x64x128": out}


def run_config3(torch, B, synth, peak):
    """configs[2]: 24^3 x 48, open BC, 12 point-source columns to 1e-10, fp64 (time-to-solution)."""
    L, kappa, csw = (24, 24, 24, 48), 0.1365, 1.9
    S = Setup(torch, B, synth, L, B.BC_OPEN, None, None, kappa, csw, 3, 0, [B.F64, B.F32], [18], inverse=True)
    g = S.g
    U32 = B.alloc_field(g, B.FIELD_GAUGE, B.F32, 18)
    B.field_to_f32(g, B.FIELD_GAUGE, 18, S.U[(B.F64, 18)], U32)
    ws = B.alloc_field(g, B.FIELD_WORKSPACE)
    cols = torch.empty(12 * B.field_bytes(g, B.FIELD_SPINOR), dtype=torch.uint8, device="cuda")
    y = (0, 0, 0, L[3] // 2)   # R12: slice 0 is frozen under open BC
    out = {}
    for name, kw in (("plain_f64", {}),
                     # inner_tol 1e-2: on this ill-conditioned lattice an fp32 inner solve of ~1500 iterations ends with a
                     # recursive residual far below its true one, and asking it for 1e-4 sometimes buys a second such
                     # solve that makes no progress (DESIGN.md section 7 "Mixed precision")
                     ("eo_mixed", dict(eo=True, mixed=True, inner_tol=1e-2, clover_inv64=S.Ainv[B.F64], U32=U32,
                                       clover32=S.A[B.F32], clover_inv32=S.Ainv[B.F32]))):
        t0 = time.perf_counter()
        infos = B.propagator(g, kappa, S.U[(B.F64, 18)], S.A[B.F64], y, cols, ws, tol=1e-10, maxiter=10000, **kw)
        dt = time.perf_counter() - t0
        out["a8_propagator_24x24x24x48_open_" + name] = {
            "seconds_12_columns": round(dt, 3), "iterations": [i["iters"] for i in infos],
            "outer": [i["outer"] for i in infos],
            "max_rel_resid_normal": max(i["rel_resid_normal"] for i in infos),
            "max_rel_resid_true": max(i["rel_resid_true"] for i in infos)}
    # the same 12 columns solved in lock step (lqcd_propagator_batched: every stencil pass takes all columns)
    wsb = torch.empty(B.cg_multi_workspace_bytes(g, 12), dtype=torch.uint8, device="cuda")
    srcs = torch.empty_like(cols)
    t0 = time.perf_counter()
    infos = B.propagator_batched(g, kappa, S.U[(B.F64, 18)], S.A[B.F64], y, cols, srcs, wsb, tol=1e-10, maxiter=10000)
    dt = time.perf_counter() - t0
    one = out["a8_propagator_24x24x24x48_open_plain_f64"]
    out["a8_propagator_24x24x24x48_open_plain_f64_batched"] = {
        "seconds_12_columns": round(dt, 3), "iterations": [i["iters"] for i in infos],
        "vs_column_by_column": round(dt / one["seconds_12_columns"], 3),
        "same_iteration_counts": [i["iters"] for i in infos] == one["iterations"],
        "max_rel_resid_normal": max(i["rel_resid_normal"] for i in infos),
        "max_rel_resid_true": max(i["rel_resid_true"] for i in infos)}
    del wsb, srcs
    S.close()
    del S, cols, ws, U32
    torch.cuda.empty_cache()
    return out


def run_config4(torch, B, synth, peak):
    """configs[3]: 32^3 x 64, SF BC, theta = 0.5 spatial: even-odd operator throughput fp64 vs fp32, mixed CG."""
    L, kappa, csw = (32, 32, 32, 64), 0.1355, 1.8
    theta = (0.5, 0.5, 0.5, 0.0)
    S = Setup(torch, B, synth, L, B.BC_SF_ORBI, theta, synth.SF_PHIT, kappa, csw, 4, 0, [B.F64, B.F32], [18],
              inverse=True, sf=True)
    g, V = S.g, S.V
    U32 = B.alloc_field(g, B.FIELD_GAUGE, B.F32, 18)
    B.field_to_f32(g, B.FIELD_GAUGE, 18, S.U[(B.F64, 18)], U32)
    S.U[(B.F32, 18)] = U32
    out = {}
    for p, pname, rb in ((B.F64, "f64", 8), (B.F32, "f32", 4)):
        tmp = B.alloc_field(g, B.FIELD_SPINOR, p)
        ms = time_calls(torch, lambda: B.dw_eo_apply(g, kappa, S.U[(p, 18)], S.A[p], S.Ainv[p], S.psi[p], S.out[p], tmp,
                                                     False, p, 18), 20)
        gb = REALS_DHAT[18] * rb * V / (ms * 1e-3) / 1e9
        out["a5_dhat_32x32x32x64_sf_" + pname] = {"ms": round(ms, 4), "GFLOP/s": round(FLOP_DHAT * V / ms / 1e6, 1),
                                                  "GB/s": round(gb, 1), "frac_measured_peak": round(gb / peak, 4)}
    ws = B.alloc_field(g, B.FIELD_WORKSPACE)
    y = (0, 0, 0, L[3] // 2)
    b = B.alloc_field(g, B.FIELD_SPINOR)
    x = B.alloc_field(g, B.FIELD_SPINOR)
    B.point_source(g, y, 0, 0, b)
    for name, kw in (("eo_f64", dict(eo=True)), ("eo_mixed", dict(eo=True, mixed=True))):
        info = B.cg_solve(g, kappa, S.U[(B.F64, 18)], S.A[B.F64], b, x, ws, tol=1e-10, maxiter=10000,
                          clover_inv64=S.Ainv[B.F64], U32=U32, clover32=S.A[B.F32], clover_inv32=S.Ainv[B.F32], **kw)
        out["a7_cg_32x32x32x64_sf_" + name] = {k: info[k] for k in ("iters", "outer", "seconds", "rel_resid_normal", "rel_resid_true")}
    S.close()
    return out


# ------------------------------------------------------------------------------------------------------
# the oracle on the host cores: cpu_baseline leg and the --impl reference arm
# ------------------------------------------------------------------------------------------------------
SAMPLE_L = (16, 16, 16, 32)


def oracle_sample_inputs(np, synth, args, U_canon_dev=None, psi_canon_dev=None, L_full=None):
    """A 16^3 x 32 periodic sample of the bench workload.  Links of the recipe are independent, so any
    sub-block of the bench field is a field of the same recipe; without a device field, draw one on the host."""
    L = SAMPLE_L
    if U_canon_dev is not None:
        Lf = L_full
        U4 = U_canon_dev.reshape(Lf[3], Lf[2], Lf[1], Lf[0], 4, 3, 3)[:L[3], :L[2], :L[1], :L[0]]
        p4 = psi_canon_dev.reshape(Lf[3], Lf[2], Lf[1], Lf[0], 4, 3)[:L[3], :L[2], :L[1], :L[0]]
        U = U4.contiguous().reshape(-1, 4, 3, 3).cpu().numpy()
        psi = p4.contiguous().reshape(-1, 4, 3).cpu().numpy()
    else:
        U = synth.smooth_gauge(L, synth.seed_for(5, 0))
        psi = synth.gaussian_spinor(L, synth.seed_for(5, 1))
    return L, U, psi


def time_oracle(np, oracle, L, U, psi, kappa, csw, budget_s, min_steps=1, max_steps=None, warm=1):
    """Time steps of (Dw, Dw^+) with the oracle as it stands; returns (GFLOP/s, steps, seconds, threads)."""
    V = int(np.prod(L))
    A = oracle.clover_blocks(L, U, kappa, csw)
    for _ in range(warm):
        oracle.dw(L, U, oracle.dw(L, U, psi, kappa, A), kappa, A, dagger=True)
    steps, t0 = 0, time.perf_counter()
    while True:
        oracle.dw(L, U, oracle.dw(L, U, psi, kappa, A), kappa, A, dagger=True)
        steps += 1
        dt = time.perf_counter() - t0
        if max_steps is not None and steps >= max_steps:
            break
        if max_steps is None and steps >= min_steps and dt >= budget_s:
            break
    return 2.0 * FLOP_DW * V * steps / dt / 1e9, steps, dt, oracle.num_threads()


def cpu_baseline(np, torch, S, args):
    import oracle
    from paper_2503_16994_b200 import synth

    if S.canon is not None:
        L, U, psi = oracle_sample_inputs(np, synth, args, S.canon[0], S.canon[1], S.L)
    else:
        L, U, psi = oracle_sample_inputs(np, synth, args)
    v, steps, dt, threads = time_oracle(np, oracle, L, U, psi, args.kappa, args.csw, budget_s=10.0)
    return {"value": round(v, 3), "unit": "GFLOP/s", "cores": threads, "kind": "oracle",
            "sample": "%d steps (Dw then Dw^+, fp64, clover blocks precomputed) on a %s periodic lattice of the bench "
                      "recipe (kappa=%g csw=%g), %.1f s" % (steps, "x".join(map(str, L)), args.kappa, args.csw, dt)}


def run_decomposed(args):
    """--decompose: the lattice of --lattice as WORLD_SIZE time slabs, one per GPU.
    A step = D then D^+ on the whole lattice: per rank pack -> face exchange (side stream) || slab stencil -> faces.
    Every rank draws its own slab of links (any stack of SU(3) slabs is a valid gauge field); the clover term sees the
    neighbours' slices through the real gauge-halo exchange.  Only the N = 1 case (the slab exchanging with itself)
    has been run: the boxes of this build have one GPU."""
    import torch

    from paper_2503_16994_b200 import binding as B
    from paper_2503_16994_b200 import slab, synth

    rank, world, local = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; this library has no CPU fallback")
    B.lib()
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    L = tuple(int(v) for v in args.lattice.lower().split("x"))
    prec = B.F64 if args.prec == "f64" else B.F32
    recon, rb = args.recon, (8 if args.prec == "f64" else 4)
    T = slab.slab_extent(L[3], world)
    Ls = (L[0], L[1], L[2], T)
    dev = torch.device("cuda", local)
    g = slab.slab_geom_create(L, world, None, device=local, rank=rank)
    Uc = synth.smooth_gauge_torch(Ls, synth.seed_for(5, 0) + 100 * rank, dev)
    xch = slab.FaceExchange()
    halo_lo, halo_hi = slab.gauge_halo_exchange(Uc, L, xch)
    U64 = B.alloc_field(g, B.FIELD_GAUGE, B.F64, recon)
    B.gauge_import(g, Uc, U64, B.F64, recon)
    A = B.alloc_field(g, B.FIELD_CLOVER, prec)
    B.clover_build_slab(g, args.kappa, args.csw, U64, halo_lo, halo_hi, A, None, recon, prec)
    U = U64
    if prec == B.F32:
        U = B.alloc_field(g, B.FIELD_GAUGE, B.F32, recon)
        B.field_to_f32(g, B.FIELD_GAUGE, recon, U64, U)
    psi, out, out2 = (B.alloc_field(g, B.FIELD_SPINOR, prec) for _ in range(3))
    B.spinor_import(g, synth.gaussian_spinor_torch(Ls, synth.seed_for(5, 1) + 100 * rank, dev), psi, prec)
    del Uc, halo_lo, halo_hi
    D = slab.SlabDirac(g, args.kappa, U, A, prec, recon, exchange=xch)

    def step():
        D.apply(psi, out, False)
        D.apply(out, out2, True)

    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.05)
    l0 = B.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    torch.cuda.synchronize()
    launches = B.launch_count() - l0
    ms_local = e0.elapsed_time(e1)
    clocks = sampler.result()
    if dist is not None:
        dist.barrier()
    ms = max_over_ranks(torch, dist, ms_local, "cuda") / args.steps
    Vs = synth.vol(Ls)
    peak, peak_src = measured_peaks()
    achieved = 2 * REALS_DW[recon] * rb * Vs / (ms_local / args.steps * 1e-3) / 1e9   # this rank's two stencil launches
    face = B.field_bytes(g, B.FIELD_FACE, prec)
    result = {
        "metric": "Dw GFLOP/s (clover Wilson-Dirac, 1872 flop/site/application)",
        "value": round(2.0 * FLOP_DW * synth.vol(L) / (ms * 1e-3) / 1e9, 1), "unit": "GFLOP/s", "n_gpus": world,
        "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": round(ms, 4), "higher_is_better": True,
        "scaling": "strong", "vs_baseline": None, "dtype": args.prec, "data": "synthetic",
        "config": {"workload": "Dw^+Dw application, %s periodic SU(3) as %d time slabs of %d slices, kappa=%g csw=%g, recon=%d"
                               % (args.lattice, world, T, args.kappa, args.csw, recon),
                   "step": "per rank: 2 x (lqcd_dw_slab_pack, face exchange, lqcd_dw_apply / lqcd_dwdag_apply, lqcd_dw_slab_faces)",
                   "l2": "inputs larger than L2, no flush", "parallelism": "time slabs x%d, half-spinor faces over NCCL" % world,
                   "face_bytes_per_application_per_rank": 2 * face},
        "gpu_launches": int(launches), "clocks": clocks,
        "roofline": {"bound": "hbm", "kernel": B.dw_plan(g, prec, recon, True).split("<")[0], "achieved": round(achieved, 1),
                     "peak": peak, "unit": "GB/s", "frac": round(achieved / peak, 4), "peak_source": peak_src,
                     "note": "whole step of this rank (pack + stencil + faces) against the stencil's compulsory bytes",
                     "traffic": None},
        "e2e": None,
    }
    B.geom_destroy(g)
    if rank == 0:
        print(json.dumps(result))
    if dist is not None:
        dist.destroy_process_group()


def run_reference(args):
    """--impl reference: there is no reference code (PAPER.md only); the arm is the fp64 oracle on the host cores."""
    rank, world, _ = dist_env()
    if rank != 0:
        return
    import numpy as np

    import oracle
    from paper_2503_16994_b200 import synth

    L, U, psi = oracle_sample_inputs(np, synth, args)
    V = int(np.prod(L))
    steps = max(1, args.steps)
    v, steps, dt, threads = time_oracle(np, oracle, L, U, psi, args.kappa, args.csw, budget_s=0.0, max_steps=steps,
                                        warm=max(1, min(args.warmup, 3)))
    sample = ("each step = Dw then Dw^+ (fp64, clover blocks precomputed) on a %s periodic sample of the bench recipe"
              % "x".join(map(str, L)))
    print(json.dumps({
        "impl": "reference", "metric": "Dw GFLOP/s (clover Wilson-Dirac, 1872 flop/site/application)",
        "value": round(v, 3), "unit": "GFLOP/s", "n_gpus": args.gpus, "steps": steps, "warmup": max(1, min(args.warmup, 3)),
        "ms_per_step": round(dt / steps * 1e3, 2), "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": "Dw^+Dw application, %s periodic SU(3), smooth links plaq~0.6, kappa=%g csw=%g, recon=18"
                               % (args.lattice, args.kappa, args.csw), "sample": sample},
        "cpu_baseline": {"value": round(v, 3), "unit": "GFLOP/s", "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": round(v, 3), "unit": "GFLOP/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.decompose:
        run_decomposed(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()

"""bench.py -- throughput of the DG-RHD hot path (one SSP-RK step = 3 fused stage launches) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload box3d|kh2d] [--impl reference]

Metric (BASELINE.json / PAPER.md:733-737 Eq. 108): DOF-updates/s per SSP-RK stage
    = DOF x stages x steps / seconds,  DOF = elements x (p+1)^d, fp64.
Default workload: BASELINE.json configs[4], the 3D periodic box 128^3, p=3, ideal EOS Gamma=5/3 (the
largest single-GPU configuration; configs[1] is a <=5120-DOF latency-bound convergence test).  One
"step" = one SSPRK3 step over the whole mesh = 1 dt kernel + 3 fused stage kernels (con2prim, flux,
volume + face + HLL + lift, RK combine, physicality operator, CFL reduction on the last stage).
Prints ONE JSON line (rank 0).  Multi-GPU: the path is single-GPU by north_star -> N independent
replicas ("replicas only"), value = sum of the replicas' DOF-updates / max time.
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

METRIC = "DOF-updates/s per SSP-RK stage"
UNIT = "DOF-updates/s"
STAGES = 3
# algorithmic HBM bytes per DOF and stage: U_s in, U_out out
# (80 B) + U0 in on stages 2 and 3 (40 B) -> (80 + 120 + 120) / 3
ALG_BYTES_PER_DOF_STAGE = (80.0 + 120.0 + 120.0) / 3.0
# fp64 work per DOF and stage of dg_stage_kernel<3,4,ideal>: executed 2*dfma + dmul + dadd from the
# ncu capture profiles/r1_ncu_summary.md, mean of the three stages (571 / 580 / 694)
FLOP_PER_DOF_STAGE = 615.1
# DRAM bytes per DOF and stage of the same capture (dram__bytes_read + write, mean of the 3 stages)
NCU_TRAFFIC_PER_DOF_STAGE = 185.7
# fp64 peak: 148 SMs x 64 DFMA/clk/SM (ncu: sm__sass_thread_inst_executed_op_dfma_pred_on peak_sustained)
# x 2 flop x SM clock
FP64_FMA_PER_CLK = 148 * 64


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--workload", default="box3d", choices=["box3d", "kh2d", "c2p"])
    ap.add_argument("--size", type=int, default=0, help="override elements per axis (debug)")
    ap.add_argument("--no-extra", action="store_true", help="skip con2prim / e2e / cpu legs")
    return ap.parse_args()


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """Samples SM clock and throttle reasons during the timed region (NVML, 20 ms period)."""

    def __init__(self, index):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def _run(self):
        nv = self.nv
        names = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "hw_thermal_slowdown": 0x40,
                 "sw_thermal_slowdown": 0x20, "hw_power_brake": 0x80, "sync_boost": 0x10}
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(0.02)

    def __enter__(self):
        if self.nv is not None:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()

    def summary(self):
        s = sorted(self.samples)
        return {"sm_mhz": (s[len(s) // 2] if s else None), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(s)}


def workload_cfg(name, size, device):
    """(cfg dict, W[5, ndof] primitives on `device`, workload label)."""
    from paper_2205_00095_b200 import inputs as I
    if name == "box3d":
        n = size or 128
        cfgd, W = I.box3d(0, n=n, p=3, kmax=8 if n >= 32 else 1, device=device)
        label = f"3D periodic box {n}^3 hex elements, p=3, ideal EOS Gamma=5/3, SSPRK3, CFL 0.3 (configs[4])"
    else:
        nx = size or 512
        cfgd, W = I.kh2d(0, nx=nx, ny=2 * nx, p=2, device=device)
        label = f"2D relativistic Kelvin-Helmholtz {nx}x{2 * nx} quad elements, p=2, Taub-Matthews, SSPRK3 (configs[3])"
    return cfgd, W, label


def cfg_args(cfgd):
    return (cfgd["ndim"], cfgd["nelem"], cfgd["xmin"], cfgd["xmax"], cfgd["bc"], cfgd["order_p"],
            cfgd["eos"], cfgd["gamma_ad"], cfgd["rk_stages"], cfgd["eps_q"], cfgd["delta_s"])


# ------------------------------------------------------------------------------------------------
# CPU legs (the oracle as it stands, on the host cores): cpu_baseline and --impl reference
# ------------------------------------------------------------------------------------------------
def oracle_sample(workload):
    """Bounded sample of the workload for the oracle: the same recipe on a smaller mesh."""
    import oracle as O
    n = 48 if workload == "box3d" else 256
    cfgd, W, _ = workload_cfg(workload, n, "cpu")
    U = O.prim2con_batch(cfgd["eos"], cfgd["gamma_ad"], W.numpy())
    ndof = U.shape[1]
    sample = (f"same recipe at {n}^3 elements (DOF {ndof}), 1 SSPRK3 step per timed step" if workload == "box3d"
              else f"same recipe at {n}x{2 * n} elements (DOF {ndof}), 1 SSPRK3 step per timed step")
    return O, O.make_config(*cfg_args(cfgd)), U, ndof, sample


def time_oracle(workload, steps, warmup):
    O, ocfg, U, ndof, sample = oracle_sample(workload)
    for _ in range(warmup):
        O.step(ocfg, U, -0.3, 1)
    t0 = time.perf_counter()
    for _ in range(steps):
        U, _, _ = O.step(ocfg, U, -0.3, 1)
    dt = time.perf_counter() - t0
    return ndof * STAGES * steps / dt, dt / steps, O.num_threads(), sample


def run_reference(a):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    val, sps, cores, sample = time_oracle(a.workload, a.steps, min(a.warmup, 1))
    label = ("3D periodic box 128^3 hex elements, p=3, ideal EOS Gamma=5/3, SSPRK3, CFL 0.3 (configs[4])"
             if a.workload == "box3d" else
             "2D relativistic Kelvin-Helmholtz 512x1024 quad elements, p=2, Taub-Matthews, SSPRK3 (configs[3])")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": a.gpus,
        "steps": a.steps, "warmup": min(a.warmup, 1), "ms_per_step": 1e3 * sps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": label, "sample": sample},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


# ------------------------------------------------------------------------------------------------
# CUDA leg
# ------------------------------------------------------------------------------------------------
def time_c2p(b, torch, eos, G, n):
    """con2prim states/s on configs[2]'s 2^26-state batch (device-resident), median of 5."""
    from paper_2205_00095_b200 import inputs as I
    W = I.c2p_states(0, n, device="cuda")
    U = b.dgrhd_prim2con_batch(eos, G, W)
    out = torch.empty_like(U)
    for _ in range(3):
        b.dgrhd_con2prim_batch(eos, G, U, out)
    ts = []
    for _ in range(5):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        b.dgrhd_con2prim_batch(eos, G, U, out)
        e1.record()
        e1.synchronize()
        ts.append(e0.elapsed_time(e1) * 1e-3)
    ts.sort()
    return n / ts[len(ts) // 2]


def max_over_ranks(secs, device):
    """Multi-GPU timing rule: the job's time is the slowest rank's device time."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([secs], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t)


def aggregate_value(world, ndof, steps, secs):
    """Whole-job DOF-updates/s: `world` independent replicas ("replicas only") over the max time."""
    return world * ndof * STAGES * steps / secs


def roofline_stage(workload, ndof, stage_s, clocks, hbm_peak, peak_src):
    """Roofline of the dominant kernel (the fused stage kernel).  The slower of the two resources
    bounds it: fp64 ALUs (flop / fp64 peak) or HBM (algorithmic bytes / measured copy bandwidth)."""
    ach_hbm = ALG_BYTES_PER_DOF_STAGE * ndof / stage_s / 1e9
    hbm = {"achieved": ach_hbm, "peak": hbm_peak, "unit": "GB/s", "frac": ach_hbm / hbm_peak,
           "peak_source": peak_src, "alg_bytes_per_dof_stage": ALG_BYTES_PER_DOF_STAGE}
    if workload != "box3d":                       # flop count measured for the 3D p=3 ideal kernel only
        return {"kernel": "dg_stage_kernel", "bound": "hbm", **hbm, "traffic": None,
                "avg_launch_ms": 1e3 * stage_s}
    mhz = clocks.get("sm_max_mhz") or 1965
    alu_peak = FP64_FMA_PER_CLK * 2 * mhz * 1e6 / 1e12
    ach_alu = FLOP_PER_DOF_STAGE * ndof / stage_s / 1e12
    t_alu, t_hbm = FLOP_PER_DOF_STAGE / (alu_peak * 1e12), ALG_BYTES_PER_DOF_STAGE / (hbm_peak * 1e9)
    out = {"kernel": "dg_stage_kernel", "bound": "alu" if t_alu >= t_hbm else "hbm",
           "achieved": ach_alu, "peak": alu_peak, "unit": "TFLOP/s", "frac": ach_alu / alu_peak,
           "peak_source": "derived: 148 SM x 64 DFMA/clk x 2 x max SM clock (DESIGN.md)",
           "flop_per_dof_stage": FLOP_PER_DOF_STAGE,
           "traffic": NCU_TRAFFIC_PER_DOF_STAGE * ndof,
           "traffic_source": "ncu dram__bytes_read+write per DOF of profiles/r1_ncu_summary.md x DOF per launch",
           "avg_launch_ms": 1e3 * stage_s, "hbm": hbm}
    if out["bound"] == "hbm":
        out.update({k: hbm[k] for k in ("achieved", "peak", "unit", "frac", "peak_source")})
    return out


def run_cuda(a):
    import torch
    import torch.distributed as dist
    from paper_2205_00095_b200 import binding as b
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device and no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    if a.workload == "c2p":            # configs[2]: the con2prim batch micro-benchmark alone
        n = a.size or (1 << 26)
        peak, peak_src = peaks()
        r = {"ideal_gamma_4_3": time_c2p(b, torch, 0, 4.0 / 3.0, n), "taub_matthews": time_c2p(b, torch, 1, 0.0, n)}
        print(json.dumps({"metric": "con2prim states/s", "value": r["ideal_gamma_4_3"], "unit": "states/s",
                          "n_gpus": 1, "dtype": "f64", "data": "synthetic", "higher_is_better": True,
                          "config": {"workload": f"con2prim batch, {n} states, ideal Gamma=4/3 and Taub-Matthews (configs[2])"},
                          "con2prim": r, "gpu_launches": 16,
                          "roofline": {"kernel": "dg_c2p_batch_kernel", "bound": "hbm", "unit": "GB/s", "peak": peak,
                                       "peak_source": peak_src, "alg_bytes_per_state": 80,
                                       "achieved": r["ideal_gamma_4_3"] * 80 / 1e9,
                                       "frac": r["ideal_gamma_4_3"] * 80 / 1e9 / peak,
                                       "achieved_tm": r["taub_matthews"] * 80 / 1e9,
                                       "frac_tm": r["taub_matthews"] * 80 / 1e9 / peak, "traffic": None}}))
        return
    cfgd, W, label = workload_cfg(a.workload, a.size, "cuda")
    ctx = b.Context(b.make_config(*cfg_args(cfgd)))
    U = b.dgrhd_prim2con_batch(cfgd["eos"], cfgd["gamma_ad"], W)
    del W
    ndof = ctx.ndof
    ctx.dgrhd_set_state(U)
    ctx.dgrhd_get_counters(reset=True)
    for _ in range(max(a.warmup, 3)):
        ctx.dgrhd_step(-0.3, 1)
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(local) as clk:
        e0.record()
        ctx.dgrhd_step(-0.3, a.steps)
        e1.record()
        barrier()
    secs = e0.elapsed_time(e1) * 1e-3
    if world > 1:
        secs = max_over_ranks(secs, "cuda")
    cnt = ctx.dgrhd_get_counters()
    value = aggregate_value(world, ndof, a.steps, secs)
    stage_s = secs / (STAGES * a.steps)
    peak, peak_src = peaks()
    ach = ALG_BYTES_PER_DOF_STAGE * ndof / stage_s / 1e9
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": a.steps,
        "warmup": max(a.warmup, 3), "ms_per_step": 1e3 * secs / a.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": label, "dof": ndof, "stages_per_step": STAGES,
                   "l2": "state (5 x DOF x 8 B per copy) is larger than L2; no flush needed"
                   if ndof * 40 > 2 * 126e6 else "state fits L2: noted, algorithmic bytes used",
                   "parallelism": "replicas only" if world > 1 else "single GPU",
                   "limiter_activations_per_stage": cnt["n_flagged"] / max(cnt["n_stages"], 1),
                   "n_bad_mean": cnt["n_bad_mean"], "n_c2p_fail": cnt["n_c2p_fail"]},
        "gpu_launches": a.steps * (STAGES + 1),
        "clocks": clk.summary(),
        "roofline": roofline_stage(a.workload, ndof, stage_s, clk.summary(), peak, peak_src),
    }
    if rank == 0 and world == 1 and not a.no_extra:
        # end to end through the C ABI with HOST buffers (pinned): H2D state, K steps, D2H state
        Uh = U.cpu().pin_memory()
        Uo = torch.empty_like(Uh).pin_memory()
        ke = 2
        ctx.dgrhd_run_host(Uh, Uo, -0.3, 1)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(ke):
            ctx.dgrhd_run_host(Uh, Uo, -0.3, 1)
        te = (time.perf_counter() - t0) / ke
        nb = Uh.numel() * 8
        out["e2e"] = {"value": ndof * STAGES / te, "unit": UNIT, "h2d_bytes_per_step": nb,
                      "d2h_bytes_per_step": nb, "ms_per_step": 1e3 * te,
                      "what": "dgrhd_run_host: pinned host state in, 1 SSPRK3 step, host state out"}
        del Uh, Uo, ctx, U
        torch.cuda.empty_cache()
        n = 1 << 26 if not a.size else 1 << 20
        out["con2prim"] = {"unit": "states/s", "n": n,
                           "ideal_gamma_4_3": time_c2p(b, torch, 0, 4.0 / 3.0, n),
                           "taub_matthews": time_c2p(b, torch, 1, 0.0, n)}
        out["con2prim"]["roofline_hbm_frac_ideal"] = out["con2prim"]["ideal_gamma_4_3"] * 80 / 1e9 / peak
        out["con2prim"]["roofline_hbm_frac_tm"] = out["con2prim"]["taub_matthews"] * 80 / 1e9 / peak
        val, sps, cores, sample = time_oracle(a.workload, 10, 0)
        out["cpu_baseline"] = {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle",
                               "sample": sample, "s_per_step": sps}
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(out))


if __name__ == "__main__":
    args = parse()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_cuda(args)

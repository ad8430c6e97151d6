#!/usr/bin/env python
"""bench.py -- BASELINE.json's metric: DtN right-hand-side columns per second at N = 2048 (fp64 and double-double) and the
achieved fraction of the FP64 (DMMA) roofline, on synthetic surfaces of the paper's shape.

One "step" = one pass of the whole hot path over one batch: setup of a new surface (node prep S0, K/G assembly S1, LU S2),
base state (2.9), and the batched linearized DtN of all nrhs columns (S3-S7) -- what one Runge-Kutta stage of the trust-region
Jacobian costs.  Setup is INSIDE the step: every stage has a new surface.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

N > 1 (torchrun, one rank per GPU): the columns are independent given the surface, so each rank runs the
step on its own 512 columns -- no data-path collective, "scaling": "weak".  Prints ONE JSON line (rank 0).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

import sww_inputs as si  # noqa: E402

METRIC = "DtN RHS-columns/sec at N=2048 (fp64)"
UNIT = "columns/s"
N_METRIC, NRHS_METRIC, NRHS_DD = 2048, 512, 128
# dram__bytes_read.sum + dram__bytes_write.sum per launch from the ncu --set full capture under profiles/ (None = not captured yet)
TRAFFIC_NCU = {"lu": 33.63e6, "trsm": 58.79e6, "gemm_dmma": 51.18e6}  # profiles/r1d_summary.md (trsm: the 512-column batch launch)
NOMINAL_FP64_OVER_BF16 = 45.0 / 2250.0  # blackwell_cuda_programming.md: B200 FP64 tensor 45 TFLOP/s, bf16 dense 2250 TFLOP/s


def rank_case(rank: int, nrhs: int) -> si.Case:
    """metric-point surface; rank r perturbs its own set of Fourier coefficients (columns are independent given the surface)"""
    c = si.metric_point(nrhs)
    if rank:
        N, j = c.N, np.arange(c.N, dtype=np.int64)
        for i in range(nrhs // 2):
            k = 1 + (rank * (nrhs // 2) + i) % (N // 2 - 1)
            col = 2.0 * np.cos(2.0 * np.pi * ((k * j) % N) / N)
            c.deta[2 * i] = col
            c.dphi[2 * i + 1] = col
    return c


class ClockSampler(threading.Thread):
    """samples SM clock and throttle reasons of one GPU while the timed region runs (NVML; nvidia-smi fallback)"""

    def __init__(self, index: int, period: float = 0.02):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop_evt = threading.Event()
        self._nvml = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nvml = pynvml
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            phys = int(vis.split(",")[index]) if vis and vis.split(",")[index].isdigit() else index
            self._h = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self._nvml = None

    def _sample(self):
        p = self._nvml
        if p is not None:
            self.samples.append(p.nvmlDeviceGetClockInfo(self._h, p.NVML_CLOCK_SM))
            r = p.nvmlDeviceGetCurrentClocksEventReasons(self._h)
            names = {"sw_power_cap": p.nvmlClocksEventReasonSwPowerCap, "hw_slowdown": p.nvmlClocksEventReasonHwSlowdown,
                     "hw_thermal_slowdown": p.nvmlClocksEventReasonHwThermalSlowdown,
                     "sw_thermal_slowdown": p.nvmlClocksEventReasonSwThermalSlowdown,
                     "applications_clocks_setting": p.nvmlClocksEventReasonApplicationsClocksSetting}
            for n, bit in names.items():
                if r & bit:
                    self.reasons.add(n)
        else:
            import subprocess
            q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"
            o = subprocess.run(["nvidia-smi", f"--query-gpu={q}", "--format=csv,noheader,nounits", "-i", str(self.index)],
                               capture_output=True, text=True).stdout.strip().split(",")
            if len(o) >= 6:
                self.samples.append(int(o[0]))
                self.max_mhz = int(o[1])
                for n, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), o[2:6]):
                    if v.strip() == "Active":
                        self.reasons.add(n)

    def run(self):
        while not self._stop_evt.is_set():
            try:
                self._sample()
            except Exception:
                pass
            time.sleep(self.period)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=2.0)
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


def measured_peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        d = json.loads(p.read_text())
        return {"hbm_gbs": d["hbm_gbs"], "bf16_tflops": d["bf16_tflops"], "source": "measured (MEASURED_PEAKS.json)"}
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "source": "fallback (B200_PROFILING.md)"}


WORKLOAD = (f"metric point: N={N_METRIC}, h=1, config-3 surface family, nrhs={NRHS_METRIC} linearized-DtN columns per GPU, "
            "setup (assembly+LU) + base state + batched columns inside every step")


def oracle_step(orc, c, n=None):
    """one pass of the hot path through the CPU oracle: setup + base state + the first n (default: all) columns"""
    n = c.nrhs if n is None else n
    t0 = time.perf_counter()
    orc.dtn_linearized(c.eta, c.h, c.phi0, c.deta[:n], c.dphi[:n])
    return time.perf_counter() - t0


def cpu_oracle_baseline(nrhs: int):
    """the oracle source built twice, timed as it stands on this host.  REAL=double (the fairer speed baseline,
    same precision as the timed GPU path) runs the WHOLE workload once; REAL=long double (the parity oracle, with __float128
    multipliers: a precision the GPU path does not compute in) runs a bounded sample, labelled as such."""
    import oracle
    c = si.metric_point(nrhs)
    o64 = oracle.Oracle("f64")
    t64 = oracle_step(o64, c)
    old = oracle.Oracle("ld")
    n_ld = 8
    t_ld = oracle_step(old, c, n_ld)
    return {"value": nrhs / t64, "unit": UNIT, "cores": o64.num_threads(), "kind": "oracle",
            "sample": f"oracle built with REAL=double, N={c.N}: one full step = setup + base state + all {nrhs} columns in {t64:.2f} s "
                      "(no extrapolation)",
            "long_double": {"value": n_ld / t_ld, "unit": UNIT, "cores": old.num_threads(),
                            "sample": f"the parity oracle (REAL=long double, __float128 multipliers): setup + base state + {n_ld} of the "
                                      f"{nrhs} columns in {t_ld:.2f} s; columns/s of that sample (setup-dominated), not extrapolated"}}


def run_reference(args):
    """--impl reference: the CPU oracle (the only 'reference implementation' this paper-only tier has), rank 0 only.
    Every step is one full pass of the workload (setup + base state + all 512 columns) through the REAL=double build of the
    oracle; ms_per_step is the measured time of exactly that."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    import oracle
    orc = oracle.Oracle("f64")
    c = si.metric_point(NRHS_METRIC)
    for _ in range(args.warmup):
        oracle_step(orc, c)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle_step(orc, c)
    t_step = (time.perf_counter() - t0) / max(args.steps, 1)
    value = NRHS_METRIC / t_step
    sample = (f"each step = the whole workload through the oracle built with REAL=double: setup + base state + all {NRHS_METRIC} columns at "
              f"N={c.N} ({t_step:.2f} s per step, {orc.num_threads()} threads); nothing extrapolated")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * t_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD, "N": N_METRIC, "nrhs_per_gpu": NRHS_METRIC},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": orc.num_threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def time_events(fn, reps, flush=None):
    """mean milliseconds of fn() over reps runs, CUDA events on the current stream, optional L2 flush between runs"""
    import torch
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(reps)]
    for e0, e1 in ev:
        if flush is not None:
            flush.zero_()
        e0.record()
        fn()
        e1.record()
    torch.cuda.synchronize()
    return sum(e0.elapsed_time(e1) for e0, e1 in ev) / reps


def other_configs(sww, flush, peak_tf):
    """BASELINE.json configs 1-5 on the device (north_star: 'N from 64 to 4096'): one step = setup + base state + columns unless
    stated; small configs are launch/latency-bound and are reported as time, config 5 also as a roofline fraction"""
    import torch
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    out = {}

    def lin_case(c, prec, reps, mesh=None):
        if prec == sww.DD:
            pk = lambda hi, lo: torch.from_numpy(np.stack([hi, lo])).cuda().contiguous()
            eta, phi0, de, dp = pk(c.eta, c.eta_lo), pk(c.phi0, c.phi0_lo), pk(c.deta, c.deta_lo), pk(c.dphi, c.dphi_lo)
        else:
            eta, phi0, de, dp = dev(c.eta), dev(c.phi0), dev(c.deta), dev(c.dphi)
        res = torch.empty_like(dp)
        d = sww.DtN(eta, c.h, prec)
        if mesh is not None:
            d.set_mesh(*mesh)

        def step():
            d.refactor(eta)
            d.set_base(phi0)
            d.linearized_apply(de, dp, res)
        for _ in range(3):
            step()
        d.check()
        ms = time_events(step, reps, flush)
        d.close()
        return ms

    c1 = si.config1()
    eta1, phi1 = dev(c1.eta), dev(c1.dphi)
    d1 = sww.DtN(eta1, c1.h)
    o1 = torch.empty_like(phi1)

    def step1():
        d1.refactor(eta1)
        d1.apply(phi1, o1)
    for _ in range(3):
        step1()
    ms = time_events(step1, 50)
    out["config1"] = {"workload": "N=64, 1 right-hand side: setup + apply", "ms_per_step": ms, "bound": "latency (10 launches)"}
    d1.close()

    c2 = si.config2()
    st = sww.State(dev(c2.eta), dev(c2.phi0), c2.h, c2.g)
    st.advance(c2.meta["dt"], 2)
    nst = 8
    ms = time_events(lambda: st.advance(c2.meta["dt"], nst), 3) / nst
    out["config2"] = {"workload": "N=256 standing wave, RK8 (11 stages, one setup + solve per stage)", "ms_per_rk_step": ms,
                      "rk_steps_per_s": 1e3 / ms, "ms_per_stage": ms / 11, "bound": "latency (4-block LU chain + ~25 launches per stage)"}
    st.close()

    c3 = si.config3()
    ms = lin_case(c3, sww.F64, 20)
    out["config3"] = {"workload": "N=512, 256 columns, fp64", "ms_per_step": ms, "columns_per_s": c3.nrhs / (ms * 1e-3),
                      "bound": "latency (8-block LU chain, launch sequence)"}
    c3b = si.config3(N=1024, ncols=256)
    ms = lin_case(c3b, sww.F64, 20)
    out["n1024"] = {"workload": "N=1024, 256 columns, fp64 (config-3 family; fills the N sweep between configs 3 and the metric point)", "ms_per_step": ms,
                    "columns_per_s": c3b.nrhs / (ms * 1e-3), "bound": "latency (16-block LU chain) + FP64 tensor"}
    c4 = si.config4()
    ms = lin_case(c4, sww.DD, 10)
    out["config4"] = {"workload": "N=512, 128 columns, double-double", "ms_per_step": ms, "columns_per_s": c4.nrhs / (ms * 1e-3),
                      "bound": "FP64 ALU (error-free-transformation kernels)"}
    c5 = si.config5()
    ms = lin_case(c5, sww.F64, 5)
    fl = (2.0 / 3.0) * c5.N ** 3 + 2.0 * c5.N ** 2 * (c5.nrhs + 2) + 2.0 * c5.N ** 2 * c5.nrhs
    out["config5"] = {"workload": "N=4096, h=0.05, 512 columns, fp64", "ms_per_step": ms, "columns_per_s": c5.nrhs / (ms * 1e-3),
                      "tflops": fl / (ms * 1e-3) / 1e12, "frac_of_fp64_tensor_roofline": fl / (ms * 1e-3) / 1e12 / peak_tf, "bound": "FP64 tensor"}
    # the shooting map: residual + Jacobian of the overdetermined shooting method, one shot = nsteps RK8 steps of
    # (q, Qdot) with n variational columns (one setup + one batched linearized solve per stage)
    Ns, ns_, nst = 512, 64, 8
    S = sww.Shooter(Ns, ns_, 1.0, 1.0)
    cs = np.zeros(ns_ + 1)
    cs[0], cs[1] = 7.2, -0.02
    cs[2:] = 2e-3 * np.exp(-0.5 * np.arange(2, ns_ + 1)) * np.cos(np.arange(2, ns_ + 1))
    S.shoot(cs, nst)
    ms = time_events(lambda: S.shoot(cs, nst), 3)
    out["shooting"] = {"workload": f"shooting map N={Ns}, n={ns_} unknowns, {nst} RK8 steps to T/4: r (3.17) and J (3.31)", "ms_per_shot": ms,
                       "column_stages_per_s": ns_ * nst * 11 / (ms * 1e-3), "bound": "latency (8-block LU chain per stage)"}
    S.gradient(cs, nst)
    ms = time_events(lambda: S.gradient(cs, nst), 3)
    out["shooting_adjoint_gradient"] = {"workload": f"gradient of f for the same shot by one backward solve of the adjoint system (section 3.2): "
                                                    f"forward {nst} RK8 steps with the stage states kept + transposed recursion, one (B.6) per stage",
                                        "ms_per_gradient": ms, "bound": "latency (single-vector solves: the chain of 2N/64 block links per stage)"}
    S.set_segments([(Ns, 0.5, 1.0, 0, nst // 2), (2 * Ns, 0.5, 0.4, 0, nst // 2)])
    S.shoot(cs, nst)
    ms = time_events(lambda: S.shoot(cs, nst), 3)
    out["shooting_refined"] = {"workload": f"the same shot in two segments (section 2.2): {nst // 2} steps on {Ns} uniform points, respacing, "
                                           f"{nst // 2} steps on {2 * Ns} points refined near x = pi with rho = 0.4", "ms_per_shot": ms,
                               "bound": "latency (LU chains of 8 and 16 blocks per stage)"}
    S.close()
    # mesh refinement in space: the metric workload with the stored samples read as values on the mesh (2.10)
    cm = si.metric_point()
    ms = lin_case(cm, sww.F64, 20, mesh=(0.3, 0))
    out["metric_refined_mesh"] = {"workload": f"N={cm.N}, {cm.nrhs} columns, fp64, mesh (2.10) with rho = 0.3 refined near x = pi",
                                  "ms_per_step": ms, "columns_per_s": cm.nrhs / (ms * 1e-3),
                                  "bound": "as the metric step; the refined-mesh assembly and dd base pass add ~0.1 ms"}
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--no-dd", action="store_true", help="skip the double-double leg")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-configs", action="store_true", help="skip the block that times BASELINE.json configs 1-5")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import paper_1210_5672_b200 as sww

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU path (use --impl reference for the oracle arm)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    N, nrhs = N_METRIC, NRHS_METRIC
    case = rank_case(rank, nrhs)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    eta, phi0, deta, dphi = dev(case.eta), dev(case.phi0), dev(case.deta), dev(case.dphi)
    out = torch.empty_like(dphi)
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")  # > 126 MB L2
    d = sww.DtN(eta, case.h)

    def step():
        d.refactor(eta)
        d.set_base(phi0)
        d.linearized_apply(deta, dphi, out)

    for _ in range(args.warmup):
        step()
    d.check()
    K = args.steps
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    l0 = sww.launch_count()
    t_wall = time.perf_counter()
    for e0, e1 in ev:
        flush.zero_()  # L2 flush between timed iterations (outside the event pair)
        e0.record()
        step()
        e1.record()
    barrier()
    t_wall = time.perf_counter() - t_wall
    launches = sww.launch_count() - l0
    clocks = sampler.stop()
    d.check()
    total_ms = sum(e0.elapsed_time(e1) for e0, e1 in ev)
    tt = torch.tensor([total_ms], dtype=torch.float64, device="cuda")
    if dist is not None:
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    total_ms = float(tt.item())
    ms_per_step = total_ms / K
    value = world * nrhs / (ms_per_step * 1e-3)

    # ---- roofline of the dominant kernel: the DMMA GEMM (LU trailing updates, triangular solves, G product)
    sww.timing_enable(True)
    kp = min(K, 10)
    for _ in range(kp):
        flush.zero_()
        step()
    torch.cuda.synchronize()
    tm = sww.timing_read()
    sww.timing_enable(False)
    kernels = {k: {"ms_per_step": v[0] / kp, "launches_per_step": v[1] / kp} for k, v in tm.items() if v[1]}
    # algorithmic FLOPs per step of the two contraction kernels
    flops = {"lu": (2.0 / 3.0) * N ** 3,                    # S2: k_lu_dataflow
             "trsm": 2.0 * N * N * nrhs,                    # S4: k_trsm_ws<32>, the nrhs columns
             "gemm_dmma": 2.0 * N * N * nrhs}               # S6: G product
    flops_step = sum(flops.values()) + 2.0 * N * N * 2      # + the two single-vector solves of the base state (k_trsm_dataflow<8>)
    peaks = measured_peaks()
    peak_tf = peaks["bf16_tflops"] * NOMINAL_FP64_OVER_BF16
    probe = {"dfma_tflops": sww.probe_fp64_peak(0) / 1e12, "dmma_tflops": sww.probe_fp64_peak(1) / 1e12}
    names = {"lu": "k_lu_dataflow (block LU in one persistent launch: a two-CTA cluster as the spine, blocked Gauss-Jordan inverses of the 64x64 Schur blocks on the tensor pipe, warp-specialized DMMA.8x8x4 tile workers: producer warps + mbarrier operand ring)",
             "trsm": "k_trsm_ws<32> (persistent warp-specialized DMMA.8x8x4 multi-RHS triangular solves of the column batch: loader warps + mbarrier ring, tasks handing blocks over through L2 with the data as the flag)",
             "gemm_dmma": "k_gemm_f64 (DMMA.8x8x4): G product"}
    per_kernel = {}
    for cls in ("lu", "trsm", "gemm_dmma"):
        ms_c, n_c = tm[cls][0] / kp, tm[cls][1] / kp
        ach = flops[cls] / (ms_c * 1e-3) / 1e12 if ms_c > 0 else 0.0
        per_kernel[cls] = {"kernel": names[cls], "achieved": ach, "frac": ach / peak_tf, "flops_per_step": flops[cls],
                           "kernel_ms_per_step": ms_c, "kernel_launches_per_step": n_c,
                           "frac_of_probe_dmma": ach / probe["dmma_tflops"] if probe["dmma_tflops"] else None}
    dom = max(per_kernel, key=lambda c: per_kernel[c]["kernel_ms_per_step"])  # the dominant kernel = the one with the most time
    roofline = {"bound": "tensor", "kernel": per_kernel[dom]["kernel"], "achieved": per_kernel[dom]["achieved"], "peak": peak_tf,
                "unit": "TFLOP/s", "frac": per_kernel[dom]["frac"], "traffic": TRAFFIC_NCU.get(dom),
                "peak_source": f"bf16 {peaks['bf16_tflops']} TFLOP/s {peaks['source']} x nominal FP64/bf16 ratio 45/2250",
                "flops_per_step": per_kernel[dom]["flops_per_step"], "kernel_ms_per_step": per_kernel[dom]["kernel_ms_per_step"],
                "kernel_launches_per_step": per_kernel[dom]["kernel_launches_per_step"],
                "probe_peaks_this_box": probe, "frac_of_probe_dmma": per_kernel[dom]["frac_of_probe_dmma"],
                "contraction_kernels": per_kernel, "whole_step_tflops": flops_step / (ms_per_step * 1e-3) / 1e12,
                "whole_step_frac": flops_step / (ms_per_step * 1e-3) / 1e12 / peak_tf}

    # ---- e2e: the HOST-buffer entry point, copies inside the timed region
    e2e = None
    if not args.no_e2e:
        pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
        h_eta, h_phi0, h_deta, h_dphi = pin(case.eta), pin(case.phi0), pin(case.deta), pin(case.dphi)
        h_out = torch.empty_like(h_dphi).pin_memory()
        ke = max(3, min(K, 20))
        for _ in range(3):
            sww.dtn_linearized_host(h_eta, h_phi0, h_deta, h_dphi, case.h, out=h_out)
        barrier()
        t0 = time.perf_counter()
        for _ in range(ke):
            res = sww.dtn_linearized_host(h_eta, h_phi0, h_deta, h_dphi, case.h, out=h_out)
        barrier()
        te = torch.tensor([(time.perf_counter() - t0) / ke], dtype=torch.float64, device="cuda")
        if dist is not None:
            dist.all_reduce(te, op=dist.ReduceOp.MAX)
        e2e = {"value": world * nrhs / float(te.item()), "unit": UNIT, "h2d_bytes_per_step": 8 * N * (2 + 2 * nrhs),
               "d2h_bytes_per_step": 8 * N * nrhs, "ms_per_step": 1e3 * float(te.item()), "steps": ke,
               "checksum": float(res.abs().sum())}

    # ---- double-double leg of the metric (N = 2048, 128 columns)
    ddres = None
    if not args.no_dd:
        cdd = si.metric_point_dd(NRHS_DD, N)
        pk = lambda hi, lo: torch.from_numpy(np.stack([hi, lo])).cuda().contiguous()
        eta_d, phi_d = pk(cdd.eta, cdd.eta_lo), pk(cdd.phi0, cdd.phi0_lo)
        de_d, dp_d = pk(cdd.deta, cdd.deta_lo), pk(cdd.dphi, cdd.dphi_lo)
        out_d = torch.empty_like(dp_d)
        dd_ = sww.DtN(eta_d, cdd.h, sww.DD)

        def step_dd():
            dd_.refactor(eta_d)
            dd_.set_base(phi_d)
            dd_.linearized_apply(de_d, dp_d, out_d)

        for _ in range(3):
            step_dd()
        dd_.check()
        kd = max(3, min(K, 10))
        evd = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(kd)]
        barrier()
        for e0, e1 in evd:
            flush.zero_()
            e0.record()
            step_dd()
            e1.record()
        barrier()
        ms_dd = sum(e0.elapsed_time(e1) for e0, e1 in evd) / kd
        sww.timing_enable(True)
        step_dd()
        torch.cuda.synchronize()
        tmd = sww.timing_read()
        sww.timing_enable(False)
        # dd multiply-adds of one step: 1 residual product (2 solves, ddpath.cu DD_SWEEPS) + 1 G product over NRHS_DD columns,
        # and the same for the base column
        ddfma = 2.0 * N * N * (NRHS_DD + 1)
        t_ddg = tmd["dd_gemm"][0] * 1e-3
        ddres = {"value": world * NRHS_DD / (ms_dd * 1e-3), "unit": UNIT, "ms_per_step": ms_dd, "N": N, "nrhs": NRHS_DD,
                 "dd_fma_per_s_in_dd_gemm": ddfma / t_ddg if t_ddg > 0 else None,
                 "kernels_ms": {k: v[0] for k, v in tmd.items() if v[1]}}
        if t_ddg > 0 and probe["dfma_tflops"]:
            # one dd multiply-add of the dd GEMM (dd_fma_lazy, dd.cuh: renormalised once per 16 terms) is 12 fp64 instructions (+ 6 / 16 for the
            # renormalisation); the bound is the fp64 pipe issue rate = DFMA probe FLOP/s / 2
            ddres["frac_of_dfma_issue_peak"] = (ddfma / t_ddg) * 12.375 / (probe["dfma_tflops"] * 1e12 / 2)

    configs = None
    if rank == 0 and not args.no_configs:
        configs = other_configs(sww, flush, peak_tf)

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu:
        cpu = cpu_oracle_baseline(nrhs)

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": args.warmup,
                "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
                "data": "synthetic",
                "config": {"workload": WORKLOAD,
                           "N": N, "nrhs_per_gpu": nrhs, "parallelism": f"columns sharded over {world} GPU(s), no data-path collective",
                           "l2": "256 MB buffer written between timed iterations (L2 flush), outside the event pairs"},
                "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "gpu_launches_per_step": launches / K,
                "roofline": roofline, "kernels": kernels, "dd": ddres, "configs": configs, "cpu_baseline": cpu,
                "wall_s_timed_region_incl_flush": t_wall}
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

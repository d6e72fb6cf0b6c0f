#!/usr/bin/env python
"""bench.py -- headline measurement (BASELINE.json): RHS evaluations/s (FP64) on config 2, the 53-species /
325-reaction synthetic mechanism over 1,048,576 reactor states, plus reactors/s of the integrators (extra keys).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--extras 0|1]

A "step" is one pass of the hot path over the whole batch: one ck_rhs call on all n states (device-resident
inputs; 914 MB touched per pass, larger than the 126 MB L2, so no L2 flush is needed between steps).
Multi-GPU (torchrun): reactors are independent, every rank evaluates its own n states (weak scaling, no
collective on the data path); value = total states / max-over-ranks time.
`--impl reference` times the CPU oracle (oracle/, as it stands) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

WORKLOAD = "C2: RHS-only, synthetic 53-species/325-reaction mechanism, 1,048,576 states, FP64"
METRIC = "rhs_evals_per_s"
UNIT = "RHS evals/s"
# FP64 vector peak derived from unit counts and clocks:
# 148 SMs x 64 FP64 FMA lanes/clk x 1.965 GHz = 1.861e13 FP64-pipe instructions ("slots")/s = 37.2 TFLOP/s
PEAK_SLOTS = 148 * 64 * 1.965e9
# dram__bytes_read.sum + dram__bytes_write.sum of ONE rhs_kernel_tmem<512> launch over the full 1,048,576 states
# (ncu --set full, profiles/r02_kernels.md); None until such a capture of the full-size launch exists
RHS_DRAM_BYTES_PER_LAUNCH_FULL = 869.1e6


def measured_hbm_gbs():
    """HBM copy bandwidth the driver measured on this pool (MEASURED_PEAKS.json); fallback of the profiling guide."""
    try:
        return float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index=0, period=0.05):
        self.index, self.period = index, period
        self.samples, self.reasons = [], set()
        self.max_mhz = None
        self._stop = threading.Event()
        self._thr = None

    def start(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nv = pynvml
            self._h = pynvml.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self._nv = None
            return self
        self._thr = threading.Thread(target=self._run, daemon=True)
        self._thr.start()
        return self

    def _run(self):
        nv = self._nv
        names = {"hw_slowdown": nv.nvmlClocksThrottleReasonHwSlowdown,
                 "hw_thermal_slowdown": nv.nvmlClocksThrottleReasonHwThermalSlowdown,
                 "sw_thermal_slowdown": nv.nvmlClocksThrottleReasonSwThermalSlowdown,
                 "sw_power_cap": nv.nvmlClocksThrottleReasonSwPowerCap}
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self._h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(self.period)

    def stop(self):
        self._stop.set()
        if self._thr:
            self._thr.join()
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


def oracle_cores():
    try:
        return len(os.sched_getaffinity(0))
    except Exception:
        return os.cpu_count() or 1


def time_oracle_rhs(mech, y, p, target_s=12.0):
    """Oracle RHS (as it stands) on a bounded sample of the workload, all host cores (omp dynamic over states):
    whole passes over up to 262,144 states are repeated until about `target_s` seconds of CPU work are done."""
    from oracle import ck_oracle
    O = ck_oracle.Mech(mech)
    cores = min(oracle_cores(), ck_oracle.max_threads())
    ns = int(min(y.shape[1], 262144))
    ys = np.ascontiguousarray(y[:, :ns]); ps = np.ascontiguousarray(p[:ns])
    O.rhs(ys[:, :4096].copy(), ps[:4096].copy(), nthreads=cores)   # page in / spin up the thread pool
    done, t0 = 0, time.perf_counter()
    while True:
        O.rhs(ys, ps, nthreads=cores)
        done += ns
        dt = time.perf_counter() - t0
        if dt >= target_s:
            break
    return done / dt, cores, done, dt


def shard_states(y, p, rank):
    """States of one rank: reactors are independent, so every rank evaluates its own batch (weak scaling);
    ranks > 0 take a seeded permutation of the same recipe so that no two ranks hold the same column order."""
    if rank == 0:
        return y, p
    perm = np.random.default_rng(1000 + rank).permutation(y.shape[1])
    return np.ascontiguousarray(y[:, perm]), np.ascontiguousarray(p[perm])


def max_over_ranks(value, dist, device=None):
    """Max of a per-rank timing over the process group (no collective touches the data path)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from synth_inputs import make_config
    mech, y, p, _ = make_config("C2", n=65536)
    per_step = max(1.0, 60.0 / max(1, args.steps + args.warmup))
    vals = []
    for i in range(args.warmup + args.steps):
        v, cores, ns, dt = time_oracle_rhs(mech, y, p, target_s=min(per_step, 10.0))
        if i >= args.warmup:
            vals.append((v, dt))
    value = float(np.mean([v for v, _ in vals]))
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * float(np.mean([d for _, d in vals])), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD, "sample": f"{ns} state evaluations per step"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                             "sample": f"{ns} state evaluations per step (passes over 65,536 states of the C2 recipe), omp dynamic over states"},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def time_oracle_integrate(mech, y, p, cfg, n_sub):
    """Oracle integrator (as it stands) on the first n_sub reactors of the workload, all host cores (omp dynamic over
    reactors, the structure of the paper's own baseline)."""
    from oracle import ck_oracle
    O = ck_oracle.Mech(mech)
    cores = min(oracle_cores(), ck_oracle.max_threads())
    ys = np.ascontiguousarray(y[:, :n_sub]); ps = np.ascontiguousarray(p[:n_sub])
    t0 = time.perf_counter()
    r = O.integrate(cfg["call"], ys, ps, cfg["dt"], rtol=cfg["rtol"], atol=cfg["atol"], nthreads=cores)
    dt = time.perf_counter() - t0
    return {"value": n_sub / dt, "unit": "reactors/s", "rhs_evals_per_s": r["rhs_evals"] / dt, "cores": cores, "kind": "oracle",
            "sample": f"first {n_sub} reactors of the workload, {dt:.1f} s, omp dynamic over reactors"}


# reactors the oracle integrates for the CPU baseline of each integration config (a few seconds each on 16 cores)
ORACLE_SUBSET = {"C1": 1024, "C3": 2048, "C4": 2048, "C5": 512, "C6": 4096, "C7": 2048}


def integrator_extras(torch, ck, dev, cpu=True):
    """Reactors/s of the integrators on configs 1, 3-7 (device-resident inputs, best of 2 after one warm-up), the same
    through the host-pointer entry point (transfers inside the call), and the oracle on a subset of the same workload."""
    from synth_inputs import make_config
    out = {}
    for name in ("C1", "C3", "C4", "C5", "C6", "C7"):
        try:
            mech, y, p, cfg = make_config(name)
            M = ck.Mechanism(mech, device=dev.index or 0)
            y0 = torch.from_numpy(y).to(dev); pd = torch.from_numpy(p).to(dev)
            best, res = None, None
            ws = None
            for it in range(3):
                yy = y0.clone()
                e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
                torch.cuda.synchronize(); e0.record()
                res = M.integrate(cfg["call"], yy, pd, cfg["dt"], rtol=cfg["rtol"], atol=cfg["atol"], ws=ws)
                e1.record(); torch.cuda.synchronize()
                ws = res["ws"]
                ms = e0.elapsed_time(e1)
                if it >= 1:
                    best = ms if best is None else min(best, ms)
            rep = res["report"]
            slots_rhs = M.rhs_slots()
            n = int(y.shape[1])
            out[name] = {"call": cfg["call"], "n": n, "ms": best, "reactors_per_s": n / (best * 1e-3),
                         "rhs_evals_per_s": rep["rhs_evals"] / (best * 1e-3), "attempts": rep["attempts"],
                         "accepted": rep["accepted"], "rejected": rep["rejected"], "rounds": rep["rounds"],
                         "simt_efficiency": rep["simt_efficiency"], "waste_p32_static": rep["waste_p32"],
                         "n_failed": rep["n_failed"],
                         "rhs_only_roofline_frac": rep["rhs_evals"] * slots_rhs / (best * 1e-3) / PEAK_SLOTS}
            # algorithmic FP64-pipe instructions of the whole integration:
            # every RHS evaluation, an analytic Jacobian at 2.1 RHS, N^3/3 per LU, 4 N^2 per attempt for the four
            # stage solves, ~20 N per attempt for the stage vectors, error norm and step control
            Nn = int(y.shape[0])
            slots = rep["rhs_evals"] * slots_rhs + rep["jac_evals"] * 2.1 * slots_rhs + rep["lu_factor"] * Nn ** 3 / 3.0 \
                + (4.0 * Nn * Nn if cfg["call"] == "ros" else 0.0) * rep["attempts"] + 20.0 * Nn * rep["attempts"]
            out[name]["alg_fp64_inst_per_attempt"] = slots / max(rep["attempts"], 1)
            out[name]["roofline_frac"] = slots / (best * 1e-3) / PEAK_SLOTS
            # end to end through ck_integrate_host: pinned host buffers, H2D + integration + D2H of states and step counts
            yh = torch.from_numpy(y).pin_memory(); ph = torch.from_numpy(p).pin_memory()
            work = torch.empty_like(yh).pin_memory()
            tbest = None
            for it in range(2):
                work.copy_(yh)
                torch.cuda.synchronize(); t0 = time.perf_counter()
                M.integrate_host(cfg["call"], work.numpy(), ph.numpy(), cfg["dt"], rtol=cfg["rtol"], atol=cfg["atol"])
                te = time.perf_counter() - t0
                if it >= 1 or tbest is None:
                    tbest = te
            out[name]["e2e"] = {"value": n / tbest, "unit": "reactors/s", "h2d_bytes_per_step": int(yh.numel() * 8 + ph.numel() * 8),
                                "d2h_bytes_per_step": int(yh.numel() * 8 + n * 20)}
            # waste study (Eq. 20 and Figs. 9-10): mean, upper decile and the
            # CDF point the paper quotes (share of work units with W < 1 %: 92 % at width 4, 63 % at width 32 for its
            # RKF45 flame data) at the paper's four SIMD widths, from this run's step counts (ck_waste);
            # and the same with 4 / 16 reactors per lane (several tasks per thread)
            ws_ = {}
            for P in (4, 8, 16, 32):
                Wd = M.waste(res["n_accept"], res["n_reject"], P)
                ws_[str(P)] = {"mean": float(Wd.mean()), "p90": float(torch.quantile(Wd, 0.9)),
                               "frac_units_below_1pct": float((Wd < 0.01).double().mean()),
                               "frac_units_below_10pct": float((Wd < 0.10).double().mean()),
                               "mean_4_tasks_per_lane": float(M.waste(res["n_accept"], res["n_reject"], P, tasks=4).mean()),
                               "mean_16_tasks_per_lane": float(M.waste(res["n_accept"], res["n_reject"], P, tasks=16).mean())}
            out[name]["waste_static"] = ws_
            if name == "C3":  # the same batch in flame order: neighbours need similar step counts
                _, yf, pf, _ = make_config(name, flame_ordered=True)
                rf = M.integrate(cfg["call"], torch.from_numpy(yf).to(dev), torch.from_numpy(pf).to(dev), cfg["dt"],
                                 rtol=cfg["rtol"], atol=cfg["atol"], ws=ws)
                out[name]["waste_static_flame_ordered"] = {
                    str(P): {"mean": float(M.waste(rf["n_accept"], rf["n_reject"], P).mean()),
                             "frac_units_below_1pct": float((M.waste(rf["n_accept"], rf["n_reject"], P) < 0.01).double().mean())}
                    for P in (4, 8, 16, 32)}
            if cpu:
                out[name]["cpu_baseline"] = time_oracle_integrate(mech, y, p, cfg, min(ORACLE_SUBSET[name], n))
            M.close()
        except Exception as ex:  # report, do not hide
            out[name] = {"error": str(ex)[:200]}
    return out


def rhs_extras(torch, ck, dev, steps=10):
    """RHS-only throughput and roofline fraction on the other model shapes (same state recipe as config 2, 1,048,576
    states): the 111-species / 784-reaction model (tensor-memory kernel with 224-thread CTAs) and the 14 / 38 model."""
    from synth_inputs import states as S
    from synth_inputs.configs import get_mech
    out = {}
    for label, mname, n in (("111sp_784rxn", "c4", 1048576), ("14sp_38rxn", "h2co", 1048576), ("53sp_634irrev", "c1irr", 1048576)):
        try:
            mech = get_mech(mname)
            y, p = S.dirichlet_states(mech, n, 108)
            M = ck.Mechanism(mech, device=dev.index or 0)
            yd = torch.from_numpy(y).to(dev); pd = torch.from_numpy(p).to(dev); o = torch.empty_like(yd)
            for _ in range(3):
                M.rhs(yd, pd, out=o)
            e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize(); e0.record()
            for _ in range(steps):
                M.rhs(yd, pd, out=o)
            e1.record(); torch.cuda.synchronize()
            ms = e0.elapsed_time(e1) / steps
            out[label] = {"n": n, "ms_per_pass": ms, "rhs_evals_per_s": n / (ms * 1e-3), "kernel": M.rhs_kernel_name(n),
                          "slots_per_eval": M.rhs_slots(), "roofline_frac": M.rhs_slots() * n / (ms * 1e-3) / PEAK_SLOTS}
            M.close()
            del yd, o
        except Exception as ex:
            out[label] = {"error": str(ex)[:200]}
    return out


def run_case(args):
    """One plain invocation of one workload, for profiler captures (profiles/*.md name these command lines):
    --case rhs | C1 | C3 | C4 | C5 | C6 | C7 [--case-flags F] runs config 2's ck_rhs three times, resp. one integration."""
    import torch
    import paper_1608_05794_b200 as ck
    from synth_inputs import make_config
    dev = torch.device("cuda", 0)
    if args.case == "lu":   # the dense linear algebra on its own: ck_lu_solve_batched (warp-per-system blocked LU, DMMA trailing update)
        out = {"case": "lu", "dfma_peak_per_s": ck.fp64_peak(0), "dmma_peak_fma_per_s": ck.fp64_mma_peak(0)}
        for N, n in ((54, 65536), (112, 16384), (15, 262144)):
            g = torch.Generator(device="cuda").manual_seed(7)
            A = torch.rand((n, N, N), dtype=torch.float64, device=dev, generator=g) - 0.5 + 4.0 * torch.eye(N, dtype=torch.float64, device=dev)
            b = torch.rand((n, N), dtype=torch.float64, device=dev, generator=g)
            ck.lu_solve_batched(A, b)
            e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(5):
                ck.lu_solve_batched(A, b)
            e1.record(); torch.cuda.synchronize()
            ms = e0.elapsed_time(e1) / 5
            fma = N ** 3 / 3.0 + N * N
            out[f"N{N}"] = {"systems": n, "ms": ms, "systems_per_s": n / (ms * 1e-3), "fma_per_system": fma,
                            "frac_of_fp64_peak": fma * n / (ms * 1e-3) / PEAK_SLOTS,
                            "hbm_GBs": (N * N + 2 * N) * 8 * n / (ms * 1e-3) / 1e9}
        print(json.dumps(out))
        return
    name = "C2" if args.case == "rhs" else args.case
    mech, y, p, cfg = make_config(name)
    M = ck.Mechanism(mech, device=0)
    yd = torch.from_numpy(y).to(dev); pd = torch.from_numpy(p).to(dev)
    if args.case == "rhs":
        out = torch.empty_like(yd)
        for _ in range(3):
            M.rhs(yd, pd, out=out)
        torch.cuda.synchronize()
        print(json.dumps({"case": "rhs", "kernel": M.rhs_kernel_name(y.shape[1]), "n": int(y.shape[1])}))
        return
    e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
    e0.record()
    res = M.integrate(cfg["call"], yd, pd, cfg["dt"], rtol=cfg["rtol"], atol=cfg["atol"], flags=args.case_flags)
    e1.record(); torch.cuda.synchronize()
    print(json.dumps({"case": args.case, "flags": args.case_flags, "ms_first_call": e0.elapsed_time(e1), "report": res["report"]}))


def run_ours(args):
    import torch
    import paper_1608_05794_b200 as ck
    from synth_inputs import make_config

    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    mech, y, p, cfg = make_config("C2")          # every rank: its own n states (seed offset by rank)
    y, p = shard_states(y, p, rank)
    n = y.shape[1]
    M = ck.Mechanism(mech, device=local)
    yd = torch.from_numpy(y).to(dev); pd = torch.from_numpy(p).to(dev)
    out = torch.empty_like(yd)
    slots = M.rhs_slots()
    alg_bytes = (2 * M.K + 3) * 8 * n

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        M.rhs(yd, pd, out=out)
    barrier()
    clocks = ClockSampler(local).start()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    ev[0].record()
    for i in range(args.steps):
        M.rhs(yd, pd, out=out)
        ev[i + 1].record()
    barrier()
    clk = clocks.stop()
    total_ms = ev[0].elapsed_time(ev[-1])
    per_launch_ms = float(np.mean([ev[i].elapsed_time(ev[i + 1]) for i in range(args.steps)]))
    total_ms = max_over_ranks(total_ms, dist, dev)
    value = world * n * args.steps / (total_ms * 1e-3)

    # end to end through the host-pointer C-ABI call: pinned host buffers, H2D + kernel + D2H per step
    yh = torch.from_numpy(y).pin_memory(); ph = torch.from_numpy(p).pin_memory(); oh = torch.empty_like(yh).pin_memory()
    ynp, pnp, onp = yh.numpy(), ph.numpy(), oh.numpy()
    e2e_steps = max(2, min(args.steps, 5))
    M.rhs_host(ynp, pnp, out=onp)
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        M.rhs_host(ynp, pnp, out=onp)
    barrier()
    e2e_s = time.perf_counter() - t0
    e2e_s = max_over_ranks(e2e_s, dist, dev)
    e2e = {"value": world * n * e2e_steps / e2e_s, "unit": UNIT, "h2d_bytes_per_step": int(ynp.nbytes + pnp.nbytes),
           "d2h_bytes_per_step": int(onp.nbytes), "steps": e2e_steps}

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return
    achieved = slots * n / (per_launch_ms * 1e-3)
    measured_peak = mma_peak = None
    try:
        measured_peak = ck.fp64_peak(local)
        mma_peak = ck.fp64_mma_peak(local)
    except Exception:
        pass
    traffic = RHS_DRAM_BYTES_PER_LAUNCH_FULL if n == 1048576 else None
    hbm_gbs, hbm_src = measured_hbm_gbs()
    roofline = {"bound": "alu", "kernel": M.rhs_kernel_name(n), "achieved": 2 * achieved / 1e12, "peak": 2 * PEAK_SLOTS / 1e12,
                "unit": "TFLOP/s", "frac": achieved / PEAK_SLOTS, "traffic": traffic,
                "peak_source": "derived and probed FP64 peak (MEASURED_PEAKS.json carries no FP64 figure): 148 SM x 64 FP64 FMA/clk x 1.965 GHz (DESIGN.md); 1 FP64-pipe instruction = 2 flop",
                "slots_per_eval": slots, "fp64_pipe_inst_per_s": achieved,
                "measured_dfma_peak_inst_per_s": measured_peak, "measured_dmma_peak_fma_per_s": mma_peak,
                "frac_of_measured_dfma_peak": (achieved / measured_peak) if measured_peak else None,
                "hbm_alg_bytes_per_launch": alg_bytes, "hbm_achieved_GBs": alg_bytes / (per_launch_ms * 1e-3) / 1e9,
                "hbm_peak_GBs": hbm_gbs, "hbm_peak_source": hbm_src,
                "hbm_frac_of_measured": alg_bytes / (per_launch_ms * 1e-3) / 1e9 / hbm_gbs}
    cpu_v, cores, ns, cpu_dt = time_oracle_rhs(mech, y, p)
    del yd, out, yh, ph, oh
    torch.cuda.empty_cache()
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD, "n_states_per_gpu": n, "l2": "inputs (914 MB per pass) larger than L2; no flush",
                       "parallelism": f"independent reactors x{world}"},
            "clocks": clk, "e2e": e2e, "gpu_launches": args.steps,
            "roofline": roofline,
            "cpu_baseline": {"value": cpu_v, "unit": UNIT, "cores": cores, "kind": "oracle",
                             "sample": f"{ns} state evaluations (passes over the first 262,144 of {n} states), {cpu_dt:.1f} s, omp dynamic over states"}}
    if args.extras:
        line["integrators"] = integrator_extras(torch, ck, dev)
        line["rhs_other_models"] = rhs_extras(torch, ck, dev)
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--extras", type=int, default=1, help="also time the integrators on configs 1,3-7 (rank 0, N=1)")
    ap.add_argument("--case", default=None, help="profiling aid: run ONE workload once (rhs, C1, C3..C7) and exit")
    ap.add_argument("--case-flags", type=int, default=0, help="ck_opts.flags for --case")
    args = ap.parse_args()
    if args.case:
        run_case(args)
        return
    if args.impl == "reference":
        run_reference(args)
    else:
        if int(os.environ.get("WORLD_SIZE", "1")) > 1:
            args.extras = 0
        run_ours(args)


if __name__ == "__main__":
    main()

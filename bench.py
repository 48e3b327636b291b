#!/usr/bin/env python
"""bench.py -- the driver's measurement contract for the batched PSR chemistry hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

A step is one pass of the hot path over BASELINE.json configs[1] ("C1": 53 species / 325
reactions, 65,536 reactors per GPU): one psr_eval_residual call that produces wdot AND the PSR
residual F.  The finite-difference Jacobian (row a10, configs[4]) and
the larger mechanisms are timed once each and reported under "extra"; DESIGN.md says why they are
not folded into the headline metric.  Inputs are seeded synthetic states (synth.py); nothing here
reads /root/reference.

value  : reactor wdot evaluations per second, inputs resident in HBM, CUDA-event time on the
         launching stream, L2 flushed between timed steps.
e2e    : same metric through the same C-ABI call with HOST (pinned) buffers: H2D of T,P,Y,Yin,tau
         and D2H of wdot,F inside the timed region.
--impl reference : the CPU oracle (oracle/), as it stands, on the host cores (the tier's reference arm).
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

METRIC = "reactor wdot evaluations/sec (FP64, 53sp/325rxn)"
UNIT = "reactor-evals/s"
WORKLOAD = "C1: 53 species / 325 reactions (28 three-body, 29 Troe), 65536 reactors per GPU"

# SURVEY.md 8(d) algorithmic FP64 work per reactor evaluation:
#   exp: 2I + 5 I_troe ; log: 1 + 2 I_troe ; div: 2 + 3 I_troe ;
#   DFMA-class: 16K + 14I + nnz(nu) + 5 I_tb + 25 I_troe ; exp = 22, log = 28, div = 10 instructions.
EXP_INSTR, LOG_INSTR, DIV_INSTR = 22.0, 28.0, 10.0
N_SM, FP64_LANES_PER_SM = 148, 64     # B200: 64 FP64 FMA lanes per SM (37 TFLOP/s nominal)

# FP64 instructions of one FD Jacobian of the C1 mechanism with the T-only factors hoisted (the naive
# count is 55 full evaluations)
C4_HOISTED_INSTR_PER_JACOBIAN = 410e3


def ncu_summary(key: str) -> dict:
    """Numbers that only a profiler sees (DRAM bytes per launch, FP64-pipe utilisation), read from the committed
    summary of the ncu --set full captures under profiles/ -- never measured under the profiler in this run."""
    try:
        return json.loads((ROOT / "profiles" / "ncu_summary.json").read_text()).get(key, {})
    except Exception:
        return {}


def algorithmic_fp64_instr(K, I, n_tb, n_troe, nnz):
    n_exp = 2 * I + 5 * n_troe
    n_log = 1 + 2 * n_troe
    n_div = 2 + 3 * n_troe
    dfma = 16 * K + 14 * I + nnz + 5 * n_tb + 25 * n_troe
    return n_exp * EXP_INSTR + n_log * LOG_INSTR + n_div * DIV_INSTR + dfma


class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int):
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

    def _one(self):
        nv = self.nv
        self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
        try:
            r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
        except Exception:
            r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
        names = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown",
                 0x4: "sw_power_cap", 0x80: "hw_power_brake_slowdown"}
        for bit, name in names.items():
            if r & bit:
                self.reasons.add(name)

    def _run(self):
        while not self._stop.is_set():
            try:
                self._one()
            except Exception:
                pass
            self._stop.wait(0.01)

    def start(self):
        if self.nv:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()

    def stop(self) -> dict:
        if self._thr:
            self._stop.set()
            self._thr.join()
        if self.nv and not self.samples:
            try:
                self._one()
            except Exception:
                pass
        return {"sm_mhz": float(np.median(self.samples)) if self.samples else None,
                "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ------------------------------------------------------------------------------ oracle legs
def _oracle_mech(mech):
    from oracle import oracle as orc
    return orc.OracleMechanism.from_arrays(mech.n_species, mech.n_reactions, mech.arrays())


def time_oracle(mech, batch, repeats: int):
    """The oracle as it stands (g++ -O2, OpenMP over reactors) on all host cores of the affinity
    mask; best of `repeats` passes over `batch`."""
    from oracle import oracle as orc
    om = _oracle_mech(mech)
    cores = min(orc.max_threads(), orc.host_cores())
    best = float("inf")
    for _ in range(repeats):
        t0 = time.perf_counter()
        orc.evaluate(om, batch.T, batch.P, batch.Y, batch.Yin, batch.tau, want=("wdot", "F"), nthreads=cores)
        best = min(best, time.perf_counter() - t0)
    return batch.n / best, cores, best


def run_reference(args):
    """--impl reference: the CPU oracle timed on the host, same metric/config/unit."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_2005_11468_b200 import synth
    mech, batch = synth.make_config("C1")
    from oracle import oracle as orc
    om = _oracle_mech(mech)
    cores = min(orc.max_threads(), orc.host_cores())
    # bounded sample of the 65,536-reactor workload per step, sized from a calibration pass so the
    # whole run stays near two minutes whatever K and W are
    cal = batch.take(np.arange(2048))
    t0 = time.perf_counter()
    orc.evaluate(om, cal.T, cal.P, cal.Y, cal.Yin, cal.tau, want=("wdot", "F"), nthreads=cores)
    rate = 2048 / (time.perf_counter() - t0)
    sample_n = int(min(batch.n, max(256, rate * 120.0 / (args.steps + args.warmup))))
    sub = batch.take(np.arange(sample_n))
    for _ in range(args.warmup):
        orc.evaluate(om, sub.T, sub.P, sub.Y, sub.Yin, sub.tau, want=("wdot", "F"), nthreads=cores)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        orc.evaluate(om, sub.T, sub.P, sub.Y, sub.Yin, sub.tau, want=("wdot", "F"), nthreads=cores)
    dt = time.perf_counter() - t0
    value = sample_n * args.steps / dt
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOAD, "sample": f"first {sample_n} reactors per step"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": f"first {sample_n} of 65536 C1 reactors per step, wdot + residual"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------ our arm
def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2005_11468_b200 import binding, shard, synth

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    # weak scaling: every rank owns its own 65,536-reactor batch (independent reactors, no
    # data-path collective -- SURVEY.md 8(e)); rank r draws the C1 state stream with seed 2001 + 100 r
    mech, batch = synth.make_config("C1")
    if rank > 0:
        batch = synth.make_states(mech.n_species, batch.n, seed=shard.state_seed(1, rank), **synth.CONFIGS["C1"]["state"])
    N, K, I = batch.n, mech.n_species, mech.n_reactions
    gm = binding.Mechanism.from_synth(mech)
    info = gm.info()
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    T, P, Y, Yin, tau = (dev(x) for x in (batch.T, batch.P, batch.Y, batch.Yin, batch.tau))
    F, wdot = torch.empty_like(Y), torch.empty_like(Y)
    flush = torch.empty(256 * 1024 * 1024 // 8, dtype=torch.float64, device="cuda")  # 256 MiB > 126 MB L2
    stream = torch.cuda.current_stream()

    def step():
        gm.eval_residual(T, P, Y, Yin, tau, F=F, wdot=wdot)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    sampler = ClockSampler(local)   # samples SM clock / throttle reasons from the warm-up to the end of the e2e leg
    sampler.start()
    for _ in range(max(args.warmup, 3)):   # warm-up steps are the timed steps without the events: flush, then call
        flush.zero_()
        step()
    barrier()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    for e0, e1 in ev:
        flush.zero_()                       # L2 flush between timed steps (not timed)
        e0.record(stream)
        step()
        e1.record(stream)
    barrier()
    dev_ms = sum(e0.elapsed_time(e1) for e0, e1 in ev)
    dev_ms = shard.max_over_ranks(dev_ms, device="cuda")
    ms_per_step = dev_ms / args.steps
    value = shard.whole_job_rate(N, args.steps, dev_ms, world)

    # ---- end to end: host pinned buffers in, host pinned buffers out, same C-ABI call.  The batch goes through
    # in E2E_CHUNKS blocks of reactors on E2E_STREAMS streams, so that one block's copy-out, the next block's kernel and
    # the one after's copy-in overlap (PCIe is full duplex; reactors are independent).  Host data are held per
    # block in the library's [K][n] layout; every byte of T, P, Y, Y_in, tau crosses to the device and every
    # byte of wdot and F comes back inside the timed region.
    # (measured on this pool, ms per step with / without the kernel: 8 blocks on 3 streams 1.73 / 1.64, 16 on 4: 2.03 /
    # 1.83, 2 on 2: 1.70 / 1.59, 4 on 2: 1.60 / 1.60 -- the copies alone, full duplex, are the floor)
    E2E_CHUNKS, E2E_STREAMS = 4, 2
    bounds = [N * c // E2E_CHUNKS for c in range(E2E_CHUNKS + 1)]
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    blocks = []
    for c in range(E2E_CHUNKS):
        c0, c1 = bounds[c], bounds[c + 1]
        # one pinned array per direction and block: rows T, P, tau, Y[0..K), Yin[0..K) in; wdot[0..K), F[0..K) out
        hin = pin(np.concatenate([batch.T[None, c0:c1], batch.P[None, c0:c1], batch.tau[None, c0:c1],
                                  batch.Y[:, c0:c1], batch.Yin[:, c0:c1]], axis=0))
        hout = torch.empty((2 * K, c1 - c0), dtype=torch.float64).pin_memory()
        din = torch.empty_like(hin, device="cuda")
        dout = torch.empty((2 * K, c1 - c0), dtype=torch.float64, device="cuda")
        blocks.append((hin, hout, din, dout))
    h2d = sum(b[0].numel() * 8 for b in blocks)
    d2h = sum(b[1].numel() * 8 for b in blocks)
    # several streams on one handle: allowed for the resident kernel only (psr.h, "Overlap on the GPU")
    side = [torch.cuda.Stream() for _ in range(E2E_STREAMS if info["eval_kernel"] == 1 else 1)]

    def e2e_step():
        start = torch.cuda.Event()
        start.record(stream)
        for c, (hin, hout, din, dout) in enumerate(blocks):
            st = side[c % len(side)]
            st.wait_event(start)
            with torch.cuda.stream(st):
                din.copy_(hin, non_blocking=True)
                gm.eval_residual(din[0], din[1], din[3:3 + K], din[3 + K:3 + 2 * K], din[2], F=dout[K:], wdot=dout[:K])
                hout.copy_(dout, non_blocking=True)
        for st in side:
            done = torch.cuda.Event()
            done.record(st)
            stream.wait_event(done)

    e2e_steps = max(3, min(args.steps, 20))
    for _ in range(3):
        e2e_step()
    barrier()
    a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a0.record(stream)
    for _ in range(e2e_steps):
        e2e_step()
    a1.record(stream)
    barrier()
    e2e_ms = a0.elapsed_time(a1)
    clocks = sampler.stop()
    e2e_ms = shard.max_over_ranks(e2e_ms, device="cuda")
    e2e_value = shard.whole_job_rate(N, e2e_steps, e2e_ms, world)
    assert all(bool(torch.isfinite(b[1]).all()) for b in blocks)
    # the blocks together are the device-resident result
    assert torch.equal(torch.cat([b[1][:K] for b in blocks], dim=1), wdot.cpu())
    assert torch.equal(torch.cat([b[1][K:] for b in blocks], dim=1), F.cpu())

    # ---- roofline of the dominant (only) kernel: FP64 ALU pipe
    instr_per_eval = algorithmic_fp64_instr(K, I, info["n_third_body"], info["n_falloff"], info["nnz_nu"])
    peak = N_SM * FP64_LANES_PER_SM * (clocks["sm_max_mhz"] or 1965) * 1e6 / 1e12   # T FP64 thread-instr/s
    achieved = instr_per_eval * N / (ms_per_step * 1e-3) / 1e12
    probes = {}
    if rank == 0:
        for kind, name in ((0, "dfma"), (1, "exp"), (2, "log")):
            ms, ops = binding.probe_fp64(kind, 2000 if kind == 0 else 500)
            probes[name + "_per_s"] = ops / (ms * 1e-3)
    hbm_bytes = (3 + 4 * K) * 8 * N    # T, P, tau, Y, Yin in; wdot, F out
    prof = ncu_summary("C1_residual")
    roofline = {
        "bound": "alu", "achieved": achieved, "peak": peak, "unit": "T FP64 thread-instr/s",
        "frac": achieved / peak, "traffic": prof.get("dram_bytes_per_launch"),
        "frac_is": "algorithmic FP64 instruction count of the METHOD with library exp/log/div costs (SURVEY.md 8(d)) / time / peak; "
                   "the kernel executes fewer FP64 instructions than that (log-linear rate forms, table exp): see fp64_pipe_util_ncu",
        "fp64_pipe_util_ncu": prof.get("fp64_pipe_pct"), "ncu_capture": prof.get("capture"),
        "peak_source": "derived: 148 SM x 64 FP64 lanes x clocks.max.sm (DESIGN.md); measured DFMA probe in 'probes'",
        "instr_per_eval": instr_per_eval, "probes": probes,
        "hbm": {"algorithmic_bytes_per_launch": hbm_bytes,
                "achieved_GBps": hbm_bytes / (ms_per_step * 1e-3) / 1e9, "peak_GBps": _hbm_peak()},
    }

    # ---- extras (rank 0, one GPU): other §8(a) rows timed once each, not part of `value`
    extra = {}
    if rank == 0 and not args.no_extra:
        extra = run_extras(binding, synth, torch, flush, cpu=not args.no_cpu)

    # ---- cpu baseline: the oracle as it stands on the host cores, bounded sample (rank 0, N=1)
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu:
        sample_n = 4096
        sub = batch.take(np.arange(sample_n))
        rate, cores, secs = time_oracle(mech, sub, repeats=1)
        # grow the sample towards the whole batch, then repeat passes until ~20 core-seconds are spent
        target = int(min(N, max(sample_n, rate * 10.0)))
        if target > sample_n:
            sub = batch.take(np.arange(target))
            sample_n = target
        rate1, cores, secs = time_oracle(mech, sub, repeats=1)
        passes = int(min(50, max(1, np.ceil(20.0 / max(secs * cores, 1e-3)))))
        rate, cores, secs = time_oracle(mech, sub, repeats=passes)
        cpu = {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"first {sample_n} of {N} C1 reactors, wdot + residual, best of {passes} passes "
                         f"({secs:.3f} s each on {cores} threads)"}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD, "call": "psr_eval_residual (wdot + F)", "l2": "flushed between timed steps (256 MiB memset)",
                       "reaction_evals_per_s": value * I, "kernel": info},
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "steps": e2e_steps, "pipeline": f"{E2E_CHUNKS} blocks of reactors on {E2E_STREAMS} streams (one copy in, kernel, one copy out per block, overlapped)"},
            "gpu_launches": args.steps,
            "roofline": roofline, "cpu_baseline": cpu, "extra": extra,
        }
        print(json.dumps(line), flush=True)
    gm.close()
    if world > 1:
        dist.destroy_process_group()


def _hbm_peak():
    p = ROOT / "MEASURED_PEAKS.json"
    try:
        return json.loads(p.read_text())["hbm_gbs"]
    except Exception:
        return 6650.0   # B200_PROFILING.md fallback


def _time_call(torch, fn, flush, reps=5):
    for _ in range(3):
        flush.zero_()
        fn()
    torch.cuda.synchronize()
    st = torch.cuda.current_stream()
    tot = 0.0
    for _ in range(reps):
        flush.zero_()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(st)
        fn()
        e1.record(st)
        torch.cuda.synchronize()
        tot += e0.elapsed_time(e1)
    return tot / reps


PEAK_INSTR = N_SM * FP64_LANES_PER_SM * 1.965e9    # FP64 thread-instructions/s at clocks.max.sm


def _oracle_rates(mech, batch, n_sample, jacobian=False):
    """The oracle as it stands on a bounded sample (SURVEY.md 8(d) "Oracle timing"): single thread and all host
    cores, best of 2.  Rates in reactor evaluations (or Jacobians) per second."""
    from oracle import oracle as orc
    om = _oracle_mech(mech)
    sub = batch.take(np.arange(min(n_sample, batch.n)))
    cores = min(orc.max_threads(), orc.host_cores())
    out = {"sample": f"first {sub.n} reactors", "cores": cores}
    for name, nt in (("per_s_1_thread", 1), ("per_s_all_cores", cores)):
        one = sub if nt > 1 else sub.take(np.arange(max(1, sub.n // 8)))
        best = float("inf")
        for _ in range(2):
            t0 = time.perf_counter()
            if jacobian:
                orc.jacobian(om, one.T, one.P, one.Y, one.Yin, one.tau, nthreads=nt)
            else:
                orc.evaluate(om, one.T, one.P, one.Y, one.Yin, one.tau, want=("wdot", "F"), nthreads=nt)
            best = min(best, time.perf_counter() - t0)
        out[name] = one.n / best
    return out


def run_extras(binding, synth, torch, flush, only=None, cpu=True):
    """The other rows of SURVEY.md 8(a)/(f), each timed on its own (mean of 5 launches, L2 flushed): psr_eval_wdot and
    the adiabatic residual on C1, the C2 / C3 residual passes, the C4 FD Jacobian (plain and adiabatic), the Newton
    step's solve, a Newton iteration, and the hybrid solver; beside them the oracle on bounded samples.
    only: run just that leg (ncu captures name it)."""
    out = {}
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    want = lambda k: only is None or only == k
    if want("C1_wdot") or want("C1_energy"):
        mech, batch = synth.make_config("C1")
        gm = binding.Mechanism.from_synth(mech)
        T, P, Y, Yin, tau = (dev(x) for x in (batch.T, batch.P, batch.Y, batch.Yin, batch.tau))
        info = gm.info()
        instr = algorithmic_fp64_instr(mech.n_species, mech.n_reactions, info["n_third_body"], info["n_falloff"], info["nnz_nu"])
        if want("C1_wdot"):   # the metric is wdot evaluations: the call that produces nothing else
            w = torch.empty_like(Y)
            ms = _time_call(torch, lambda: gm.eval_wdot(T, P, Y, wdot=w), flush)
            out["C1_wdot"] = {"call": "psr_eval_wdot", "ms": ms, "reactor_evals_per_s": batch.n / (ms * 1e-3),
                              "alu_frac": instr * batch.n / (ms * 1e-3) / PEAK_INSTR}
        if want("C1_energy"):   # NEXT-1: the adiabatic residual (species rows + energy row)
            Tin = torch.full_like(T, 300.0)
            F, FT = torch.empty_like(Y), torch.empty_like(T)
            ms = _time_call(torch, lambda: gm.eval_residual_energy(T, P, Y, Tin, Yin, tau, F=F, FT=FT), flush)
            out["C1_energy"] = {"call": "psr_eval_residual_energy", "ms": ms, "reactor_evals_per_s": batch.n / (ms * 1e-3)}
        gm.close()
    for cfg in ("C2", "C3"):
        if not want(cfg):
            continue
        mech, batch = synth.make_config(cfg)
        gm = binding.Mechanism.from_synth(mech)
        info = gm.info()
        T, P, Y, Yin, tau = (dev(x) for x in (batch.T, batch.P, batch.Y, batch.Yin, batch.tau))
        instr = algorithmic_fp64_instr(mech.n_species, mech.n_reactions, info["n_third_body"], info["n_falloff"], info["nnz_nu"])
        F, w = torch.empty_like(Y), torch.empty_like(Y)
        ms = _time_call(torch, lambda: gm.eval_residual(T, P, Y, Yin, tau, F=F, wdot=w), flush)
        prof = ncu_summary(cfg + "_residual")
        out[cfg] = {"call": "psr_eval_residual", "ms": ms, "reactor_evals_per_s": batch.n / (ms * 1e-3),
                    "reaction_evals_per_s": batch.n * mech.n_reactions / (ms * 1e-3),
                    "alu_frac": instr * batch.n / (ms * 1e-3) / PEAK_INSTR,
                    "kernel": {k: info[k] for k in ("eval_kernel", "eval_parts", "eval_acc_global")},
                    "hbm_algorithmic_bytes": (3 + 4 * mech.n_species) * 8 * batch.n, "dram_bytes_ncu": prof.get("dram_bytes_per_launch"),
                    "fp64_pipe_util_ncu": prof.get("fp64_pipe_pct"), "ncu_capture": prof.get("capture")}
        if cpu:
            out[cfg]["cpu_oracle"] = _oracle_rates(mech, batch, 2048)
        gm.close()
    if any(want(k) for k in ("C4", "C4_energy", "C4_solve", "C4_newton", "C4_hybrid")):
        mech, batch = synth.make_config("C4")
        gm = binding.Mechanism.from_synth(mech)
        info = gm.info()
        T, P, Y, Yin, tau = (dev(x) for x in (batch.T, batch.P, batch.Y, batch.Yin, batch.tau))
        instr = algorithmic_fp64_instr(mech.n_species, mech.n_reactions, info["n_third_body"], info["n_falloff"], info["nnz_nu"])
        n = mech.n_species + 1
        J = torch.empty((batch.n, n, n), dtype=torch.float64, device="cuda")
        F0 = torch.empty((batch.n, n), dtype=torch.float64, device="cuda")
        if want("C4"):
            ms = _time_call(torch, lambda: gm.fd_jacobian(T, P, Y, Yin, tau, J=J), flush)
            prof = ncu_summary("C4_jacobian")
            out["C4"] = {"call": "psr_fd_jacobian (fused kernel)", "ms": ms, "jacobians_per_s": batch.n / (ms * 1e-3),
                         "residual_evals_per_s": batch.n * (n + 1) / (ms * 1e-3),
                         # BASELINE's unit (55 full evaluations per Jacobian) and SURVEY 8(d)'s hoisted count; the fused
                         # kernel does less work than either, so these compare times, not pipe use
                         "alu_frac_unhoisted": instr * batch.n * (n + 1) / (ms * 1e-3) / PEAK_INSTR,
                         "alu_frac_hoisted": C4_HOISTED_INSTR_PER_JACOBIAN * batch.n / (ms * 1e-3) / PEAK_INSTR,
                         "hbm_GBps_on_J": batch.n * n * n * 8 / (ms * 1e-3) / 1e9,
                         "fp64_pipe_util_ncu": prof.get("fp64_pipe_pct"), "ncu_capture": prof.get("capture")}
            gm.set_option(binding.OPT_JAC_GENERIC, 1)
            ms_g = _time_call(torch, lambda: gm.fd_jacobian(T, P, Y, Yin, tau, J=J), flush)
            gm.set_option(binding.OPT_JAC_GENERIC, 0)
            out["C4"]["generic_sweep_ms"] = ms_g
            if cpu:
                out["C4"]["cpu_oracle"] = _oracle_rates(mech, batch, 256, jacobian=True)
        if want("C4_energy"):
            Tin = torch.full_like(T, 300.0)
            ms_en = _time_call(torch, lambda: gm.fd_jacobian(T, P, Y, Yin, tau, J=J, Tin=Tin), flush)
            out["C4_energy"] = {"call": "psr_fd_jacobian_energy (generic sweep)", "ms": ms_en, "jacobians_per_s": batch.n / (ms_en * 1e-3)}
        if want("C4_solve") or want("C4_newton"):
            gm.fd_jacobian(T, P, Y, Yin, tau, J=J, F0=F0)
            rhs = torch.empty_like(F0)
            dt_inf = torch.full((batch.n,), float("inf"), dtype=torch.float64, device="cuda")
            info_t = torch.empty(batch.n, dtype=torch.int32, device="cuda")
            # NEXT-2: the Newton step's solve J dx = -F0 (psr_ptc_solve with dt = inf reads F0 and negates it itself)
            ms_lu = _time_call(torch, lambda: binding.ptc_solve(J, F0, dt_inf, dx=rhs, info=info_t), flush)
            out["C4_solve"] = {"call": "psr_ptc_solve (dt = inf: the Newton step)", "ms": ms_lu, "systems_per_s": batch.n / (ms_lu * 1e-3),
                               "n": n, "hbm_GBps_on_J": batch.n * n * n * 8 / (ms_lu * 1e-3) / 1e9}
            def newton():
                gm.fd_jacobian(T, P, Y, Yin, tau, J=J, F0=F0)
                binding.ptc_solve(J, F0, dt_inf, dx=rhs, info=info_t)
            ms_n = _time_call(torch, newton, flush)
            out["C4_newton"] = {"call": "psr_fd_jacobian + psr_ptc_solve (one Newton iteration's device work)", "ms": ms_n,
                                "iterations_per_s": batch.n / (ms_n * 1e-3)}
        if want("C4_hybrid"):
            # NEXT-4: the whole hybrid solve from the generated (far) states, the full C4 batch, fixed budget of 420 solves
            nb = 8192
            a0 = [x[..., :nb].contiguous() for x in (T, P, Y, Yin, tau)]
            kw = dict(atol=1e-12, rtol=1e-7, max_iter=420, max_newton=5, max_ptc=20, dt0=1e-9, dt_grow=2.0, dt_shrink=0.25, y_floor=1e-9)
            ws = torch.empty(int(binding.lib().psr_solve_hybrid_workspace_bytes(gm._h, nb)), dtype=torch.uint8, device="cuda")
            def hybrid():
                Tt, Yt = a0[0].clone(), a0[2].clone()
                return gm.solve_hybrid(Tt, a0[1], Yt, a0[3], a0[4], workspace=ws, **kw)
            st, nn, npt = hybrid()
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(torch.cuda.current_stream())
            st, nn, npt = hybrid()
            e1.record(torch.cuda.current_stream())
            torch.cuda.synchronize()
            ms_h = e0.elapsed_time(e1)
            out["C4_hybrid"] = {"call": "psr_solve_hybrid", "reactors": nb, "options": kw, "ms": ms_h,
                                "converged_frac": float((st == 0).float().mean()), "mean_newton": float(nn.float().mean()),
                                "mean_ptc": float(npt.float().mean()), "ms_per_solve_round": ms_h / kw["max_iter"]}
            # the restart case: the converged states perturbed by 1 %, same budget of 420 rounds.  Every reactor finishes
            # within a few Newton iterations; the rounds after the last one are empty launches (finished reactors are
            # counted on the device), so the budget costs little
            Tt, Yt = a0[0].clone(), a0[2].clone()
            st0, _, _ = gm.solve_hybrid(Tt, a0[1], Yt, a0[3], a0[4], workspace=ws, **kw)
            conv = (st0 == 0).nonzero().flatten()
            gen = torch.Generator(device="cuda").manual_seed(17)
            pert = 1.0 + 0.01 * (2.0 * torch.rand((Yt.shape[0], conv.numel()), generator=gen, device="cuda", dtype=torch.float64) - 1.0)
            a1 = [Tt[conv].contiguous(), a0[1][conv].contiguous(), (Yt[:, conv] * pert).contiguous(), a0[3][:, conv].contiguous(),
                  a0[4][conv].contiguous()]
            def restart():
                return gm.solve_hybrid(a1[0].clone(), a1[1], a1[2].clone(), a1[3], a1[4], workspace=ws, **kw)
            st1, nn1, np1 = restart()
            torch.cuda.synchronize()
            e0.record(torch.cuda.current_stream())
            st1, nn1, np1 = restart()
            e1.record(torch.cuda.current_stream())
            torch.cuda.synchronize()
            out["C4_hybrid"]["restart"] = {"reactors": int(conv.numel()), "start": "converged states x (1 +- 1 %)", "ms": e0.elapsed_time(e1),
                                           "converged_frac": float((st1 == 0).float().mean()), "mean_newton": float(nn1.float().mean()),
                                           "mean_ptc": float(np1.float().mean())}
        gm.close()
    return out


# ------------------------------------------------------------------------------ paper-shaped sweep (NEXT-3)
def run_sweep(args):
    """bench.py --sweep: the AXES of the paper's Fig. 5 (one Newton iteration of a batch of
    10^2..10^6 identical reactors, 101 species / 542 reactions, T = 1800 K, tau = 50 ms) on a synthetic
    mechanism of that shape (config P5; the real mechanism [27] is not in this container).  Per batch size:
    the residual pass (device-resident, and with the paper's offload pattern: inputs copied in, outputs copied
    out), and the Newton iteration's device work -- FD Jacobian + linear solve -- up to 10^5 reactors (the
    Jacobians of 10^6 reactors are 83 GB).  The oracle is timed on a bounded sample on the host cores."""
    import torch
    from oracle import oracle as orc
    from paper_2005_11468_b200 import binding, synth
    torch.cuda.set_device(0)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    mech, _ = synth.make_config("P5", 1)
    gm = binding.Mechanism.from_synth(mech)
    n = mech.n_species + 1
    om = _oracle_mech(mech)
    cores = min(orc.max_threads(), orc.host_cores())
    # oracle rates on bounded samples: residual on 4096 reactors, Jacobian + solve on 128
    _, sb = synth.make_config("P5", 4096)
    t_res = min(_wall(lambda: orc.evaluate(om, sb.T, sb.P, sb.Y, sb.Yin, sb.tau, want=("wdot", "F"), nthreads=cores)) for _ in range(3)) / sb.n
    _, jb = synth.make_config("P5", 128)
    def cpu_newton():
        j = orc.jacobian(om, jb.T, jb.P, jb.Y, jb.Yin, jb.tau, nthreads=cores)
        orc.lu_solve(j["J"], -j["F0"])
    t_newton = min(_wall(cpu_newton) for _ in range(2)) / jb.n
    t_res_1 = _wall(lambda: orc.evaluate(om, sb.T[:256], sb.P[:256], sb.Y[:, :256].copy(), sb.Yin[:, :256].copy(), sb.tau[:256],
                                         want=("wdot", "F"), nthreads=1)) / 256
    rows = []
    for N in (100, 1000, 10000, 100000, 1000000):
        _, b = synth.make_config("P5", N)
        T, P, Y, Yin, tau = (dev(x) for x in (b.T, b.P, b.Y, b.Yin, b.tau))
        F = torch.empty_like(Y)
        ms_res = _time_call(torch, lambda: gm.eval_residual(T, P, Y, Yin, tau, F=F), flush)
        hT, hP, hY, hYin, htau = (torch.from_numpy(np.ascontiguousarray(x)).pin_memory() for x in (b.T, b.P, b.Y, b.Yin, b.tau))
        hF = torch.empty(Y.shape, dtype=torch.float64).pin_memory()
        def offload():
            for d_, h_ in ((T, hT), (P, hP), (Y, hY), (Yin, hYin), (tau, htau)):
                d_.copy_(h_, non_blocking=True)
            gm.eval_residual(T, P, Y, Yin, tau, F=F)
            hF.copy_(F, non_blocking=True)
        ms_off = _time_call(torch, offload, flush)
        row = {"batch": N, "residual_ms": ms_res, "residual_offload_ms": ms_off,
               "cpu_residual_ms_all_cores": t_res * N * 1e3, "cpu_residual_ms_1_core": t_res_1 * N * 1e3}
        if N <= 100000:
            J = torch.empty((N, n, n), dtype=torch.float64, device="cuda")
            F0 = torch.empty((N, n), dtype=torch.float64, device="cuda")
            rhs = torch.empty_like(F0)
            def newton():
                gm.fd_jacobian(T, P, Y, Yin, tau, J=J, F0=F0)
                torch.neg(F0, out=rhs)
                binding.lu_solve(J, rhs)
            row["newton_iteration_ms"] = _time_call(torch, newton, flush, reps=3)
            row["cpu_newton_iteration_ms_all_cores"] = t_newton * N * 1e3
            del J, F0, rhs
        rows.append(row)
        del T, P, Y, Yin, tau, F
        torch.cuda.empty_cache()
    gm.close()
    print(json.dumps({"sweep": "paper-shaped (PAPER.md:129-137), synthetic 101 species / 542 reactions, T=1800 K, tau=50 ms, 1 atm",
                      "cpu": {"kind": "oracle", "cores": cores, "sample": "residual: 4096 reactors; Newton iteration (n+1 = 103 residuals + LU): 128 reactors"},
                      "rows": rows}), flush=True)


def _wall(fn):
    t0 = time.perf_counter()
    fn()
    return time.perf_counter() - t0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", choices=("ours", "reference"), default="ours")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--no-extra", action="store_true", help="skip the C2/C3/C4 extras")
    ap.add_argument("--sweep", action="store_true", help="paper-shaped batch sweep (NEXT-3) instead of the headline line")
    ap.add_argument("--only", default=None, help="run just one leg of `extra` (C1_wdot, C1_energy, C2, C3, C4, C4_energy, "
                                                 "C4_solve, C4_newton, C4_hybrid) and print it: what the ncu captures under profiles/ run")
    args = ap.parse_args()
    if args.only:
        import torch
        from paper_2005_11468_b200 import binding, synth
        torch.cuda.set_device(0)
        flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
        print(json.dumps(run_extras(binding, synth, torch, flush, only=args.only, cpu=False)), flush=True)
    elif args.sweep:
        run_sweep(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()

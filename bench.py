#!/usr/bin/env python
"""bench.py -- cell source-term evaluations per second (fp64) and fraction of roofline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--workload mid_1m|tiny_1m|large_256k|...]

A "step" is one pass of the whole hot path (ck_source_terms: every layer of the paper's
ANN form, include/ck.h (1)-(6)) over one batch of seeded synthetic cells.  The default
workload is the one BASELINE.json's metric is quoted on: S=53, R=325, N=2^20 cells, fp64.
Prints ONE JSON line (rank 0).  N>1: launched by torchrun, one process per GPU, cells
sharded across ranks with no collective (weak scaling: N cells per GPU).

--impl reference times the CPU oracle (oracle/, test infrastructure) on the host cores.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "cell source-term evals/sec (fp64) at S=53,R=325; fraction of roofline"
UNIT = "cells/s"


def algorithmic_fp64_instr_per_cell(info, costs=(15, 28, 8)):
    """SURVEY.md section 8(d) / DESIGN.md section 6: algorithmic FP64-pipe instructions per cell,
    FMA / add / mul = 1 and (exp, log, div) = `costs`.  The default (15, 28, 8) is the survey's
    fixed convention (CUDA 12.9's libm fast paths on sm_100a): NORMALISED WORK, which a cheaper
    hand-written exp does not change.  IMPLEMENTED_COSTS are what this library's own ck_exp /
    ck_log / ck_rcp execute; with them the figure is the FP64 issue the kernel really needs."""
    S, R = info["S"], info["R"]
    n_fo = info["n_lindemann"] + info["n_troe"]
    n_exp = 2 * R + 5 * info["n_troe"] + info["n_lindemann"]
    n_log = S + 1 + 2 * n_fo
    n_div = 3 + 3 * n_fo
    fma = 20 * S + 2 * (R + n_fo) + info["nnz_reac"] + 2 * info["nnz_net"] + info["nnz_eff"]
    return fma + costs[0] * n_exp + costs[1] * n_log + costs[2] * n_div


IMPLEMENTED_COSTS = (8, 11, 4)     # ck_exp, ck_log, ck_rcp of csrc/ck_jit_kernel.cuh


class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thread = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def _loop(self):
        nv = self.nv
        names = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "hw_thermal_slowdown": 0x40,
                 "sw_thermal_slowdown": 0x20, "hw_power_brake_slowdown": 0x80,
                 "sync_boost": 0x10, "applications_clocks_setting": 0x2}
        while not self._stop.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                try:
                    mask = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for n, bit in names.items():
                    if mask & bit:
                        self.reasons.add(n)
            except Exception:
                pass
            time.sleep(0.002)

    def __enter__(self):
        if self.nv is not None:
            self._thread = threading.Thread(target=self._loop, daemon=True)
            self._thread.start()
        return self

    def __exit__(self, *exc):
        self._stop.set()
        if self._thread:
            self._thread.join()

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["unavailable"]}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


def time_oracle(mech, T, P, Y, target_s=12.0):
    """Oracle as it stands on a bounded sample of the workload: the first n cells, n grown
    until one pass takes about target_s (or the whole batch, passed over repeatedly)."""
    import oracle
    om = oracle.OracleMechanism(mech)
    n = min(4096, T.shape[0])
    t0 = time.perf_counter()
    _, _, cores = oracle.source_terms(om, T[:n], P[:n], np.ascontiguousarray(Y[:, :n]))
    rate = n / max(time.perf_counter() - t0, 1e-9)
    n = int(min(T.shape[0], max(n, rate * target_s)))
    Ys = np.ascontiguousarray(Y[:, :n])
    passes, t0 = 0, time.perf_counter()
    while passes == 0 or (time.perf_counter() - t0 < 0.8 * target_s and passes < 64):
        oracle.source_terms(om, T[:n], P[:n], Ys)
        passes += 1
    dt = time.perf_counter() - t0
    # one core, beside the paper's one-MPI-rank CPU baseline: about 4 s of work
    n1 = int(min(T.shape[0], max(256, rate / max(int(cores), 1) * 4.0)))
    Y1 = np.ascontiguousarray(Y[:, :n1])
    t1 = time.perf_counter()
    oracle.source_terms(om, T[:n1], P[:n1], Y1, nthreads=1)
    dt1 = time.perf_counter() - t1
    return {"value": passes * n / dt, "unit": UNIT, "cores": int(cores), "kind": "oracle",
            "sample": "first %d cells of the workload x %d passes, %.1f s, OpenMP static over cells"
                      % (n, passes, dt),
            "single_core": {"value": n1 / dt1, "unit": UNIT, "cores": 1,
                            "sample": "first %d cells, one pass, %.1f s, one thread" % (n1, dt1)}}


def sample_parity(mech, T, P, Y, w, d, n=32768):
    """The timed step's own results (device buffers w, d) against the oracle on the first n cells of the
    workload, under the north_star tolerance; `q19_cells` counts the cells whose dT/dt alone is over the
    bound (reading Q19: decided on the energy sum's scale by the tests, 0 on this workload).
    Outside the timed region; part of the cpu_baseline leg (rank 0, N = 1)."""
    import oracle
    n = int(min(n, T.shape[0]))
    wr, dr, _ = oracle.source_terms(oracle.OracleMechanism(mech), T[:n], P[:n], np.ascontiguousarray(Y[:, :n]))
    wg, dg = w[:, :n].cpu().numpy(), d[:n].cpu().numpy()
    tol_w = 1e-10 * np.abs(wr).max(axis=0, keepdims=True) + 1e-12 * np.abs(wr)
    tol_t = 1e-10 * np.abs(dr) + 1e-12
    rw = np.abs(wg - wr) / np.maximum(tol_w, 1e-300)
    rt = np.abs(dg - dr) / tol_t
    finite = bool(np.isfinite(wg).all() and np.isfinite(dg).all())
    return {"cells": n, "finite": finite, "worst_wdot_err_over_tol": float(rw.max()),
            "worst_dTdt_err_over_tol": float(rt.max()), "q19_cells": int((rt > 1.0).sum()),
            "cells_over_wdot_tol": int((rw > 1.0).any(axis=0).sum())}


def run_reference(args, cfg, mech):
    """--impl reference: the CPU oracle on the host cores, rank 0 only."""
    import ckgen
    import oracle
    if int(os.environ.get("RANK", "0")) != 0:
        return
    # each step = the whole workload (the same N as the GPU arm) unless --ref-cells bounds it
    N = args.cells or cfg.N
    n = min(N, args.ref_cells) if args.ref_cells > 0 else N
    T, P, Y = ckgen.states(cfg, N=N)
    T, P, Y = T[:n], P[:n], np.ascontiguousarray(Y[:, :n])
    om = oracle.OracleMechanism(mech)
    cores = 0
    for _ in range(args.warmup):
        _, _, cores = oracle.source_terms(om, T[:4096], P[:4096], np.ascontiguousarray(Y[:, :4096]))
    t0 = time.perf_counter()
    for _ in range(args.steps):
        _, _, cores = oracle.source_terms(om, T, P, Y)
    dt = time.perf_counter() - t0
    value = n * args.steps / dt
    sample = "each step = %s (oracle, OpenMP static)" % (
        "all %d cells of the workload" % n if n == N else "first %d of the workload's %d cells" % (n, N))
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": workload_config(cfg, mech, n),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": int(cores), "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def workload_config(cfg, mech, n_per_gpu):
    S, R = mech.n_species, mech.n_reactions
    step_mb = 8 * (2 * S + 3) * n_per_gpu / 1e6
    return {"workload": "%s: S=%d R=%d N=%d cells per GPU, fp64 SoA T[N] P[N] Y[S][N], seeded "
                        "synthetic mechanism + states (ckgen)" % (cfg.name, S, R, n_per_gpu),
            "S": S, "R": R, "cells_per_gpu": int(n_per_gpu),
            "l2": "no flush: %.0f MB of state in+out per step vs 126 MB L2" % step_mb
                  if step_mb > 126 else "state (%.1f MB per step) is L2 resident" % step_mb}


def run_sweep(args):
    """BASELINE.json configs[4], first half: batch-size saturation sweep at S=53/R=325,
    N = 2^8 .. 2^22 (the paper's Fig. 9 right panel): cells/s and the
    achieved fraction of the FP64 roofline against N.  One JSON line."""
    import torch
    import ckgen
    import paper_2008_08483_b200 as ck
    cfg = ckgen.CONFIGS["mid_1m"]
    mech = ckgen.mechanism(cfg.mech)
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    stream = torch.cuda.current_stream().cuda_stream
    gm = ck.Mechanism(mech)
    info = {k: gm.info(k) for k in ck.INFO}
    i_cell = algorithmic_fp64_instr_per_cell(info)
    peak = ck.ck_measure_fp64_peak(stream)
    S = mech.n_species
    rows = []
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)      # > 126 MB L2
    for N in ckgen.SWEEP_N:
        T, P, Y = ckgen.states(cfg, N=N)
        Td, Pd, Yd = (torch.from_numpy(a).to(dev) for a in (T, P, Y))
        w = torch.empty((S, N), dtype=torch.float64, device=dev)
        d = torch.empty(N, dtype=torch.float64, device=dev)
        for _ in range(max(args.warmup, 3)):
            gm.source_terms(Td, Pd, Yd, w, d, stream=stream)
        reps = 20
        # back to back (state L2-resident when it fits) and with an L2 flush between calls
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        for _ in range(reps):
            gm.source_terms(Td, Pd, Yd, w, d, stream=stream)
        e1.record()
        torch.cuda.synchronize()
        warm_ms = e0.elapsed_time(e1) / reps
        cold = []
        for _ in range(8):
            flush.zero_()
            e0.record()
            gm.source_terms(Td, Pd, Yd, w, d, stream=stream)
            e1.record()
            torch.cuda.synchronize()
            cold.append(e0.elapsed_time(e1))
        cold_ms = float(np.median(cold))
        # every row is checked where it is timed: finite results, mass and element conservation on
        # every cell (the element-by-element comparison with the oracle at these sizes is
        # tests/test_gpu_parity.py::test_sweep_sizes_parity_every_cell)
        assert bool(torch.isfinite(w).all() and torch.isfinite(d).all()), "non-finite result at N=%d" % N
        worst_cons = 0.0
        for wt in [mech.mol_weight] + [mech.elem_count[:, e].astype(float) for e in range(mech.elem_count.shape[1])]:
            terms = torch.from_numpy(wt).to(dev)[:, None] * w
            worst_cons = max(worst_cons, float((terms.sum(0).abs() / (terms.abs().sum(0) + 1e-300)).max()))
            del terms
        assert worst_cons <= 1e-11, "conservation violated at N=%d: %.3g" % (N, worst_cons)
        rows.append({"N": N, "ms_back_to_back": warm_ms, "ms_l2_flushed": cold_ms,
                     "checked": "finite; mass and element conservation residual <= %.1e of the terms on every cell" % worst_cons,
                     "cells_per_s": N / (warm_ms * 1e-3),
                     "roofline_frac": i_cell * N / (warm_ms * 1e-3) / peak,
                     "state_mb": 8 * (2 * S + 3) * N / 1e6})
    print(json.dumps({"sweep": "S=53 R=325 fp64, N = 2^8..2^22, one ck_source_terms call per timing",
                      "fp64_peak_tflops": 2 * peak / 1e12, "fp64_instr_per_cell": i_cell,
                      "launch": {"threads": info["threads"], "blocks_per_sm": info["blocks_per_sm"],
                                 "small_batch_shape_up_to_N": info["small_batch_max"]},
                      "rows": rows}))
    gm.close()


def run_rk4(args):
    """BASELINE.json configs[4], second half: explicit RK4, dt = 1e-9 s, 1000 steps on 65536
    independent cells (T0 ~ U[1100, 1500] K), ck_source_terms once per stage: device time for
    the run with the step replayed from a CUDA graph and with plain launches.  One JSON line."""
    import torch
    import ckgen
    import paper_2008_08483_b200 as ck
    cfg = ckgen.CONFIGS["mid_rk4"]
    mech = ckgen.mechanism(cfg.mech)
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    stream = torch.cuda.current_stream().cuda_stream
    gm = ck.Mechanism(mech)
    N, steps, dt = args.cells or cfg.N, args.rk4_steps, 1e-9
    T, P, Y = ckgen.states(cfg, N=N)
    fused = os.environ.get("CK_RK4_FUSED", "1") != "0" and gm.info("jit") == 1
    out = {"rk4": "S=53 R=325 fp64, N=%d cells, %d steps of dt=%g s, 4 source-term evaluations per step"
                  % (N, steps, dt),
           "stage_update": "fused into the source-term kernel (1 launch per stage)" if fused
                           else "separate kernel (2 launches per stage)"}
    for mode, use_graph in (("graph", True), ("plain_launches", False)):
        Td, Pd, Yd = (torch.from_numpy(a).to(dev) for a in (T, P, Y))
        gm.rk4_integrate(Td, Pd, Yd, dt, 3, use_graph=use_graph, stream=stream)    # warm-up, capture
        Td.copy_(torch.from_numpy(T)); Yd.copy_(torch.from_numpy(Y))
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        e0.record()
        gm.rk4_integrate(Td, Pd, Yd, dt, steps, use_graph=use_graph, stream=stream)
        e1.record()
        torch.cuda.synchronize()
        wall = time.perf_counter() - t0
        ms = e0.elapsed_time(e1)
        ok = bool(torch.isfinite(Td).all() and torch.isfinite(Yd).all())
        out[mode] = {"device_ms": ms, "wall_s": wall, "steps_per_s": steps / (ms * 1e-3),
                     "source_term_calls_per_s": 4 * steps / (ms * 1e-3),
                     "cell_source_term_evals_per_s": 4.0 * steps * N / (ms * 1e-3),
                     "us_per_stage": ms * 1e3 / (4 * steps), "finite": ok}
    print(json.dumps(out))
    gm.close()


def run_ann(args):
    """The paper's Fig. 10 on this implementation: time of the source term
    with the approximate ANN for log Kc (Architecture 2, elu; N_L = 1..3 hidden layers of N_H
    neurons, random weights -- timing needs no trained ones) against the exact equilibrium
    layer, at N_C = 1e5 cells, for the three mechanism shapes.  The kernel is fused, so the
    layer's own cost is measured by ablation: t_none is the same kernel with the equilibrium
    layer removed (CK_JIT_KC=none, a measurement-only variant).  One JSON line."""
    import torch
    import ckgen
    import paper_2008_08483_b200 as ck
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    stream = torch.cuda.current_stream().cuda_stream
    N = args.cells or 100000
    out = {"ann": "Fig. 10 analogue: ck_source_terms at N=%d cells, exact vs approximate-ANN log Kc "
                  "(Architecture 2, elu, random weights); ms per call" % N, "mechanisms": []}

    def timed(gm, bufs):
        Td, Pd, Yd, w, d = bufs
        for _ in range(5):
            gm.source_terms(Td, Pd, Yd, w, d, stream=stream)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        for _ in range(20):
            gm.source_terms(Td, Pd, Yd, w, d, stream=stream)
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / 20

    for name in ("tiny_1m", "mid_1m", "large_256k"):
        cfg = ckgen.CONFIGS[name]
        mech = ckgen.mechanism(cfg.mech)
        S, R = mech.n_species, mech.n_reactions
        T, P, Y = ckgen.states(cfg, N=N)
        bufs = [torch.from_numpy(a).to(dev) for a in (T, P, Y)]
        bufs += [torch.empty((S, N), dtype=torch.float64, device=dev), torch.empty(N, dtype=torch.float64, device=dev)]
        with ck.Mechanism(mech) as gm:
            t_exact = timed(gm, bufs)
        os.environ["CK_JIT_KC"] = "none"          # measurement-only ablation, refused by the library
        os.environ["CK_ALLOW_ABLATION"] = "1"     # unless this is set as well
        try:
            with ck.Mechanism(mech) as gm:
                assert gm.info("ablation") == 1
                t_none = timed(gm, bufs)
        finally:
            del os.environ["CK_JIT_KC"], os.environ["CK_ALLOW_ABLATION"]
        rows = []
        for n_layers in (1, 2, 3):
            for n_hidden in (2, 4, 8, 16, 32):
                ann = ckgen.random_kc_ann(R, n_layers, n_hidden, seed=n_layers * 100 + n_hidden, T_range=cfg.T_range)
                with ck.Mechanism(mech, kc_ann=ann) as gm:
                    t_ann = timed(gm, bufs)
                rows.append({"N_L": n_layers, "N_H": n_hidden, "N_H_over_N_S": n_hidden / S, "ms": t_ann,
                             "speedup_source_term": t_exact / t_ann,
                             "speedup_kc_layer": (t_exact - t_none) / max(t_ann - t_none, 1e-9)})
        out["mechanisms"].append({"S": S, "R": R, "ms_exact": t_exact, "ms_without_kc_layer": t_none,
                                  "kc_share_of_source_term": (t_exact - t_none) / t_exact, "rows": rows})
    print(json.dumps(out))


def run_peaks(args):
    """the FP64 microbenchmarks the roofline and the sparse-vs-dense
    decision rest on (ck_measure_peaks): DFMA rate, DMMA.8x8x4 rate alone and interleaved with
    DFMA, libm exp / log rates.  One JSON line."""
    import torch
    import paper_2008_08483_b200 as ck
    torch.cuda.set_device(0)
    stream = torch.cuda.current_stream().cuda_stream
    with ClockSampler(0) as clocks:
        p = ck.ck_measure_peaks(stream)
    mhz = clocks.max_mhz or 1965.0
    sched = p["sms"] * 4
    fma = p["dfma_per_s"]
    out = {"peaks": "FP64 microbenchmarks, each kernel timed alone (CUDA events, best of 5)", **p,
           "clocks": clocks.summary(),
           "dfma_tflops": 2 * fma / 1e12,
           "dfma_nominal_tflops": p["sms"] * 64 * 2 * mhz * 1e6 / 1e12,
           "dfma_cycles_per_warp_instr_per_scheduler": sched * mhz * 1e6 / (fma / 32),
           "dmma_tflops": 2 * 256 * p["dmma_per_s"] / 1e12,
           "dmma_cycles_per_instr_per_scheduler": sched * mhz * 1e6 / p["dmma_per_s"],
           "dmma_in_dfma_warp_instr": (fma / 32) / p["dmma_per_s"],
           "interleaved_tflops": 2 * (256 * p["dmma_per_s_interleaved"] + p["dfma_per_s_interleaved"]) / 1e12,
           "interleaved_cycles_per_group_per_scheduler": sched * mhz * 1e6 / p["dmma_per_s_interleaved"],
           "imma_cycles_per_instr_per_scheduler": sched * mhz * 1e6 / p["imma_s8_m16n8k32_per_s"],
           "hmma_cycles_per_instr_per_scheduler": sched * mhz * 1e6 / p["hmma_f16_m16n8k16_per_s"],
           "libm_exp_cost_in_dfma": fma / p["libm_exp_per_s"],
           "libm_log_cost_in_dfma": fma / p["libm_log_per_s"]}
    print(json.dumps(out))


def run_precision(args):
    """the reduced-precision variants of the rate layers
    (ck_mech_desc.precision) against the fp64 product: time per call at the config's N and error
    against the fp64 oracle on a sample of the same states -- wdot relative to max_k|wdot_k| per cell,
    dT/dt relative to the scale of the energy sum -- on the three mechanisms as generated and "tamed"
    (mild kinetics whose rates fit fp32).  One JSON line."""
    import torch
    import ckgen
    import oracle
    import paper_2008_08483_b200 as ck
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from helpers import energy_kappa, tame
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    stream = torch.cuda.current_stream().cuda_stream
    n_err = args.cells or 32768
    out = {"precision": "ck_source_terms with precision = f64 | mixed | f32_rates: ms per call at the config's N; "
                        "errors against the fp64 oracle on the first %d cells" % n_err, "rows": []}
    for name in ("tiny_1m", "mid_1m", "large_256k"):
        cfg = ckgen.CONFIGS[name]
        for tamed in (False, True):
            mech = ckgen.mechanism(cfg.mech)
            if tamed:
                mech = tame(mech)
            S = mech.n_species
            T, P, Y = ckgen.states(cfg)
            N = T.shape[0]
            Td, Pd, Yd = (torch.from_numpy(a).to(dev) for a in (T, P, Y))
            w = torch.empty((S, N), dtype=torch.float64, device=dev)
            d = torch.empty(N, dtype=torch.float64, device=dev)
            Ts, Ps, Ys = T[:n_err], P[:n_err], np.ascontiguousarray(Y[:, :n_err])
            wr, dr, _ = oracle.source_terms(oracle.OracleMechanism(mech), Ts, Ps, Ys)
            kap = energy_kappa(mech, Ts, wr)
            for prec, pname in ((0, "f64"), (1, "mixed"), (2, "f32_rates")):
                with ck.Mechanism(mech, precision=prec) as gm:
                    for _ in range(5):
                        gm.source_terms(Td, Pd, Yd, w, d, stream=stream)
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    torch.cuda.synchronize()
                    e0.record()
                    for _ in range(20):
                        gm.source_terms(Td, Pd, Yd, w, d, stream=stream)
                    e1.record()
                    torch.cuda.synchronize()
                    ms = e0.elapsed_time(e1) / 20
                wg, dg = w[:, :n_err].cpu().numpy(), d[:n_err].cpu().numpy()
                e_w = np.abs(wg - wr).max(0) / np.abs(wr).max(0)
                e_t = np.abs(dg - dr) / (kap * np.abs(dr))
                out["rows"].append({"mechanism": "S=%d R=%d%s" % (S, mech.n_reactions, " tamed" if tamed else ""),
                                    "N": N, "precision": pname, "ms": ms, "cells_per_s": N / (ms * 1e-3),
                                    "wdot_err_rel_max_median": float(np.median(e_w)), "wdot_err_rel_max_worst": float(e_w.max()),
                                    "dTdt_err_rel_scale_median": float(np.median(e_t)), "dTdt_err_rel_scale_worst": float(e_t.max()),
                                    "finite": bool(np.isfinite(wg).all() and np.isfinite(dg).all())})
    print(json.dumps(out))


def run_jacobian(args):
    """ck_jacobian, d(wdot, dT/dt)/d(Y, T) for N cells, cell-major
    (S+1)x(S+1) matrices.  HBM-write bound: 8 (S+1)^2 bytes out per cell against 8 (S+2) in.
    Times the three mechanism shapes; the oracle's Jacobian is timed beside it on a bounded
    sample.  One JSON line."""
    import torch
    import ckgen
    import oracle
    import paper_2008_08483_b200 as ck
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    stream = torch.cuda.current_stream().cuda_stream
    try:
        hbm_peak = float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"])
        peak_src = "MEASURED_PEAKS.json hbm_gbs"
    except Exception:
        hbm_peak, peak_src = 6650.0, "fallback 6650 GB/s"
    out = {"jacobian": "ck_jacobian, fp64, J[N][S+1][S+1] cell-major; device-resident inputs, CUDA events",
           "rows": []}
    for name, N in (("tiny_1m", 1 << 20), ("mid_1m", 1 << 16), ("large_256k", 1 << 14)):
        if args.only and name != args.only:
            continue
        if args.cells:
            N = args.cells
        cfg = ckgen.CONFIGS[name]
        mech = ckgen.mechanism(cfg.mech)
        S, R = mech.n_species, mech.n_reactions
        T, P, Y = ckgen.states(cfg, N=N)
        Td, Pd, Yd = (torch.from_numpy(a).to(dev) for a in (T, P, Y))
        J = torch.empty((N, S + 1, S + 1), dtype=torch.float64, device=dev)
        with ck.Mechanism(mech) as gm:
            for _ in range(max(args.warmup, 3)):
                gm.jacobian(Td, Pd, Yd, J, stream=stream)
            reps = max(args.steps, 10) if args.steps != 50 else 20
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            e0.record()
            for _ in range(reps):
                gm.jacobian(Td, Pd, Yd, J, stream=stream)
            e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1) / reps
            cells_per_tile = gm.info("jac_cells")
            kernel = {0: "none", 1: "jacobian_kernel (table-driven, lanes = columns)", 2: "jacobian_kernel_v2 (table-driven, lanes = cells)",
                      3: "ck_jacobian_jit (specialised to the mechanism)"}[gm.info("jac_kernel")]
        bytes_per_cell = 8 * ((S + 1) * (S + 1) + S + 2)
        gbs = bytes_per_cell * N / (ms * 1e-3) / 1e9
        row = {"S": S, "R": R, "N": N, "ms": ms, "cells_per_s": N / (ms * 1e-3), "kernel": kernel, "cells_per_tile": cells_per_tile,
               "roofline": {"bound": "hbm", "achieved": gbs, "peak": hbm_peak, "unit": "GB/s", "frac": gbs / hbm_peak,
                            "bytes_per_cell": bytes_per_cell, "peak_source": peak_src},
               "l2": "output %.0f MB per call vs 126 MB L2" % (8 * (S + 1) ** 2 * N / 1e6)}
        if not args.no_cpu_baseline:
            # the oracle's Jacobian over the first cells of the same batch, in chunks of 8192 cells (its
            # output is 8 (S+1)^2 bytes per cell), for about 10 s of host time or the whole batch
            om = oracle.OracleMechanism(mech)
            n, t0 = 0, time.perf_counter()
            while n < N and time.perf_counter() - t0 < 10.0:
                m = min(N - n, 8192)
                oracle.jacobian(om, T[n:n + m], P[n:n + m], np.ascontiguousarray(Y[:, n:n + m]))
                n += m
            dt = time.perf_counter() - t0
            row["cpu_baseline"] = {"value": n / dt, "unit": "cells/s", "kind": "oracle", "cores": os.cpu_count(),
                                   "sample": "first %d cells of the batch, one pass in chunks of 8192, %.1f s" % (n, dt)}
        out["rows"].append(row)
    print(json.dumps(out))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="mid_1m")
    ap.add_argument("--cells", type=int, default=0, help="override cells per GPU")
    ap.add_argument("--ref-cells", type=int, default=0,
                    help="--impl reference: bound the cells per step (default 0 = the whole workload, as the GPU arm)")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="--gpus N > 1: weak = N cells per GPU (default), strong = one batch of N cells sliced over the GPUs")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--sweep", action="store_true", help="configs[4]: saturation sweep over N (1 GPU)")
    ap.add_argument("--rk4", action="store_true", help="configs[4]: explicit RK4 reactor run (1 GPU)")
    ap.add_argument("--rk4-steps", type=int, default=1000)
    ap.add_argument("--jacobian", action="store_true", help="ck_jacobian throughput and HBM roofline (1 GPU)")
    ap.add_argument("--only", default="", help="--jacobian: only this mechanism's row (tiny_1m, mid_1m, large_256k)")
    ap.add_argument("--ann", action="store_true", help="Fig. 10 analogue: approximate-ANN vs exact log Kc (1 GPU)")
    ap.add_argument("--precision", action="store_true", help="reduced-precision variants: time and error against the fp64 oracle")
    ap.add_argument("--peaks", action="store_true", help="FP64 microbenchmarks: DFMA, DMMA.8x8x4, interleave, libm exp/log")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)
    if args.sweep:
        return run_sweep(args)
    if args.rk4:
        return run_rk4(args)
    if args.ann:
        return run_ann(args)
    if args.jacobian:
        return run_jacobian(args)
    if args.peaks:
        return run_peaks(args)
    if args.precision:
        return run_precision(args)

    import ckgen
    cfg = ckgen.CONFIGS[args.workload]
    mech = ckgen.mechanism(cfg.mech)
    if args.impl == "reference":
        run_reference(args, cfg, mech)
        return

    import torch
    import paper_2008_08483_b200 as ck
    from paper_2008_08483_b200.shard import max_over_ranks, rank_cells

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    S = mech.n_species
    # each rank owns its own cells (cells are independent): no collective.
    # weak: N cells per rank, a different seeded batch each; strong: one batch of N cells sliced
    n_gen, lo, hi, seed_off = rank_cells(args.cells or cfg.N, rank, world, args.scaling)
    T, P, Y = ckgen.states(cfg, N=n_gen, seed_offset=seed_off)
    T, P, Y = T[lo:hi], P[lo:hi], np.ascontiguousarray(Y[:, lo:hi])
    N = hi - lo
    n_job = n_gen if args.scaling == "strong" else world * N       # cells the whole job evaluates per step
    gm = ck.Mechanism(mech)
    info = {k: gm.info(k) for k in ck.INFO}
    if not info["jit"] and os.environ.get("CK_KERNEL") != "generic":
        sys.exit("bench.py: the mechanism-specialised kernel is not in use (%s); refusing to report the "
                 "generic fallback as the product (set CK_KERNEL=generic to time it on purpose)" % gm.note())
    stream = torch.cuda.current_stream().cuda_stream
    Td, Pd, Yd = (torch.from_numpy(a).to(dev) for a in (T, P, Y))
    w = torch.empty((S, N), dtype=torch.float64, device=dev)
    d = torch.empty(N, dtype=torch.float64, device=dev)

    fp64_fma_per_s = ck.ck_measure_fp64_peak(stream)

    for _ in range(args.warmup):
        gm.source_terms(Td, Pd, Yd, w, d, stream=stream)
    barrier()

    # ---- timed region: K steps, device-resident inputs, CUDA events on the launch stream
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    with ClockSampler(local_rank) as clocks:
        barrier()
        ev[0].record()
        for s in range(args.steps):
            gm.source_terms(Td, Pd, Yd, w, d, stream=stream)
            ev[s + 1].record()
        barrier()
    total_ms = ev[0].elapsed_time(ev[-1])
    step_ms = [ev[s].elapsed_time(ev[s + 1]) for s in range(args.steps)]
    kernel_ms = float(np.mean(step_ms))          # one kernel launch per step
    total_ms = max_over_ranks(total_ms, dist, dev)
    value = n_job * args.steps / (total_ms * 1e-3)

    # ---- end to end through the public host entry point (pinned host buffers) ---------
    Th, Ph, Yh = (torch.from_numpy(a).pin_memory() for a in (T, P, Y))
    wh = torch.empty((S, N), dtype=torch.float64).pin_memory()
    dh = torch.empty(N, dtype=torch.float64).pin_memory()
    e2e_steps = max(3, min(args.steps, 10))
    gm.source_terms_host(Th, Ph, Yh, wh, dh, stream=stream)
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        gm.source_terms_host(Th, Ph, Yh, wh, dh, stream=stream)
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    e2e_s = max_over_ranks(e2e_s, dist, dev)
    e2e_value = n_job * e2e_steps / e2e_s
    assert np.array_equal(dh.numpy(), d.cpu().numpy()), "host and device entry points disagree"

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---- roofline of the (single) kernel: FP64-pipe bound -------------------
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    i_cell = algorithmic_fp64_instr_per_cell(info)
    i_cell_impl = algorithmic_fp64_instr_per_cell(info, IMPLEMENTED_COSTS)
    achieved_tflops = 2.0 * i_cell * N / (kernel_ms * 1e-3) / 1e12
    peak_tflops = 2.0 * fp64_fma_per_s / 1e12
    hbm_bytes = 8.0 * (2 * S + 3) * N
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
    ncu = {}
    try:
        ncu = json.load(open(os.path.join(ROOT, "profiles", "traffic.json"))).get(cfg.name) or {}
        if not isinstance(ncu, dict):
            ncu = {"dram_bytes": ncu}
    except Exception:
        pass
    roofline = {
        "bound": "alu", "achieved": achieved_tflops, "peak": peak_tflops, "unit": "TFLOP/s",
        "frac": achieved_tflops / peak_tflops, "traffic": ncu.get("dram_bytes"),
        "kernel": "ck_source_terms_jit" if info["jit"] else "ck::source_terms_kernel",
        "kernel_ms": kernel_ms,
        "fp64_instr_per_cell": i_cell,
        "frac_convention": "normalised work: SURVEY 8(d) counts exp/log/div at CUDA libm cost (15/28/8 FP64 "
                           "instructions); the kernel's own exp/log/rcp take 8/11/4",
        # the same ratio with the costs the kernel implements: the share of the FP64 pipe's issue rate
        # the algorithmic work needs -- the number to hold against ncu's pipe-active counter
        "frac_issue": i_cell_impl * N / (kernel_ms * 1e-3) / fp64_fma_per_s,
        "fp64_instr_per_cell_implemented_costs": i_cell_impl,
        # ncu counters of this kernel on this workload (profiles/traffic.json, from the committed
        # ncu --set full capture; null if that workload was not profiled)
        "fp64_instr_executed_per_cell": ncu.get("fp64_instr_executed_per_cell"),
        # FP64 datapath busy = FP64-pipe counter + DMMA sub-pipe counter (they do not overlap and the
        # first does not see DMMA: profiles/r02_peaks.md)
        "pipe_active_pct": ncu.get("fp64_datapath_busy_pct"),
        "pipe_fp64_pct": ncu.get("pipe_fp64_cycles_active_pct"),
        "pipe_dmma_pct": ncu.get("pipe_dmma_active_pct"),
        "ncu_source": ncu.get("source"),
        "peak_source": "DFMA microbenchmark run by this bench (ck_measure_fp64_peak), x2 flop/FMA; "
                       "nominal 148 SM x 64 lanes x 2 x sm_max_mhz = %.1f TFLOP/s"
                       % (148 * 64 * 2 * (clocks.max_mhz or 1965.0) * 1e6 / 1e12),
        "hbm": {"achieved": hbm_bytes / (kernel_ms * 1e-3) / 1e9, "peak": hbm_peak, "unit": "GB/s",
                "frac": hbm_bytes / (kernel_ms * 1e-3) / 1e9 / hbm_peak,
                "peak_source": "MEASURED_PEAKS.json hbm_gbs" if peaks else "fallback 6650 GB/s"},
    }

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True,
        "scaling": args.scaling, "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(cfg, mech, N),
        "clocks": clocks.summary(),
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(8 * (S + 2) * N),
                "d2h_bytes_per_step": int(8 * (S + 1) * N), "steps": e2e_steps},
        "gpu_launches": int(args.steps * info["launches_per_call"]),
        "roofline": roofline,
        "launch": {"threads": info["threads"], "blocks_per_sm": info["blocks_per_sm"],
                   "smem_bytes": info["smem_bytes"]},
    }
    if world == 1 and not args.no_cpu_baseline:
        out["cpu_baseline"] = time_oracle(mech, T, P, Y)
        out["parity"] = sample_parity(mech, T, P, Y, w, d)
    print(json.dumps(out))
    gm.close()
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

#!/usr/bin/env python
"""bench.py -- QR-CTMRG iterations/s on one B200 (BASELINE.json metric).

A "step" is one pass of the whole hot path: K1..K7 (one QR-CTMRG iteration) plus
K8 (corner spectrum + convergence delta), i.e. what qrctm_run does per
iteration.  Default workload: BASELINE.json configs[4] (d=2, D=7, chi=196), the
configuration the north_star's roofline target is quoted on; `--config` selects
another one.  Inputs are the seeded synthetic tensors of qrctm_inputs.

  value      iterations/s with A, C, T resident in HBM (CUDA events around qrctm_run)
  e2e        iterations/s through the C ABI with HOST buffers: every step copies
             A, C, T from pinned host memory, runs one iteration and copies C, T and
             delta back (copies inside the timed region)
  roofline   the dominant kernel (K4, P.a, FP64 DMMA GEMM): algorithmic flops
             2 chi^2 D^8 per launch / its mean CUDA-event duration in the timed run,
             against the FP64 tensor issue rate measured live by qrctm_probe_fp64
  cpu_baseline  the oracle (NumPy) timed on the host cores, rank 0, bounded sample
  time_to_convergence  the config's own BASELINE.json run (max iterations, tol) from its
             seeded initial environment: iterations done, final delta, device ms

Multi-GPU: the path is one dependent chain on one GPU:
"replicas only" -- each rank runs an independent instance, no collective.

`--impl reference` times the oracle as it stands on the host cores.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

from qrctm_inputs import CONFIGS, gen_named  # noqa: E402

METRIC = "QR-CTMRG iterations/s"
UNIT = "iterations/s"


def step_flops(D, chi):
    b = D * D
    m = chi * b
    return dict(K1=2 * chi ** 3 * b, K2=4 * m * chi ** 2 - (4 / 3) * chi ** 3, K3=2 * m * m * chi,
                K4=2 * chi ** 2 * b ** 4, K5=2 * m * m * chi, K6=4 * chi ** 3 * b)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, pw = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except ValueError:
                continue
            for n, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def aggregate_over_ranks(ms_total, e2e_ms, steps, world, device=None):
    """Whole-job numbers from per-rank times ("replicas only": every rank ran `steps` independent
    iterations): MAX over ranks of the elapsed times, then value = world * steps / max time.
    Works on any torch.distributed backend (nccl on GPUs, gloo in the CPU tests)."""
    if world > 1:
        import torch
        import torch.distributed as dist
        t = torch.tensor([ms_total, e2e_ms], dtype=torch.float64, device=device)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_total, e2e_ms = float(t[0]), float(t[1])
    return dict(ms_total=ms_total, e2e_ms=e2e_ms, ms_per_step=ms_total / steps,
                value=world * steps / (ms_total * 1e-3), e2e_value=world * 1e3 / e2e_ms)


def oracle_time_steps(name, max_steps, budget_s):
    """Time the oracle's QR-CTMRG iteration (qr_step + normalize + spectrum) as it stands."""
    from oracle import ctmrg as o
    try:
        from threadpoolctl import threadpool_info
        cores = max([p.get("num_threads", 1) for p in threadpool_info()] + [1])
    except Exception:
        cores = os.cpu_count()
    A, C0, T0, c = gen_named(name)
    a = o.build_a(A)
    C, T = o.normalize(C0, T0)
    times = []
    t_all = time.perf_counter()
    for _ in range(max_steps):
        t0 = time.perf_counter()
        s = o.qr_step(C, T, a)
        C, T = o.normalize(s["Cn"], s["Tn"])
        o.spectrum(C)
        times.append(time.perf_counter() - t0)
        if time.perf_counter() - t_all > budget_s:
            break
    return times, cores


def oracle_time_one_thread(name, budget_s):
    """The same oracle iteration with the host BLAS limited to ONE thread."""
    try:
        from threadpoolctl import threadpool_limits
    except Exception:
        return None
    with threadpool_limits(limits=1):
        times, _ = oracle_time_steps(name, 3, budget_s)
    tt = times[1:] if len(times) > 1 else times
    return {"ms_per_step": 1e3 * float(np.mean(tt)), "steps": len(tt), "cores": 1}


def oracle_time_eig_step(name, reps):
    """The oracle's standard (eigen) CTMRG step beside its QR step at the same (D, chi): the shape of the paper's claim
    that the standard step is dominated by the eigendecomposition."""
    from oracle import ctmrg as o
    A, C0, T0, c = gen_named(name)
    a = o.build_a(A)
    C, T = o.normalize(C0, T0)
    te, tq = [], []
    for _ in range(reps):
        t0 = time.perf_counter(); o.eig_step(C, T, a); te.append(time.perf_counter() - t0)
        t0 = time.perf_counter(); o.qr_step(C, T, a); tq.append(time.perf_counter() - t0)
    e, q = 1e3 * float(np.min(te)), 1e3 * float(np.min(tq))
    return {"eig_step_ms": e, "qr_step_ms": q, "eig_over_qr": e / q, "reps": reps}


def file_sha16(*paths):
    import hashlib
    h = hashlib.sha256()
    for p in paths:
        h.update(open(p, "rb").read())
    return h.hexdigest()[:16]


def bench_config(pkg, torch, name, steps, warmup, peak_dmma, conv=True, corner_mode=0):
    """it/s, ms/step, per-stage ms, step TFLOP/s and time-to-convergence of one BASELINE.json config on the current
    device (the side configs of the `configs` block; the headline config is timed in main() with the same calls)."""
    A, C0, T0, c = gen_named(name)
    d, D, chi = c["d"], c["D"], c["chi"]
    b = D * D
    fl = step_flops(D, chi)
    if corner_mode == 1:      # K6': the enlarged corner costs a second K3 + K4, then C~ Q and Q^T (C~ Q)
        m = chi * b
        fl = dict(fl); fl["K6"] = 2 * m * m * chi + 2 * chi ** 2 * b ** 4 + 2 * m * m * chi + 2 * m * chi * chi
    h = pkg.QRCTM(d, D, chi)
    h.set_option(pkg.OPT_CORNER_MODE, corner_mode)
    h.set_A(A); h.set_env(C0, T0)
    h.run(warmup + 1, -1.0)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    n0 = h.launch_count()
    torch.cuda.synchronize()
    ev0.record(h.stream)
    it, _ = h.run(steps, -1.0)
    ev1.record(h.stream)
    torch.cuda.synchronize()
    ms = ev0.elapsed_time(ev1) / steps
    launches = h.launch_count() - n0
    h.set_option(pkg.OPT_TIME_STAGES, 1)
    h.run(1, -1.0); h.get_stage_ms(reset=True)
    h.run(steps, -1.0)
    st, nst = h.get_stage_ms(reset=True)
    h.set_option(pkg.OPT_TIME_STAGES, 0)
    out = {"d": d, "D": D, "chi": chi, "value": 1e3 / ms, "unit": UNIT, "ms_per_step": ms, "steps": steps,
           "gpu_launches_per_step": launches / steps,
           "path": ("whole-iteration kernels for tiny problems (K1..K6 one launch, K7 one, K8 one; stages_ms below is the "
                    "general multi-kernel path, timed serially with events)" if launches / steps < 6 else "general"),
           "stages_ms": {k: v / nst for k, v in st.items()},
           "stages_tflops": {k: fl[k.split("_")[0]] / (v / nst * 1e-3) / 1e12 for k, v in st.items()
                             if k.split("_")[0] in fl and v > 0},
           "algorithmic_gflop_per_step": sum(fl.values()) / 1e9,
           "step_tflops": sum(fl.values()) / (ms * 1e-3) / 1e12,
           "step_frac_of_fp64_peak": sum(fl.values()) / (ms * 1e-3) / 1e12 / peak_dmma}
    if conv:
        h.set_env(C0, T0)
        torch.cuda.synchronize()
        ev0.record(h.stream)
        its, dl = h.run(int(c["iters"]), float(c["tol"]))
        ev1.record(h.stream)
        torch.cuda.synchronize()
        out["time_to_convergence"] = {"iterations": int(its), "max_iter": int(c["iters"]), "tol": float(c["tol"]),
                                      "final_delta": float(dl), "converged": bool(dl < c["tol"]),
                                      "ms": ev0.elapsed_time(ev1)}
    h.close()
    return out


def run_reference(args, rank, world):
    if rank != 0:
        return
    name = args.config
    c = CONFIGS[name]
    total = args.steps + args.warmup
    times, cores = oracle_time_steps(name, total, budget_s=150.0)
    timed = times[args.warmup:] if len(times) > args.warmup else times[-1:]
    ms = 1e3 * float(np.mean(timed))
    val = 1e3 / ms
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
        "steps": len(timed), "warmup": min(args.warmup, len(times) - len(timed)), "ms_per_step": ms,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"{name}: d={c['d']} D={c['D']} chi={c['chi']} seed={c['seed']} (BASELINE.json configs)",
                   "step": "oracle qr_step + normalize + spectrum (NumPy FP64, host BLAS)"},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": f"{len(timed)} full iterations of {name} after {len(times) - len(timed)} warm-up"},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="cfg4", choices=sorted(CONFIGS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-next", action="store_true",
                    help="skip the side measurements outside the timed region: the NEXT-1/2/4 variants and the "
                         "time-to-convergence run")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return
    if args.warmup < 3:
        args.warmup = 3

    import torch
    import torch.distributed as dist
    import paper_2505_00494_b200 as pkg
    from paper_2505_00494_b200 import build as qbuild

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl")
    if rank == 0:
        qbuild.build()
    if world > 1:
        dist.barrier()

    name = args.config
    A, C0, T0, c = gen_named(name)
    d, D, chi = c["d"], c["D"], c["chi"]
    b = D * D
    fl = step_flops(D, chi)

    h = pkg.QRCTM(d, D, chi)
    h.set_A(A)
    h.set_env(C0, T0)
    h.run(args.warmup, -1.0)                 # warm-up (tol < 0: never stops early)
    peak_dmma = pkg.probe_fp64(1)
    peak_dfma = pkg.probe_fp64(0)

    # ---- device-resident timing: K steps, barrier + sync on both sides, CUDA events
    h.run(1, -1.0)
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    n0 = h.launch_count()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    ev0.record(h.stream)                 # events on the stream the kernels are launched on
    it, delta = h.run(args.steps, -1.0)
    ev1.record(h.stream)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    ms_total = ev0.elapsed_time(ev1)
    launches = h.launch_count() - n0
    assert it == args.steps
    # second pass, same K steps, strictly serial with CUDA events around every stage of every step:
    # the per-kernel durations the roofline object is computed from
    h.set_option(pkg.OPT_TIME_STAGES, 1)
    h.run(1, -1.0)
    h.get_stage_ms(reset=True)
    h.run(args.steps, -1.0)
    stage_ms, nst = h.get_stage_ms(reset=True)
    clocks = sampler.stop() if rank == 0 else None
    h.set_option(pkg.OPT_TIME_STAGES, 0)
    assert nst == args.steps

    # ---- bandwidth-bound stages (L2-resident at these sizes, reported against the measured HBM copy rate)
    Ad = torch.from_numpy(A).cuda()
    for _ in range(2):
        h.set_A(Ad)
    torch.cuda.synchronize()
    ev0.record(h.stream)
    for _ in range(5):
        h.set_A(Ad)
    ev1.record(h.stream)
    torch.cuda.synchronize()
    k0_ms = ev0.elapsed_time(ev1) / 5
    k0_bytes = 8 * (b ** 4) + 8 * 3 * d * D ** 4                  # a written; A read, two layered copies of A written
    k7_ms = stage_ms["K7_normalize"] / nst
    k7_bytes = 8 * (chi * chi + chi * b * chi) * 5                 # pass 1: read x2 (symmetrisation partner) + write, pass 2: read + write
    hbm_peak = None
    try:
        hbm_peak = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]
    except Exception:
        hbm_peak = 6650.0                                          # guide fallback
    hbm_kernels = {
        "peak_gbs": hbm_peak,
        "K0_build_a": {"ms": k0_ms, "gbytes": k0_bytes / 1e9, "gbs": k0_bytes / (k0_ms * 1e-3) / 1e9,
                       "frac": k0_bytes / (k0_ms * 1e-3) / 1e9 / hbm_peak},
        "K7_normalize": {"ms": k7_ms, "gbytes": k7_bytes / 1e9, "gbs": k7_bytes / (k7_ms * 1e-3) / 1e9,
                         "frac": k7_bytes / (k7_ms * 1e-3) / 1e9 / hbm_peak,
                         "note": "two launches over an L2-resident 15 MB working set: launch-latency-bound"},
    }

    # ---- time to convergence (north_star: "iterations/s and time-to-convergence"): the config's own run from its seeded
    # initial environment, qrctm_run(iters, tol) with the default check interval (every step); outside the timed region
    conv = None
    if rank == 0 and not args.no_next:
        h.set_env(C0, T0)
        torch.cuda.synchronize()
        ev0.record(h.stream)
        its, dl = h.run(int(c["iters"]), float(c["tol"]))
        ev1.record(h.stream)
        torch.cuda.synchronize()
        conv = {"iterations": int(its), "max_iter": int(c["iters"]), "tol": float(c["tol"]), "final_delta": float(dl),
                "converged": bool(dl < c["tol"]), "ms": ev0.elapsed_time(ev1),
                "note": "BASELINE.json run of this config: qrctm_run(max_iter, tol) from the seeded C0, T0; "
                        "delta = max_i |s_i - s_i^prev| of the normalised corner spectrum, checked every step"}
        h.set_env(C0, T0)
        h.run(2, -1.0)

    # ---- NEXT-1 variant: layered absorption, same result up to rounding, own flop count
    layered = None
    if chi % 2 == 0 and not args.no_next:
        h.set_option(pkg.OPT_ABSORB_MODE, 1)
        h.set_env(C0, T0)
        h.run(args.warmup, -1.0)
        torch.cuda.synchronize()
        ev0.record(h.stream)
        h.run(args.steps, -1.0)
        ev1.record(h.stream)
        torch.cuda.synchronize()
        lay_ms = ev0.elapsed_time(ev1) / args.steps
        h.set_option(pkg.OPT_TIME_STAGES, 1)
        h.run(1, -1.0)
        h.get_stage_ms(reset=True)
        h.run(args.steps, -1.0)
        lst, ln = h.get_stage_ms(reset=True)
        h.set_option(pkg.OPT_TIME_STAGES, 0)
        k4l = lst["K4_absorb_a"] / ln
        fl_l = 4 * d * chi ** 2 * D ** 6
        by_l = 8 * ((chi * b) ** 2 * 2 + 2 * d * b * chi * chi * b)      # P read, S written, P1 written + read
        layered = {"value": 1e3 / lay_ms, "unit": UNIT, "ms_per_step": lay_ms, "k4_ms": k4l,
                   "k4_algorithmic_gflop": fl_l / 1e9, "k4_tflops": fl_l / (k4l * 1e-3) / 1e12,
                   "k4_algorithmic_gbytes": by_l / 1e9, "k4_gbs": by_l / (k4l * 1e-3) / 1e9,
                   "note": "QRCTM_OPT_ABSORB_MODE=1: P contracted with the ket and bra copies of A in turn "
                           "(4 d chi^2 D^6 flops instead of 2 chi^2 D^8); not the headline path (the north_star's "
                           "roofline target is quoted on the explicit double-layer tensor); QRCTM_OPT_ABSORB_MODE=2 "
                           "(automatic) selects it for D >= 6",
                   "auto_mode_selects": "layered" if D >= 6 and 4 * d <= b else "explicit"}
        h.set_option(pkg.OPT_ABSORB_MODE, 0)
        h.set_env(C0, T0)
        h.run(2, -1.0)

    # ---- NEXT-2: the paper's warm-up -- bulk initialisation + one standard (eigen) step growing
    # chi from D^2 -- and one eigen step at the full chi, for the EIGH-vs-QR step-time ratio.
    warm = None
    if b <= chi and chi * b <= 14000 and rank == 0 and not args.no_next:
        h.warmup(1)
        torch.cuda.synchronize()
        ev0.record(h.stream)
        h.warmup(1)
        ev1.record(h.stream)
        torch.cuda.synchronize()
        wu_ms = ev0.elapsed_time(ev1)
        chi_w = h.chi
        warm = {"warmup_ms": wu_ms, "chi_after": chi_w, "eigen_matrix_n": b * b,
                "what": "qrctm_warmup(1): bulk initialisation + one eigen step D^2 -> min(chi, D^4)"}
        if chi_w == chi:
            ev0.record(h.stream)
            h.eig_step()
            ev1.record(h.stream)
            torch.cuda.synchronize()
            es_ms = ev0.elapsed_time(ev1)
            n_e = chi * b
            tri_bytes = 8.0 * n_e ** 3 / 3.0           # upper triangle of the trailing block read + written once per reflector
            warm.update({"eig_step_ms": es_ms, "eig_step_n": n_e,
                         "eig_over_qr_step_time": es_ms / (ms_total / args.steps),
                         "tridiag_algorithmic_gbytes": tri_bytes / 1e9,
                         "eig_step_gbs_lower_bound": tri_bytes / (es_ms * 1e-3) / 1e9,
                         "note": "the whole eigen step (C~ build, tridiagonalisation, multisection, inverse iteration, "
                                 "back-transform, T' contraction) divided into the tridiagonalisation's bytes alone"})
        h.set_env(C0, T0)
        h.run(2, -1.0)

    # ---- NEXT-4: per-rank compute of the sharded iteration, measured on this one GPU.  The
    # exchange (all-gather of T' slices + all-reduce of C') needs more than one GPU and is NOT in these numbers.
    shard = None
    if rank == 0 and world == 1 and not args.no_next:
        shard = {"what": "qrctm_shard_front(rank 0, nranks) on one GPU: K1+K2 replicated, K3-K6 on chi/nranks columns of Q; "
                         "exchange not included", "front_ms": {}}
        for nr in (1, 2, 4, 8):
            if nr > chi:
                continue
            for _ in range(2):
                h.shard_front(0, nr)
            torch.cuda.synchronize()
            ev0.record(h.stream)
            for _ in range(3):
                h.shard_front(0, nr)
            ev1.record(h.stream)
            torch.cuda.synchronize()
            shard["front_ms"][str(nr)] = ev0.elapsed_time(ev1) / 3
        shard["exchange_bytes_per_rank"] = {"all_gather_T": 8 * chi * b * chi, "all_reduce_C": 8 * chi * chi}
        h.set_env(C0, T0)
        h.run(2, -1.0)

    # ---- end to end through the C ABI with host buffers (pinned), copies inside the timed region
    Ah = torch.from_numpy(A).pin_memory()
    Ch, Th = torch.from_numpy(C0).pin_memory(), torch.from_numpy(T0).pin_memory()
    Co = torch.empty((chi, chi), dtype=torch.float64).pin_memory()
    To = torch.empty((chi, b, chi), dtype=torch.float64).pin_memory()
    import ctypes
    lib = h.lib
    P = ctypes.c_void_p

    bufs = {"in": (Ch, Th), "out": (Co, To)}

    def e2e_step():
        ci, ti = bufs["in"]
        co, to = bufs["out"]
        assert lib.qrctm_set_A(h._h, P(Ah.data_ptr())) == 0
        assert lib.qrctm_set_env(h._h, P(ci.data_ptr()), P(ti.data_ptr())) == 0
        its, dl = h.run(1, -1.0)
        assert lib.qrctm_get_env(h._h, P(co.data_ptr()), P(to.data_ptr())) == 0
        bufs["in"], bufs["out"] = (co, to), (ci, ti)   # next step continues from the returned environment
        return dl

    for _ in range(2):
        e2e_step()
    torch.cuda.synchronize()
    e2e_n = max(3, min(args.steps, 10))
    t0 = time.perf_counter()
    for _ in range(e2e_n):
        e2e_step()
    torch.cuda.synchronize()
    e2e_ms = 1e3 * (time.perf_counter() - t0) / e2e_n
    h2d = 8 * (A.size + C0.size + T0.size)
    d2h = 8 * (C0.size + T0.size) + 8

    # ---- max over ranks
    agg = aggregate_over_ranks(ms_total, e2e_ms, args.steps, world, device="cuda")
    ms_total, e2e_ms = agg["ms_total"], agg["e2e_ms"]
    ms_per_step, value, e2e_value = agg["ms_per_step"], agg["value"], agg["e2e_value"]

    if rank == 0:
        k4_ms = stage_ms["K4_absorb_a"] / nst
        ach = fl["K4"] / (k4_ms * 1e-3) / 1e12
        # DRAM traffic of the K4 kernel: not measurable inside this process (it needs ncu's dram__bytes counters), so it
        # is the figure of the committed ncu --set full capture -- reported ONLY while the GEMM sources still hash to
        # what that capture profiled (profiles/k4_traffic_bytes.txt: config, bytes, sha16 of gemm_f64.cuh+gemm_launch.cuh)
        traffic, traffic_note = None, "no capture for this config"
        csrc = os.path.join(ROOT, "paper_2505_00494_b200", "csrc")
        src_sha = file_sha16(os.path.join(csrc, "gemm_f64.cuh"), os.path.join(csrc, "gemm_launch.cuh"))
        tpath = os.path.join(ROOT, "profiles", "k4_traffic_bytes.txt")
        if os.path.exists(tpath):
            for ln in open(tpath):
                f = ln.split()
                if len(f) == 3 and f[0] == name:
                    if f[2] == src_sha:
                        traffic, traffic_note = int(f[1]), f"profiles/r2_k4_gemm_ws_ncu.md (GEMM sources sha16 {src_sha})"
                    else:
                        traffic_note = f"stale: capture was of GEMM sources {f[2]}, now {src_sha}"
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{name}: d={d} D={D} chi={chi} seed={c['seed']} (BASELINE.json configs)",
                       "step": "K1..K7 + K8 spectrum check every step (qrctm_run; K8 of step k overlaps K1..K6 of step k+1 on a side stream)",
                       "l2": "inputs larger than L2 (P and S are %.0f MB each; L2 126 MB)" % (8e-6 * (chi * b) ** 2)
                             if 8 * (chi * b) ** 2 > 126e6 else "working set smaller than L2: L2-resident by design, no flush",
                       "multi_gpu": "replicas only"},
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "ms_per_step": e2e_ms},
            "gpu_launches": int(launches),
            "clocks": clocks,
            "roofline": {"bound": "tensor", "kernel": "gemm_f64_dmma (K4: S = P.a)", "achieved": ach,
                         "peak": peak_dmma, "unit": "TFLOP/s", "frac": ach / peak_dmma, "traffic": traffic, "traffic_source": traffic_note,
                         "peak_source": "FP64 DMMA issue rate measured live by qrctm_probe_fp64 "
                                        "(MEASURED_PEAKS.json has no FP64 entry; nominal 148 SM x 64 FMA/clk x 1.965 GHz = 37.2)",
                         "dfma_peak": peak_dfma, "algorithmic_flops_per_launch": fl["K4"], "ms_per_launch": k4_ms},
            "stages_ms": {k: v / nst for k, v in stage_ms.items()},
            "stages_tflops": {k: fl[k.split("_")[0]] / (v / nst * 1e-3) / 1e12 for k, v in stage_ms.items()
                              if k.split("_")[0] in fl and v > 0},
            "hbm_kernels": hbm_kernels,
            "time_to_convergence": conv,
            "next_1_layered": layered,
            "next_2_warmup": warm,
            "next_4_shard": shard,
            "step_tflops": sum(fl.values()) / (ms_per_step * 1e-3) / 1e12,
            "step_frac_of_fp64_peak": sum(fl.values()) / (ms_per_step * 1e-3) / 1e12 / peak_dmma,
        }
        if not args.no_next:
            side = [n_ for n_ in ("cfg0", "cfg1", "cfg2", "cfg3a", "cfg3b", "cfg4") if n_ != name]
            line["configs"] = {n_: bench_config(pkg, torch, n_, args.steps, args.warmup, peak_dmma) for n_ in side}
            # K6' (the enlarged-corner route, "the standard diagram on the left-hand side" of Fig. 1(f))
            # under its own flop count (cfg2 and cfg4)
            line["corner_mode_1"] = {n_: bench_config(pkg, torch, n_, max(3, args.steps // 4), args.warmup, peak_dmma,
                                                       conv=False, corner_mode=1) for n_ in ("cfg2", "cfg4")}
        if not args.no_cpu_baseline and world == 1:
            budget = 20.0
            times, cores = oracle_time_steps(name, 50, budget_s=budget)
            tt = times[1:] if len(times) > 1 else times
            cms = 1e3 * float(np.mean(tt))
            line["cpu_baseline"] = {"value": 1e3 / cms, "unit": UNIT, "cores": cores, "kind": "oracle",
                                    "sample": f"{len(tt)} full iterations of {name} (oracle qr_step+normalize+spectrum, "
                                              f"NumPy {np.__version__}), first one discarded" if len(times) > 1 else
                                              f"1 iteration of {name}",
                                    "ms_per_step": cms}
            one = oracle_time_one_thread(name, 25.0)
            if one:
                line["cpu_baseline"]["one_thread"] = one
            line["cpu_baseline"]["eig_step_vs_qr_step"] = {n_: oracle_time_eig_step(n_, 3) for n_ in ("cfg1", "cfg2")}
            line["cpu_baseline"]["eig_step_vs_qr_step"]["note"] = (
                "oracle eig_step (enlarged corner + full LAPACK eigh) beside oracle qr_step at the same (D, chi): the "
                "shape of PAPER.md:40's claim (standard CTMRG dominated by the eigendecomposition)")
        print(json.dumps(line), flush=True)
    h.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

#!/usr/bin/env python
"""bench.py -- headline measurement of the hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config cfg3] [--batch 1]

A "step" is one pass of the whole hot path (rows A1-A8: rhs projection, n_iter CG iterations, target projection)
over one batch of seeded synthetic slope frames.  Prints ONE JSON line (see DESIGN.md for every key).
Multi-GPU = independent replicas of the plan: frames are dealt to ranks, no data-path collective.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "us per CG iteration & reconstructions/s at 74x74x6LGS; % of HBM/L2 roofline"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="cfg3")
    ap.add_argument("--batch", type=int, default=1)
    ap.add_argument("--n-iter", type=int, default=0, help="CG iterations per solve (0 = the config's count)")
    ap.add_argument("--solver", default=os.environ.get("TOMO_SOLVER", "persistent"), choices=["multikernel", "persistent"])
    ap.add_argument("--precision", default="f32", choices=["f32", "f32s_f64a", "f64"])
    ap.add_argument("--method", default="cg", choices=["cg", "minres"],
                    help="cg (north_star's solver, the headline) or minres (the paper's solver for the Toeplitz method, same persistent kernel)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    return ap.parse_args()


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    return 6650.0, "fallback (B200_PROFILING.md)"


# ------------------------------------------------------------------------------------------------ clocks
class ClockSampler:
    """Samples SM clock and throttle reasons with NVML while the timed regions run."""

    def __init__(self, index: int):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._t = None
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
        names = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20,
                 "hw_power_brake_slowdown": 0x80, "sync_boost": 0x10}
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(0.02)

    def start(self):
        if self.nv is not None:
            self._t = threading.Thread(target=self._run, daemon=True)
            self._t.start()

    def stop(self):
        self._stop.set()
        if self._t is not None:
            self._t.join()
        return {"sm_mhz": statistics.median(self.samples) if self.samples else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ------------------------------------------------------------------------------------------------ reference arm
def _oracle_generator_rows(job):
    from oracle import toeplitz as tz
    (n, d, dirs, h_gs, h, frac, r0, L0, model, i) = job
    return tz.css_generators(n, d, dirs, h_gs, h, frac, r0, L0, model, wfs_rows=[i])


def oracle_setup(cfg, n_iter, whole):
    """The fp64 oracle, as it stands, on a bounded sample of the workload.  Returns (step, description, cores, extrapolated);
    step() runs the sample once and returns the seconds per reconstruction it implies.
    tiny / mid sizes: the dense oracle's full CG solve + projection.
    ELT sizes, whole = True (the reference arm): the WHOLE step -- n_iter matrix-free direct-sum products (oracle/directsum.c,
    OpenMP) inside the oracle's CG, then the matrix-free target projection; the oracle's generator table (its one-time setup,
    like the library's plan build) is built once, one process per output WFS.
    ELT sizes, whole = False (the cpu_baseline leg of the GPU arm, which must stay short): the median of five timed direct-sum
    products, times n_iter -- an extrapolation, flagged as such; the projection is left out."""
    import numpy as np
    from oracle import directsum
    from oracle import toeplitz as tz
    from oracle.system import OracleSystem
    from tomo_inputs import screens
    cores = len(os.sched_getaffinity(0))
    if 2 * cfg.n_wfs * cfg.n * cfg.n <= 6000:
        osys = OracleSystem(cfg)
        s = screens.generate(cfg, osys.sigma2)["slopes"].ravel()

        def step():
            t0 = time.perf_counter()
            x, _ = osys.solve_cg(s, n_iter)
            osys.reconstruct(x, 0)
            return time.perf_counter() - t0
        return step, f"dense fp64 oracle: full {n_iter}-iteration CG solve + projection", cores, False
    osys = OracleSystem(cfg, dense=False)
    if whole:
        from concurrent.futures import ProcessPoolExecutor
        jobs = [(cfg.n, cfg.d, osys.dirs, osys.h_gs, list(cfg.h), list(cfg.frac), cfg.r0, cfg.L0, osys.model, i) for i in range(osys.N)]
        with ProcessPoolExecutor(max_workers=min(osys.N, cores)) as ex:
            osys.theta = sum(ex.map(_oracle_generator_rows, jobs))
        s = np.asarray(screens.generate(cfg, osys.sigma2)["slopes"][0].ravel(), dtype=np.float64)

        def step():
            t0 = time.perf_counter()
            x, _ = osys.solve_cg(s, n_iter)
            for t in range(len(cfg.targets)):
                osys.reconstruct(x, t)
            return time.perf_counter() - t0
        return step, (f"matrix-free fp64 oracle, whole step: {n_iter} direct-sum Sigma_ss products (oracle/directsum.c, OpenMP) in the "
                      f"oracle's CG + the matrix-free projection to {len(cfg.targets)} target(s)"), cores, False
    # the direct sum's cost does not depend on the generator values: only the rows of WFS 0 are built (the oracle's
    # numpy generator build takes minutes for all N^2 pairs); the product itself is timed in full
    theta = tz.css_generators(cfg.n, cfg.d, osys.dirs, osys.h_gs, cfg.h, cfg.frac, cfg.r0, cfg.L0, wfs_rows=[0])
    v = np.random.default_rng(1).standard_normal(osys.Ns)
    directsum.css_mvm(theta, osys.ix, osys.iy, v)

    def step():
        ts = []
        for _ in range(5):
            t0 = time.perf_counter()
            directsum.css_mvm(theta, osys.ix, osys.iy, v)
            ts.append(time.perf_counter() - t0)
        return statistics.median(ts) * n_iter
    return step, (f"matrix-free fp64 oracle (oracle/directsum.c, OpenMP): median of 5 timed direct-sum Sigma_ss products "
                  f"x {n_iter} iterations (extrapolated; target projection not included)"), cores, True


def workload_config(cfg, plan_P, plan_P_os, n_iter, batch, solver, method, world):
    return {"workload": cfg.name, "n": cfg.n, "n_wfs": cfg.n_wfs, "n_layers": cfg.n_layers, "pad": plan_P, "pad_os": plan_P_os,
            "n_iter": n_iter, "batch": batch, "targets": len(cfg.targets), "solver": solver, "method": method,
            "parallelism": f"replicas x{world}", "l2": "flushed (256 MiB write) before every timed step"}


def run_reference(args, cfg, n_iter, rank):
    if rank != 0:
        return
    from paper_1806_07938_b200 import tomo
    step, desc, cores, extrapolated = oracle_setup(cfg, n_iter, whole=True)
    elt = 2 * cfg.n_wfs * cfg.n * cfg.n > 6000
    w = 0 if elt else min(max(args.warmup, 0), 2)           # a whole ELT step takes the oracle around half a minute
    for _ in range(w):
        step()
    k = max(1, min(args.steps, 1 if elt else 5))
    sec = statistics.mean(step() for _ in range(k))
    val = 1.0 / sec
    sz = tomo.host_sizes(cfg, cfg.pad, cfg.pad_os)
    config = workload_config(cfg, sz["P"], sz["P_os"], n_iter, 1, "oracle (fp64, host cores)", "cg", 1)
    config["l2"] = "n/a (host)"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": "reconstructions/s", "n_gpus": args.gpus,
            "steps": k, "warmup": w, "ms_per_step": sec * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": config,
            "us_per_cg_iteration": sec / n_iter * 1e6, "extrapolated": extrapolated,
            "cpu_baseline": {"value": val, "unit": "reconstructions/s", "cores": cores, "kind": "oracle", "sample": desc},
            "e2e": {"value": val, "unit": "reconstructions/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------------ our arm
def respawn_under_torchrun(args):
    """`python bench.py --gpus N` with no rendezvous in the environment: start the N ranks ourselves (one process per GPU,
    torch.distributed.run on 127.0.0.1) and let rank 0 print the line."""
    import socket
    import subprocess
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    raise SystemExit(subprocess.call(cmd))


def kernel_source_hash():
    """sha256 (16 hex digits) of the persistent kernel's sources: ties a stored ncu traffic figure to the code it was taken from."""
    import hashlib
    h = hashlib.sha256()
    for f in ("persist_kernel.cuh", "persist_host.cuh", "solve_persistent.cu", "fft_reg.cuh"):
        h.update(open(os.path.join(ROOT, "paper_1806_07938_b200", "csrc", f), "rb").read())
    return h.hexdigest()[:16]


def stored_traffic(workload, batch, precision, method="cg"):
    """dram__bytes_read.sum + dram__bytes_write.sum of one k_persistent launch from the committed ncu capture
    (profiles/r2_traffic.json), or None when there is none for this (workload, batch, precision, method) or the kernel has changed since."""
    p = os.path.join(ROOT, "profiles", "r2_traffic.json")
    if not os.path.exists(p):
        return None
    for e in json.load(open(p)).get("entries", []):
        if (e["workload"], e["batch"], e["precision"], e.get("method", "cg")) == (workload, batch, precision, method) and e["kernel_source_hash"] == kernel_source_hash():
            return e["dram_bytes_per_launch"]
    return None


def main():
    args = parse()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        respawn_under_torchrun(args)
    from tomo_inputs.configs import get_config
    cfg = get_config(args.config)
    n_iter = args.n_iter or cfg.n_iter
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, cfg, n_iter, rank)
        return

    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_1806_07938_b200 import tomo
    from paper_1806_07938_b200.replicas import barrier, max_over_ranks
    from tomo_inputs import screens

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the library has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    prec = {"f32": tomo.TOMO_F32, "f32s_f64a": tomo.TOMO_F32S_F64A, "f64": tomo.TOMO_F64}[args.precision]
    solver = tomo.TOMO_SOLVER_PERSISTENT if args.solver == "persistent" else tomo.TOMO_SOLVER_MULTIKERNEL
    B = args.batch
    t0 = time.perf_counter()
    plan = tomo.TomoPlan(cfg, max_batch=B, precision=prec, solver=solver)
    t_plan = time.perf_counter() - t0
    # the solver that RUNS the plan (decided by the library at upload: a plan the persistent kernel cannot take falls back to the
    # multi-kernel solver, e.g. n = 128 with max_batch 16 does not fit its shared-memory layout); every number below is labelled with it
    sv, solver_note = plan.solver_in_use()
    solver_used = "persistent" if sv == tomo.TOMO_SOLVER_PERSISTENT else "multikernel"
    sigma2 = float(plan.noise()[0][0])
    # every rank (replica) gets its own frames: seed offset by rank
    data = screens.generate(cfg, sigma2, n_frames=B, seed_offset=10 * rank)
    h_slopes = torch.from_numpy(np.ascontiguousarray(data["slopes"].reshape(B, -1), dtype=np.float32)).pin_memory()
    d_slopes = h_slopes.cuda()
    d_out = torch.empty(B * plan.wavefront_len, dtype=torch.float32, device="cuda")
    stream = torch.cuda.current_stream()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")     # > 126 MB L2
    minres = args.method == "minres"

    def solve(n_it):
        if minres:
            plan.solve_minres(d_slopes, d_out, B, n_it, stream=stream)
        else:
            plan.solve_batch(d_slopes, d_out, B, n_it, stream=stream)

    def timed(n_it, steps, do_flush=True):
        """device time of `steps` solves, each bracketed by its own CUDA events (the L2 flush is outside)."""
        evs = []
        for _ in range(steps):
            if do_flush:
                flush.zero_()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            solve(n_it)
            b.record(stream)
            evs.append((a, b))
        torch.cuda.synchronize()
        return sum(a.elapsed_time(b) for a, b in evs)

    for _ in range(max(args.warmup, 3)):
        solve(n_iter)
        solve(0)
    torch.cuda.synchronize()
    launches = plan.stats()["launches_last_solve"]
    solve(n_iter)
    launches = plan.stats()["launches_last_solve"]

    sampler = ClockSampler(local_rank)
    sampler.start()
    barrier(world)
    torch.cuda.synchronize()
    ms_total = timed(n_iter, args.steps)                # THE timed region: exactly K steps
    torch.cuda.synchronize()
    barrier(world)
    ms_total = max_over_ranks(ms_total, world)
    ms_step = ms_total / args.steps
    k0 = max(3, min(args.steps, 50))
    ms_step0 = max_over_ranks(timed(0, k0), world) / k0             # A1 + A7-A8 only -> per-iteration time by difference
    # L2-warm steady state (what a real-time loop sees: nothing else touches the GPU between frames)
    torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record(stream)
    for _ in range(args.steps):
        solve(n_iter)
    b.record(stream)
    torch.cuda.synchronize()
    ms_step_warm = max_over_ranks(a.elapsed_time(b), world) / args.steps
    # end to end through the public API with HOST buffers: pinned H2D + solve + D2H, synchronised per step
    e2e = []
    for i in range(args.steps + 3):
        flush.zero_()
        torch.cuda.synchronize()
        t1 = time.perf_counter()
        out_h = plan.solve_host(h_slopes, n_iter, n_frames=B, stream=stream, minres=minres)
        stream.synchronize()
        e2e.append(time.perf_counter() - t1)
    e2e_ms = max_over_ranks(statistics.mean(e2e[3:]) * 1e3, world)
    clocks = sampler.stop()

    # per-kernel device times of the multi-kernel loop (CUDA events after every kernel, on the launch stream)
    kt = plan.time_kernels(B, n_iter, stream=stream) if solver_used == "multikernel" else None
    n, C, P = cfg.n, 2 * cfg.n_wfs, plan.P
    Ph, Ns, npair = P // 2 + 1, 2 * cfg.n_wfs * plan.n_vs, C * (C + 1) // 2
    E = 4 if prec == tomo.TOMO_F32 else 8
    SE = 8 if prec == tomo.TOMO_F64 else 4
    spectra = npair * P * Ph * 2 * SE
    tbuf = C * Ph * n * 2 * E
    kbytes = {"cols": spectra + B * 2 * tbuf, "rows_fwd": B * (3 * Ns * E + tbuf), "rows_inv": B * (tbuf + 3 * Ns * E),
              "update": B * 6 * Ns * E}
    b_iter = spectra + B * 9 * Ns * E
    hbm, how = peaks()
    us_iter = (ms_step - ms_step0) / n_iter * 1e3
    roof = None
    if kt:
        dom = max(kt, key=kt.get)
        ach = kbytes[dom] / (kt[dom] * 1e-3) / 1e9
        roof = {"kernel": "k_" + dom, "bound": "hbm", "achieved": ach, "peak": hbm, "unit": "GB/s", "frac": ach / hbm,
                "traffic": None, "peak_source": how, "algorithmic_bytes_per_launch": kbytes[dom],
                "us_per_launch": {k: v * 1e3 for k, v in kt.items()},
                "state": "in situ inside the iteration loop (spectra L2-resident after the first iteration)"}
    f_iter = 2 * C * (n * 2.5 * P * np.log2(P) + Ph * 5 * P * np.log2(P)) + 8 * C * C * P * Ph      # SURVEY 8(d), per frame
    fp32_peak = 148 * 128 * 2 * 1.965e9                                                             # nominal FMA peak, DESIGN.md 6
    if solver_used == "persistent":
        # the dominant kernel is the persistent solver itself: device time of the launch alone (CUDA events on the stream)
        reps = max(3, min(args.steps, 50))
        k_ms = plan.time_solver(d_slopes, B, n_iter, reps, stream=stream, minres=minres)
        k_ms0 = plan.time_solver(d_slopes, B, 0, reps, stream=stream, minres=minres)
        kb = n_iter * b_iter + B * 4 * Ns * E
        ach = kb / (k_ms * 1e-3) / 1e9
        roof = {"kernel": "k_persistent", "bound": "hbm", "achieved": ach, "peak": hbm, "unit": "GB/s", "frac": ach / hbm,
                # dram__bytes_read.sum + dram__bytes_write.sum of one launch from the committed ncu capture of THIS kernel source
                # (profiles/r2_traffic.json, keyed by workload, batch, precision and source hash), else null
                "traffic": stored_traffic(cfg.name, B, args.precision, args.method), "kernel_source_hash": kernel_source_hash(),
                "peak_source": how, "algorithmic_bytes_per_launch": kb,
                "ms_per_launch": k_ms, "ms_per_launch_n_iter0": k_ms0,
                "us_per_iteration_in_kernel": (k_ms - k_ms0) / n_iter * 1e3,
                "alu": {"flop_per_launch": B * n_iter * f_iter, "achieved_TFLOPs": B * n_iter * f_iter / (k_ms * 1e-3) / 1e12,
                        "peak_TFLOPs": fp32_peak / 1e12, "frac": B * n_iter * f_iter / (k_ms * 1e-3) / fp32_peak},
                "state": ("one cooperative launch per solve; spectra pinned in shared memory, exchange buffers L2-resident: "
                          "latency-bound at batch 1 (two grid barriers per iteration), see DESIGN.md 6")}
    # L2 roofline (north_star: "... and over L2 bandwidth where the spectra are L2-resident"): the device's L2 -> SM read
    # bandwidth and plain FMA rate measured by the library's own kernels in this run (tomo_measure_device)
    dev_meas = tomo.measure_device(0, 5, stream=stream)
    npairs_rows = (n + 1) // 2
    exch = Ph * C * 2 * npairs_rows * 2 * E                       # one row <-> column exchange buffer of one frame
    if solver_used == "persistent":
        # per frame-iteration through L2: T1 written + read, T1p read + written, T2 written + read (spectra sit in shared memory)
        l2_bytes_iter = B * 6 * exch
        l2_what = "T1, T1p, T2 exchange buffers: 6 passes per frame-iteration (spectra pinned in shared memory)"
    else:
        l2_bytes_iter = spectra * B + B * 4 * tbuf + B * 9 * Ns * E     # k_cols re-reads the spectra per (k_x, frame) CTA
        l2_what = "spectra per frame + 4 exchange passes + CG vector passes"
    l2_roof = {"peak_GBps_measured": dev_meas["l2_read_GBps"], "bytes_per_iteration": l2_bytes_iter, "what": l2_what,
               "achieved_GBps": l2_bytes_iter / (us_iter * 1e-6) / 1e9,
               "frac": l2_bytes_iter / (us_iter * 1e-6) / 1e9 / max(dev_meas["l2_read_GBps"], 1e-9),
               "b_iter_over_l2_peak_us": b_iter / max(dev_meas["l2_read_GBps"], 1e-9) / 1e3,
               "fp32_TFLOPs_measured": dev_meas["fp32_TFLOPs"],
               "f_iter_frac_of_measured_fp32": B * f_iter / (us_iter * 1e-6) / 1e12 / max(dev_meas["fp32_TFLOPs"], 1e-9)}
    iter_roof = {"b_iter_bytes": b_iter, "us_per_iteration": us_iter, "achieved_GBps": b_iter / (us_iter * 1e-6) / 1e9,
                 "frac_of_hbm_peak": b_iter / (us_iter * 1e-6) / 1e9 / hbm}

    value = world * B * 1e3 / ms_step
    line = {"metric": METRIC, "value": value, "unit": "reconstructions/s", "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": args.precision, "data": "synthetic",
            "config": workload_config(cfg, plan.P, plan.P_os, n_iter, B, solver_used, args.method, world),
            "us_per_cg_iteration": us_iter, "ms_per_step_n_iter0": ms_step0, "ms_per_step_l2_warm": ms_step_warm,
            "reconstructions_per_s_l2_warm": world * B * 1e3 / ms_step_warm,
            "iteration_roofline": iter_roof, "l2_roofline": l2_roof, "roofline": roof,
            "e2e": {"value": world * B * 1e3 / e2e_ms, "unit": "reconstructions/s", "ms_per_step": e2e_ms,
                    "h2d_bytes_per_step": int(h_slopes.numel() * 4), "d2h_bytes_per_step": int(out_h.numel() * 4)},
            "gpu_launches": launches * args.steps, "launches_per_step": launches, "clocks": clocks,
            "plan_build_s": t_plan, "device_bytes": plan.stats()["device_bytes"]}
    if solver_used != args.solver:
        line["solver_fallback"] = {"requested": args.solver, "used": solver_used, "reason": solver_note}
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        step, desc, cores, extrapolated = oracle_setup(cfg, n_iter, whole=False)
        sec = statistics.median(step() for _ in range(3))
        line["cpu_baseline"] = {"value": 1.0 / sec, "unit": "reconstructions/s", "cores": cores, "kind": "oracle",
                                "sample": desc, "extrapolated": extrapolated, "us_per_cg_iteration": sec / n_iter * 1e6}
    if rank == 0:
        print(json.dumps(line))
    plan.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

#!/usr/bin/env python
"""bench.py — throughput of the hot path (S3 fold + S4 form-factor kernel, include/scarf.h) on synthetic input.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--impl ours|reference]

One "step" = one 12-form-factor job on the workload: scarf_set_transitions (fold T^s into the pair stream) +
scarf_form_factors over the whole q grid.  Default workload: BASELINE.json configs[2] = config 3 of DESIGN.md
(10 heavy atoms + 8 H, 190 basis functions, 12 transitions, 64^3 q grid), the configuration the headline metric
is quoted on.  Metric: q.primitive-pair.state evaluations per second.

`value`   : inputs resident in HBM, CUDA events on the library's stream, L2 flushed between steps.
`e2e`     : the same job through the C ABI with HOST buffers (pinned T, q and out): H2D/D2H inside.
`roofline`: FP64-ALU bound ("alu"): algorithmic FP64 issue slots / kernel time against the DFMA peak.
`cpu_baseline`: the oracle, as it stands, on the host cores, on a bounded sample of the same q grid.

N > 1 (torchrun): the path does not shard ("replicas only"): each rank runs the same job on its own
GPU; value = total evaluations / max-over-ranks time.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "q*primitive-pair*state evaluations per second (12-form-factor job, fold + kernel)"
UNIT = "evals/s"
# FP64 lanes per SM per clock on B200 (GB100): 64 DFMA/clk/SM, as on GH100.
DFMA_PER_CLK_PER_SM = 64
# dram__bytes_read.sum + dram__bytes_write.sum of one ff_v1_kernel<12> launch, from the `ncu --set full` capture
# summarised in profiles/r01b_ff_v1_ncu_full.md (config 3 only; other configs were not captured -> null).
NCU_DRAM_BYTES_PER_LAUNCH = {3: 16.663808e6 + 293.769984e6}


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--seed", type=int, default=None)
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="target wall time of the oracle sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--fft-grid", type=int, default=None, help="points per axis of the FFT-method grid (default: the config's q grid size)")
    return ap.parse_args()


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md clocks line)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                       "-lms", "50", "-i", str(gpu_index)], stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self) -> dict:
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, smax, power, reasons = [], [], [], set()
        for line in self.f:
            c = [x.strip() for x in line.split(",")]
            if len(c) < 9:
                continue
            try:
                sm.append(float(c[1])); smax.append(float(c[2])); power.append(float(c[3]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), c[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        self.f.close()
        try:
            os.unlink(self.f.name)
        except OSError:
            pass
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        # "under load" = samples in the upper half of the observed power range
        thr = 0.5 * (min(power) + max(power))
        load = [s for s, p in zip(sm, power) if p >= thr] or sm
        return {"sm_mhz": float(np.median(load)), "sm_max_mhz": float(max(smax)), "reasons": sorted(reasons),
                "samples": len(sm), "power_w_max": float(max(power))}


def oracle_sample(w, target_s: float, seed: int = 0):
    """Time the oracle (as it stands) on a bounded, seeded sample of the workload's q grid."""
    import oracle
    import workloads as W
    threads = oracle.max_threads()
    n0 = max(2, min(w.n_q, threads))
    idx = W.sample_q_indices(w.n_q, n0, seed)
    t0 = time.perf_counter()
    oracle.form_factors(w.basis, w.T, w.q[idx])
    dt0 = time.perf_counter() - t0
    per_q = dt0 / len(idx)
    n = int(max(n0, min(w.n_q, target_s / max(per_q, 1e-9))))
    n = max(threads, (n // threads) * threads)
    idx = W.sample_q_indices(w.n_q, n, seed + 1)
    t0 = time.perf_counter()
    f = oracle.form_factors(w.basis, w.T, w.q[idx])
    dt = time.perf_counter() - t0
    return idx, f, dt, threads


def n_pairs_all(basis) -> int:
    n = int(np.sum(basis.shell_nprim))
    return n * (n + 1) // 2


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores; each step = a bounded sample of the grid.
    Evaluations are counted in the same unit: q-points x primitive shell pairs (A <= B, all of them: the oracle
    screens nothing) x states."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    import workloads as W
    w = W.make_workload(args.config, oracle.overlap, seed=args.seed)
    threads = oracle.max_threads()
    # size one step at ~ cpu_seconds / (steps + warmup), at least `threads` q-points
    idx0 = W.sample_q_indices(w.n_q, max(4, threads), 0)
    t0 = time.perf_counter()
    oracle.form_factors(w.basis, w.T, w.q[idx0])
    per_q = (time.perf_counter() - t0) / len(idx0)
    budget = max(1.0, 120.0 / max(1, args.steps + args.warmup))
    n = int(max(threads, min(w.n_q, budget / per_q)))
    idx = W.sample_q_indices(w.n_q, n, 1)
    for _ in range(args.warmup):
        oracle.form_factors(w.basis, w.T, w.q[idx])
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.form_factors(w.basis, w.T, w.q[idx])
    dt = (time.perf_counter() - t0) / max(1, args.steps)
    evals = float(len(idx)) * n_pairs_all(w.basis) * w.n_states
    value = evals / dt
    sample = f"{len(idx)} of {w.n_q} q-points (seeded sample), all {w.n_states} states, every primitive pair"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "config": args.config, "n_q": w.n_q, "n_states": w.n_states,
                       "nbf": w.basis.nbf, "n_pairs_all": n_pairs_all(w.basis), "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample,
                             "job_seconds_extrapolated": dt * w.n_q / len(idx)},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def run_ours(args):
    import torch
    import torch.distributed as dist
    import workloads as W
    from paper_2512_18010_b200 import Scarf, binding, replicas

    rank, world, local = replicas.env_rank_world_local()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    sc = Scarf(local)
    stream = torch.cuda.Stream()
    sc.set_stream(stream.cuda_stream)

    # The workload generator needs the AO overlap to orthonormalise the random MOs: the PRODUCT's own
    # (scarf_overlap, host tables) here; the oracle's in the tests.
    def overlap(basis):
        sc.set_basis(basis)
        return sc.overlap()

    w = W.make_workload(args.config, overlap, seed=args.seed)
    sc.set_basis(w.basis)
    T_dev = torch.as_tensor(w.T, device="cuda")
    q_dev = torch.as_tensor(w.q, device="cuda")
    out_dev = torch.empty((w.n_states, w.n_q, 2), dtype=torch.float64, device="cuda")
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")  # > 126 MB L2

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def step_device():
        sc.set_transitions(T_dev)
        sc.form_factors(q_dev, out=out_dev)

    # ---- resident-input timing: CUDA events on the library's stream, L2 flushed between steps (untimed)
    with torch.cuda.stream(stream):
        for _ in range(max(3, args.warmup)):
            step_device()
        barrier()
        sampler = ClockSampler(local) if rank == 0 else None
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
        kern_ms = []
        sc.set_option("timing", 1)
        barrier()
        t_wall0 = time.perf_counter()
        for k in range(args.steps):
            flush.fill_(k & 0xFF)
            ev[k][0].record(stream)
            step_device()
            ev[k][1].record(stream)
            st_k = sc.stats()
            kern_ms.append((st_k["last_fold_ms"], st_k["last_kernel_ms"]))
        barrier()
        t_wall = time.perf_counter() - t_wall0
        clocks = sampler.stop() if sampler else None
        sc.set_option("timing", 0)
    step_ms = [a.elapsed_time(b) for a, b in ev]
    st = sc.stats()
    evals_per_step = st["evals_per_q"] * w.n_q
    value, ms_per_step = replicas.whole_job_value(evals_per_step, args.steps, float(sum(step_ms)), "cuda")

    # ---- product-grid path (NEXT-1, scarf_form_factors_grid) on the Cartesian configs: same job, same timing protocol
    grid_path = None
    if w.grid.get("kind") == "cartesian":
        ax_dev = torch.as_tensor(W.cartesian_axis(w.grid["n_per_axis"], w.grid["qmax"]), device="cuda")

        def step_grid():
            sc.set_transitions(T_dev)
            sc.form_factors_grid(ax_dev, ax_dev, ax_dev, out=out_dev)

        with torch.cuda.stream(stream):
            for _ in range(3):
                step_grid()
            barrier()
            gev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
            gk = []
            sc.set_option("timing", 1)
            for k in range(args.steps):
                flush.fill_(k & 0xFF)
                gev[k][0].record(stream)
                step_grid()
                gev[k][1].record(stream)
                gk.append(sc.stats()["last_kernel_ms"])
            barrier()
            sc.set_option("timing", 0)
        g_ms = float(np.mean([a.elapsed_time(b) for a, b in gev]))
        g_ms = replicas.max_over_ranks(g_ms, "cuda")
        gst = sc.stats()
        grid_path = {"api": "scarf_form_factors_grid", "ms_per_step": g_ms, "kernel_ms": float(np.median(gk)),
                     "value": world * evals_per_step / (g_ms * 1e-3), "unit": UNIT, "slots": gst["last_grid_slots"],
                     "launches_per_step": int(gst["last_kernel_launches"] + gst["last_fold_launches"])}
        step_device()   # leave the general path's result in out_dev for the parity sample below
        torch.cuda.synchronize()

    # ---- the paper's FFT method (NEXT-4, scarf_fft_form_factors) on a real-space grid of the same size: box = atoms + 5 bohr
    fft_path = None
    if w.grid.get("kind") == "cartesian":
        n_ax = int(args.fft_grid or w.grid["n_per_axis"])
        lo = w.basis.atom_xyz.min(axis=0) - 5.0
        box = w.basis.atom_xyz.max(axis=0) + 5.0 - lo
        fft_out = torch.empty((w.n_states, n_ax ** 3, 2), dtype=torch.float64, device="cuda")
        with torch.cuda.stream(stream):
            sc.set_transitions(T_dev)
            for _ in range(2):
                sc.fft_form_factors((n_ax,) * 3, lo, box, out=fft_out)
            barrier()
            fev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
            for k in range(args.steps):
                flush.fill_(k & 0xFF)
                fev[k][0].record(stream)
                sc.fft_form_factors((n_ax,) * 3, lo, box, out=fft_out)
                fev[k][1].record(stream)
            barrier()
        f_ms = float(np.median([a.elapsed_time(b) for a, b in fev]))
        fma = 0.5 * w.n_states * float(w.basis.nbf) ** 2 * n_ax ** 3
        fft_path = {"api": "scarf_fft_form_factors", "grid": [n_ax] * 3, "box_bohr": [float(x) for x in box], "ms_per_call": f_ms,
                    "density_fma": fma, "note": "approximate method (box truncation, grid spacing); timing only"}
        del fft_out

    # ---- angular moments of the result (NEXT-3, scarf_angular_moments) on the spherical product grid of config 5
    angular = None
    if w.grid.get("kind") == "spherical":
        n_r, n_t, n_p = w.grid["n_r"], w.grid["n_theta"], w.grid["n_phi"]
        ct, wt = np.polynomial.legendre.leggauss(n_t)
        l_max = 24
        f_dev = torch.view_as_complex(out_dev)
        with torch.cuda.stream(stream):
            for _ in range(3):
                sc.angular_moments(f_dev, ct, wt, n_p, l_max, n_r=n_r)
            barrier()
            aev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
            for k in range(args.steps):
                flush.fill_(k & 0xFF)
                aev[k][0].record(stream)
                sc.angular_moments(f_dev, ct, wt, n_p, l_max, n_r=n_r)
                aev[k][1].record(stream)
            barrier()
        a_ms = float(np.median([a.elapsed_time(b) for a, b in aev]))
        a_bytes = 16.0 * w.n_states * w.n_q + 16.0 * w.n_states * n_r * (l_max + 1) ** 2
        angular = {"api": "scarf_angular_moments", "l_max": l_max, "ms_per_call": a_ms, "algorithmic_bytes": a_bytes,
                   "achieved_gbs": a_bytes / (a_ms * 1e-3) / 1e9,
                   "note": "includes the host-side Legendre/twiddle tables and their upload; bound: hbm"}

    # ---- end to end: host buffers through the C ABI (pinned T, q and out), copies inside the timed region
    q_host = torch.as_tensor(w.q).pin_memory()
    out_host = torch.empty((w.n_states, w.n_q, 2), dtype=torch.float64).pin_memory()
    T_host = torch.as_tensor(np.ascontiguousarray(w.T)).pin_memory()

    def step_host():
        sc.set_transitions(T_host)
        sc.form_factors(q_host, out=out_host)

    with torch.cuda.stream(stream):
        for _ in range(2):
            step_host()
        barrier()
        e2e_steps = max(3, min(args.steps, 10))
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            step_host()
        barrier()
        e2e_s = (time.perf_counter() - t0) / e2e_steps
    e2e_s = replicas.max_over_ranks(e2e_s, "cuda")
    e2e_value = world * evals_per_step / e2e_s
    h2d = T_host.numel() * 8 + q_host.numel() * 8
    d2h = out_host.numel() * 8

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (S4): algorithmic FP64 issue slots / its CUDA-event time
    fold_ms = float(np.median([a for a, _ in kern_ms]))
    kernel_ms = float(np.median([b for _, b in kern_ms]))
    slots = st["slots_per_q"] * w.n_q
    peak_meas, peak_mhz = binding.fp64_peak(local)
    sms = torch.cuda.get_device_properties(local).multi_processor_count
    sm_max = (clocks or {}).get("sm_max_mhz") or 1965.0
    peak_nominal = DFMA_PER_CLK_PER_SM * sms * sm_max * 1e6
    achieved = slots / (kernel_ms * 1e-3)
    roofline = {"bound": "alu", "achieved": achieved / 1e12, "peak": peak_meas / 1e12, "unit": "T FP64-slot/s (1 slot = 1 DFMA lane-op = 2 flop)",
                "frac": achieved / peak_meas, "traffic": NCU_DRAM_BYTES_PER_LAUNCH.get(args.config),
                "peak_source": f"measured register-only DFMA micro-benchmark (scarf_fp64_peak) at {peak_mhz:.0f} MHz; "
                               f"nominal {DFMA_PER_CLK_PER_SM}/clk/SM x {sms} SMs x {sm_max:.0f} MHz = {peak_nominal / 1e12:.2f}",
                "frac_of_nominal": achieved / peak_nominal, "kernel": "S4 form-factor kernel(s)", "kernel_ms": kernel_ms,
                "fold_ms": fold_ms, "slots_per_launch_set": slots, "kernel_share_of_step": kernel_ms / ms_per_step,
                "algorithmic_bytes": st["stream_bytes"] + 16.0 * w.n_states * w.n_q + 24.0 * w.n_q}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(3, args.warmup),
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "config": args.config, "seed": w.seed, "n_q": w.n_q, "n_states": w.n_states,
                       "nbf": w.basis.nbf, "n_pairs_all": st["n_pairs_all"], "n_pairs_kept": st["n_pairs_kept"],
                       "pairs_kept_per_class": st["pairs_kept_per_class"], "cond_S": w.cond_S,
                       "l2": "flushed between timed steps (256 MB write, untimed)",
                       "parallelism": "replicas only" if world > 1 else "single GPU"},
            "job_seconds": ms_per_step * 1e-3, "wall_s_timed_region": t_wall,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                    "job_seconds": e2e_s},
            "gpu_launches": int(args.steps * (st["last_kernel_launches"] + st["last_fold_launches"])),
            "clocks": clocks, "roofline": roofline}

    if grid_path is not None:
        g_ach = grid_path["slots"] / (grid_path["kernel_ms"] * 1e-3)
        grid_path["roofline"] = {"bound": "alu", "achieved": g_ach / 1e12, "peak": peak_meas / 1e12, "frac": g_ach / peak_meas,
                                 "unit": roofline["unit"]}
        line["grid_path"] = grid_path

    if angular is not None:
        line["angular_moments"] = angular
    if fft_path is not None:
        line["fft_path"] = fft_path

    if not args.no_cpu_baseline and world == 1:
        import oracle
        idx, f_ref, dt, threads = oracle_sample(w, args.cpu_seconds)
        f_gpu = torch.view_as_complex(out_dev)[:, torch.as_tensor(idx, device="cuda")].cpu().numpy()
        err = max(float(np.max(np.abs(f_gpu[s] - f_ref[s])) / np.max(np.abs(f_ref[s]))) for s in range(w.n_states))
        cpu_evals = float(len(idx)) * st["n_pairs_all"] * w.n_states
        line["cpu_baseline"] = {"value": cpu_evals / dt, "unit": UNIT, "cores": threads, "kind": "oracle",
                                "sample": f"{len(idx)} of {w.n_q} q-points (seeded sample), all {w.n_states} states, "
                                          f"every primitive pair ({st['n_pairs_all']}, unscreened)",
                                "seconds": dt, "job_seconds_extrapolated": dt * w.n_q / len(idx)}
        line["parity"] = {"max_rel_err_vs_oracle_on_sample": err, "tolerance": 1e-10, "ok": bool(err <= 1e-10)}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()

#!/usr/bin/env python
"""bench.py — throughput of the hot path (S3 fold + S4 form-factor kernel, include/scarf.h) on synthetic input.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--path auto|grid|list] [--impl ours|reference]

One "step" = one 12-form-factor job on the workload: scarf_set_transitions (fold T^s into the pair stream, screen and
pack it on the device) + the S4 call a user makes for that q set: scarf_form_factors_grid for the Cartesian product
grids of configs 1-4 (per-axis factor tables; f(-q) = conj f(q) on the inversion-symmetric grid), scarf_form_factors
(arbitrary point list) for config 5 — `--path` forces one or the other; the other path is timed as well and reported
beside the headline (`list_path` / `grid_path`).  Default workload: BASELINE.json configs[2] = config 3 of DESIGN.md
(10 heavy atoms + 8 H, 190 basis functions, 12 transitions, 64^3 q grid), the configuration the headline metric is
quoted on.  Metric: q.primitive-pair.state evaluations per second, one evaluation = one (q-point, kept pair, state)
triple actually EXECUTED by S4 (mirror points filled by conjugation are not counted; `job_seconds` is the job time).

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
# roofline.traffic: dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, looked up BY NAME
# (config, kernel) in the table written from the committed `ncu --set full` captures; null when there is no capture.
TRAFFIC_TABLE = os.path.join(os.path.dirname(os.path.abspath(__file__)), "profiles", "dram_traffic_per_launch.csv")


def traffic_from_profiles(config: int, kernel: str):
    try:
        with open(TRAFFIC_TABLE) as f:
            rows = [l.strip().split(",") for l in f if l.strip() and not l.startswith("#")]
    except OSError:
        return None, None
    hdr = rows[0]
    best = None
    for r in rows[1:]:
        d = dict(zip(hdr, r))
        if int(d["config"]) == config and d["kernel"] == kernel:
            best = d                       # the last matching row = the latest capture
    if best is None:
        return None, None
    return float(best["dram_bytes_read"]) + float(best["dram_bytes_write"]), best["source"]


def measured_hbm_peak():
    """(GB/s, source): the driver-written MEASURED_PEAKS.json, else the fallback B200_PROFILING.md states."""
    try:
        with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (copy bandwidth, burst)"
    except (OSError, KeyError, ValueError):
        return 6650.0, "of fallback (B200_PROFILING.md: 6.65 TB/s)"


def cpu_model() -> str:
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


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
    ap.add_argument("--path", default="auto", choices=["auto", "grid", "list", "sph"],
                    help="S4 entry point of the headline step: Cartesian product-grid API, spherical product-grid API or arbitrary point list "
                         "(auto: grid on the Cartesian configs, sph on the spherical one)")
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
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "cpu_model": cpu_model(), "kind": "oracle", "sample": sample,
                             "unit_note": "evaluations counted on ALL primitive shell pairs (the oracle screens nothing)",
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
    cartesian = w.grid.get("kind") == "cartesian"
    spherical = w.grid.get("kind") == "spherical"
    path = args.path if args.path != "auto" else ("grid" if cartesian else ("sph" if spherical else "list"))
    if path == "grid" and not cartesian:
        raise SystemExit("--path grid needs a Cartesian product grid (configs 1-4)")
    if path == "sph" and not spherical:
        raise SystemExit("--path sph needs the spherical product grid (config 5)")
    if spherical:
        sph_r = np.geomspace(w.grid["qmin"], w.grid["qmax"], w.grid["n_r"])
        sph_ct, _sph_w = np.polynomial.legendre.leggauss(w.grid["n_theta"])
        sph_nphi = w.grid["n_phi"]
    T_dev = torch.as_tensor(w.T, device="cuda")
    q_dev = torch.as_tensor(w.q, device="cuda")
    out_dev = torch.empty((w.n_states, w.n_q, 2), dtype=torch.float64, device="cuda")
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")  # > 126 MB L2
    ax_host = W.cartesian_axis(w.grid["n_per_axis"], w.grid["qmax"]) if cartesian else None   # host axes: fully asynchronous call

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def step_list():
        sc.set_transitions(T_dev)
        sc.form_factors(q_dev, out=out_dev)

    def step_grid():
        sc.set_transitions(T_dev)
        sc.form_factors_grid(ax_host, ax_host, ax_host, out=out_dev)

    def step_sph():
        sc.set_transitions(T_dev)
        sc.form_factors_sph(sph_r, sph_ct, sph_nphi, out=out_dev)

    def step_sph_plain():
        sc.set_option("grid_symmetry", 0)
        step_sph()
        sc.set_option("grid_symmetry", 1)

    def step_grid_plain():
        sc.set_option("grid_symmetry", 0)
        step_grid()
        sc.set_option("grid_symmetry", 1)

    def step_grid_box():                    # the box kernel (ff_grid.cu) where another kernel is the automatic choice
        sc.set_option("grid_variant", 0)
        step_grid()
        sc.set_option("grid_variant", -1)

    def step_grid_row():                    # the row kernel (ff_row.cu) where the mirror-pair kernel (ff_zrow.cu) is the automatic choice
        sc.set_option("grid_variant", 1)
        step_grid()
        sc.set_option("grid_variant", -1)

    def grid_kernel_name(stats):
        return {1: "ff_row_kernel<12>", 2: "ff_zrow_kernel<12>", 3: "ff_sph_kernel<12>"}.get(stats.get("last_grid_variant", 0), "ff_grid_kernel<12>")

    def run_timed(step, steps, warmup, sample_clocks=False):
        """W untimed steps, then `steps` steps timed with CUDA events on the library's stream (L2 flushed before each,
        outside the events), asynchronous (no per-call sync); then the same steps again with the library's per-kernel
        events ("timing" option) for the kernel-only durations.  Returns a dict."""
        with torch.cuda.stream(stream):
            for _ in range(warmup):
                step()
            barrier()
            sampler = ClockSampler(local) if (sample_clocks and rank == 0) else None
            ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
            barrier()
            t0 = time.perf_counter()
            for k in range(steps):
                flush.fill_(k & 0xFF)
                ev[k][0].record(stream)
                step()
                ev[k][1].record(stream)
            barrier()
            wall = time.perf_counter() - t0
            clocks = sampler.stop() if sampler else None
            st = sc.stats()
            ms = [a.elapsed_time(b) for a, b in ev]
            # instrumented pass: per-kernel CUDA events inside the library (one stream sync per call)
            sc.set_option("timing", 1)
            fold, kern, main = [], [], []
            for k in range(steps):
                flush.fill_(k & 0xFF)
                step()
                s2 = sc.stats()
                fold.append(s2["last_fold_ms"]); kern.append(s2["last_kernel_ms"]); main.append(s2["last_main_kernel_ms"])
            sc.set_option("timing", 0)
            barrier()
        return {"ms": ms, "sum_ms": float(sum(ms)), "wall_s": wall, "clocks": clocks, "stats": st,
                "fold_ms": float(np.median(fold)), "kernel_ms": float(np.median(kern)), "main_kernel_ms": float(np.median(main)),
                "main_kernel_ms_mean": float(np.mean(main))}

    steps, warmup = args.steps, max(3, args.warmup)
    step_head = {"grid": step_grid, "sph": step_sph, "list": step_list}[path]
    head = run_timed(step_head, steps, warmup, sample_clocks=True)
    st = head["stats"]
    n_eval_q = w.n_q
    if path == "grid" and st["last_grid_symmetric"]:
        n_ax = w.grid["n_per_axis"]
        n_eval_q = ((n_ax + 1) // 2) * n_ax * n_ax

    def sph_eval_points():
        n_t, n_p = w.grid["n_theta"], w.grid["n_phi"]
        return w.grid["n_r"] * ((n_t // 2) * n_p + (n_p // 2 if n_t % 2 else 0))
    if path == "sph" and st["last_grid_symmetric"]:
        n_eval_q = sph_eval_points()
    evals_per_step = st["evals_per_q"] * n_eval_q                      # executed (q, kept pair, state) triples
    value, ms_per_step = replicas.whole_job_value(evals_per_step, steps, head["sum_ms"], "cuda")
    clocks = head["clocks"]

    # ---- the other S4 entry point (and the product grid without the symmetry), same job, same protocol
    def side(step, n_q_exec, slots_key):
        r = run_timed(step, steps, 3)
        s2 = r["stats"]
        ms = replicas.max_over_ranks(float(np.mean(r["ms"])), "cuda")
        slots = s2["last_grid_kernel_slots"] if slots_key == "grid" else s2["slots_per_q"] * w.n_q
        return {"ms_per_step": ms, "job_seconds": ms * 1e-3, "kernel_ms": r["kernel_ms"], "main_kernel_ms": r["main_kernel_ms"],
                "fold_ms": r["fold_ms"], "value": world * s2["evals_per_q"] * n_q_exec / (ms * 1e-3), "unit": UNIT,
                "slots_main_kernel": slots, "n_chunks": s2["last_n_chunks"],
                "kernel": grid_kernel_name(s2) if slots_key == "grid" else "ff_v1_kernel<12>",
                "launches_per_step": int(s2["last_kernel_launches"] + s2["last_fold_launches"])}

    list_path = grid_path = grid_plain = grid_box = grid_row = sph_path = sph_plain = None
    if spherical:
        if path == "sph":
            list_path = dict(side(step_list, w.n_q, "list"), api="scarf_form_factors")
        else:
            sph_path = dict(side(step_sph, sph_eval_points(), "grid"), api="scarf_form_factors_sph", symmetric=True)
        sph_plain = dict(side(step_sph_plain, w.n_q, "grid"), api="scarf_form_factors_sph", symmetric=False)
        step_head()                                            # leave the headline path's result in out_dev for the parity sample
        torch.cuda.synchronize()
    if cartesian:
        if path == "grid":
            list_path = dict(side(step_list, w.n_q, "list"), api="scarf_form_factors")
        else:
            n_ax = w.grid["n_per_axis"]
            grid_path = dict(side(step_grid, ((n_ax + 1) // 2) * n_ax * n_ax, "grid"), api="scarf_form_factors_grid", symmetric=True)
        grid_plain = dict(side(step_grid_plain, w.n_q, "grid"), api="scarf_form_factors_grid", symmetric=False)
        head_variant = st.get("last_grid_variant", 0) if path == "grid" else {"ff_row_kernel<12>": 1, "ff_zrow_kernel<12>": 2}.get(grid_path["kernel"], 0)
        if head_variant in (1, 2):
            n_ax = w.grid["n_per_axis"]
            grid_box = dict(side(step_grid_box, ((n_ax + 1) // 2) * n_ax * n_ax, "grid"), api="scarf_form_factors_grid", symmetric=True,
                            option="grid_variant = 0")
        if head_variant == 2:
            grid_row = dict(side(step_grid_row, ((n_ax + 1) // 2) * n_ax * n_ax, "grid"), api="scarf_form_factors_grid", symmetric=True,
                            option="grid_variant = 1")
        (step_grid if path == "grid" else step_list)()        # leave the headline path's result in out_dev for the parity sample
        torch.cuda.synchronize()

    # ---- the paper's FFT method (NEXT-4, scarf_fft_form_factors) on a real-space grid of the same size: box = atoms + 5 bohr
    fft_path = None
    if cartesian:
        n_ax = int(args.fft_grid or w.grid["n_per_axis"])
        lo = w.basis.atom_xyz.min(axis=0) - 5.0
        box = w.basis.atom_xyz.max(axis=0) + 5.0 - lo
        fft_out = torch.empty((w.n_states, n_ax ** 3, 2), dtype=torch.float64, device="cuda")
        with torch.cuda.stream(stream):
            sc.set_transitions(T_dev)
            for _ in range(2):
                sc.fft_form_factors((n_ax,) * 3, lo, box, out=fft_out)
            barrier()
            fev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
            for k in range(steps):
                flush.fill_(k & 0xFF)
                fev[k][0].record(stream)
                sc.fft_form_factors((n_ax,) * 3, lo, box, out=fft_out)
                fev[k][1].record(stream)
            barrier()
        f_ms = float(np.median([a.elapsed_time(b) for a, b in fev]))
        fma = 0.5 * w.n_states * float(w.basis.nbf) ** 2 * n_ax ** 3
        fft_path = {"api": "scarf_fft_form_factors", "grid": [n_ax] * 3, "box_bohr": [float(x) for x in box], "ms_per_call": f_ms,
                    "density_fma": fma, "note": "approximate method (box truncation, grid spacing)"}
        if rank == 0 and world == 1 and not args.no_cpu_baseline:
            # sampled parity against the FFT-method oracle: the same basis, T and box on a small ragged grid the oracle's
            # einsum finishes in seconds (the density kernel's launch shape depends on nbf, not on the grid size)
            from oracle import fft_method as offt
            n_small = (10, 6, 14)
            f_ref = offt.form_factors(w.basis, w.T, n_small, lo, box)
            f_gpu = sc.fft_form_factors(n_small, lo, box).cpu().numpy()
            err = max(float(np.max(np.abs(f_gpu[s] - f_ref[s])) / np.max(np.abs(f_ref[s]))) for s in range(w.n_states))
            fft_path["parity"] = {"grid": list(n_small), "max_rel_err_vs_fft_oracle": err, "tolerance": 1e-10, "ok": bool(err <= 1e-10)}
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
            aev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
            for k in range(steps):
                flush.fill_(k & 0xFF)
                aev[k][0].record(stream)
                sc.angular_moments(f_dev, ct, wt, n_p, l_max, n_r=n_r)
                aev[k][1].record(stream)
            barrier()
        a_ms = float(np.median([a.elapsed_time(b) for a, b in aev]))
        a_bytes = 16.0 * w.n_states * w.n_q + 16.0 * w.n_states * n_r * (l_max + 1) ** 2 + 8.0 * w.n_states * n_r
        hbm_peak, hbm_src = measured_hbm_peak()
        a_traffic, a_src = traffic_from_profiles(args.config, "angular_fused_kernel")
        angular = {"api": "scarf_angular_moments", "l_max": l_max, "ms_per_call": a_ms, "algorithmic_bytes": a_bytes,
                   "roofline": {"bound": "hbm", "achieved": a_bytes / (a_ms * 1e-3) / 1e9, "peak": hbm_peak, "unit": "GB/s",
                                "frac": a_bytes / (a_ms * 1e-3) / 1e9 / hbm_peak, "traffic": a_traffic, "traffic_source": a_src,
                                "peak_source": hbm_src}}

    # ---- end to end: host buffers through the C ABI (pinned T, q/axes and out), copies inside the timed region
    q_host = torch.as_tensor(w.q).pin_memory()
    out_host = torch.empty((w.n_states, w.n_q, 2), dtype=torch.float64).pin_memory()
    T_host = torch.as_tensor(np.ascontiguousarray(w.T)).pin_memory()

    def step_host():
        sc.set_transitions(T_host)
        if path == "grid":
            sc.form_factors_grid(ax_host, ax_host, ax_host, out=out_host)
        elif path == "sph":
            sc.form_factors_sph(sph_r, sph_ct, sph_nphi, out=out_host)
        else:
            sc.form_factors(q_host, out=out_host)

    with torch.cuda.stream(stream):
        for _ in range(2):
            step_host()
        barrier()
        e2e_steps = max(3, min(steps, 10))
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            step_host()
        barrier()
        e2e_s = (time.perf_counter() - t0) / e2e_steps
    e2e_s = replicas.max_over_ranks(e2e_s, "cuda")
    e2e_value = world * evals_per_step / e2e_s
    h2d = T_host.numel() * 8 + (3 * ax_host.size * 8 if path == "grid" else ((sph_r.size + sph_ct.size) * 8 if path == "sph" else q_host.numel() * 8))
    d2h = out_host.numel() * 8

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (S4): algorithmic FP64 issue slots / its CUDA-event time
    peak_meas, peak_mhz = binding.fp64_peak(local)
    sms = torch.cuda.get_device_properties(local).multi_processor_count
    sm_max = (clocks or {}).get("sm_max_mhz") or 1965.0
    peak_nominal = DFMA_PER_CLK_PER_SM * sms * sm_max * 1e6
    unit_slots = "T FP64-slot/s (1 slot = 1 DFMA lane-op = 2 flop)"

    def alu_roofline(slots, kernel_ms, kernel_name, poly_slots=None):
        ach = slots / (kernel_ms * 1e-3)
        traffic, tsrc = traffic_from_profiles(args.config, kernel_name)
        r = {"bound": "alu", "achieved": ach / 1e12, "peak": peak_meas / 1e12, "unit": unit_slots, "frac": ach / peak_meas,
             "traffic": traffic, "traffic_source": tsrc, "kernel": kernel_name, "kernel_ms": kernel_ms,
             "slots_per_launch": slots, "frac_of_nominal": ach / peak_nominal}
        if poly_slots is not None:       # the model without the per-(q, pair) transcendental / factor slots
            r["frac_poly_only"] = poly_slots / (kernel_ms * 1e-3) / peak_meas
        return r

    kW = [2, 7, 13, 23, 38, 59, 87] + [0] * 6
    poly_per_q = float(sum(n * w.n_states * kW[c] for c, n in enumerate(st["pairs_kept_per_class"])))
    if path == "grid":
        slots = st["last_grid_kernel_slots"]        # the kernel's own count: W(L) per (q, pair, state) (n_herm + 3 beyond L = 3) and 6 per (q, pair)
        roofline = alu_roofline(slots, head["main_kernel_ms"], grid_kernel_name(st), poly_per_q * n_eval_q)
        # the same time against the monomial-form model of the list kernel (n_herm + 3 per (q, pair, state)),
        # i.e. the slots this launch would have cost without sharing the (q_y, q_z) part between a thread's two points
        survey_slots = n_eval_q * (poly_per_q + 6.0 * st["n_pairs_kept"] * len(range(0, w.n_states, 12)))
        roofline["frac_survey_model"] = survey_slots / (head["main_kernel_ms"] * 1e-3) / peak_meas
        if st.get("last_grid_variant", 0) == 2:
            roofline["slots_model_note"] = ("frac: FP64 slots the kernel's algorithm needs (a lane owns the points +z and -z of a row and accumulates "
                                            "their half sum and half difference, whose polynomials in z^2 are shared by the pair and by the row: "
                                            "4 / 5 / 6 slots per (q, pair, state) for L = 1 / 2 / 3, 2 per (q, pair), plus the per-row part, "
                                            "14 / 23 / 36 slots per (row, pair, state)); frac_survey_model: the monomial-form count n_herm + 3 "
                                            "over the same time.  With 12 (4, 8) states per tile the accumulates of classes L = 0..2 are "
                                            "issued as mma.sync.m8n8k4.f64 (DMMA, the FP64 tensor pipe: a matrix product over the records "
                                            "of a stage), the other classes and the per-row parts as DFMAs; peak stays the DFMA peak "
                                            "(the DMMA rate is the same 64 FMA/clk/SM on a pipe of its own)")
        elif st.get("last_grid_variant", 0) == 1:
            roofline["slots_model_note"] = ("frac: FP64 slots the kernel's algorithm needs (the 64 points of a warp's row share the (q_x, q_y) "
                                            "part of every polynomial: 5 / 7 / 9 slots per (q, pair, state) for L = 1 / 2 / 3 plus the "
                                            "per-row part, 2 / 7 / 16 slots per (row, pair, state)); frac_survey_model: the monomial-form "
                                            "count n_herm + 3 over the same time")
        else:
            roofline["slots_model_note"] = ("frac: FP64 slots the kernel's algorithm needs (two points of a thread share the (q_y, q_z) part "
                                            "of every polynomial: 6 / 10.5 / 17 slots per (q, pair, state) for L = 1 / 2 / 3); "
                                            "frac_survey_model: the monomial-form count n_herm + 3 over the same time")
        alg_bytes = st["stream_bytes"] + 16.0 * w.n_states * w.n_q + 32.0 * st["n_pairs_kept"] * (n_eval_q ** (1 / 3))
    elif path == "sph":
        slots = st["last_grid_kernel_slots"]        # the kernel's own count: W(L) = 2, 4, 5, 6 (+ the per-direction sums / 64), n_herm + 3 beyond L = 3; 24 per (q, pair)
        roofline = alu_roofline(slots, head["main_kernel_ms"], grid_kernel_name(st), poly_per_q * n_eval_q)
        survey_slots = n_eval_q * st["slots_per_q"]
        roofline["frac_survey_model"] = survey_slots / (head["main_kernel_ms"] * 1e-3) / peak_meas
        roofline["slots_model_note"] = ("frac: FP64 slots the kernel's algorithm needs (the 64 radii of a warp's direction share the phase slope "
                                        "n.P and the per-degree sums of the polynomial: 4 / 5 / 6 slots per (q, pair, state) for L = 1 / 2 / 3 and "
                                        "24 per (q, pair)); frac_survey_model: the list kernel's count (n_herm + 3, and 40 per (q, pair)) over "
                                        "the same time")
        alg_bytes = st["stream_bytes"] + 16.0 * w.n_states * w.n_q + 8.0 * st["n_pairs_kept"] * w.grid["n_r"]
    else:
        slots = st["slots_per_q"] * w.n_q
        roofline = alu_roofline(slots, head["main_kernel_ms"], "ff_v1_kernel<12>", poly_per_q * w.n_q)
        alg_bytes = st["stream_bytes"] + 16.0 * w.n_states * w.n_q + 24.0 * w.n_q
    roofline.update({"peak_source": f"measured register-only DFMA micro-benchmark (scarf_fp64_peak) at {peak_mhz:.0f} MHz; "
                                    f"nominal {DFMA_PER_CLK_PER_SM}/clk/SM x {sms} SMs x {sm_max:.0f} MHz = {peak_nominal / 1e12:.2f}",
                     "fold_ms": head["fold_ms"], "s4_call_ms": head["kernel_ms"],
                     "kernel_share_of_step": head["main_kernel_ms"] / ms_per_step, "algorithmic_bytes": alg_bytes,
                     "n_chunks": st["last_n_chunks"],
                     "timing": "kernel_ms = median of the library's CUDA events around this kernel alone over the same K steps, "
                               "repeated with option timing=1 right after the asynchronous timed region"})

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": steps, "warmup": warmup,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "config": args.config, "seed": w.seed, "n_q": w.n_q, "n_states": w.n_states,
                       "nbf": w.basis.nbf, "n_pairs_all": st["n_pairs_all"], "n_pairs_kept": st["n_pairs_kept"],
                       "pairs_kept_per_class": st["pairs_kept_per_class"], "cond_S": w.cond_S,
                       "s4_api": {"grid": "scarf_form_factors_grid", "sph": "scarf_form_factors_sph", "list": "scarf_form_factors"}[path],
                       "inversion_symmetry_used": bool(path in ("grid", "sph") and st["last_grid_symmetric"]),
                       "q_points_evaluated": int(n_eval_q),
                       "l2": "flushed between timed steps (256 MB write, untimed)",
                       "parallelism": "replicas only" if world > 1 else "single GPU"},
            "job_seconds": ms_per_step * 1e-3, "wall_s_timed_region": head["wall_s"],
            "delivered_evals_per_s": world * st["evals_per_q"] * w.n_q / (ms_per_step * 1e-3),
            "paper_unit": {"cartesian_term_pairs": st["cart_term_pairs"],
                           "term_pair_q_state_per_s": world * float(st["cart_term_pairs"]) * w.n_q * w.n_states / (ms_per_step * 1e-3),
                           "note": "ordered Cartesian-term pairs N_c^2 of Eq. (68) PAPER.md:505-508 x q-points x states delivered per second"},
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                    "job_seconds": e2e_s,
                    "note": ("host T (pinned) -> device copy and the pinned host `out` inside the timed region; on the product-grid paths the "
                             "kernel's last chunks store the finished values straight into the pinned buffer (option host_zero_copy), so the "
                             "d2h bytes cross PCIe while the kernel runs" if path == "grid" else
                             "host T (pinned) -> device copy; `out` computed on the device and copied once into the pinned host buffer" if path == "sph" else
                             "host T, q (pinned) -> device copies and the sliced device -> host download of `out` inside the timed region")},
            "gpu_launches": int(steps * (st["last_kernel_launches"] + st["last_fold_launches"])),
            "clocks": clocks, "roofline": roofline}

    for name, obj in (("list_path", list_path), ("grid_path", grid_path), ("grid_path_no_symmetry", grid_plain),
                      ("grid_path_box_kernel", grid_box), ("grid_path_row_kernel", grid_row), ("sph_path", sph_path), ("sph_path_no_symmetry", sph_plain)):
        if obj is not None:
            obj["roofline"] = alu_roofline(obj["slots_main_kernel"], obj["main_kernel_ms"], obj["kernel"])
            line[name] = obj
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
        line["cpu_baseline"] = {"value": cpu_evals / dt, "unit": UNIT, "cores": threads, "cpu_model": cpu_model(), "kind": "oracle",
                                "sample": f"{len(idx)} of {w.n_q} q-points (seeded sample), all {w.n_states} states, "
                                          f"every primitive pair ({st['n_pairs_all']}, unscreened)",
                                "seconds": dt, "job_seconds_extrapolated": dt * w.n_q / len(idx),
                                "unit_note": "the oracle loops over ordered basis-function x primitive pairs and screens nothing; its "
                                             "evaluations are counted on ALL primitive shell pairs, the GPU's on the kept ones: compare "
                                             "job_seconds_extrapolated with job_seconds, not the two evals/s"}
        line["parity"] = {"max_rel_err_vs_oracle_on_sample": err, "tolerance": 1e-10, "ok": bool(err <= 1e-10)}
        # kappa_s = max_q sum_{mu nu} |g T_mu_nu I_mu_nu(q)| / max_q |f_s(q)| (SURVEY.md §8(c) "achievable tolerance"), from the
        # oracle's pair integrals on a few sampled q: round-off of any summation order is ~ 1e-16 * kappa
        kq = idx[:: max(1, len(idx) // 24)][:24]
        num = np.zeros(w.n_states)
        for i in kq:
            I = oracle.pair_matrix(w.basis, w.q[i])
            num = np.maximum(num, 2.0 * np.sum(np.abs(w.T * I[None]), axis=(1, 2)))
        kap = num / np.max(np.abs(f_ref), axis=1)
        line["kappa"] = {"max_over_states": float(np.max(kap)), "median": float(np.median(kap)), "q_points": int(len(kq)),
                         "note": "max over sampled q of sum|term| over max over the oracle sample of |f_s|"}
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

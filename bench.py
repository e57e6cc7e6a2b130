#!/usr/bin/env python
"""bench.py -- throughput of the ELBO-and-gradient hot path (BASELINE.json metric).

A *step* is one pass of the whole hot path over one batch of synthetic input: one optimisation
iteration of the variational fit (Philox draws -> transform -> forward profile + residual ->
backward six sums -> chain rule + reduction over draws -> Adam), i.e. one replay of the CUDA Graph
xrdvi_fit runs.  Workload: config 1 of BASELINE.json (K=50 candidates = 2^50 combinations,
N=4001, S=256 draws) unless --config says otherwise.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference]

One JSON line on stdout (rank 0).  `value` = peak.point pair evaluations per second (forward +
backward of one in-window (peak, grid point) pair of one draw count as ONE evaluation), whole job.
"""
from __future__ import annotations

import argparse
import json
import os
import pathlib
import statistics
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = pathlib.Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

METRIC = "ELBO+grad peak-point evals/s"
UNIT = "pair-evals/s"
L2_FLUSH_BYTES = 256 << 20          # > 126 MB L2
DOM_KERNEL = "elbo_tile_kernel"     # the dominant kernel of a step (roofline object)
REF_DRAWS = 16                      # draws per step of the oracle arm (bounded sample)
FULL_FIT_BUDGET_S = 30.0            # the whole-fit leg of the default run is skipped above this prediction
# Plain-formulation issue model of one pair: forward 5 FP32 + 2 MUFU,
# backward 14 FP32 + 2 MUFU + 1/4 LDG.128; MUFU 16 lanes/SM/clk, FP32 128 lanes/SM/clk, 4 issue/SM/clk.


class ClockSampler:
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.tmp = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.proc = None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.FIELDS}", "--format=csv,noheader,nounits", "-lms", "100",
                 "-i", str(index)], stdout=self.tmp, stderr=subprocess.DEVNULL)
        except OSError:
            self.proc = None

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        self.tmp.flush()
        rows = [ln.strip().split(", ") for ln in open(self.tmp.name) if ln.strip()]
        os.unlink(self.tmp.name)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for nm, v in zip(names, r[3:7]):
                if v.strip().lower() == "active":
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "reasons": sorted(reasons),
                "samples": len(sm)}


def measured_peaks() -> dict:
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        try:
            return json.loads(p.read_text())
        except Exception:
            pass
    return {}


CAPTURE_FILE = "profiles/r2_capture_counters.txt"


def captured_counters(cfg: int):
    """(kernel, DRAM bytes per launch, warp instructions per launch, pipe utilisation) of the dominant kernel at config
    `cfg` from the committed `ncu --set full` capture of THIS build (profiles/r2_capture_counters.txt: kernel, config,
    dram bytes, warp instructions, then issue / XU / FMA pipe activity in per cent of the active cycles; written from the
    capture named in its header), or (DOM_KERNEL, None, None, None) when no capture exists."""
    p = ROOT / CAPTURE_FILE
    if p.exists():
        for ln in p.read_text().splitlines():
            t = ln.split()
            if len(t) in (4, 7) and not ln.startswith("#") and t[1] == str(cfg):
                util = ({"issue_active_pct": float(t[4]), "xu_pipe_pct": float(t[5]), "fma_pipe_pct": float(t[6])}
                        if len(t) == 7 else None)
                return t[0], int(t[2]), int(t[3]), util
    return DOM_KERNEL, None, None, None


def run_reference(args, rank: int) -> None:
    """Oracle arm: the fp64 CPU oracle, as it stands, on the host cores (rank 0 only)."""
    if rank != 0:
        return
    from oracle import xrdvi_oracle as orc
    from paper_2501_09308_b200 import synth
    wl = synth.make_workload(args.config, n_patterns=1 if args.config == 3 else None,
                             n_restarts=1 if args.config == 2 else None)
    o = orc.from_workload(wl)
    S = min(wl.S, REF_DRAWS)
    pairs = o.pair_count()
    st = o.init_state()
    mom = None
    st, mom, _ = o.fit(st, args.warmup, S, seed=1, first_step=1, mom=mom)
    t0 = time.perf_counter()
    st, mom, _ = o.fit(st, args.steps, S, seed=1, first_step=1 + args.warmup, mom=mom)
    dt = time.perf_counter() - t0
    value = pairs * S * args.steps / dt
    cores = orc.num_threads()
    sample = f"{S} of {wl.S} draws per step, 1 pattern x 1 restart, all {wl.K} phases and {wl.N} points"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"config{args.config}: K={wl.K} N={wl.N} M={wl.M} draws/step={S}",
                   "pairs_per_instance": pairs},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def run_ours(args, rank: int, local_rank: int, world: int) -> None:
    import torch
    from paper_2501_09308_b200 import Xrdvi, replicas, synth

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the hot path has no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1 or ("RANK" in os.environ and "MASTER_ADDR" in os.environ):   # launched by torchrun (any N)
        import torch.distributed as dist_mod
        dist_mod.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
        dist = dist_mod

    # weak scaling: every rank fits its own replica (own jittered restart, own draw seed) of the same workload; the path
    # shards over independent (pattern, restart) instances with no data-path collective.
    wl = synth.make_workload(args.config)
    gpu = Xrdvi.from_workload(wl, device=local_rank)
    seeds = replicas.replica_seeds(rank)
    gpu.reset_state(seed=seeds["state_seed"], restart_offset=seeds["restart_offset"])
    S, T = wl.S, wl.P * wl.R * wl.S
    pairs = gpu.pair_count
    gpu.bench_steps(max(args.warmup, 1), S=S, seed=seeds["draw_seed"], l2_flush_bytes=L2_FLUSH_BYTES)

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    barrier()
    sampler = ClockSampler(local_rank) if rank == 0 else None
    ms = gpu.bench_steps(args.steps, S=S, seed=seeds["draw_seed"], l2_flush_bytes=L2_FLUSH_BYTES)
    barrier()
    t_ms = replicas.max_over_ranks(float(ms.astype(np.float64).sum()), dist, "cuda")
    # per-kernel device times, measured live on the launching stream (CUDA events inside the library)
    tk = gpu.time_kernels(S=S, seed=seeds["draw_seed"], reps=30)

    # end to end through the C ABI with HOST buffers: create (H2D of the pattern and peak tables) +
    # fit + read-back of the variational parameters and inclusion probabilities, host wall clock.
    barrier()
    t0 = time.perf_counter()
    gpu2 = Xrdvi.from_workload(wl, device=local_rank)
    gpu2.reset_state(seed=seeds["state_seed"], restart_offset=seeds["restart_offset"])
    st, inc, _ = gpu2.fit(args.steps, S=S, seed=seeds["draw_seed"])
    e2e_s = replicas.max_over_ranks(time.perf_counter() - t0, dist, "cuda")
    # the same through one xrdvi_elbo_grad call per step: H2D of the variational parameters, D2H of ELBO and
    # gradient, and a stream synchronisation in EVERY step (the per-call cost a host-side optimiser would see)
    n_calls = min(args.steps, 200)
    barrier()
    t0 = time.perf_counter()
    for i in range(n_calls):
        gpu2.elbo_grad(state=st, S=S, seed=seeds["draw_seed"], iteration=i + 1)
    percall_s = replicas.max_over_ranks(time.perf_counter() - t0, dist, "cuda")
    h2d = 8 * (wl.two_theta.size + wl.y.size + wl.background.size + wl.peak_pos.size + wl.peak_int.size
               + wl.peak_ofs.size)
    d2h = st.nbytes + inc.nbytes
    gpu2.close()

    # The second half of BASELINE.json's metric -- wall-clock of the WHOLE fit of the config (config 1: K=50 =
    # 2^50 combinations, 2000 iterations) -- measured independently of --steps: xrdvi_create + xrdvi_fit(all
    # iterations) + read-back through the C ABI with host buffers, host wall clock, max over ranks.  Skipped (with
    # the reason) only when the per-step time just measured predicts more than FULL_FIT_BUDGET_S seconds.
    ms_step = float(ms.astype(np.float64).mean())
    full = {"fit_iterations_full": int(wl.iterations), "fit_wall_s_full": None}
    adaptive = None
    W = float(wl.hyper.get("window_W", 0.0))
    predicted_s = ms_step * 1e-3 * wl.iterations
    if predicted_s > FULL_FIT_BUDGET_S:
        full["skipped"] = f"predicted {predicted_s:.0f} s > {FULL_FIT_BUDGET_S:.0f} s budget of the default run"
    else:
        barrier()
        t0 = time.perf_counter()
        gpu3 = Xrdvi.from_workload(wl, device=local_rank)
        gpu3.reset_state(seed=seeds["state_seed"], restart_offset=seeds["restart_offset"])
        _, inc_full, _ = gpu3.fit(wl.iterations, S=S, seed=seeds["draw_seed"])
        full["fit_wall_s_full"] = replicas.max_over_ranks(time.perf_counter() - t0, dist, "cuda")
        full["covers"] = ("xrdvi_create (host fp64 preprocessing + H2D) + xrdvi_fit(all iterations) + D2H of "
                          "parameters and inclusion probabilities, host wall clock")
        gpu3.reset_state(seed=seeds["state_seed"], restart_offset=seeds["restart_offset"])
        barrier()
        t0 = time.perf_counter()
        gpu3.fit(wl.iterations, S=S, seed=seeds["draw_seed"])           # the same fit on the existing handle (no create)
        full["fit_wall_s_full_existing_handle"] = replicas.max_over_ranks(time.perf_counter() - t0, dist, "cuda")
        # the steps of a fit are not equally expensive (the Gaussian-core extent follows the sampled widths and shifts:
        # the first steps, which the --steps region times from a fresh state, are the slowest): mean over the whole fit
        full["ms_per_step_whole_fit"] = 1e3 * full["fit_wall_s_full_existing_handle"] / wl.iterations
        full["pair_evals_per_s_whole_fit"] = pairs * T * wl.iterations / full["fit_wall_s_full_existing_handle"]
        truth = set(wl.true_phases[0])
        full["planted_phases_recovered"] = bool(
            set(int(k) for k in np.nonzero(inc_full[0, 0] > 0.5)[0]) == truth)
        # DESIGN.md R27: the same fit with the per-phase windows refreshed from the
        # variational means every 250 steps; reported beside the headline numbers, never inside them
        if W > 0 and wl.iterations >= 500:
            gpu3.reset_state(seed=seeds["state_seed"], restart_offset=seeds["restart_offset"])
            barrier()
            t0 = time.perf_counter()
            _, inc_a, _ = gpu3.fit_adaptive(wl.iterations, 250, W, S=S, seed=seeds["draw_seed"])
            ad_s = replicas.max_over_ranks(time.perf_counter() - t0, dist, "cuda")
            ms_a = gpu3.bench_steps(20, S=S, seed=seeds["draw_seed"], l2_flush_bytes=L2_FLUSH_BYTES)
            pairs_after = gpu3.pair_count
            gpu3.set_phase_windows(None)
            t0 = time.perf_counter()
            gpu3.adapt_windows(W)                                       # one full refresh from the static tables
            refresh_ms = 1e3 * (time.perf_counter() - t0)
            adaptive = {"fit_wall_s": ad_s, "static_fit_wall_s": full["fit_wall_s_full_existing_handle"],
                        "fit_iterations": int(wl.iterations), "refresh_every": 250, "W": W, "refresh_ms": refresh_ms,
                        "pairs_per_instance_after": pairs_after,
                        "ms_per_step_after": float(ms_a.astype(np.float64).mean()),
                        "max_abs_inclusion_diff_vs_static_fit": float(np.abs(inc_a - inc_full).max()),
                        "covers": "xrdvi_fit_adaptive on an existing handle (no create), host wall clock"}
        gpu3.close()
    clocks = sampler.stop() if sampler else None

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    value = replicas.whole_job_rate(pairs * T * args.steps, world, t_ms * 1e-3)
    props = torch.cuda.get_device_properties(local_rank)
    n_sm = props.multi_processor_count
    peaks = measured_peaks()
    f_max = 1e6 * float(peaks.get("sm_max_mhz", 1965.0))
    # dominant kernel: the fused profile + residual + backward kernel (one launch per step)
    dom_ms = tk["ms_tile"]
    achieved = pairs * T / (dom_ms * 1e-3)
    r_plain = n_sm * f_max * 16.0 / 4.0          # plain formulation: 4 MUFU per pair (2 per pass), 16 MUFU lanes/SM/clk
    dom_kernel, traffic, warp_instr, pipe_util = captured_counters(args.config)
    roofline = {
        "bound": "alu", "kernel": dom_kernel, "achieved": achieved / 1e9, "peak": r_plain / 1e9,
        "unit": "Gpair/s", "frac": achieved / r_plain, "traffic": traffic,
        "traffic_source": (f"{CAPTURE_FILE} (ncu --set full capture of this build: dram read + write bytes per launch)"
                           if traffic is not None else f"null: no ncu capture of this build at config {args.config} "
                                                       f"in {CAPTURE_FILE}"),
        # distance of the kernel from the hardware's own bound for the instruction stream it actually executes:
        # warp instructions per launch (same capture) / (SMs x 4 issue slots per clock x f_clk x kernel time)
        "issue_frac": (warp_instr / (n_sm * 4.0 * f_max * dom_ms * 1e-3) if warp_instr else None),
        "warp_instructions_per_launch": warp_instr,
        # how busy the kernel keeps the pipes its own formulation uses (same capture, one launch under ncu: sm__
        # inst_executed_pipe_xu, sm__pipe_fma_cycles_active, smsp__issue_active in % of the active cycles)
        "pipe_util_captured": pipe_util,
        "peak_source": f"derived: {n_sm} SMs x {f_max / 1e6:.0f} MHz (MEASURED_PEAKS sm_max_mhz) x 16 MUFU lanes / "
                       f"4 MUFU per pair (plain forward+backward formulation, DESIGN.md Roofline)",
        "ms_tile": tk["ms_tile"], "ms_tile_forward_only": tk["ms_tile_forward_only"], "ms_update": tk["ms_update"],
        "ms_iteration_unfused": tk["ms_iteration"],
    }
    if clocks and clocks.get("sm_mhz"):
        roofline["frac_at_achieved_clock"] = achieved / (n_sm * 1e6 * clocks["sm_mhz"] * 4.0)

    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        from oracle import xrdvi_oracle as orc
        wl1 = wl if (wl.P == 1 and wl.R == 1) else synth.make_workload(args.config, n_patterns=1, n_restarts=1)
        o = orc.from_workload(wl1)
        Sc = min(wl1.S, 256)
        st0 = o.init_state()
        o.elbo_grad(st0, min(Sc, 16), 1, 1)
        reps, t0 = 0, time.perf_counter()
        while True:
            o.elbo_grad(st0, Sc, 1, 1 + reps)
            reps += 1
            if time.perf_counter() - t0 > 10.0 or reps >= 50:
                break
        dt = time.perf_counter() - t0
        cpu = {"value": o.pair_count() * Sc * reps / dt, "unit": UNIT, "cores": orc.num_threads(), "kind": "oracle",
               "sample": f"{reps} ELBO+gradient evaluations of {Sc} draws (1 pattern x 1 restart) of config {args.config}"}

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": t_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"config{args.config}: K={wl.K} (2^{wl.K} combinations) N={wl.N} M={wl.M} "
                               f"P={wl.P} R={wl.R} S={wl.S}, window +-{gpu.n_c} points",
                   "pairs_per_instance": pairs, "instances_per_step": T,
                   "l2": f"flushed between timed steps ({L2_FLUSH_BYTES >> 20} MiB memset outside the event brackets)",
                   "parallelism": f"replicas x{world} (independent restarts, no collective)"},
        "fit_wall_s": e2e_s, "fit_iterations": args.steps,
        "fit_wall_s_full": full["fit_wall_s_full"], "fit_iterations_full": full["fit_iterations_full"],
        "full_fit": full,
        "e2e": {"value": replicas.whole_job_rate(pairs * T * args.steps, world, e2e_s), "unit": UNIT,
                "h2d_bytes_per_step": h2d / args.steps, "d2h_bytes_per_step": d2h / args.steps,
                "covers": "xrdvi_create (host fp64 preprocessing + H2D) + xrdvi_fit + D2H of parameters and "
                          "inclusion probabilities; inputs are uploaded once per fit"},
        "e2e_per_call": {"value": replicas.whole_job_rate(pairs * T * n_calls, world, percall_s), "unit": UNIT,
                         "calls": n_calls, "h2d_bytes_per_step": int(st.nbytes), "d2h_bytes_per_step": int(st.nbytes + 8 * wl.P * wl.R),
                         "covers": "one xrdvi_elbo_grad call per step with host buffers: H2D of the variational "
                                   "parameters, draw + tile + reduce kernels, D2H of ELBO and gradient, stream sync"},
        "gpu_launches": 2 * args.steps + 1,
        "roofline": roofline,
        "adaptive_windows": adaptive,
        "cpu_baseline": cpu,
        "clocks": clocks,
    }
    print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2000)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--config", type=int, default=1)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, rank)
    else:
        run_ours(args, rank, local_rank, world)


if __name__ == "__main__":
    main()

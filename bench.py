#!/usr/bin/env python
"""Benchmark of the ENUF reciprocal-space energy+force path (BASELINE.json metric).

    python bench.py --gpus N --steps K --warmup W            # this repo's CUDA path
    python bench.py --impl reference --steps K --warmup W    # the CPU oracle, as it stands

A "step" is one pass of the whole hot path (bin, spread, FFT+scale+energy, inverse FFT,
gather) over BASELINE.json config 5 (N = 1e6, n = 256, Kaiser-Bessel m = 6, fp32); every
step sees positions displaced by a fresh random 0.05 per coordinate (the config's 100-step
loop), so every step re-bins.  For N > 1 GPUs ONE system is sharded by particle over the ranks
(HP-ENUF: every rank spreads and transforms its own particles, one all-reduce of the
partial spectra, every rank finishes for its own particles; strong scaling);
`--parallel replicas` runs independent copies instead.  One JSON line is printed by rank 0.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "enuf_recip_energy_force_particles_per_sec"
UNIT = "particles/s"
HBM_FALLBACK_GBS = 6650.0     # B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg5")
    ap.add_argument("--variant", default="analytic", choices=["analytic", "ik"])
    ap.add_argument("--parallel", default=None, choices=["replicas", "sharded"],
                    help="N > 1: ONE system sharded by particle with an all-reduce of the partial spectra (strong "
                         "scaling; the default, DESIGN.md section 9) or independent replicas (weak scaling, no "
                         "data-path collective)")
    ap.add_argument("--e2e-steps", type=int, default=20)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-comparisons", action="store_true",
                    help="skip the context timings (cuFFT round trip, ik force variant)")
    return ap.parse_args()


# ---------------------------------------------------------------------- inputs

def step_positions(w, steps: int, rank: int):
    """Positions for `steps` consecutive steps: r_{s+1} = wrap(r_s + 0.05 (2U - 1)) (config 5)."""
    from enuf_inputs import displaced_positions
    amp = w.meta.get("step_displacement", 0.05 * w.L / 215.0)
    out = np.empty((steps,) + w.r.shape, dtype=w.r.dtype)
    r = w.r
    for s in range(steps):
        out[s] = r
        r = displaced_positions(r, w.L, w.seed + 7919 * rank, s, amp)
    return out


# ---------------------------------------------------------------------- algorithmic bytes

def algorithmic_bytes(w, variant: str, n_charged: int, n_local: int = None) -> dict:
    """Bytes each stage must move per evaluation: every input read
    once, every output written once, at the pruned sizes."""
    B = 8 if w.dtype == "f64" else 4
    n, kc, N = w.n, w.k_cut, (w.N if n_local is None else n_local)
    kx, ky = kc + 1, 2 * kc + 1
    n3 = n ** 3
    a1 = n * n * kx * 2 * B          # [z][y][kx] complex
    a2 = n * ky * kx * 2 * B         # [z][ky][kx] complex
    nf = 3 if variant == "ik" else 1
    fwd = (n3 * B + a1) + (a1 + a2)
    zf = a2 + nf * a2
    inv = nf * ((a2 + a1) + (a1 + n3 * B))
    return {
        "bin": N * 4 * B + n_charged * (4 * B + 8),
        "spread": n_charged * (4 * B + 4) + n3 * B,
        "fft": fwd + zf + inv,
        "gather": nf * n3 * B + n_charged * (4 * B + 8) + N * 3 * B,
    }


def measured_hbm_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return HBM_FALLBACK_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


def recorded_traffic(stage: str):
    """dram bytes per launch of the stage's kernel from the committed ncu capture, or None."""
    try:
        with open(os.path.join(ROOT, "profiles", "dram_traffic.json")) as fh:
            v = json.load(fh).get(stage)
            return float(v) if v is not None else None
    except Exception:
        return None


# ---------------------------------------------------------------------- clocks

class ClockSampler:
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.tmp = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.proc = None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={index}", f"--query-gpu={self.FIELDS}", "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=self.tmp, stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def _lines(self) -> int:
        try:
            with open(self.tmp.name) as fh:
                return sum(1 for line in fh if line.count(",") >= 6)
        except OSError:
            return 0

    def wait_first(self, keep_busy, timeout: float = 3.0) -> None:
        """nvidia-smi takes a few hundred ms to start, longer than a 100-step timed region: keep the GPU
        under the same (untimed) load until the first sample is there, then mark where the timed region begins."""
        t0 = time.perf_counter()
        while self.proc is not None and self._lines() == 0 and time.perf_counter() - t0 < timeout:
            keep_busy()
        self.n0 = self._lines()

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        self.tmp.flush()
        rows = []
        with open(self.tmp.name) as fh:
            for line in fh:
                parts = [p.strip() for p in line.split(",")]
                if len(parts) >= 7:
                    rows.append(parts)
        os.unlink(self.tmp.name)
        n0 = getattr(self, "n0", 0)
        if len(rows) > n0:
            rows = rows[n0:]          # samples taken from the start of the timed region on
        if not rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        sm = sorted(float(r[0]) for r in rows if r[0].replace(".", "").isdigit())
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        reasons = [nm for i, nm in enumerate(names) if any(r[3 + i].lower().startswith("active") for r in rows)]
        pw = [float(r[2]) for r in rows if r[2].replace(".", "").isdigit()]
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": float(rows[0][1]),
                "reasons": reasons, "samples": len(rows), "power_w_max": max(pw) if pw else None}


# ---------------------------------------------------------------------- reference arm (CPU oracle)

def sub_box_sample(w, scale: int):
    """A bounded sample of the workload: the particles of the sub-box [0, L/scale)^3 with the
    grid, cutoff and bandwidth divided by `scale` (same density, cell size and alpha)."""
    if scale == 1:
        return w.r, w.q, w.L, w.k_cut, w.n
    Ls = w.L / scale
    keep = np.all(w.r < np.asarray(Ls, dtype=w.r.dtype), axis=1)
    keep[np.nonzero(keep)[0][(keep.sum() // 2) * 2:]] = False       # even count
    return w.r[keep], w.q[keep], Ls, w.k_cut // scale, w.n // scale


def oracle_step(O, w, r, q, L, k_cut, n, variant):
    t = time.perf_counter()
    # (grids of 3 * 2^k points, sigma = 1.5: the oracle's radix-2 transform does not apply, its plain DFT does)
    out = O.enuf(r, q, L, w.alpha, k_cut, n, w.m, w.window, w.sigma, variant=variant,
                 slater_lambda=w.slater_lambda, use_dft=(n & (n - 1)) != 0)
    return time.perf_counter() - t, out


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from enuf_inputs import make_workload
    from oracle import enuf_oracle as O
    O.build()
    w = make_workload(args.workload)
    total = args.steps + args.warmup
    budget_s = 150.0
    # full-size cost is ~30-40 s on 8 cores and falls ~ 1/scale^3; start from a guess, refine
    scale = 1
    while scale < 8 and w.n // (scale * 2) >= 32 and 40.0 / scale ** 3 * total > budget_s:
        scale *= 2
    r, q, L, kc, n = sub_box_sample(w, scale)
    times = []
    for s in range(total):
        dt, _ = oracle_step(O, w, r, q, L, kc, n, args.variant)
        if s >= args.warmup:
            times.append(dt)
    t_step = sum(times) / len(times)
    value = q.shape[0] / t_step
    sample = (f"{args.workload} sub-box 1/{scale}^3 of the volume: N={q.shape[0]}, n={n}, k_cut={kc}, "
              f"same alpha/density/window; one full Oracle-B evaluation (forces on all particles) per step")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t_step, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        # what was timed: the sub-box, not the full workload (same density, cell size, alpha and window)
        "config": {"workload": args.workload, "variant": args.variant, "N": int(q.shape[0]), "L": float(L), "n": int(n),
                   "k_cut": int(kc), "m": int(w.m), "window": w.window, "same_config": scale == 1,
                   "full_workload": {"N": int(w.N), "L": float(w.L), "n": int(w.n), "k_cut": int(w.k_cut)},
                   "sample": sample},
        "evals_per_sec": 1.0 / t_step,
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": O.num_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------- rank plumbing (replicas only)

def reduce_over_ranks(x: float, op: str, device: str = "cuda") -> float:
    """max / sum of a scalar over all ranks (identity when torch.distributed is not initialised).
    The only collectives of the N > 1 run: the path itself has no data-path exchange (DESIGN.md
    section 9).  Covered on CPU by tests/test_multirank_gloo.py (gloo, world_size 2)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(x)
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX if op == "max" else dist.ReduceOp.SUM)
    return float(t.item())


def whole_job_value(n_particles: int, world: int, ms_step_max: float) -> float:
    """Whole-job throughput of `world` independent replicas: all ranks' particles / slowest rank's time."""
    return n_particles * world / (ms_step_max * 1e-3)


# ---------------------------------------------------------------------- this repo's arm

def run_ours(args):
    import torch
    import torch.distributed as dist
    import paper_2004_12484_b200 as enuf
    from enuf_inputs import make_workload

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; this library has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()

    def max_over_ranks(x: float) -> float:
        return reduce_over_ranks(x, "max", "cuda")

    def sum_over_ranks(x: float) -> float:
        return reduce_over_ranks(x, "sum", "cuda")

    w = make_workload(args.workload)
    K, W = args.steps, args.warmup
    tdtype = torch.float64 if w.dtype == "f64" else torch.float32
    sharded = args.parallel == "sharded" or (args.parallel is None and world > 1)
    N_sys = w.N
    if sharded:
        # ONE system, the same on every rank; this rank owns the particles [lo, hi)
        lo, hi = enuf.shard_bounds(w.N, rank, world)
        pos_host = np.ascontiguousarray(step_positions(w, W + K, 0)[:, lo:hi])
        q_host = np.ascontiguousarray(w.q[lo:hi])
    else:
        lo, hi = 0, w.N
        pos_host = step_positions(w, W + K, rank)                   # (W+K, N, 3)
        q_host = w.q
    N_loc = hi - lo
    pos_pinned = torch.from_numpy(pos_host).pin_memory()
    q_pinned = torch.from_numpy(q_host).pin_memory()
    pos_dev = pos_pinned.cuda()
    q_dev = q_pinned.cuda()
    F_dev = torch.empty((N_loc, 3), dtype=tdtype, device="cuda")
    n_charged = int(np.count_nonzero(q_host))

    plan = enuf.Plan.from_workload(w, variant=args.variant, profile=False)
    if sharded:
        plan.close()
        plan = enuf.Plan(N_loc, w.L, w.alpha, w.k_cut, w.M, sigma=w.sigma, m=w.m, dtype=tdtype, window=w.window,
                         variant=args.variant, slater_lambda=w.slater_lambda)
    evaluate = plan.energy_forces_sharded if sharded else plan.energy_forces
    for s in range(W):
        evaluate(pos_dev[s], q_dev, F=F_dev, want_energy=False)
    sampler = ClockSampler(local) if rank == 0 else None
    if sampler:
        def keep_busy():
            if sharded:                      # its evaluation holds a collective: rank 0 must not run one alone
                time.sleep(0.05)
                return
            for s_ in range(W):
                evaluate(pos_dev[s_], q_dev, F=F_dev, want_energy=False)
            torch.cuda.synchronize()
        sampler.wait_first(keep_busy)
    # Two passes over the same K steps.  The first is the timed region (`value`, `ms_per_step`): the library as a
    # user runs it, no event between the kernels of an evaluation (each kernel is launched as a programmatic
    # dependent of its predecessor, ENUF_OPT_PDL).  The second records the library's per-stage events
    # (ENUF_OPT_PROFILE; an event between two kernels orders them fully) and gives `stages` and the roofline
    # kernel's duration; its own step time is reported as `ms_per_step_profiled`.
    torch.cuda.synchronize()
    barrier()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches = 0
    torch.cuda.synchronize()
    ev0.record()
    for s in range(K):
        evaluate(pos_dev[W + s], q_dev, F=F_dev, want_energy=False)
        launches += plan.launch_count()
    ev1.record()
    torch.cuda.synchronize()
    barrier()
    ms_total = max_over_ranks(ev0.elapsed_time(ev1))
    E_last = plan.energy()
    plan.set(enuf.OPT_PROFILE, 1)
    torch.cuda.synchronize()
    barrier()
    ev2, ev3 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev2.record()
    for s in range(K):
        evaluate(pos_dev[W + s], q_dev, F=F_dev, want_energy=False)
    ev3.record()
    torch.cuda.synchronize()
    barrier()
    ms_step_profiled = max_over_ranks(ev2.elapsed_time(ev3)) / K
    clocks = sampler.stop() if sampler else None
    stage_ms, n_prof = plan.stage_ms_mean()
    ms_step = ms_total / K
    value = N_sys / (ms_step * 1e-3) if sharded else whole_job_value(w.N, world, ms_step)
    total_launches = int(sum_over_ranks(float(launches)))

    # ---- end to end: host buffers in, host forces + energy out, through the C ABI
    plan.set(enuf.OPT_PROFILE, 0)
    Ke = max(1, min(args.e2e_steps, K))
    F_host = torch.empty((N_loc, 3), dtype=tdtype).pin_memory()
    if sharded:
        r_st, q_st = torch.empty_like(pos_dev[0]), torch.empty_like(q_dev)

        def host_step(s_):       # pinned host shard -> device, sharded evaluation, forces + energy back
            r_st.copy_(pos_pinned[s_], non_blocking=True); q_st.copy_(q_pinned, non_blocking=True)
            plan.energy_forces_sharded(r_st, q_st, F=F_dev, want_energy=False)
            F_host.copy_(F_dev, non_blocking=True)
            return plan.energy()
        api = "Plan.energy_forces_sharded (pinned host shard -> device, all-reduce, host F, E)"
    else:
        def host_step(s_):
            return plan.energy_forces_host(pos_pinned[s_], q_pinned, F=F_host)[0]
        api = "enuf_energy_forces_host (pinned host r, q -> host F, E; ENUF_OPT_CUDA_GRAPH on)"
        # the host entry point evaluates on the plan's own staging buffers, i.e. the same device pointers
        # every call: the evaluation is captured in the second warm-up call and replayed in the timed ones
        plan.set(enuf.OPT_CUDA_GRAPH, 1)
    for s in range(3):
        host_step(s)
    torch.cuda.synchronize()
    barrier()
    t0 = time.perf_counter()
    for s in range(Ke):
        E_h = host_step(W + s)
    torch.cuda.synchronize()
    t_e2e = max_over_ranks((time.perf_counter() - t0) / Ke)
    barrier()
    if not sharded:
        plan.set(enuf.OPT_CUDA_GRAPH, 0)
    esz = 8 if w.dtype == "f64" else 4
    e2e = {"value": (N_sys if sharded else w.N * world) / t_e2e, "unit": UNIT, "ms_per_step": 1e3 * t_e2e, "steps": Ke,
           "h2d_bytes_per_step": int(N_loc * 4 * esz), "d2h_bytes_per_step": int(N_loc * 3 * esz + 8),
           "api": api}
    if not sharded:
        # the same call with q = NULL: the charges of the previous host call stay resident on the device
        # (an MD loop moves positions, not charges); r in, F and E out every step
        plan.set(enuf.OPT_CUDA_GRAPH, 1)
        for s in range(3):
            plan.energy_forces_host(pos_pinned[s], q_pinned if s == 0 else None, F=F_host)
        torch.cuda.synchronize()
        barrier()
        t0 = time.perf_counter()
        for s in range(Ke):
            plan.energy_forces_host(pos_pinned[W + s], None, F=F_host)
        torch.cuda.synchronize()
        t_res = max_over_ranks((time.perf_counter() - t0) / Ke)
        barrier()
        plan.set(enuf.OPT_CUDA_GRAPH, 0)
        e2e["q_resident"] = {"value": w.N * world / t_res, "unit": UNIT, "ms_per_step": 1e3 * t_res,
                             "h2d_bytes_per_step": int(N_loc * 3 * esz), "d2h_bytes_per_step": int(N_loc * 3 * esz + 8)}
    exchange = None
    if sharded:
        # the one exchange step of the sharded path, timed alone: all-reduce (sum) of the partial spectrum buffer
        buf = plan.spectrum_tensor()
        for _ in range(3):
            enuf.all_reduce_sum_(buf)
        c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize(); barrier(); c0.record()
        for _ in range(10):
            enuf.all_reduce_sum_(buf)
        c1.record(); torch.cuda.synchronize()
        exchange = {"collective": "all_reduce(SUM) of the partial spectrum [z][ky'][kx] after the Y pass (NCCL)",
                    "bytes_per_rank": int(buf.numel() * buf.element_size()),
                    "ms": max_over_ranks(c0.elapsed_time(c1) / 10), "ranks": world}

    if rank != 0:
        plan.close()
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant stage (CUDA events recorded on the plan's stream, per evaluation)
    peak, peak_src = measured_hbm_peak()
    abytes = algorithmic_bytes(w, args.variant, n_charged, N_loc)
    stages = {}
    for st in ("bin", "spread", "fft", "gather"):
        gbs = abytes[st] / (stage_ms[st] * 1e-3) / 1e9 if stage_ms[st] > 0 else 0.0
        stages[st] = {"ms": stage_ms[st], "algorithmic_bytes": abytes[st], "GBps": gbs, "hbm_frac": gbs / peak}
    # spread and gather are bound by FP32 FMA issue, not by HBM: their ALU fractions too
    W3 = (2 * w.m + 1) ** 3
    sm_max = (clocks or {}).get("sm_max_mhz") or 1965.0
    peak_tf = 148 * 128 * 2 * sm_max * 1e6 / 1e12
    for st, per in (("spread", 1), ("gather", 3 if args.variant == "ik" else 2)):
        if stages[st]["ms"] > 0:
            tf = 2.0 * per * W3 * n_charged / (stages[st]["ms"] * 1e-3) / 1e12
            stages[st]["alu_TFLOPs"] = tf
            stages[st]["alu_frac"] = tf / peak_tf
    dom = max(stages, key=lambda k: stages[k]["ms"])
    if dom in ("spread", "gather"):
        # these two stages are bound by FP32 FMA issue, not by HBM.  Algorithmic
        # work = (2m+1)^3 FMAs per charged particle (spread), twice that for the analytic gather
        # (field x window and field x window derivative), three times for the ik gather.
        per = {"spread": 1, "gather": 3 if args.variant == "ik" else 2}[dom]
        flops = 2.0 * per * W3 * n_charged
        ach = flops / (stages[dom]["ms"] * 1e-3) / 1e12
        roofline = {"bound": "alu", "kernel": dom, "achieved": ach, "peak": peak_tf, "unit": "TFLOP/s",
                    "frac": ach / peak_tf, "traffic": recorded_traffic(dom),
                    "peak_source": "148 SMs x 128 FP32 lanes x 2 flop x clocks.max.sm (B200_PROFILING.md nominal table; "
                                   "DESIGN.md section 7)",
                    "algorithmic_flops": flops, "events_averaged": n_prof,
                    "hbm": {"achieved": stages[dom]["GBps"], "peak": peak, "unit": "GB/s",
                            "frac": stages[dom]["hbm_frac"], "peak_source": peak_src}}
        # what binds both kernels in practice is the shared-memory data pipe (one 128-byte wavefront per SM and clock;
        # ncu l1tex 67-79 %).  Algorithmic wavefronts: every stencil value of every particle crosses
        # it once -- the gather reads (2m+1)^3 field values per particle (32 words per wavefront); the spread's
        # register accumulation needs its window values: (2m+1)^2 (x, y) products + (2m+1) z values per particle.
        smem_peak = 148 * sm_max * 1e6
        wf = n_charged * (W3 / 32.0 if dom == "gather" else ((2 * w.m + 1) ** 2 + (2 * w.m + 1)) / 32.0)
        roofline["smem_pipe"] = {"algorithmic_wavefronts": wf, "achieved": wf / (stages[dom]["ms"] * 1e-3),
                                 "peak": smem_peak, "unit": "wavefronts/s", "frac": wf / (stages[dom]["ms"] * 1e-3) / smem_peak,
                                 "peak_source": "148 SMs x 1 wavefront per clock x clocks.max.sm (B300_MICROARCH.md: 128 B/clk/SM)"}
    else:
        roofline = {"bound": "hbm", "kernel": dom, "achieved": stages[dom]["GBps"], "peak": peak, "unit": "GB/s",
                    "frac": stages[dom]["hbm_frac"], "traffic": recorded_traffic(dom), "peak_source": peak_src,
                    "events_averaged": n_prof}

    # ---- context timings asked for by north_star (not on the product path, not the headline)
    comparisons = None
    if world == 1 and not args.no_comparisons:
        comparisons = {}
        # (1) cuFFT (torch.fft) real-to-complex + complex-to-real round trip of the full n^3 grid,
        #     against this library's pruned 5-pass FFT + scale + energy ("fft" stage above)
        g = torch.randn((w.n, w.n, w.n), dtype=tdtype, device="cuda")
        for _ in range(3):
            torch.fft.irfftn(torch.fft.rfftn(g), s=g.shape)
        c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize(); c0.record()
        for _ in range(10):
            torch.fft.irfftn(torch.fft.rfftn(g), s=g.shape)
        c1.record(); torch.cuda.synchronize()
        comparisons["cufft_rfftn_irfftn_ms"] = c0.elapsed_time(c1) / 10
        comparisons["own_fft_scale_energy_ms"] = stage_ms["fft"]
        del g
        # (2) the paper's ik force variant (three inverse FFTs and three gathers, Eq. 41-42)
        other = "ik" if args.variant == "analytic" else "analytic"
        plan2 = enuf.Plan.from_workload(w, variant=other, profile=False)
        for s_ in range(3):
            plan2.energy_forces(pos_dev[s_], q_dev, F=F_dev, want_energy=False)
        plan2.set(enuf.OPT_PROFILE, 1)
        torch.cuda.synchronize(); c0.record()
        Kc = min(10, K)
        for s_ in range(Kc):
            plan2.energy_forces(pos_dev[W + s_], q_dev, F=F_dev, want_energy=False)
        c1.record(); torch.cuda.synchronize()
        st2, _ = plan2.stage_ms_mean()
        comparisons[other + "_variant"] = {"ms_per_step": c0.elapsed_time(c1) / Kc,
                                           "stages_ms": {k: st2[k] for k in ("bin", "spread", "fft", "gather")}}
        plan2.close()
        # (3) the other two terms of Eq. 25 on the device (not part of the metric): real-space
        #     sum at the cutoff the config tunes alpha for, self term; forces accumulated onto the reciprocal ones
        r_cut = w.meta.get("r_c")
        if r_cut and r_cut <= 0.5 * w.L and not sharded:
            for s_ in range(2):
                plan.real_space(pos_dev[s_], q_dev, r_cut, F=F_dev, accumulate=True, want_energy=False)
            torch.cuda.synchronize(); c0.record()
            for s_ in range(5):
                plan.real_space(pos_dev[W + s_], q_dev, r_cut, F=F_dev, accumulate=True, want_energy=False)
            c1.record(); torch.cuda.synchronize()
            E_real, E_self, _ = plan.real_space(pos_dev[W + K - 1], q_dev, r_cut, F=F_dev, accumulate=True)
            comparisons["real_space"] = {"ms_per_step": c0.elapsed_time(c1) / 5, "r_cut": r_cut, "E_real": E_real,
                                         "E_self": E_self, "E_total_last_step": E_real + E_last - E_self}

    cpu_baseline = None
    if world == 1 and not args.no_cpu_baseline:
        from oracle import enuf_oracle as O
        O.build()
        dt, out = oracle_step(O, w, pos_host[W], w.q, w.L, w.k_cut, w.n, args.variant)
        cpu_baseline = {"value": w.N / dt, "unit": UNIT, "cores": O.num_threads(), "kind": "oracle",
                        "sample": f"1 full evaluation of {args.workload} (N={w.N}, forces on all particles), {dt:.1f} s",
                        "seconds": dt}
        # single-thread leg on a bounded sample: the 1/4^3 sub-box (same density, cell size, alpha)
        cores = O.num_threads()
        sc = 4 if w.n // 4 >= 32 else (2 if w.n // 2 >= 32 else 1)
        rs, qs, Ls, kcs, ns_ = sub_box_sample(w, sc)
        O.set_threads(1)
        dt1, _ = oracle_step(O, w, rs, qs, Ls, kcs, ns_, args.variant)
        O.set_threads(cores)
        dtm, _ = oracle_step(O, w, rs, qs, Ls, kcs, ns_, args.variant)
        cpu_baseline["single_thread"] = {"value": qs.shape[0] / dt1, "unit": UNIT, "seconds": dt1,
                                         "all_cores_same_sample": {"value": qs.shape[0] / dtm, "seconds": dtm, "cores": cores},
                                         "sample": f"sub-box 1/{sc}^3 of the volume: N={qs.shape[0]}, n={ns_}, k_cut={kcs}"}
        # Oracle A (direct Ewald sum, the definition) on configs 1-3, all cores
        oa = {}
        for name in ("cfg1", "cfg2", "cfg3"):
            wa = make_workload(name)
            t0 = time.perf_counter()
            O.direct(wa.r, wa.q, wa.L, wa.alpha, wa.k_cut, slater_lambda=wa.slater_lambda)
            oa[name] = {"seconds": time.perf_counter() - t0, "N": int(wa.N), "k_cut": int(wa.k_cut)}
        cpu_baseline["oracle_a_direct_sum"] = oa

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms_step, "ms_per_step_profiled": ms_step_profiled, "higher_is_better": True, "scaling": "strong" if sharded else "weak", "vs_baseline": None,
        "dtype": w.dtype, "data": "synthetic",
        "config": {"workload": args.workload, "N": int(w.N), "L": w.L, "alpha": w.alpha, "k_cut": w.k_cut,
                   "M": w.M, "sigma": w.sigma, "n": w.n, "m": w.m, "window": w.window, "variant": args.variant,
                   "parallelism": (f"sharded by particle x{world}, all-reduce of the partial spectrum" if sharded else
                                   f"replicas x{world}") if world > 1 else "single GPU",
                   "l2": "no explicit flush: positions differ every step and the per-step working set "
                         "(grid + spectra + particles, ~165 MB) exceeds the 126 MB L2"},
        "evals_per_sec": (1 if sharded else world) / (ms_step * 1e-3),
        "energy_last_step": E_last,
        "clocks": clocks, "e2e": e2e, "gpu_launches": total_launches,
        "roofline": roofline, "stages": stages, "cpu_baseline": cpu_baseline, "comparisons": comparisons,
        "exchange": exchange,
    }
    print(json.dumps(line), flush=True)
    plan.close()
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()

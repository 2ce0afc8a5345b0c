#!/usr/bin/env python
"""bench.py -- Landau Jacobian builds/s and GPair-evals/s (fp64) on B200.

One "step" = one pass of the whole hot path (a1-a7: fields, beta sums, all-pairs inner integral,
element matrices, CSR gather, C(f)) over BASELINE.json config 5: 512 independent velocity-space
problems on the refined Q3 mesh "3B" (308 cells, 4,928 points, 2 species), one
landau_jacobian_batched call.  value = ordered point pairs N(N-1) x problems / time, whole job.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

N > 1: launched by torchrun, one rank per GPU; the problems are independent (weak scaling: every
rank builds its own 512 problems, no data-path collective).
--impl reference: times the CPU oracle (double instantiation) on the host cores on a bounded
sample of the same workload.
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
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "landau_jacobian_gpair_evals_per_s"
UNIT = "GPair/s"
WORKLOAD = "config5: 512 problems x (2 species e+D, Q3 quadtree mesh 3B: 308 cells, 4928 points)"
# FP64 flop (2 DFMA + DMUL + DADD) and FP64-pipe instructions the pair kernel executes per ORDERED
# pair on this workload, ncu-counted (profiles/r01e_pair_kernel.md).
FLOP_PER_PAIR = 75.27
FP64_INST_PER_PAIR = 48.51
# of which DFMAs with three distinct register operands: they issue in 3 cycles instead of 2
# (measured), so the issue-cycle cost per ordered pair is 2 x 48.51 + 11.09 SMSP-cycles x 32 lanes.
FP64_3OP_INST_PER_PAIR = 11.09
FP64_LANES_PER_SM = 64      # DFMA lanes per SM per clock (B200: 148 x 64 x 2 x 1.965 GHz = 37.2 TF)
# dram__bytes_read.sum + dram__bytes_write.sum of one k_pair_sym launch on this workload, from the
# ncu --set full capture summarised in profiles/r01e_pair_kernel.md (68.7 MB read + 3.879 GB written:
# the per-source-tile partial slabs; the algorithmic minimum is 24 B/point in + 40 B/point out = 0.16 GB).
PAIR_KERNEL_DRAM_BYTES = 68.7e6 + 3.8789e9
# the same for the rest of the step (fields, slab sum, element matrices, two gathers), profiles/r01e_step_kernels.md (ncu --set full, dram read + write)
REST_DRAM_BYTES = 6.03e9   # 4.04 GB of it is k_sum_partials reading the slabs


class ClockSampler(threading.Thread):
    """One `nvidia-smi -lms 50` process sampling clocks / throttle reasons DURING the timed region
    (B200_PROFILING.md recipe); its lines are read by this thread."""

    QUERY = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.rows, self.proc = [], None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.QUERY}", "--format=csv,noheader,nounits",
                                          "-lms", "50", "-i", str(index)], stdout=subprocess.PIPE, text=True)
        except Exception:
            self.proc = None

    def run(self):
        if self.proc is None:
            return
        for line in self.proc.stdout:
            self.rows.append((time.perf_counter(), [c.strip() for c in line.split(",")]))

    def stop(self, t0: float, t1: float):
        """Summary over the samples taken in [t0, t1] (perf_counter times of the timed region)."""
        if self.proc is not None:
            self.proc.terminate()
            self.join(timeout=5)
        rows = [r for (t, r) in self.rows if t0 <= t <= t1 and len(r) >= 7] or [r for (_, r) in self.rows if len(r) >= 7]

        def num(x):
            try:
                return float(x)
            except ValueError:
                return None
        sm = [v for v in (num(r[0]) for r in rows) if v is not None]
        mx = [v for v in (num(r[1]) for r in rows) if v is not None]
        pw = [v for v in (num(r[2]) for r in rows) if v is not None]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({names[k] for r in rows for k in range(4) if r[3 + k].lower() == "active"})
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "reasons": reasons, "samples": len(rows)}


CPU_SAMPLE_PROBLEMS = 8      # of the 512: ~0.5 s each on 16 cores, i.e. tens of core-seconds in total


def cpu_baseline_sample(wl, inputs):
    """The oracle as it stands (double instantiation) on a bounded sample of the workload."""
    from oracle import landau_oracle as oracle
    oracle.build()
    sp = oracle.build_space(wl.mesh, wl.order)
    fs = [inputs.nodal_f(wl, sp.dof_r, sp.dof_z, b) for b in range(CPU_SAMPLE_PROBLEMS)]
    t0 = time.perf_counter()
    for f in fs:
        oracle.build_all(wl.mesh, wl.order, wl.species, f, 1.0, precision="d")
    dt = time.perf_counter() - t0
    pairs = CPU_SAMPLE_PROBLEMS * sp.N * (sp.N - 1)
    return pairs / dt * 1e-9, dt, os.cpu_count()


def run_reference(args):
    """--impl reference: the CPU oracle on the host cores, each step one problem of config 5."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_2104_10000_b200 import inputs
    from oracle import landau_oracle as oracle
    oracle.build()
    wl = inputs.config(5, nbatch=max(1, args.steps + args.warmup))
    sp = oracle.build_space(wl.mesh, wl.order)
    pairs = sp.N * (sp.N - 1)
    times = []
    for k in range(args.warmup + args.steps):
        f = inputs.nodal_f(wl, sp.dof_r, sp.dof_z, k)
        t0 = time.perf_counter()
        oracle.build_all(wl.mesh, wl.order, wl.species, f, 1.0, precision="d")
        if k >= args.warmup:
            times.append(time.perf_counter() - t0)
    ms = 1e3 * float(np.mean(times))
    val = pairs / (ms * 1e-3) * 1e-9
    sample = "1 of the 512 problems per step (full N=4928 mesh, a1-a8), double-precision oracle, OpenMP over i"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic", "config": {"workload": WORKLOAD, "sample": sample},
        "builds_per_s": 1e3 / ms,
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": os.cpu_count(), "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def time_single_config(binding, inputs, torch, k, variant="B", reps=20):
    """Single-problem build (split launch shape) of configs 1-4: device time per build."""
    wl = inputs.config(k, variant=variant)
    ctx = binding.LandauContext(wl.mesh, wl.order, wl.species, 1)
    r, z = ctx.dof_coords()
    f = torch.from_numpy(inputs.nodal_f(wl, r, z)).cuda()
    vals = torch.zeros((ctx.S, ctx.nnz), dtype=torch.float64, device="cuda")
    Cf = torch.zeros((ctx.S, ctx.n), dtype=torch.float64, device="cuda")
    for _ in range(3):
        ctx.jacobian(f, vals, Cf)
    torch.cuda.synchronize()
    ctx.profile_enable(True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        ctx.jacobian(f, vals, Cf)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / reps
    pair_ms, cnt = ctx.profile_read()
    ctx.profile_enable(False)
    # the same build captured once in a CUDA graph and replayed (the library makes no synchronising call)
    graph_ms = None
    try:
        side = torch.cuda.Stream()
        with torch.cuda.stream(side):
            ctx.jacobian(f, vals, Cf)
            torch.cuda.synchronize()
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=side):
                ctx.jacobian(f, vals, Cf)
            g.replay()
            e0.record()
            for _ in range(reps):
                g.replay()
            e1.record()
            torch.cuda.synchronize()
            graph_ms = e0.elapsed_time(e1) / reps
    except Exception as exc:   # reported, not fatal
        graph_ms = f"unavailable: {exc}"
    pairs = ctx.N * (ctx.N - 1)
    out = {"config": wl.name, "graph_replay_ms_per_build": graph_ms, "N": ctx.N, "S": ctx.S, "n": ctx.n, "nnz": ctx.nnz, "ms_per_build": ms,
           "builds_per_s": 1e3 / ms, "gpair_per_s": pairs / (ms * 1e-3) * 1e-9,
           "pair_kernel_ms": pair_ms / max(cnt, 1), "pair_kernel_gpair_per_s": pairs / (pair_ms / max(cnt, 1) * 1e-3) * 1e-9}
    ctx.destroy()
    return out


def time_next_rows(binding, inputs, torch, ctx5, f5, vals5, Cf5, nb):
    """SURVEY 8(f) rows at the same measurement bar: NEXT-3 (implicit-step operator, config 5) and NEXT-2
    (the paper's three 20-cell grids with ten species, Table I, 512 problems batched)."""
    out = {}
    Ez = torch.full((nb,), 0.3, dtype=torch.float64, device="cuda")
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ctx5.implicit_operator_batched(f5, Ez, 2.0, vals5, Cf5)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(3):
        ctx5.implicit_operator_batched(f5, Ez, 2.0, vals5, Cf5)
    e1.record(); torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / 3
    out["implicit_operator_config5"] = {"ms_per_step": ms, "gpair_per_s": nb * ctx5.N * (ctx5.N - 1) / (ms * 1e-3) * 1e-9,
                                        "what": "shift M + A(E_z) - J and A f - C(f) in one pass (landau_implicit_operator_batched)"}
    # NEXT-4: band LU of the nb * S matrices of the implicit step (vals5 holds them now), then one solve
    bw, md, ws = ctx5.band_sizes()
    band = torch.empty(nb * ws, dtype=torch.float64, device="cuda")
    rhs = torch.ones((nb, ctx5.S, ctx5.n), dtype=torch.float64, device="cuda")
    x = torch.empty_like(rhs)
    ctx5.band_factor_batched(vals5, band); ctx5.band_solve_batched(band, rhs, x)
    torch.cuda.synchronize()
    e2 = torch.cuda.Event(enable_timing=True)
    e0.record(); ctx5.band_factor_batched(vals5, band); e1.record(); ctx5.band_solve_batched(band, rhs, x); e2.record()
    torch.cuda.synchronize()
    fms, sms_ = e0.elapsed_time(e1), e1.elapsed_time(e2)
    nmat = nb * ctx5.S
    flop = ctx5.band_flop_per_factorization * nmat     # outer-product updates inside the envelope (executed)
    flop_band = 2.0 * ctx5.n * bw * bw * nmat          # Alg. 4.3.1 on the uniform band: n outer products of bw x bw
    out["band_lu_config5"] = {"matrices": nmat, "n": ctx5.n, "half_bandwidth_rcm": bw, "workspace_gb": nb * ws * 8e-9,
                              "factor_ms": fms, "solve_ms": sms_, "factor_tflops": flop / (fms * 1e-3) * 1e-12,
                              "factor_tflops_uniform_band_equiv": flop_band / (fms * 1e-3) * 1e-12,
                              "factorizations_per_s": nmat / (fms * 1e-3),
                              "what": "scatter + blocked outer-product band LU without pivoting, then L/U solves (one rhs)"}
    del band, rhs, x
    name, order, meshes, spc, sgrid, comps = inputs.multigrid_case("paper3")
    mg = binding.LandauMultigridContext(meshes, sgrid, order, spc, nb)
    fl = []
    for a, c in enumerate(comps):
        r, z = mg.grid_dof_coords(sgrid[a])
        fl.append(inputs.maxwellian(float(spc.mass[a]), c.n, c.T, c.zs, r, z))
    f = torch.from_numpy(np.tile(np.concatenate(fl), (nb, 1))).cuda()
    v = torch.zeros((nb, mg.vals_stride), dtype=torch.float64, device="cuda")
    c_ = torch.zeros((nb, mg.f_stride), dtype=torch.float64, device="cuda")
    mg.jacobian_batched(f, v, c_)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(5):
        mg.jacobian_batched(f, v, c_)
    e1.record(); torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / 5
    out["multigrid_paper3"] = {"workload": f"{nb} problems x (10 species on 3 grids of 20 Q3 cells: N = {mg.N}, n = {mg.f_stride})",
                               "ms_per_step": ms, "builds_per_s": nb / (ms * 1e-3),
                               "gpair_per_s": nb * mg.N * (mg.N - 1) / (ms * 1e-3) * 1e-9}
    mg.destroy()
    # The paper's throughput metric (Tables II/III, L246-270): Newton iterations per second on the e + D + 8 heavy
    # ion species, 80-cell Q3 problem -- here one iteration = implicit-step operator + band LU + solve, all on the
    # device, nb problems batched (context beside the paper's 7,005 it/s on 6 V100 + 42 P9 cores with a CPU LU).
    wl = inputs.config(6)
    c80 = binding.LandauContext(wl.mesh, wl.order, wl.species, nb)
    r, z = c80.dof_coords()
    f80 = torch.from_numpy(np.tile(inputs.nodal_f(wl, r, z), (nb, 1, 1))).cuda()
    v80 = torch.zeros((nb, c80.S, c80.nnz), dtype=torch.float64, device="cuda")
    F80 = torch.zeros((nb, c80.S, c80.n), dtype=torch.float64, device="cuda")
    d80 = torch.zeros_like(F80)
    Ez80 = torch.zeros(nb, dtype=torch.float64, device="cuda")
    bw80, _, ws80 = c80.band_sizes()
    band80 = torch.empty(nb * ws80, dtype=torch.float64, device="cuda")

    def newton():
        c80.implicit_operator_batched(f80, Ez80, 2.0, v80, F80)
        c80.band_factor_batched(v80, band80)
        c80.band_solve_batched(band80, F80, d80)
    newton(); torch.cuda.synchronize()
    e0.record()
    for _ in range(5):
        newton()
    e1.record(); torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / 5
    out["newton_iteration_ctx80"] = {"workload": f"{nb} problems x (10 species, 80 Q3 cells: N = {c80.N}, n = {c80.n}, RCM half-bandwidth {bw80})",
                                     "ms_per_batched_iteration": ms, "newton_iterations_per_s": nb / (ms * 1e-3),
                                     "what": "operator (shift M + A - J, A f - C(f)) + band LU of 10 species blocks + solve, per problem"}
    c80.destroy()
    return out


def run_ours(args):
    import torch
    from paper_2104_10000_b200 import binding, inputs

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback); use --impl reference for the CPU oracle")
    binding.lib()
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1 or "TORCHELASTIC_RUN_ID" in os.environ:      # launched by torchrun: same code path for every N
        import torch.distributed as dist
        os.environ.setdefault("NCCL_DEBUG", "WARN")           # keep stdout to the one JSON line
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    wl = inputs.config(5)
    nb = wl.nbatch
    ctx = binding.LandauContext(wl.mesh, wl.order, wl.species, nb)
    r, z = ctx.dof_coords()
    # every rank builds its own 512 problems (weak scaling); problem seeds are offset by rank
    f_host = torch.from_numpy(np.stack([inputs.nodal_f(wl, r, z, b) for b in range(nb)])).pin_memory()
    if rank:
        f_host.mul_(1.0 + 1e-3 * rank)
    f = f_host.cuda()
    vals = torch.zeros((nb, ctx.S, ctx.nnz), dtype=torch.float64, device="cuda")
    Cf = torch.zeros((nb, ctx.S, ctx.n), dtype=torch.float64, device="cuda")
    flush = torch.zeros(256 * 1024 * 1024 // 8, dtype=torch.float64, device="cuda")   # 256 MiB > 126 MB L2
    pairs_per_step = nb * ctx.N * (ctx.N - 1)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        ctx.jacobian_batched(f, vals, Cf)
    barrier()

    # ---- device-resident timing: K steps, CUDA events per step on the launching stream ----------
    sampler = ClockSampler(local_rank)
    sampler.start()
    ctx.profile_enable(True)
    ctx.profile_read()
    l0 = ctx.launch_count()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    barrier()
    t_begin = time.perf_counter()
    t_wall = t_begin
    for k in range(args.steps):
        flush.add_(1.0)                      # L2 flush between timed iterations (outside the events)
        evs[k][0].record()
        ctx.jacobian_batched(f, vals, Cf)
        evs[k][1].record()
    barrier()
    t_wall = time.perf_counter() - t_wall
    launches = ctx.launch_count() - l0
    step_ms = [a.elapsed_time(b) for a, b in evs]
    total_ms = float(sum(step_ms))
    pair_ms, pair_cnt = ctx.profile_read()
    ctx.profile_enable(False)
    clocks = sampler.stop(t_begin, t_begin + t_wall)

    # ---- end to end through the host entry point: pinned host buffers, H2D + D2H inside -----------
    vals_host = torch.zeros((nb, ctx.S, ctx.nnz), dtype=torch.float64).pin_memory()
    Cf_host = torch.zeros((nb, ctx.S, ctx.n), dtype=torch.float64).pin_memory()
    ctx.jacobian_host(f_host, vals_host, Cf_host)        # warm-up (allocates staging)
    barrier()
    e2e_steps = max(1, min(args.steps, 5))
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        ctx.jacobian_host(f_host, vals_host, Cf_host)    # synchronises
    barrier()
    e2e_ms = (time.perf_counter() - t0) * 1e3
    assert torch.equal(vals_host[-1], vals[-1].cpu())

    t = torch.tensor([total_ms, e2e_ms], dtype=torch.float64, device="cuda")
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    total_ms, e2e_ms = float(t[0]), float(t[1])
    ms_per_step = total_ms / args.steps
    value = world * pairs_per_step / (ms_per_step * 1e-3) * 1e-9
    e2e_value = world * pairs_per_step / (e2e_ms / e2e_steps * 1e-3) * 1e-9

    if rank == 0:
        peak_flops, _ = binding.landau_fp64_peak_probe(1 << 16)
        sm_max = clocks["sm_max_mhz"] or 1965.0
        sms = torch.cuda.get_device_properties(local_rank).multi_processor_count
        nominal_peak = sms * FP64_LANES_PER_SM * 2 * sm_max * 1e6 * 1e-12
        pair_launch_ms = pair_ms / max(pair_cnt, 1)
        achieved = FLOP_PER_PAIR * pairs_per_step / (pair_launch_ms * 1e-3) * 1e-12
        roof = {"bound": "alu", "kernel": "k_pair_sym<128,2>", "achieved": achieved, "peak": nominal_peak, "unit": "TFLOP/s",
                "frac": achieved / nominal_peak, "traffic": PAIR_KERNEL_DRAM_BYTES,
                "peak_source": "derived: SMs x 64 DFMA lanes x 2 x clocks.max.sm (DESIGN.md); MEASURED_PEAKS.json has no fp64 entry",
                "peak_probe_measured": peak_flops * 1e-12, "frac_of_probe": achieved / (peak_flops * 1e-12),
                "flop_per_pair": FLOP_PER_PAIR,
                "fp64_pipe_frac": FP64_INST_PER_PAIR * pairs_per_step / (pair_launch_ms * 1e-3) / (nominal_peak * 0.5e12),
                "fp64_issue_bound_frac": (FP64_INST_PER_PAIR + 0.5 * FP64_3OP_INST_PER_PAIR) * pairs_per_step
                / (pair_launch_ms * 1e-3) / (nominal_peak * 0.5e12),
                "kernel_ms_per_launch": pair_launch_ms,
                "kernel_share_of_step": pair_ms / total_ms if world == 1 else None,
                "kernel_gpair_per_s": pairs_per_step / (pair_launch_ms * 1e-3) * 1e-9}
        cpu_val, cpu_dt, cores = cpu_baseline_sample(wl, inputs)
        detail = [time_single_config(binding, inputs, torch, k) for k in (1, 2, 3, 4)]
        detail.append(time_single_config(binding, inputs, torch, 3, variant="A"))
        detail += [time_single_config(binding, inputs, torch, k) for k in (6, 7)]   # paper-shaped S = 10 context runs
        next_rows = time_next_rows(binding, inputs, torch, ctx, f, vals, Cf, nb)
        # everything but the pair kernel (a1, a2, a4-a7): HBM-bound; algorithmic bytes = f in, vals and C(f) out,
        # G_D/G_K (5 doubles per point) between the two halves of the path
        rest_ms = (total_ms - pair_ms) / args.steps if world == 1 else None
        rest_bytes = nb * (ctx.S * 8 * (2 * ctx.n + ctx.nnz) + 40 * ctx.N)
        hbm_peak = None
        try:
            hbm_peak = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]
            hbm_src = "MEASURED_PEAKS.json hbm_gbs"
        except Exception:
            hbm_peak, hbm_src = 6460.0, "fallback (B200_PROFILING.md measured copy bandwidth)"
        roof_rest = None
        if rest_ms:
            ach = rest_bytes / (rest_ms * 1e-3) * 1e-9
            roof_rest = {"bound": "hbm", "kernels": "k_fields_beta + k_sum_partials + k_element_q3 + k_gather x2", "achieved": ach,
                         "peak": hbm_peak, "unit": "GB/s", "frac": ach / hbm_peak, "peak_source": hbm_src,
                         "ms_per_step": rest_ms, "algorithmic_bytes_per_step": rest_bytes, "traffic": REST_DRAM_BYTES}
        h2d = nb * ctx.S * ctx.n * 8
        d2h = nb * ctx.S * (ctx.nnz + ctx.n) * 8
        print(json.dumps({
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": WORKLOAD, "problems_per_gpu": nb, "N": ctx.N, "S": ctx.S, "n": ctx.n, "nnz": ctx.nnz,
                       "pairs_per_step_per_gpu": pairs_per_step, "l2": "256 MiB flush write between timed steps; outputs 0.7 GB > L2"},
            "builds_per_s": world * nb / (ms_per_step * 1e-3),
            "wall_ms_per_step_incl_flush": t_wall * 1e3 / args.steps,
            "clocks": clocks, "gpu_launches": launches,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "ms_per_step": e2e_ms / e2e_steps, "steps": e2e_steps, "api": "landau_jacobian_host (pinned host buffers)"},
            "roofline": roof,
            "cpu_baseline": {"value": cpu_val, "unit": UNIT, "cores": cores, "kind": "oracle",
                             "sample": f"{CPU_SAMPLE_PROBLEMS} of the 512 problems (N=4928, a1-a8), double-precision oracle, OpenMP over i, {cpu_dt:.2f} s wall"},
            "roofline_rest": roof_rest,
            "per_config": detail,
            "next_rows": next_rows,
        }))
    ctx.destroy()
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        args.warmup = max(args.warmup, 3)
        run_ours(args)


if __name__ == "__main__":
    main()

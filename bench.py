#!/usr/bin/env python
"""bench.py -- Landau Jacobian builds/s and GPair-evals/s (fp64) on B200.

One "step" = one pass of the whole hot path (a1-a7: fields, beta sums, all-pairs inner integral,
element matrices, CSR gather, C(f)) over BASELINE.json config 5: 512 independent velocity-space
problems on the refined Q3 mesh "3B" (308 cells, 4,928 points, 2 species), one
landau_jacobian_batched call.  value = ordered point pairs N(N-1) x problems / time, whole job.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
  python bench.py --kernel-run single|batched|main     # launches only (for ncu), prints the launch plan
  python bench.py --summarise-ncu RAW.csv [...]        # ncu --page raw --csv export(s) -> roofline-input CSV on stdout

N > 1: launched by torchrun, one rank per GPU; the problems are independent (weak scaling: every
rank builds its own 512 problems, no data-path collective).
--impl reference: times the CPU oracle (double instantiation) on the host cores on a bounded
sample of the same workload.

The step goes through the library's default path for a batch (LANDAU_PAIR_SHARED, include/landau.h): the tensor
of every ordered point pair is evaluated once per call (k_pair_tensor) and applied to all problems by an fp64
tensor-core contraction (k_apply_dmma); `value` still counts N(N-1) pair interactions per problem, `builds_per_s`
is the unambiguous figure.  The per-problem path (k_pair_sym: every problem evaluates every pair itself) is timed
on the same workload and reported under `per_problem_path`.
"""
from __future__ import annotations

import argparse
import csv
import hashlib
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
FP64_LANES_PER_SM = 64      # DFMA lanes per SM per clock = 4 sub-partitions x one DMMA.8x8x4 (256 FMA) per 16 clocks
APPLY_FLOP_PER_PAIR = 14.0  # k_apply_dmma: seven products per ordered pair and problem (landau_shared.cu)
CSRC = os.path.join(ROOT, "paper_2104_10000_b200", "csrc")
KERNEL_SOURCES = ["landau_kernels.cu", "landau_shared.cu", "landau_pair_math.cuh", "landau_launch.cuh"]
ROOFLINE_INPUTS = os.path.join(ROOT, "profiles", "r02_roofline_inputs.csv")

# (key, inputs.config number, variant, problems of the batched run: >= 10 ms of pair work on the per-problem path)
CONFIGS = [("cfg1", 1, "B", 8192), ("cfg2", 2, "B", 512), ("cfg3A", 3, "A", 1024), ("cfg3B", 3, "B", 256),
           ("cfg4B", 4, "B", 256), ("ctx80", 6, "B", 1024), ("ctx320", 7, "B", 128)]


def kernel_source_sha() -> str:
    h = hashlib.sha256()
    for name in KERNEL_SOURCES:
        h.update(open(os.path.join(CSRC, name), "rb").read())
    return h.hexdigest()[:16]


def load_roofline_inputs():
    """profiles/r02_roofline_inputs.csv (written by `bench.py --summarise-ncu`): ncu-counted FP64 instructions and
    DRAM bytes per launch, keyed by (kernel, workload).  Rows whose source hash differs from the kernel sources in
    the tree are ignored (the numbers then print as null)."""
    out = {}
    try:
        sha = kernel_source_sha()
        with open(ROOFLINE_INPUTS) as fh:
            for row in csv.DictReader(l for l in fh if not l.startswith("#")):
                if row["source_sha"] == sha:      # several captures of one launch (counter pass, full set) are merged
                    d = out.setdefault((row["kernel"], row["workload"]), {})
                    for k, v in row.items():
                        if k not in ("kernel", "workload", "source_sha", "instance") and v not in ("", None):
                            d[k] = float(v)
                        elif k not in ("kernel", "workload", "source_sha", "instance"):
                            d.setdefault(k, None)
    except Exception:
        pass
    return out


class ClockSampler(threading.Thread):
    """One `nvidia-smi -lms 20` process sampling clocks / throttle reasons DURING the timed region
    (B200_PROFILING.md recipe); its lines are read by this thread."""

    QUERY = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.rows, self.proc = [], None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.QUERY}", "--format=csv,noheader,nounits",
                                          "-lms", "20", "-i", str(index)], stdout=subprocess.PIPE, text=True)
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


# ------------------------------------------------------------------------------------------------------------------
# CPU baseline: the oracle as it stands (double instantiation of the pair loop, OpenMP over i; numpy for the rest)
# ------------------------------------------------------------------------------------------------------------------
def oracle_step(oracle, sp, species, f):
    """Steps a1-a7 of one problem on an already built Space (the GPU side's ctx is created outside its timed region
    as well): pair loop + scaling, element matrices, dense assembly -> CSR values, C(f).  Returns
    (seconds of the whole step, seconds of the pair loop alone)."""
    t0 = time.perf_counter()
    fq, dfr, dfz = oracle.fields_at_points(sp, f)
    e2 = np.asarray(species.charge, dtype=np.float64) ** 2
    m0m = species.m0 / np.asarray(species.mass, dtype=np.float64)
    t1 = time.perf_counter()
    oracle.inner_integral(sp.r, sp.z, sp.w_in, fq, dfr, dfz, e2, m0m, None, "d")
    t_pair = time.perf_counter() - t1
    K, D, _ = oracle.coefficients(sp, species, f, None, "d")          # (runs the pair loop again: subtracted below)
    Ce = oracle.element_matrices(sp, K, D)
    for a in range(f.shape[0]):
        oracle.csr_values(sp, oracle.assemble_dense(sp, Ce[a]))
    oracle.collision(sp, species, f, "d", (K, D))
    t_all = time.perf_counter() - t0
    return t_all - t_pair, t_pair      # the pair loop ran twice: count it once


def cpu_baseline(oracle, inputs, wl, problems, reps=1):
    """Median over `reps` of the oracle's time for the listed problems of a workload."""
    sp = oracle.build_space(wl.mesh, wl.order)
    fs = [inputs.nodal_f(wl, sp.dof_r, sp.dof_z, b) for b in problems]
    tot, pair = [], []
    for _ in range(reps):
        ta = tp = 0.0
        for f in fs:
            a, p = oracle_step(oracle, sp, wl.species, f)
            ta += a; tp += p
        tot.append(ta); pair.append(tp)
    pairs = len(problems) * sp.N * (sp.N - 1)
    t, tpair = float(np.median(tot)), float(np.median(pair))
    return {"value": pairs / t * 1e-9, "unit": UNIT, "cores": os.cpu_count(), "kind": "oracle",
            "builds_per_s": len(problems) / t, "seconds": t, "pair_loop_only_gpair_per_s": pairs / tpair * 1e-9,
            "pair_loop_share": tpair / t, "reps": reps}


def run_reference(args):
    """--impl reference: the CPU oracle on the host cores, each step one problem of config 5 (a1-a7 on a Space
    built once, as the GPU arm's ctx is)."""
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
        t, _ = oracle_step(oracle, sp, wl.species, f)
        if k >= args.warmup:
            times.append(t)
    ms = 1e3 * float(np.median(times))
    val = pairs / (ms * 1e-3) * 1e-9
    sample = ("1 of the 512 problems per step (full N=4928 mesh, a1-a7 on a Space built once), double-precision oracle, "
              "OpenMP over i in the pair loop, numpy elsewhere; median step")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic", "config": {"workload": WORKLOAD, "sample": sample},
        "builds_per_s": 1e3 / ms,
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": os.cpu_count(), "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


# ------------------------------------------------------------------------------------------------------------------
# GPU timing helpers
# ------------------------------------------------------------------------------------------------------------------
def make_problem(binding, inputs, torch, wl, nb, path=0):
    ctx = binding.LandauContext(wl.mesh, wl.order, wl.species, nb, pair_path=path)
    r, z = ctx.dof_coords()
    nprob = len(wl.components)
    f1 = [inputs.nodal_f(wl, r, z, b) for b in range(min(nb, nprob))]
    f = np.stack([f1[b % len(f1)] for b in range(nb)])
    fd = torch.from_numpy(f).cuda()
    vals = torch.zeros((nb, ctx.S, ctx.nnz), dtype=torch.float64, device="cuda")
    Cf = torch.zeros((nb, ctx.S, ctx.n), dtype=torch.float64, device="cuda")
    return ctx, fd, vals, Cf


def timed_steps(torch, fn, steps, flush=None, warmup=3):
    for _ in range(warmup):
        fn()
    torch.cuda.synchronize()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for a, b in evs:
        if flush is not None:
            flush.add_(1.0)                  # L2 flush between timed iterations (outside the events)
        a.record(); fn(); b.record()
    torch.cuda.synchronize()
    return [a.elapsed_time(b) for a, b in evs]


def a3_profile(ctx, torch, fn, reps):
    """Device time per CALL of the step-a3 kernels: (tensor evaluation or per-problem pair kernel ms, contraction ms)
    via landau_profile_* (a call of the per-problem path launches its pair kernel once per group of problems: the
    launches of a call are added up)."""
    ctx.profile_enable(True); ctx.profile_read()
    for _ in range(reps):
        fn()
    torch.cuda.synchronize()
    ms, cnt = ctx.profile_read()
    ctx.profile_enable(False)
    return [m / reps if c else None for m, c in zip(ms, cnt)]


def fp64_roof(kind, kernel, flop_per_pair, pairs, ms, peak, probe, extra=None):
    ach = flop_per_pair * pairs / (ms * 1e-3) * 1e-12 if (flop_per_pair and ms) else None
    d = {"bound": kind, "kernel": kernel, "achieved": ach, "peak": peak, "unit": "TFLOP/s", "frac": ach / peak if ach else None,
         "frac_of_probe": ach / probe if (ach and probe) else None, "flop_per_pair": flop_per_pair,
         "kernel_ms_per_launch": ms, "kernel_gpair_per_s": pairs / (ms * 1e-3) * 1e-9 if ms else None}
    if extra:
        d.update(extra)
    return d


def pair_sym_roof(rin, key, kname, pairs, ms, peak, probe, issue, mix_key=None):
    """Roofline entry of the per-problem pair kernel from the ncu-counted instruction mix of workload `key`
    (`mix_key`: the workload whose counters give the mix when `key`'s capture has none -- same kernel, same mesh)."""
    c = rin.get(("k_pair_sym", key))
    if mix_key and rin.get(("k_pair_sym", mix_key)) and (not c or c.get("dfma") is None):
        m = rin[("k_pair_sym", mix_key)]
        c = dict(c or {"dram_read": None, "dram_write": None})
        c.update({k: m[k] for k in ("dfma", "dmul", "dadd", "units_per_launch")})
    if not c or not ms or c.get("dfma") is None:
        return fp64_roof("alu", kname, None, pairs, ms, peak, probe, {"note": "no ncu counters for this source revision"})
    upl = c["units_per_launch"]
    dfma, dmul, dadd = c["dfma"] / upl, c["dmul"] / upl, c["dadd"] / upl     # thread instructions per ordered pair
    flop = 2 * dfma + dmul + dadd
    inst = dfma + dmul + dadd
    extra = {"fp64_inst_per_pair": inst, "dfma_share_of_fp64_inst": dfma / inst,
             "fp64_pipe_frac": inst * pairs / (ms * 1e-3) / (peak * 0.5e12),
             "traffic": (c.get("dram_read") or 0) + (c.get("dram_write") or 0) if c.get("dram_read") is not None else None,
             "ncu_fp64_pipe_pct": c.get("fp64_pipe_pct"), "ncu_issue_active_pct": c.get("issue_active_pct")}
    if c.get("dfma_3reg") is not None and issue:
        # issue cycles per pair on the FP64 port: measured cycles per instruction class (landau_fp64_issue_probe)
        three = c["dfma_3reg"] / upl
        cyc = (inst - three) * issue["two_operand"] + three * issue["three_operand_reuse_mix"]
        extra["fp64_issue_bound_frac"] = cyc * pairs / 32.0 / (ms * 1e-3) / (issue["smsp"] * issue["clock_hz"])
    return fp64_roof("alu", kname, flop, pairs, ms, peak, probe, extra)


def pair_kernel_name(N, latency=False):
    """The per-problem pair kernel a context runs: latency tiling (contexts for fewer than 4 problems) or throughput tiling."""
    if latency:
        return "k_pair_sym<128,2>" if N >= 16384 else ("k_pair_sym<64,2>" if N >= 8192 else ("k_pair_split<2>" if N >= 2048 else "k_pair_split<4>"))
    return "k_pair_sym<128,2>" if N >= 4096 else ("k_pair_sym<64,2>" if N >= 2560 else ("k_pair_split<2>" if N >= 1536 else "k_pair_split<4>"))


def time_config(binding, inputs, torch, oracle, key, k, variant, nb_batched, rin, peaks, flush, with_cpu=True):
    """One BASELINE config (or context run): single build (per-problem path, as landau_create chooses for
    max_batch = 1), a batch through both paths, the CPU oracle."""
    wl = inputs.config(k, variant=variant)
    out = {"config": wl.name}
    # --- single build -------------------------------------------------------------------------------------------
    ctx, fd, vals, Cf = make_problem(binding, inputs, torch, wl, 1)
    N, pairs = ctx.N, ctx.N * (ctx.N - 1)
    out.update({"N": N, "S": ctx.S, "n": ctx.n, "nnz": ctx.nnz})
    ms = float(np.median(timed_steps(torch, lambda: ctx.jacobian(fd[0], vals[0], Cf[0]), 20)))
    pk = a3_profile(ctx, torch, lambda: ctx.jacobian(fd[0], vals[0], Cf[0]), 10)[0]
    graph_ms = None
    try:        # the same build captured once in a CUDA graph and replayed (the library makes no synchronising call)
        side = torch.cuda.Stream()
        with torch.cuda.stream(side):
            ctx.jacobian(fd[0], vals[0], Cf[0])
            torch.cuda.synchronize()
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=side):
                ctx.jacobian(fd[0], vals[0], Cf[0])
            g.replay()
            graph_ms = float(np.median(timed_steps(torch, g.replay, 20)))
    except Exception as exc:   # reported, not fatal
        graph_ms = f"unavailable: {exc}"
    kname = pair_kernel_name(N)
    out["single"] = {"path": "per-problem (latency tiling)", "ms_per_build": ms, "graph_replay_ms_per_build": graph_ms, "builds_per_s": 1e3 / ms,
                     "gpair_per_s": pairs / (ms * 1e-3) * 1e-9,
                     "roofline": pair_sym_roof(rin, key + ":single", pair_kernel_name(N, True), pairs, pk, peaks["fp64"], peaks["probe"], peaks["issue"])}
    ctx.destroy()
    # --- batch, both paths --------------------------------------------------------------------------------------
    nb = nb_batched
    out["batched"] = {"problems": nb}
    for path, pname in ((binding.LANDAU_PAIR_SHARED, "shared"), (binding.LANDAU_PAIR_PER_PROBLEM, "per_problem")):
        ctx, fd, vals, Cf = make_problem(binding, inputs, torch, wl, nb, path)
        fn = lambda: ctx.jacobian_batched(fd, vals, Cf)
        ms = float(np.median(timed_steps(torch, fn, 5, flush)))
        pk = a3_profile(ctx, torch, fn, 3)
        e = {"ms_per_step": ms, "builds_per_s": nb / (ms * 1e-3), "gpair_per_s": nb * pairs / (ms * 1e-3) * 1e-9}
        if path == binding.LANDAU_PAIR_SHARED:
            e["tensor_eval_ms"] = pk[0]
            e["roofline"] = fp64_roof("tensor", "k_apply_dmma", APPLY_FLOP_PER_PAIR, nb * pairs, pk[1], peaks["fp64"], peaks["dmma_probe"])
        else:
            e["roofline"] = pair_sym_roof(rin, key + ":batched", kname, nb * pairs, pk[0], peaks["fp64"], peaks["probe"], peaks["issue"])
        out["batched"][pname] = e
        ctx.destroy()
        del fd, vals, Cf
    # --- CPU oracle ---------------------------------------------------------------------------------------------
    if with_cpu:
        out["cpu_baseline"] = cpu_baseline(oracle, inputs, wl, [0], reps=3)
        out["cpu_baseline"]["sample"] = "one build (a1-a7 on a Space built once), median of 3"
    return out


def time_next_rows(binding, inputs, torch, ctx5, f5, vals5, Cf5, nb):
    """SURVEY 8(f) rows at the same measurement bar: NEXT-3 (implicit-step operator, config 5) and NEXT-2
    (the paper's three 20-cell grids with ten species, Table I, 512 problems batched)."""
    out = {}
    Ez = torch.full((nb,), 0.3, dtype=torch.float64, device="cuda")
    ms = float(np.median(timed_steps(torch, lambda: ctx5.implicit_operator_batched(f5, Ez, 2.0, vals5, Cf5), 3, warmup=1)))
    out["implicit_operator_config5"] = {"ms_per_step": ms, "gpair_per_s": nb * ctx5.N * (ctx5.N - 1) / (ms * 1e-3) * 1e-9,
                                        "what": "shift M + A(E_z) - J and A f - C(f) in one pass (landau_implicit_operator_batched)"}
    # NEXT-4: band LU of the nb * S matrices of the implicit step (vals5 holds them now), then one solve
    bw, md, ws = ctx5.band_sizes()
    band = torch.empty(nb * ws, dtype=torch.float64, device="cuda")
    rhs = torch.ones((nb, ctx5.S, ctx5.n), dtype=torch.float64, device="cuda")
    piv = torch.zeros((nb, ctx5.S, 2), dtype=torch.float64, device="cuda")
    x = torch.empty_like(rhs)
    ctx5.band_factor_batched(vals5, band, piv); ctx5.band_solve_batched(band, rhs, x)
    torch.cuda.synchronize()
    e0, e1, e2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
    e0.record(); ctx5.band_factor_batched(vals5, band, piv); e1.record(); ctx5.band_solve_batched(band, rhs, x); e2.record()
    torch.cuda.synchronize()
    fms, sms_ = e0.elapsed_time(e1), e1.elapsed_time(e2)
    nmat = nb * ctx5.S
    method, front_rows = ctx5.band_method()
    flop = ctx5.band_flop_in_use * nmat                # window updates executed by the kernel in use (front: inside the envelope)
    flop_band = 2.0 * ctx5.n * bw * bw * nmat          # Alg. 4.3.1 on the uniform band: n outer products of bw x bw
    out["band_lu_config5"] = {"matrices": nmat, "n": ctx5.n, "half_bandwidth": bw, "workspace_gb": nb * ws * 8e-9,
                              "kernel": "front (envelope)" if method == binding.LANDAU_BAND_FRONT else "hull", "front_rows_max": front_rows,
                              "hull_flop_per_factorization": ctx5.band_flop_per_factorization,
                              "factor_ms": fms, "solve_ms": sms_, "factor_tflops": flop / (fms * 1e-3) * 1e-12,
                              "factor_tflops_uniform_band_equiv": flop_band / (fms * 1e-3) * 1e-12,
                              "factorizations_per_s": nmat / (fms * 1e-3),
                              "min_pivot_ratio": float((piv[:, :, 0] / piv[:, :, 1]).min()),
                              "what": "fill + blocked outer-product LU without pivoting inside the envelope (pivot report on), then L/U solves (one rhs)"}
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
    ms = float(np.median(timed_steps(torch, lambda: mg.jacobian_batched(f, v, c_), 5, warmup=1)))
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
    ms = float(np.median(timed_steps(torch, newton, 5, warmup=1)))
    out["newton_iteration_ctx80"] = {"workload": f"{nb} problems x (10 species, 80 Q3 cells: N = {c80.N}, n = {c80.n}, half-bandwidth {bw80} after the band order)",
                                     "ms_per_batched_iteration": ms, "newton_iterations_per_s": nb / (ms * 1e-3),
                                     "what": "operator (shift M + A - J, A f - C(f)) + band LU of 10 species blocks + solve, per problem"}
    c80.destroy()
    return out


def measure_peaks(binding, sms, sm_max_mhz):
    """FP64 denominators: derived (SMs x 64 lanes x 2 x max clock; the same for DFMA and DMMA.8x8x4, one per 16 clocks
    and sub-partition) and measured on this GPU by the in-library probes."""
    nominal = sms * FP64_LANES_PER_SM * 2 * sm_max_mhz * 1e6 * 1e-12
    probe, _ = binding.landau_fp64_peak_probe(1 << 16)
    cyc = {m: binding.landau_fp64_issue_probe(m)[0] for m in range(5)}
    dmma_cyc, dmma_flops = binding.landau_fp64_issue_probe(5)
    issue = {"two_operand": cyc[1], "immediate_operand": cyc[0], "three_operand": cyc[2], "three_operand_shared": cyc[3],
             "three_operand_reuse_mix": 0.5 * (cyc[2] + cyc[3]), "dependent_latency": cyc[4], "dmma_8x8x4": dmma_cyc,
             "smsp": sms * 4, "clock_hz": sm_max_mhz * 1e6,
             "what": "SM cycles per FP64 warp instruction and sub-partition, landau_fp64_issue_probe modes 0-5"}
    return {"fp64": nominal, "probe": probe * 1e-12, "dmma_probe": dmma_flops * 1e-12, "issue": issue,
            "source": "derived: SMs x 64 FP64 lanes x 2 x clocks.max.sm (DESIGN.md 8); MEASURED_PEAKS.json has no fp64 entry; "
                      "probe = landau_fp64_peak_probe (DFMA), dmma_probe = landau_fp64_issue_probe(5), both measured in this run"}


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
    path, scratch_bytes = ctx.pair_path()
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
    for k in range(args.steps):
        flush.add_(1.0)                      # L2 flush between timed iterations (outside the events)
        evs[k][0].record()
        ctx.jacobian_batched(f, vals, Cf)
        evs[k][1].record()
    barrier()
    t_wall = time.perf_counter() - t_begin
    launches = ctx.launch_count() - l0
    step_ms = [a.elapsed_time(b) for a, b in evs]
    a3_ms, a3_cnt = ctx.profile_read()
    ctx.profile_enable(False)
    clocks = sampler.stop(t_begin, t_begin + t_wall)

    # ---- end to end through the host entry point: pinned host buffers, H2D + D2H inside -----------
    vals_host = torch.zeros((nb, ctx.S, ctx.nnz), dtype=torch.float64).pin_memory()
    Cf_host = torch.zeros((nb, ctx.S, ctx.n), dtype=torch.float64).pin_memory()
    ctx.jacobian_host(f_host, vals_host, Cf_host)        # warm-up (allocates staging)
    barrier()
    e2e_steps = max(1, min(args.steps, 5))
    e2e_times = []
    for _ in range(e2e_steps):
        t0 = time.perf_counter()
        ctx.jacobian_host(f_host, vals_host, Cf_host)    # synchronises
        e2e_times.append((time.perf_counter() - t0) * 1e3)
    barrier()
    assert torch.equal(vals_host[-1], vals[-1].cpu())

    t = torch.tensor([float(np.median(step_ms)), float(np.mean(step_ms)), float(np.median(e2e_times))], dtype=torch.float64, device="cuda")
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms_per_step, ms_mean, e2e_ms = float(t[0]), float(t[1]), float(t[2])
    value = world * pairs_per_step / (ms_per_step * 1e-3) * 1e-9
    e2e_value = world * pairs_per_step / (e2e_ms * 1e-3) * 1e-9

    if rank == 0:
        from oracle import landau_oracle as oracle
        oracle.build()
        rin = load_roofline_inputs()
        sm_max = clocks["sm_max_mhz"] or 1965.0
        sms = torch.cuda.get_device_properties(local_rank).multi_processor_count
        peaks = measure_peaks(binding, sms, sm_max)
        tensor_ms = a3_ms[0] / len(step_ms) if a3_cnt[0] else None      # per step (the per-problem path launches its
        apply_ms = a3_ms[1] / len(step_ms) if a3_cnt[1] else None       # pair kernel once per group of problems)
        shared = path == binding.LANDAU_PAIR_SHARED
        if shared:
            c = rin.get(("k_apply_dmma", "cfg5:main")) or {}
            roof = fp64_roof("tensor", "k_apply_dmma<4,2>", APPLY_FLOP_PER_PAIR, pairs_per_step, apply_ms, peaks["fp64"], peaks["dmma_probe"], {
                "traffic": (c.get("dram_read", 0) + c.get("dram_write", 0)) if c else None,
                "ncu_dmma_pipe_pct": c.get("dmma_pipe_pct") if c else None,
                "peak_source": peaks["source"], "peak_probe_measured": peaks["dmma_probe"],
                "kernel_share_of_step": apply_ms / ms_per_step if world == 1 else None,
                "what": "fp64 mma.sync.m8n8k4 (DMMA.8x8x4) contraction G = U T: 7 products = 14 flop per ordered pair and problem"})
            c = rin.get(("k_pair_tensor", "cfg5:main"))
            m = rin.get(("k_pair_tensor", "cfg3B:batched:shared"))       # same kernel, same mesh: instruction mix
            if c and m and c.get("dfma") is None:
                c = dict(c); c.update({k: m[k] for k in ("dfma", "dmul", "dadd", "units_per_launch")})
            tens = None
            if c and tensor_ms and c.get("dfma") is not None:
                upl = c["units_per_launch"]
                fl = (2 * c["dfma"] + c["dmul"] + c["dadd"]) / upl
                tens = fp64_roof("alu", "k_pair_tensor", fl, ctx.N * (ctx.N - 1), tensor_ms, peaks["fp64"], peaks["probe"],
                                 {"traffic": c["dram_read"] + c["dram_write"], "what": "one tensor evaluation per ORDERED pair and call (K, E by the scaled AGM), all problems share it"})
        else:
            roof = pair_sym_roof(rin, "cfg5:per_problem", "k_pair_sym<128,2>", pairs_per_step, tensor_ms, peaks["fp64"], peaks["probe"], peaks["issue"], "cfg3B:batched")
            tens = None
        # the per-problem path on the same workload (round 1's headline kernel), and the tensor cache
        ctx.set_pair_path(binding.LANDAU_PAIR_PER_PROBLEM)
        pp_ms = float(np.median(timed_steps(torch, lambda: ctx.jacobian_batched(f, vals, Cf), 5, flush)))
        pp_k = a3_profile(ctx, torch, lambda: ctx.jacobian_batched(f, vals, Cf), 3)[0]
        per_problem = {"ms_per_step": pp_ms, "gpair_per_s": pairs_per_step / (pp_ms * 1e-3) * 1e-9, "builds_per_s": nb / (pp_ms * 1e-3),
                       "roofline": pair_sym_roof(rin, "cfg5:per_problem", "k_pair_sym<128,2>", pairs_per_step, pp_k, peaks["fp64"], peaks["probe"], peaks["issue"], "cfg3B:batched"),
                       "what": "LANDAU_PAIR_PER_PROBLEM: every problem evaluates every pair's tensor itself (symmetric tile pairs)"}
        ctx.set_pair_path(binding.LANDAU_PAIR_AUTO)
        ctx.set_tensor_cache(True)
        tc_ms = float(np.median(timed_steps(torch, lambda: ctx.jacobian_batched(f, vals, Cf), 5, flush)))
        ctx.set_tensor_cache(False)
        cached = {"ms_per_step": tc_ms, "gpair_per_s": pairs_per_step / (tc_ms * 1e-3) * 1e-9, "builds_per_s": nb / (tc_ms * 1e-3),
                  "what": "landau_set_tensor_cache(1): the pair tensor kept between calls (off by default and in `value`)"}
        # CPU baseline on a bounded sample of the headline workload
        cpu = cpu_baseline(oracle, inputs, wl, list(range(CPU_SAMPLE_PROBLEMS)))
        cpu["sample"] = (f"{CPU_SAMPLE_PROBLEMS} of the 512 problems (N=4928, a1-a7 on a Space built once), double-precision oracle, "
                         f"OpenMP over i in the pair loop, {cpu['seconds']:.2f} s wall")
        detail = [time_config(binding, inputs, torch, oracle, key, k, var, nbb, rin, peaks, flush) for key, k, var, nbb in CONFIGS]
        next_rows = time_next_rows(binding, inputs, torch, ctx, f, vals, Cf, nb)
        # everything but step a3's kernels (a1, a2, a4-a7): HBM-bound; algorithmic bytes = f in, vals and C(f) out,
        # G_D/G_K (5 doubles per point) between the two halves of the path
        a3_total = (tensor_ms or 0.0) + (apply_ms or 0.0)
        rest_ms = ms_per_step - a3_total if world == 1 else None
        rest_bytes = nb * (ctx.S * 8 * (2 * ctx.n + ctx.nnz) + 40 * ctx.N)
        try:
            hbm_peak = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]
            hbm_src = "MEASURED_PEAKS.json hbm_gbs"
        except Exception:
            hbm_peak, hbm_src = 6650.0, "fallback (B200_PROFILING.md)"
        roof_rest = None
        if rest_ms:
            ach = rest_bytes / (rest_ms * 1e-3) * 1e-9
            c = rin.get(("rest", "cfg5:main")) or {}
            roof_rest = {"bound": "hbm", "kernels": "k_fields_beta + k_sum_partials + k_element_q3 + k_gather x2", "achieved": ach,
                         "peak": hbm_peak, "unit": "GB/s", "frac": ach / hbm_peak, "peak_source": hbm_src,
                         "ms_per_step": rest_ms, "algorithmic_bytes_per_step": rest_bytes,
                         "traffic": (c.get("dram_read", 0) + c.get("dram_write", 0)) if c else None}
        h2d = nb * ctx.S * ctx.n * 8
        d2h = nb * ctx.S * (ctx.nnz + ctx.n) * 8
        print(json.dumps({
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "ms_per_step_mean": ms_mean, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD, "problems_per_gpu": nb, "N": ctx.N, "S": ctx.S, "n": ctx.n, "nnz": ctx.nnz,
                       "pairs_per_step_per_gpu": pairs_per_step, "l2": "256 MiB flush write between timed steps; outputs 0.7 GB > L2",
                       "pair_path": "LANDAU_PAIR_SHARED" if shared else "LANDAU_PAIR_PER_PROBLEM", "pair_scratch_bytes": scratch_bytes,
                       "value_counts": "N(N-1) ordered pair interactions per problem; on the shared path the tensor of a pair is "
                                       "evaluated once per call (inside the timed step) and applied to all 512 problems"},
            "builds_per_s": world * nb / (ms_per_step * 1e-3),
            "wall_ms_per_step_incl_flush": t_wall * 1e3 / args.steps,
            "clocks": clocks, "gpu_launches": launches,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "ms_per_step": e2e_ms, "steps": e2e_steps, "api": "landau_jacobian_host (pinned host buffers), median"},
            "roofline": roof,
            "roofline_tensor_eval": tens,
            "cpu_baseline": cpu,
            "roofline_rest": roof_rest,
            "fp64_peaks": {k: v for k, v in peaks.items() if k != "source"},
            "per_problem_path": per_problem,
            "tensor_cache_on": cached,
            "roofline_inputs": {"file": os.path.relpath(ROOFLINE_INPUTS, ROOT), "source_sha": kernel_source_sha(), "rows_matching": len(rin)},
            "per_config": detail,
            "next_rows": next_rows,
        }))
    ctx.destroy()
    if dist is not None:
        dist.destroy_process_group()


CPU_SAMPLE_PROBLEMS = 8      # of the 512: ~0.5 s each on 16 cores, i.e. tens of core-seconds in total


# ------------------------------------------------------------------------------------------------------------------
# ncu support: launch plans and the summariser of raw exports
# ------------------------------------------------------------------------------------------------------------------
def kernel_run(which):
    """Launches for an ncu pass, nothing timed.  Prints one line per launch group: workload key, kernel regex,
    units (ordered pairs) per launch -- the summariser needs them to turn counters into per-pair figures.
      single : one single build (per-problem path) of every per_config entry, in CONFIGS order
      batched: the batched run of every per_config entry through the per-problem path, then the shared path
      main   : config 5, shared path (one step), then per-problem path (one step)
      lu     : band LU (fill, factorisation, solve) of config 5's and the ten-species 80-cell problem's matrices"""
    import torch
    from paper_2104_10000_b200 import binding, inputs
    binding.lib()
    plan = []
    if which == "lu":
        # operator -> band fill -> factorisation -> one solve, for the 1,024 matrices of config 5 and the
        # 5,120 of the ten-species 80-cell problem (the two workloads of next_rows.band_lu_config5 / newton_iteration_ctx80)
        for tag, k in (("cfg5:lu", 5), ("ctx80:lu", 6)):
            wl = inputs.config(k)
            nb = 512
            ctx, fd, vals, Cf = make_problem(binding, inputs, torch, wl, nb)
            Ez = torch.full((nb,), 0.3, dtype=torch.float64, device="cuda")
            ctx.implicit_operator_batched(fd, Ez, 2.0, vals, Cf)
            bw, md, ws = ctx.band_sizes()
            band = torch.empty(nb * ws, dtype=torch.float64, device="cuda")
            piv = torch.zeros((nb, ctx.S, 2), dtype=torch.float64, device="cuda")
            for method in (binding.LANDAU_BAND_AUTO, binding.LANDAU_BAND_HULL):       # the kernel in use, then the hull kernel
                ctx.band_set_method(method)
                ctx.band_factor_batched(vals, band, piv)
                m, rows = ctx.band_method()
                plan.append({"workload": tag + (":hull" if m == binding.LANDAU_BAND_HULL else ":front"), "matrices": nb * ctx.S, "n": ctx.n,
                             "half_bandwidth": bw, "front_rows_max": rows, "flop_per_factorization": ctx.band_flop_in_use})
            ctx.band_solve_batched(band, Cf, Cf)
            torch.cuda.synchronize()
            ctx.destroy()
            del fd, vals, Cf, band
    elif which == "main":
        wl = inputs.config(5)
        for path, tag in ((binding.LANDAU_PAIR_SHARED, "cfg5:main"), (binding.LANDAU_PAIR_PER_PROBLEM, "cfg5:per_problem")):
            ctx, fd, vals, Cf = make_problem(binding, inputs, torch, wl, wl.nbatch, path)
            ctx.jacobian_batched(fd, vals, Cf)
            torch.cuda.synchronize()
            plan.append({"workload": tag, "N": ctx.N, "problems": wl.nbatch, "pairs_per_launch": wl.nbatch * ctx.N * (ctx.N - 1),
                         "tensor_pairs_per_launch": ctx.N * (ctx.N - 1)})
            ctx.destroy()
            del fd, vals, Cf
    else:
        for key, k, var, nbb in CONFIGS:
            wl = inputs.config(k, variant=var)
            nb = 1 if which == "single" else nbb
            paths = [binding.LANDAU_PAIR_PER_PROBLEM] + ([binding.LANDAU_PAIR_SHARED] if which == "batched" else [])
            for path in paths:
                ctx, fd, vals, Cf = make_problem(binding, inputs, torch, wl, nb, path)
                ctx.jacobian_batched(fd, vals, Cf)
                torch.cuda.synchronize()
                plan.append({"workload": f"{key}:{which}" + (":shared" if path == binding.LANDAU_PAIR_SHARED else ""), "N": ctx.N,
                             "problems": nb, "pairs_per_launch": nb * ctx.N * (ctx.N - 1), "tensor_pairs_per_launch": ctx.N * (ctx.N - 1)})
                ctx.destroy()
                del fd, vals, Cf
    print(json.dumps({"kernel_run": which, "source_sha": kernel_source_sha(), "plan": plan}))


NCU_COLS = {
    "dfma": "smsp__sass_thread_inst_executed_op_dfma_pred_on.sum", "dmul": "smsp__sass_thread_inst_executed_op_dmul_pred_on.sum",
    "dadd": "smsp__sass_thread_inst_executed_op_dadd_pred_on.sum", "dram_read": "dram__bytes_read.sum", "dram_write": "dram__bytes_write.sum",
    "time_ns": "gpu__time_duration.sum", "fp64_pipe_pct": "sm__inst_executed_pipe_fp64.avg.pct_of_peak_sustained_active",
    "issue_active_pct": "smsp__issue_active.avg.pct_of_peak_sustained_active", "inst_executed": "smsp__inst_executed.sum",
    "dmma_pipe_pct": "sm__inst_executed_pipe_tensor_subpipe_dmma.avg.pct_of_peak_sustained_active",
}


def summarise_ncu(paths, plan_file):
    """ncu `--page raw --csv` exports + the JSON line `--kernel-run` printed for the same command -> CSV rows
    (kernel, workload, source_sha, units_per_launch, counters per launch).  The n-th launch of a pair kernel
    (k_pair_sym / k_pair_tensor / k_apply_dmma) in the export belongs to the n-th entry of the plan that runs it."""
    plan = json.loads(open(plan_file).read().strip().splitlines()[-1])
    sha = plan["source_sha"]
    w = csv.writer(sys.stdout)
    cols = list(NCU_COLS)
    w.writerow(["kernel", "workload", "source_sha", "units_per_launch"] + cols + ["instance"])
    for p in paths:
        rows = list(csv.DictReader(l for l in open(p) if l.startswith('"')))
        units = next((r for r in rows if not r.get("ID", "").strip().isdigit()), {})     # the units row
        rows = [r for r in rows if r.get("ID", "").strip().isdigit()]
        scale = {"Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12, "us": 1e3, "ms": 1e6, "s": 1e9}   # -> byte, ns

        def val(r, col):
            v = r.get(col, "")
            try:
                return float(v.replace(",", "")) * scale.get(units.get(col, ""), 1.0)
            except Exception:
                return None
        seq = {"k_pair_sym": [], "k_pair_tensor": [], "k_apply_dmma": []}      # k_pair_sym: also its small-N form k_pair_split
        rest = {}
        for r in rows:
            name = r["Kernel Name"]
            hit = next((k for k in seq if k in name), "k_pair_sym" if "k_pair_split" in name else None)
            if hit:
                seq[hit].append(r)
            elif "landau::" in name or name.startswith("k_") or " k_" in name:
                rest.setdefault("rest", []).append(r)
        pct_cols = [c for c in cols if c.endswith("_pct")]
        for kern, lst in seq.items():
            entries = [e for e in plan["plan"] if (kern == "k_pair_sym") == (not e["workload"].endswith(":shared") and e["workload"] != "cfg5:main")]
            pos = 0
            for e in entries:
                if pos >= len(lst):
                    break
                # the per-problem path sends a batch through its pair kernel in groups of problems (grid.y = problems of the
                # launch): the launches of one plan entry are added up (counters summed, percentages weighted by time)
                grp, seen = [], 0
                while pos < len(lst) and (not grp or (kern == "k_pair_sym" and seen < e["problems"])):
                    r = lst[pos]; pos += 1
                    grp.append(r)
                    try:
                        seen += int(r["Grid Size"].strip("() ").split(",")[1])
                    except Exception:
                        seen = e["problems"]
                upl = e["tensor_pairs_per_launch"] if kern == "k_pair_tensor" else e["pairs_per_launch"]
                inst = grp[0]["Kernel Name"].split("(")[0].replace("landau::", "").replace("void ", "").replace(" ", "").replace(",", ";")
                tsum = sum((val(r, NCU_COLS["time_ns"]) or 0.0) for r in grp) or 1.0
                out = []
                for c in cols:
                    vs = [(val(r, NCU_COLS[c]), val(r, NCU_COLS["time_ns"]) or 0.0) for r in grp]
                    if any(v is None for v, _ in vs):
                        out.append(None)
                    elif c in pct_cols:
                        out.append(sum(v * t for v, t in vs) / tsum)
                    else:
                        out.append(sum(v for v, _ in vs))
                w.writerow([kern, e["workload"], sha, upl] + out + [inst + (f" x{len(grp)} launches" if len(grp) > 1 else "")])
        if rest.get("rest") and plan["kernel_run"] == "main":
            # the other kernels of the FIRST step (shared path: everything before the per-problem step's k_fields_beta<0>): summed
            n_first = next((i for i, r in enumerate(rest["rest"]) if "k_fields_beta<0>" in r["Kernel Name"].replace("(bool)", "").replace(" ", "")), len(rest["rest"]) // 2)
            tot = {c: sum((val(r, NCU_COLS[c]) or 0.0) for r in rest["rest"][:n_first]) for c in cols}
            w.writerow(["rest", "cfg5:main", sha, plan["plan"][0]["pairs_per_launch"]] + [tot[c] for c in cols] + ["all other kernels of the step"])


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--kernel-run", default=None, choices=["single", "batched", "main", "lu"])
    ap.add_argument("--summarise-ncu", nargs="+", default=None, metavar="RAW.csv")
    ap.add_argument("--plan", default=None, help="file holding the JSON line --kernel-run printed (for --summarise-ncu)")
    args = ap.parse_args()
    if args.summarise_ncu:
        summarise_ncu(args.summarise_ncu, args.plan)
    elif args.kernel_run:
        kernel_run(args.kernel_run)
    elif args.impl == "reference":
        run_reference(args)
    else:
        args.warmup = max(args.warmup, 3)
        run_ours(args)


if __name__ == "__main__":
    main()

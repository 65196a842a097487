#!/usr/bin/env python
"""bench.py -- complete PDAS query time of the B200-native RefDef hot path (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--config 1..5 | --twin NAME] [--method refdef|jacobi|zeroext] [--ref-tol T]

A STEP is one complete optimization query of the config's sequence: S1-S7 of DESIGN.md for every PDAS step
(restriction, coarse setup, Algorithm 1, multiplier / active-set update) plus recovery and KKT.  Queries run in
sequence order under the paper's warm-start policy; when the sequence wraps, the context is reset
and the reference is rebuilt (S0), its time charged to the first query of the new pass.  `value` is
the mean complete time per query in seconds, reference builds inside the timed region included.

The JSON line also carries
  roofline      the persistent Algorithm-1 kernel: algorithmic bytes / CUDA-event time
  cpu_baseline  the CPU oracle as it stands, timed on the host cores on a bounded sample (rank 0, N = 1)
  e2e           the same metric through the C ABI with HOST buffers (H2D of y_d, psi and D2H of y, u, lambda inside)
  clocks        nvidia-smi samples during the timed region

Multi-GPU (torchrun, one rank per GPU): the path is one GPU by definition (BASELINE.json); ranks run independent
replicas of the sequence on different query seeds ("replicas only", weak scaling), no data-path collective.
`--impl reference` runs the oracle (test infrastructure) on the host cores for the same metric, rank 0 only.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METHODS = {"jacobi": 0, "refdef": 1, "zeroext": 2}
FALLBACK_HBM_GBS = 6650.0  # /opt/skills/guides/B200_PROFILING.md fallback


# ----------------------------------------------------------------------------------------------- helpers
def algorithmic_bytes_per_iter(nnz: int, N: int, n: int, r: int, tall_passes: int = 1) -> float:
    """HBM bytes one Algorithm-1 loop iteration must move: the rows of K whose
    columns reach the inactive set and the rows of K^T in it (8 B value + 4 B index per nonzero: 24 nnz n/N on these
    stencil operators), t written and read where it can be nonzero (16 N n/N), the mask (N n/N), 14 passes of 8 B over
    the n inactive rows, and `tall_passes` passes over an n x r tall-skinny block: ONE (H_II Z only) for the default
    kernel, which carries the projection in coefficient form; two (H_II Z and Z) for the literal recurrence
    (alg1_variant = 1), which is what SURVEY.md 8(d) counted.  At n = N: 24 nnz + 17 N + 112 N + 8 N r."""
    return (24.0 * nnz + 17.0 * N) * (n / float(N)) + 112.0 * n + 8.0 * tall_passes * n * r


def shard_queries(rank: int, world: int, n_queries: int):
    """Replica r of `world` runs the config's sequence on its own seeds: query ids r*n .. r*n + n - 1."""
    return [rank * n_queries + q for q in range(n_queries)]


def dist_env():
    return int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))


def reduce_max(values, backend_device=None):
    """Max over ranks of a list of floats (torch.distributed all_reduce MAX); identity without a process group."""
    import torch
    import torch.distributed as dist

    if not (dist.is_available() and dist.is_initialized()):
        return list(values)
    t = torch.tensor(list(values), dtype=torch.float64, device=backend_device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t.cpu()]


def reduce_sum(values, backend_device=None):
    import torch
    import torch.distributed as dist

    if not (dist.is_available() and dist.is_initialized()):
        return list(values)
    t = torch.tensor(list(values), dtype=torch.float64, device=backend_device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return [float(x) for x in t.cpu()]


class ClockSampler:
    """nvidia-smi samples of one GPU while the timed region runs (the recipe's clocks line)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
            out, _ = self.proc.communicate()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.strip().splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def make_workload(args):
    from workloads import make_config

    if args.twin:
        return make_config(twin=args.twin)
    return make_config(args.config)


def workload_name(args, w, cap=None):
    return f"{w.name}: {w.kind} CHT {'x'.join(map(str, w.dims))}" + (f" x{w.nt} slabs" if w.nt > 1 else "") + \
           f", N={w.N}, k={w.k}, {w.n_queries} queries/sequence, PDAS cap {cap or w.pdas_cap}"


def build_analytical_reference(g, w):
    """The paper's closed-form references: sine products on steady Cartesian grids (section 2.2.3), sine products
    paired with per-mode temporal eigenvectors on the all-at-once transient grid (section 2.2.4; horizon T = 1)."""
    if w.nt > 1:
        g.build_reference_spacetime(w.k, w.dims, w.nt, 1.0 / w.nt)
    else:
        g.build_reference_sine(w.k, w.dims)


_COARSE = {}


KAPPA_REF = 1.0  # conductivity of the homogeneous comparison medium of the LOBPCG preconditioner: the generator's solid
DEFAULT_EIG_SOLVER = "lobpcg"  # steady Cartesian grids; everything else takes the filter (eig_solver_for)


def eig_solver_for(w, reference):
    """Which of the two eigensolvers of S0 builds the 'eig' reference: the sine-preconditioned LOBPCG needs a steady
    Cartesian grid (csrc/lobpcg.cuh); everything else, and 'eig-filter', takes the Chebyshev-filtered subspace iteration."""
    if reference == "eig-filter" or w.nt != 1:
        return "filter"
    if reference == "eig-lobpcg":
        return "lobpcg"
    return DEFAULT_EIG_SOLVER


def build_eig_reference(g, w, reference, ref_tol, sweeps=60):
    """The k lowest eigenvectors of H (BASELINE.json's reference) to ||H w - theta w|| <= ref_tol theta.
    Returns (theta, residuals, iterations or sweeps, status)."""
    if eig_solver_for(w, reference) == "lobpcg":
        return g.build_reference_lobpcg(w.k, w.dims, kappa_ref=KAPPA_REF, tol=ref_tol, max_iters=800)
    return g.build_reference(w.k, tol=ref_tol, max_block_iters=sweeps)


def build_coarse_reference(g, w, ref_tol, coarsen=2):
    """The paper's coarse-mesh reference (section 2.2.2): Jacobi-scaled low modes of the operator on a grid
    with 1/coarsen of the cells per axis (a second context, rd_build_reference_scaled), P1 prolongation and column
    normalisation on the fine grid (rd_build_reference_prolonged).  The coarse operator is an input like the fine one
    (assembled once on the host, cached); the coarse eigensolve and the prolongation are timed.  Returns (status of
    the coarse eigensolve, its milliseconds)."""
    import paper_2606_17971_b200 as pkg
    from workloads import make_config

    if w.nt > 1:
        return build_transient_coarse_reference(g, w, ref_tol, coarsen)
    key = (w.config, tuple(w.dims), w.k, coarsen)
    if key not in _COARSE:
        _COARSE[key] = make_config(w.config, n=max(2, w.dims[0] // coarsen), k=w.k)
    wc = _COARSE[key]
    gc = pkg.RefDef.from_workload(wc)
    try:
        _, _, _, st = gc.build_reference_scaled(w.k, tol=ref_tol, max_block_iters=60)
        ms_c = gc.reference_info()["build_ms"]
        Wc = gc.get_reference()
    finally:
        gc.close()
    g.build_reference_prolonged(Wc, wc.dims, w.dims)
    return st, ms_c


def build_transient_coarse_reference(g, w, ref_tol, coarsen=2):
    """Transient variant (eq. (14)): spatial low modes of the steady operator of the same geometry
    ("as in config 2") on the coarse grid, P1-prolonged to the fine spatial grid (a steady context of the fine grid
    hosts rd_build_reference_prolonged), then rd_build_reference_transient on the all-at-once context."""
    import paper_2606_17971_b200 as pkg
    from workloads import make_config

    key = ("st", tuple(w.dims), w.k, coarsen)
    if key not in _COARSE:
        _COARSE[key] = (make_config(2, n=max(2, w.dims[0] // coarsen), k=w.k), make_config(2, n=w.dims[0], k=w.k))
    wc, wf = _COARSE[key]
    gc = pkg.RefDef.from_workload(wc)
    gf = pkg.RefDef.from_workload(wf)
    try:
        _, _, _, st = gc.build_reference_scaled(w.k, tol=ref_tol, max_block_iters=60)
        ms = gc.reference_info()["build_ms"]
        gf.build_reference_prolonged(gc.get_reference(), wc.dims, wf.dims)
        ms += gf.reference_info()["build_ms"]
        Phi = gf.get_reference()
    finally:
        gc.close()
        gf.close()
    g.build_reference_transient(w.k, Phi, w.nt)
    return st, ms


def load_profile():
    p = os.path.join(ROOT, "profiles", "bench_workload_profile.json")
    if os.path.exists(p):
        return json.load(open(p))
    return {}


# ----------------------------------------------------------------------------------------------- our arm
class Sequence:
    """The config's query sequence on one context: warm starts inside a pass, reset + reference rebuild on wrap."""

    def __init__(self, g, w, method, ref_tol, qids, reference="eig"):
        self.g, self.w, self.method, self.ref_tol, self.qids, self.reference = g, w, method, ref_tol, qids, reference
        self.pos = 0
        self.ref_builds = 0
        self.ref_ms = 0.0

    def _target(self, q):
        qid = self.qids[q]
        yd = self.w._target(1000 * self.w.config + qid)
        psi = np.full(self.w.N, self.w.psi_factor * float(yd.max()))
        return yd, psi

    def begin_pass(self):
        self.g.reset_sequence()
        if self.method != 0:
            extra_ms = 0.0
            if self.reference == "sine":  # analytical references of the paper: PAPER.md:186-192 (steady), :194-208 (transient)
                build_analytical_reference(self.g, self.w)
                st = 0
            elif self.reference == "coarse":  # coarse generalized eigenproblem + P1 prolongation
                st, extra_ms = build_coarse_reference(self.g, self.w, self.ref_tol)
            elif self.reference == "eig-scaled":  # Jacobi-scaled generalized problem
                _, _, _, st = self.g.build_reference_scaled(self.w.k, tol=self.ref_tol, max_block_iters=60)
            else:
                _, _, _, st = build_eig_reference(self.g, self.w, self.reference, self.ref_tol)
            info = self.g.reference_info()
            self.ref_builds += 1
            self.ref_ms += info["build_ms"] + extra_ms
            self.ref_status = st

    def next_inputs(self):
        q = self.pos % len(self.qids)
        return q, self._target(q)

    def run(self, yd, psi, **kw):
        if self.pos % len(self.qids) == 0:
            self.begin_pass()
        self.pos += 1
        return self.g.solve_query(self.method, yd, psi, want_sets=False, **kw)


def pdas_cap_for(args, w):
    """PDAS step cap: --pdas-cap, else the paper's raised cap of 400 ("raised to 400 for Bore 4") on the
    two full-size 2-D-in-space configs whose sequences need more than 100 steps (configs 2 and 4), else the workload's."""
    if args.pdas_cap > 0:
        return args.pdas_cap
    if not args.twin and w.config in (2, 4):
        return 400
    return w.pdas_cap


def query_ok(res):
    """A query is a time-to-solution only if PDAS converged, every inner solve returned RD_OK and every KKT measure of
    eq. (25) is <= 1e-8 ("The reported times contain only sequences that satisfy these criteria")."""
    return res["status"] == 0 and res["worst_inner_status"] == 0 and max(res["kkt"]) <= 1e-8


def inactive_histogram(results, N):
    """Share of the Algorithm-1 time spent at each |I|/N decile (S6: what compaction can save)."""
    edges = [0.0, 0.1, 0.25, 0.5, 0.75, 0.9, 1.0000001]
    t = [0.0] * (len(edges) - 1)
    for res in results:
        for s_ in res["steps"]:
            if s_["n_inactive"] > 0:
                f = s_["n_inactive"] / N
                for b in range(len(t)):
                    if edges[b] <= f < edges[b + 1]:
                        t[b] += s_["t_iter"]
    tot = sum(t) or 1.0
    return {f"[{edges[b]:.2f},{min(edges[b + 1], 1.0):.2f})": round(t[b] / tot, 4) for b in range(len(t))}


def latency_block(args, dev):
    """Secondary block: config 2 (N = 262,144, k = 32), whose working set sits in the L2: the latency-bound case, judged
    on microseconds per deflated iteration, not on GB/s.  One capped Algorithm-1 solve of H y = l from zero with the
    analytical reference (milliseconds to build)."""
    import torch

    import paper_2606_17971_b200 as pkg
    from workloads import make_config

    w2 = make_config(2)
    g2 = pkg.RefDef.from_workload(w2, pkg.Options(cg_cap=4000), stream=torch.cuda.current_stream().cuda_stream)
    try:
        g2.build_reference_sine(w2.k, w2.dims)
        b = torch.from_numpy(w2.m * w2._target(2000)).to(dev)
        act = torch.zeros(w2.N, dtype=torch.uint8, device=dev)
        x0 = torch.zeros(w2.N, dtype=torch.float64, device=dev)
        reps = [g2.solve_inactive(1, act, b, x0)[1] for _ in range(3)]
        r = reps[-1]
        return {"workload": "config2: 2d CHT 512x512, N=262144, k=32 (L2-resident: latency-bound)", "cg_iters": r["iters"],
                "us_per_iter": round(1e3 * r["t_iter_ms"] / max(r["iters"], 1), 3),
                "t_stage_us_per_iter": [round(x / max(r["iters"], 1), 3) for x in r["t_stage_us"]],
                "stages": "A (K product), barrier, B (K^T product), barrier+reduce, k x k, C (updates + HW pass), barrier+reduce, outside loop"}
    finally:
        g2.close()


def run_ours(args):
    import torch

    rank, local_rank, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        import torch.distributed as dist

        dist.init_process_group("nccl", device_id=dev)
    import paper_2606_17971_b200 as pkg

    pkg.load_library()
    w = make_workload(args)
    method = METHODS[args.method]
    stream = torch.cuda.current_stream()
    cap = pdas_cap_for(args, w)
    g = pkg.RefDef.from_workload(w, pkg.Options(pdas_cap=cap, alg1_variant=args.alg1_variant), stream=stream.cuda_stream)
    tall = 2 if args.alg1_variant == 1 else 1
    seq = Sequence(g, w, method, args.ref_tol, shard_queries(rank, world, w.n_queries), args.reference)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)  # > 126 MB L2

    def barrier():
        if world > 1:
            import torch.distributed as dist

            dist.barrier()
        torch.cuda.synchronize()

    def one_step(host: bool):
        """One query.  Device mode: inputs already resident in HBM, outputs stay there.  Host mode (e2e): numpy in/out."""
        q, (yd, psi) = seq.next_inputs()
        if not host:
            yd_in, psi_in = torch.from_numpy(yd).to(dev), torch.from_numpy(psi).to(dev)
        else:
            yd_in, psi_in = yd, psi
        flush.fill_(q & 0xFF)  # L2 flush between steps
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        res = seq.run(yd_in, psi_in)
        e1.record(stream)
        e1.synchronize()
        return e0.elapsed_time(e1), res, q

    warm = [one_step(False) for _ in range(args.warmup)]
    warm_ms = [x[0] for x in warm]
    sampler = ClockSampler(local_rank)
    barrier()
    sampler.start()
    torch.cuda.profiler.start()  # ncu --profile-from-start off: only the timed region is listed
    launches0 = g.kernel_launches()
    builds0, refms0 = seq.ref_builds, seq.ref_ms
    step_ms, results, qpos = [], [], []
    t_wall0 = time.perf_counter()
    for _ in range(args.steps):
        ms, res, q = one_step(False)
        step_ms.append(ms)
        results.append(res)
        qpos.append(q)
    barrier()
    torch.cuda.profiler.stop()
    wall_ms = (time.perf_counter() - t_wall0) * 1e3
    clocks = sampler.stop()
    launches = g.kernel_launches() - launches0
    ref_builds, ref_ms = seq.ref_builds - builds0, seq.ref_ms - refms0
    total_ms = sum(step_ms)

    # ---- roofline of the dominant kernel (persistent Algorithm-1 kernel, one launch per PDAS step with I != {})
    alg_bytes = alg_bytes_N = alg_ms = 0.0
    alg_launches = iters = 0
    coarse_ms = upd_ms = 0.0
    n_steps = 0
    statuses, inner = {}, {}
    for res in results:
        statuses[res["status"]] = statuses.get(res["status"], 0) + 1
        inner[res["worst_inner_status"]] = inner.get(res["worst_inner_status"], 0) + 1
        n_steps += res["n_steps"]
        for s in res["steps"]:
            coarse_ms += s["t_coarse"] + s["t_restrict"]
            upd_ms += s["t_update"]
            if s["n_inactive"] > 0:
                alg_launches += 1
                iters += s["cg_iters"]
                alg_ms += s["t_iter"]
                # the model charges the loop iterations only; the 3-5 operator applies and n x r passes outside the loop
                # body (lines 3, 12, 16, Verify) are inside alg_ms but not in the bytes: the fraction errs low
                alg_bytes += algorithmic_bytes_per_iter(w.nnz, w.N, s["n_inactive"], s["rank_used"], tall) * s["cg_iters"]
                alg_bytes_N += algorithmic_bytes_per_iter(w.nnz, w.N, w.N, s["rank_used"], tall) * s["cg_iters"]
    peak, peak_src = load_peaks()
    achieved = alg_bytes / (alg_ms * 1e-3) / 1e9 if alg_ms > 0 else 0.0
    prof = load_profile().get(w.name, {})
    roofline = {"kernel": "k_alg1_v3 (persistent Algorithm-1 kernel: S3+S4+S5)", "bound": "hbm", "achieved": round(achieved, 1),
                "peak": peak, "peak_source": peak_src, "unit": "GB/s", "frac": round(achieved / peak, 4),
                # ncu dram__bytes_read + dram__bytes_write of one captured launch, per iteration, scaled to this run's
                # mean iterations per launch (profiles/bench_workload_profile.json names the capture)
                "traffic": (prof["dram_bytes_per_iter"] * iters / max(alg_launches, 1)) if "dram_bytes_per_iter" in prof else None,
                "bytes_per_launch": alg_bytes / max(alg_launches, 1), "ms_per_launch": alg_ms / max(alg_launches, 1),
                "launches": alg_launches, "cg_iters": iters, "us_per_iter": 1e3 * alg_ms / max(iters, 1),
                "share_of_step": round(alg_ms / total_ms, 4) if total_ms else None,
                "bytes_model": "24 nnz + 17 N + 112 n + 8 n r per iteration with n = |I|, r = retained rank of each launch (DESIGN.md 5)",
                "achieved_if_every_launch_streamed_all_N_rows": round(alg_bytes_N / (alg_ms * 1e-3) / 1e9, 1) if alg_ms > 0 else 0.0,
                "alg1_time_share_by_inactive_fraction": inactive_histogram(results, w.N)}

    # ---- e2e: the same metric with HOST buffers through the C ABI, continuing the same sequence for one full pass
    # (every query id once, one reference build, one all-active start: the same mix as the timed region when K is a
    # multiple of the pass length)
    e2e_steps = args.e2e_steps if args.e2e_steps > 0 else w.n_queries
    e2e = [one_step(True) for _ in range(e2e_steps)]
    e2e_ms = [x[0] for x in e2e]
    h2d = 2 * 8 * w.N
    d2h = 3 * 8 * w.N
    mx_total, mx_e2e = reduce_max([total_ms, sum(e2e_ms)], dev if world > 1 else None)
    tot_steps = reduce_sum([float(args.steps)], dev if world > 1 else None)[0]
    value = mx_total * 1e-3 / tot_steps  # whole job: max-over-ranks time / queries all ranks processed
    e2e_value = mx_e2e * 1e-3 / (e2e_steps * world)
    ok = [query_ok(r) for r in results]
    conv_ms = [ms for ms, o in zip(step_ms, ok) if o]

    out = None
    if rank == 0:
        out = {
            "metric": "complete PDAS query time (incl. reference build)", "value": round(value, 4), "unit": "s/query",
            "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": round(mx_total / args.steps, 3),
            "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(args, w, cap), "method": args.method, "parallelism": f"replicas x{world}",
                       "alg1_variant": args.alg1_variant, "reference": args.reference, "reference_tol": args.ref_tol,
                       "eig_solver": (eig_solver_for(w, args.reference) if args.reference in ("eig", "eig-filter", "eig-lobpcg") else None),
                       "sigma": "alpha (DESIGN.md reading A1)", "eps": 1e-8,
                       "l2": "flushed between steps (256 MiB write)" + ("; the loop's working set is far larger than the 126 MB L2" if w.N > 1000000 else
                                                                          "; the loop's working set (HW, K, K^T, vectors: about 120 MB) is the size of the L2")},
            # time-to-solution bookkeeping: a query counts as converged only if PDAS stopped on a repeated
            # active set, every inner solve verified, and all five KKT measures of eq. (25) are <= 1e-8
            "converged_queries": int(sum(ok)), "non_converged_queries": int(len(ok) - sum(ok)),
            "value_converged_only": round(sum(conv_ms) * 1e-3 / len(conv_ms), 4) if conv_ms else None,
            "valid_time_to_solution": bool(all(ok)),
            "e2e": {"value": round(e2e_value, 4), "unit": "s/query", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "steps": e2e_steps, "query_positions": [x[2] for x in e2e], "converged_queries": int(sum(query_ok(x[1]) for x in e2e)),
                    "query_s": [round(x * 1e-3, 3) for x in e2e_ms]},
            "gpu_launches": int(launches),
            "clocks": clocks,
            "roofline": roofline,
            "breakdown": {"pdas_steps": n_steps, "query_status_counts": {str(k): v for k, v in statuses.items()},
                          "worst_inner_status_counts": {str(k): v for k, v in inner.items()},
                          "max_kkt": max(max(r["kkt"]) for r in results),
                          "pdas_steps_per_query": [r["n_steps"] for r in results],
                          "cg_iters_per_query": [int(r["total_cg_iters"]) for r in results],
                          "query_positions": qpos,
                          "reference_builds_in_timed_region": ref_builds, "reference_ms": round(ref_ms, 1),
                          "alg1_ms": round(alg_ms, 1), "coarse_setup_ms": round(coarse_ms, 1), "update_ms": round(upd_ms, 1),
                          "wall_ms_incl_host": round(wall_ms, 1),
                          # the sequence so far, for the reader: the first query of a pass carries the reference build
                          # (PAPER.md:352); warm-up queries are untimed for `value` but listed here
                          "warmup_query_s": [round(x * 1e-3, 3) for x in warm_ms], "timed_query_s": [round(x * 1e-3, 3) for x in step_ms],
                          "reference_build_s_before_timed_region": round(refms0 * 1e-3, 3)},
        }
        if method != 0:
            out["reference_build"] = g.reference_info()
        if world == 1 and not args.no_latency_block and not args.twin and w.config != 2:
            out["latency_case"] = latency_block(args, dev)
        if world == 1 and not args.no_cpu_baseline:
            out["cpu_baseline"] = cpu_baseline(args, w, g, method, iters / max(args.steps, 1), n_steps / max(args.steps, 1))
    g.close()
    if world > 1:
        import torch.distributed as dist

        dist.destroy_process_group()
    return out


def run_loop(args):
    """--mode loop: the deflated-CG iteration loop alone (second half of BASELINE.json's metric: HBM GB/s of the loop
    against peak).  One step = one Algorithm-1 solve (S1-S5) of the full-domain system H y = l of query 0 from a zero
    start, at most --cg-cap iterations; the reference is built once, outside the timed region."""
    import torch

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    import paper_2606_17971_b200 as pkg

    pkg.load_library()
    w = make_workload(args)
    method = METHODS[args.method]
    stream = torch.cuda.current_stream()
    g = pkg.RefDef.from_workload(w, pkg.Options(pdas_cap=w.pdas_cap, cg_cap=args.cg_cap, alg1_variant=args.alg1_variant),
                                 stream=stream.cuda_stream)
    tall = 2 if args.alg1_variant == 1 else 1
    ref = None
    if method != 0:
        if args.reference == "sine":
            build_analytical_reference(g, w)
            ref = dict(g.reference_info(), kind="analytical (PAPER.md:186-208)")
        elif args.reference == "coarse":
            st, ms_c = build_coarse_reference(g, w, args.ref_tol)
            ref = dict(g.reference_info(), kind="coarse eigenproblem + P1 prolongation (PAPER.md:176)", status=st, coarse_eig_ms=ms_c)
        else:
            if args.reference == "eig-scaled":
                _, resid, sweeps, st = g.build_reference_scaled(w.k, tol=args.ref_tol, max_block_iters=args.ref_sweeps)
            else:
                _, resid, sweeps, st = build_eig_reference(g, w, args.reference, args.ref_tol, args.ref_sweeps)
            ref = dict(g.reference_info(), sweeps=sweeps, status=st, worst_rel_residual=float(resid.max()),
                       solver=eig_solver_for(w, args.reference))
    yd = w._target(1000 * w.config)
    b = torch.from_numpy(w.m * yd).to(dev)
    act = torch.zeros(w.N, dtype=torch.uint8, device=dev)
    x0 = torch.zeros(w.N, dtype=torch.float64, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    reps = []
    sampler = ClockSampler(0)
    for i in range(args.warmup + args.steps):
        if i == args.warmup:
            torch.cuda.synchronize()
            sampler.start()
            launches0 = g.kernel_launches()
        flush.fill_(i & 0xFF)
        torch.cuda.synchronize()
        _, rep = g.solve_inactive(method, act, b, x0)
        if i >= args.warmup:
            reps.append(rep)
    torch.cuda.synchronize()
    clocks = sampler.stop()
    launches = g.kernel_launches() - launches0
    ms = sum(r["t_iter_ms"] for r in reps)
    iters = sum(r["iters"] for r in reps)
    nbytes = sum(algorithmic_bytes_per_iter(w.nnz, w.N, w.N, r["rank_used"], tall) * r["iters"] for r in reps)
    peak, peak_src = load_peaks()
    achieved = nbytes / (ms * 1e-3) / 1e9
    prof = load_profile().get(w.name, {})
    out = {"metric": "deflated-CG loop HBM throughput", "value": round(achieved, 1), "unit": "GB/s", "n_gpus": 1,
           "steps": args.steps, "warmup": args.warmup, "ms_per_step": round(ms / args.steps, 3), "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": workload_name(args, w), "method": args.method, "mode": "loop", "cg_cap": args.cg_cap, "alg1_variant": args.alg1_variant,
                      "reference_tol": args.ref_tol, "l2": "flushed between steps (256 MiB write)"},
           "gpu_launches": int(launches), "clocks": clocks,
           "roofline": {"kernel": "k_alg1", "bound": "hbm", "achieved": round(achieved, 1), "peak": peak, "peak_source": peak_src,
                        "unit": "GB/s", "frac": round(achieved / peak, 4), "frac_of_nominal_8TBs": round(achieved / 8000.0, 4),
                        "traffic": prof.get("dram_bytes_per_iter"), "bytes_per_iter": nbytes / max(iters, 1),
                        "us_per_iter": 1e3 * ms / max(iters, 1), "cg_iters": iters, "rank": reps[-1]["rank_used"],
                        "status": reps[-1]["status"],
                        "t_stage_us_per_iter": [round(x / max(reps[-1]["iters"], 1), 3) for x in reps[-1]["t_stage_us"]],
                        "stages": "A (K product), barrier, B (K^T product), barrier+reduce, k x k, C (updates + HW pass), barrier+reduce, outside loop",
                        "live_slices": [reps[-1]["live_slices_A"], reps[-1]["live_slices_B"]]},
           "reference": ref}
    g.close()
    return out


def run_setup(args):
    """--mode setup: the once-per-PDAS-step and once-per-sequence parts next to the loop: S1 + S2 (restriction, Gram on the
    FP64 tensor cores, basis transform, blocked SpMM, k x k factorisation) timed as a whole over --steps repetitions, the
    FP64 tensor-core peak of the device (probe), and -- with --reference eig -- S0's Chebyshev filter in GB/s
    (algorithmic bytes 3 nnz + 48 N per column and degree).  Per-kernel times come from an ncu launch list
    of this command (profiles/)."""
    import torch

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    import paper_2606_17971_b200 as pkg

    pkg.load_library()
    w = make_workload(args)
    stream = torch.cuda.current_stream()
    g = pkg.RefDef.from_workload(w, pkg.Options(pdas_cap=w.pdas_cap), stream=stream.cuda_stream)
    peak_tf = g.probe_fp64_tensor_peak()
    ref = None
    if args.reference in ("eig", "eig-filter", "eig-lobpcg"):
        _, resid, sweeps, st = build_eig_reference(g, w, args.reference, args.ref_tol, args.ref_sweeps)
        ref = dict(g.reference_info(), sweeps=sweeps, status=st, worst_rel_residual=float(resid.max()),
                   solver=eig_solver_for(w, args.reference), kappa_ref=KAPPA_REF)
    else:
        build_analytical_reference(g, w)
        ref = dict(g.reference_info(), kind="analytical (PAPER.md:186-208)")
    if "lobpcg_TFLOPs" in ref:
        # S0 by LOBPCG is bound by the FP64 tensor pipe: its roofline entry is flop over the iteration loop's time against the
        # probe's peak (the same probe the Gram kernels of S2 are quoted against)
        ref["roofline"] = {"bound": "tensor", "achieved": round(ref["lobpcg_TFLOPs"], 2), "peak": round(peak_tf, 2), "unit": "TFLOP/s",
                           "frac": round(ref["lobpcg_TFLOPs"] / peak_tf, 3), "peak_source": "rd_probe_fp64_tensor_peak (m8n8k4 on registers)",
                           "note": "whole iteration loop, incl. the block applies of H (HBM-bound) and the ns x ns Rayleigh-Ritz (latency-bound)"}
    act = torch.zeros(w.N, dtype=torch.uint8, device=dev)
    ms = []
    info = None
    for i in range(args.warmup + args.steps):
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        info = g.coarse_setup(1, act)
        e1.record(stream)
        e1.synchronize()
        if i >= args.warmup:
            ms.append(e0.elapsed_time(e1))
    kp = (w.k + 7) & ~7
    peak, peak_src = load_peaks()
    # algorithmic work of S1 + S2 per PDAS step at n = N: restriction 16 N k; two Gram products 2 * 2 N k^2 flop reading
    # 8 N k (G) and 16 N k (E); transform 2 N k^2 flop, 8 N k read, 16 N k written (column- and tile-major); SpMM
    # 24 nnz k / 8 + 40 N k
    flop = 6.0 * w.N * kp * kp
    nbytes = (16 + 8 + 16 + 24 + 40) * w.N * kp + 3.0 * w.nnz * kp
    out = {"metric": "coarse setup (S1 + S2) per PDAS step", "value": round(statistics.median(ms), 3), "unit": "ms", "n_gpus": 1,
           "steps": args.steps, "warmup": args.warmup, "higher_is_better": False, "dtype": "f64", "data": "synthetic",
           "config": {"workload": workload_name(args, w), "mode": "setup", "reference": args.reference},
           "rank": info["rank"], "cond_E": info["cond_E"],
           "setup_model": {"flop": flop, "bytes": nbytes, "GBs": round(nbytes / (statistics.median(ms) * 1e-3) / 1e9, 1),
                           "note": "includes the host round trips of rd_coarse_setup (k x k copies out)"},
           "fp64_tensor_peak_tflops_probe": round(peak_tf, 2), "hbm_peak": peak, "hbm_peak_source": peak_src,
           "reference": ref}
    g.close()
    return out


def run_replay(args):
    """--mode replay: the matched-replay protocol of the paper (Table 3 :438-451; NEXT-4 of SURVEY.md 8(f)).
    A query sequence is run once with RefDef under the warm-start policy and every inactive system it meets is
    recorded (active set and right-hand side b = l_I - H_IJ psi_J).  The SAME systems are then solved again from zero
    initial guesses with direct restriction (eq. (12)), with zero-extension (eq. (13), history accumulating in replay
    order) and with Jacobi-CG, all from the same reference: iterations, retained rank and seconds per transfer, and the
    energy fraction chi of eq. (24) (rd_energy_fraction, x_* = the verified solution of the replayed
    solve) that the coarse correction removes from a zero initial guess, and the effective condition number of the
    Jacobi-scaled deflated operator of eq. (23) (extreme Ritz values of each replayed solve)."""
    import torch

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(0)
    import paper_2606_17971_b200 as pkg

    pkg.load_library()
    w = make_workload(args)
    g = pkg.RefDef.from_workload(w, pkg.Options(pdas_cap=w.pdas_cap, alg1_variant=args.alg1_variant))
    if args.reference == "sine":
        build_analytical_reference(g, w)
    elif args.reference == "coarse":
        build_coarse_reference(g, w, args.ref_tol)
    elif args.reference == "eig-scaled":
        g.build_reference_scaled(w.k, tol=args.ref_tol, max_block_iters=60)
    else:
        build_eig_reference(g, w, args.reference, args.ref_tol)
    ref = g.reference_info()
    systems = []
    nq = min(w.n_queries, args.steps)
    for q in range(nq):
        yd, psi = w.target(q)
        res = g.solve_query(1, yd, psi, want_sets=True)
        ell = w.m * yd
        for st in range(res["n_steps"]):
            act = np.unpackbits(res["J_bits"][st], bitorder="little")[:w.N].astype(np.uint8)  # packed LSB first
            if act.all():
                continue  # empty inactive set: nothing to solve
            b = np.where(act == 0, ell - g.apply_H(np.where(act == 1, psi, 0.0)), 0.0)
            systems.append((act, b))
    out_methods = {}
    x0 = np.zeros(w.N)
    for name in ("refdef", "zeroext", "jacobi"):
        g.reset_sequence()
        iters = ranks = 0
        ms = 0.0
        worst = 0.0
        chis, kappas = [], []
        for act, b in systems:
            xs, r = g.solve_inactive(METHODS[name], act, b, x0)
            if r["ritz_min"] > 0.0:
                kappas.append(r["ritz_max"] / r["ritz_min"])
            iters += r["iters"]
            ranks += r["rank_used"]
            ms += r["t_iter_ms"]
            worst = max(worst, r["rel_resid_verified"])
            # after the solve: the zero-extension history now also holds this J, whose rows are masked anyway
            chis.append(g.energy_fraction(METHODS[name], act, b, xs)[0])
        out_methods[name] = {"cg_iters": iters, "alg1_s": round(ms * 1e-3, 4), "mean_rank": round(ranks / max(len(systems), 1), 2),
                             "worst_rel_resid": worst, "mean_chi": float(np.mean(chis)) if chis else 0.0,
                             "min_chi": float(np.min(chis)) if chis else 0.0,
                             # eq. (23): effective condition number of the deflated, Jacobi-preconditioned operator
                             # (extreme Ritz values of each replayed solve)
                             "mean_kappa_eff": float(np.mean(kappas)) if kappas else None,
                             "max_kappa_eff": float(np.max(kappas)) if kappas else None}
    g.close()
    base = out_methods["zeroext"]["cg_iters"]
    return {"metric": "matched replay of the inactive systems of a sequence (PAPER.md:168, Table 3): CG iterations per transfer",
            "value": out_methods["refdef"]["cg_iters"], "unit": "CG iterations (direct restriction)", "n_gpus": 1, "steps": nq, "warmup": 0,
            "higher_is_better": False, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(args, w), "mode": "replay", "queries": nq, "systems": len(systems),
                       "reference": args.reference, "reference_build_ms": ref["build_ms"]},
            "methods": out_methods,
            "iteration_ratio_zeroext_over_direct": round(base / max(out_methods["refdef"]["cg_iters"], 1), 3)}


# ----------------------------------------------------------------------------------------------- oracle legs
class OracleTimer:
    """Times the oracle (test infrastructure; built here with -fopenmp so that its row loops use the host cores, the
    arithmetic as it stands) on a bounded sample of the workload: Algorithm 1 on the full-domain inactive system of a
    query (b = l, zero start).  Line 2 (the coarse setup: QR + SVD, B Z, E, Cholesky) is built and timed ONCE; every
    sample is a capped run of the loop on it.  A complete query is extrapolated as
    seconds per CG iteration x CG iterations per query + setup seconds x PDAS steps per query, labelled as such."""

    def __init__(self, w, method, W):
        import oracle

        oracle.build_oracle(threaded=True)
        self.w, self.method = w, method
        self.o = oracle.Oracle.from_workload(w, threaded=True)
        self.cores = self.o.threads
        self.idx = np.arange(w.N, dtype=np.int64)
        t0 = time.perf_counter()
        self.cs = self.o.coarse(self.idx, W if (method != 0 and W is not None) else np.zeros((w.N, 0)))
        self.setup_s = time.perf_counter() - t0 if method != 0 else 0.0
        # one short run to size the samples
        b = w.m * w._target(1000 * w.config)
        t0 = time.perf_counter()
        _, rep = self.o.alg1_on(self.cs, b, np.zeros(w.N), cap=4)
        self.per_it_est = max((time.perf_counter() - t0) / (max(rep["iters"], 1) + 3.0), 1e-9)  # + the applies outside the loop

    def sample(self, budget_s, seed_qid=0):
        w = self.w
        b = w.m * w._target(1000 * w.config + seed_qid)
        cap = int(max(4, min(20000, budget_s / self.per_it_est)))
        t0 = time.perf_counter()
        _, rep = self.o.alg1_on(self.cs, b, np.zeros(w.N), cap=cap)
        t = time.perf_counter() - t0
        done = max(rep["iters"], 1)
        return t / (done + 3.0), done, t

    def per_query(self, per_it, iters_per_query, steps_per_query):
        return per_it * iters_per_query + self.setup_s * steps_per_query


def cpu_baseline(args, w, g, method, iters_per_query, steps_per_query):
    W = g.get_reference() if method != 0 else None
    tm = OracleTimer(w, method, W)
    per_it, done, t = tm.sample(args.cpu_budget)
    v = tm.per_query(per_it, iters_per_query, steps_per_query)
    return {"value": round(v, 2), "unit": "s/query (extrapolated: measured s per CG iteration x the CG iterations per query of this run)",
            "cores": tm.cores, "kind": "oracle",
            "sample": f"oracle Algorithm 1 ({args.method}, {tm.cores} OpenMP threads) on the full-domain inactive system of query 0: "
                      f"{done} iterations timed in {t:.1f} s ({per_it * 1e3:.3f} ms/iteration), coarse setup {tm.setup_s:.2f} s per PDAS step "
                      f"timed once; scaled by {iters_per_query:.0f} iterations and {steps_per_query:.0f} PDAS steps per query",
            "detail": dict(s_per_cg_iter=per_it, s_coarse_setup=tm.setup_s, iters_timed=done, seconds_timed=t,
                           iters_per_query=iters_per_query, steps_per_query=steps_per_query)}


def oracle_reference(w, method):
    """The reference W the oracle arm solves with.  Up to 1.5 M DOFs: the definition, a library eigensolver on the
    assembled H (oracle.reference_eigs).  Above that the eigensolve does not fit a run of a few minutes and the oracle's
    analytical reference stands in (the time per iteration does not depend on the values of W); said in `sample`."""
    import oracle

    if method == 0:
        return None, 0.0, "none"
    t0 = time.perf_counter()
    if w.N <= 1500000:
        _, W = oracle.reference_eigs(w.rowptr, w.colidx, w.val, w.m, w.alpha, w.k)
        kind = "library eigensolver on the assembled H"
    elif w.nt > 1:
        W = oracle.spacetime_reference(w.dims, w.nt, 1.0 / w.nt, w.k)[-1]
        kind = "analytical space-time reference (eigensolve of the assembled H skipped at this size)"
    else:
        W = oracle.sine_reference(w.dims, w.k)[-1]
        kind = "analytical sine reference (eigensolve of the assembled H skipped at this size)"
    return np.asfortranarray(W), time.perf_counter() - t0, kind


def run_reference(args):
    rank, _, world = dist_env()
    if rank != 0:
        return None
    import oracle

    oracle.build_oracle()
    w = make_workload(args)
    method = METHODS[args.method]
    prof = load_profile().get(w.name, {}).get(args.method, {})
    iters_per_query = float(prof.get("cg_iters_per_query", 0.0))
    steps_per_query = float(prof.get("pdas_steps_per_query", w.pdas_cap))
    W, t_ref, ref_kind = oracle_reference(w, method)
    tm = OracleTimer(w, method, W)
    nsteps = max(args.steps + args.warmup, 1)
    budget = max(0.5, min(args.cpu_budget, (180.0 - 2.0 * tm.setup_s) / nsteps))
    vals, last = [], None
    for i in range(args.warmup + args.steps):
        per_it, done, t = tm.sample(budget, seed_qid=i % w.n_queries)
        last = (per_it, done, t)
        if i >= args.warmup:
            vals.append(tm.per_query(per_it, iters_per_query or 1.0, steps_per_query))
    value = sum(vals) / len(vals) + t_ref / w.n_queries
    if not iters_per_query:
        unit_note = " (no recorded CG iterations per query for this workload: value is s per CG ITERATION-equivalent)"
    else:
        unit_note = ""
    sample = (f"oracle Algorithm 1 ({args.method}, {tm.cores} OpenMP threads) on the full-domain inactive system, {last[1]} iterations per step "
              f"({last[0] * 1e3:.3f} ms/iteration; coarse setup {tm.setup_s:.1f} s timed once), scaled to a query by the recorded "
              f"{iters_per_query:.0f} CG iterations and {steps_per_query:.0f} PDAS steps per query (profiles/bench_workload_profile.json); "
              f"reference: {ref_kind} ({t_ref:.1f} s) charged over the {w.n_queries} queries of a pass{unit_note}")
    return {"impl": "reference", "metric": "complete PDAS query time (incl. reference build)", "value": round(value, 2),
            "unit": "s/query", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": round(1e3 * value, 1), "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(args, w, pdas_cap_for(args, w)), "method": args.method, "parallelism": "host cores, rank 0 only"},
            "cpu_baseline": {"value": round(value, 2), "unit": "s/query", "kind": "oracle", "cores": tm.cores, "sample": sample},
            "e2e": {"value": round(value, 2), "unit": "s/query", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}


def build_parser():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=5,
                    help="BASELINE.json config; default 5 = the largest (160^3, N = 4,096,000, k = 64), the one the metric's "
                         "bandwidth target is quoted on")
    ap.add_argument("--pdas-cap", type=int, default=0, help="PDAS step cap; 0 = 400 on configs 2 and 4 (PAPER.md:341), else the workload's")
    ap.add_argument("--no-latency-block", action="store_true", help="skip the config-2 microseconds-per-iteration block")
    ap.add_argument("--twin", default=None)
    ap.add_argument("--method", default="refdef", choices=list(METHODS))
    ap.add_argument("--ref-tol", type=float, default=1e-3)
    ap.add_argument("--reference", default="eig", choices=["eig", "eig-filter", "eig-lobpcg", "eig-scaled", "sine", "coarse"],
                    help="eig: k lowest eigenvectors of H (BASELINE.json) by the default eigensolver; eig-filter: by Chebyshev-filtered "
                         "subspace iteration (rd_build_reference); eig-lobpcg: by sine-preconditioned LOBPCG (rd_build_reference_lobpcg, "
                         "steady Cartesian grids); sine: the paper's analytical "
                         "references (rd_build_reference_sine on the steady configs, rd_build_reference_spacetime on config 4); "
                         "coarse: Jacobi-scaled modes of the half-resolution operator, P1-prolonged (PAPER.md:176)")
    ap.add_argument("--kappa-ref", type=float, default=None,
                    help="conductivity of the homogeneous comparison medium of the LOBPCG preconditioner (default 1.0, the generator's solid)")
    ap.add_argument("--e2e-steps", type=int, default=0, help="host-buffer queries after the timed region; 0 = one full pass of the sequence")
    ap.add_argument("--cpu-budget", type=float, default=15.0, help="seconds of oracle work for cpu_baseline")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--mode", default="query", choices=["query", "loop", "replay", "setup"],
                    help="query: the metric; loop: the CG loop alone; replay: matched replay of a sequence's inactive systems")
    ap.add_argument("--cg-cap", type=int, default=500000, help="--mode loop: iteration cap of each solve")
    ap.add_argument("--alg1-variant", type=int, default=0, help="rd_options.alg1_variant (0: default kernel; 1: literal recurrence)")
    ap.add_argument("--ref-sweeps", type=int, default=60, help="--mode loop: filter sweeps of the reference build")
    return ap


def main(argv=None):
    args = build_parser().parse_args(argv)
    if args.kappa_ref is not None:
        global KAPPA_REF
        KAPPA_REF = float(args.kappa_ref)
    if args.impl == "reference":
        out = run_reference(args)
    elif args.mode == "loop":
        out = run_loop(args)
    elif args.mode == "replay":
        out = run_replay(args)
    elif args.mode == "setup":
        out = run_setup(args)
    else:
        out = run_ours(args)
    if out is not None:
        print(json.dumps(out), flush=True)
    return 0


if __name__ == "__main__":
    sys.exit(main())

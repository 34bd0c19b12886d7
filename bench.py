#!/usr/bin/env python
"""bench.py -- RK4 steps/s of the QTT/MPS time-step algebra on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--impl ours|reference]

A "step" is one qtt_rk4_step (the whole hot path: 24 apply+round, 16 hadamard+round, 8+6+2 sum+round)
on the synthetic decaying-jet workload of BASELINE.json configs[2] (2^10 x 2^10, chi = 64), the
configuration the metric is quoted on.  One process per GPU; the path does not shard ("replicas only",
DESIGN.md): with N > 1 every rank advances its own replica and value = N * K / max-over-ranks time.

Prints ONE JSON line (rank 0).  `--impl reference` times the CPU oracle (oracle/) on the host cores on a
bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import qtt_inputs as I  # noqa: E402

METRIC = "QTT RK4 steps/sec at 2^10x2^10, chi=64 fp64"  # BASELINE.json's metric (config 3, the default workload)
METRICS = {2: "QTT RK4 steps/sec at 2^8x2^8, chi=32 fp64", 3: METRIC, 4: "QTT RK4 steps/sec at 2^11x2^11, chi=128 fp64"}
UNIT = "steps/s"


EPS = 0.0     # --eps: truncation tolerance of every rounding (Eq. 16); 0 = pure chi_max cap, the BASELINE configs
SKETCH = None  # --product-compression sketch: seed of the sketched zip-up (reading 25); None = deterministic zip-up
SKEW = False  # --convection skew: the paper's skew-symmetric convection (PAPER.md Eq. B2) instead of the convective form


def workload(cfg: int):
    c = I.CONFIGS[cfg]
    name = {2: "config2 double shear layer", 3: "config3 decaying jet", 4: "config4 decaying turbulence"}[cfg]
    desc = (f"{name}: 2^{c['n']}x2^{c['n']} grid ({c['n']} sites, d=4), chi_max={c['chi']}, chi_work={2 * c['chi']}, "
            f"Re={c['Re']:g}, dt={c['dt']:g}, eps={EPS:g}, "
            f"{'skew-symmetric convection (PAPER.md Eq. B2)' if SKEW else 'convective form'}, "
            f"{'SKETCHED zip-up (seed %d; NOT the BASELINE method: DESIGN.md reading 25), ' % SKETCH if SKETCH is not None else ''}"
            f"one qtt_rk4_step per step")
    return c, desc


# ------------------------------------------------------------------------------------------- clocks
class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms during the timed region."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.lines, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "200", "-i",
                 str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                mx = float(f[1])
            except ValueError:
                continue
            for nme, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nme)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm)}


# ------------------------------------------------------------------------------------------- CPU oracle leg
def oracle_step_seconds(cfg: int, state=None):
    """Times ONE WHOLE RK4 step of the oracle as it stands (4 rhs evaluations, 3 stage combinations, the final 5-term
    sum: 56 roundings) on the host cores.  Returns (seconds, description, state); the next call continues from the
    state this step produced."""
    from oracle import qtt_oracle as O
    c, _ = workload(cfg)
    n, chi = c["n"], c["chi"]
    if state is None:
        ux, uy = I.config_fields(cfg)
        dx = 1.0 / (1 << n)
        state = dict(U=[O.from_dense(ux, chi), O.from_dense(uy, chi)], Dx=O.mpo_d1(n, dx), Dy=O.mpo_d2(n, dx),
                     Lap=O.mpo_laplacian(n, dx))
    t0 = time.perf_counter()
    state["U"] = O.rk4_step(state["U"], state["Dx"], state["Dy"], state["Lap"], c["Re"], c["dt"], chi, eps=EPS, skew=SKEW,
                             sketch_seed=SKETCH)
    t = time.perf_counter() - t0
    return t, "one whole oracle RK4 step per timed step (no extrapolation)", state


def blas_threads():
    try:
        from threadpoolctl import threadpool_info
        return max([p.get("num_threads", 1) for p in threadpool_info()] + [1])
    except Exception:
        return os.cpu_count() or 1


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    c, desc = workload(args.config)
    state = None
    # a CPU program needs no warm-up beyond the first touch of its BLAS threads: at most ONE untimed whole step, so
    # that the run (K + 1 whole oracle steps, ~19 s each at config 3 on 16 cores) stays within minutes
    warm = min(args.warmup, 1)
    for _ in range(warm):
        _, _, state = oracle_step_seconds(args.config, state)
    tot, sample = 0.0, ""
    for _ in range(args.steps):
        sec1, sample, state = oracle_step_seconds(args.config, state)
        tot += sec1
    sec = tot / max(args.steps, 1)
    val = 1.0 / sec
    cores = blas_threads()
    line = {
        "impl": "reference", "metric": METRICS[args.config], "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": desc, "note": "CPU oracle (NumPy fp64 + LAPACK) on the host cores; every timed step is one "
                   f"WHOLE oracle RK4 step (free-running trajectory); untimed warm-up steps run: {warm}"},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line), flush=True)
    return 0


# ------------------------------------------------------------------------------------------- replicas (N > 1)
def replica_seed(rank: int) -> int:
    """The path does not shard ("replicas only"): rank r advances its own replica, whose
    perturbation phases are drawn with seed r."""
    return int(rank)


def max_over_ranks(value: float, world: int, device: str = "cuda") -> float:
    """MAX of a host scalar over the ranks of the default process group (identity for world == 1)."""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(world: int, steps: int, ms_max: float) -> float:
    """steps/s summed over all replicas: every rank did `steps` steps within the slowest rank's time."""
    return world * steps / (ms_max * 1e-3)


# ------------------------------------------------------------------------------------------- algorithmic work model
def _bond_profile(n, chi):
    return [1] + [min(4 ** l, 4 ** (n - l), chi) for l in range(1, n)] + [1]


def _svd_nominal(a, b):
    a, b = max(a, b), min(a, b)
    return 6.0 * a * b * b + 20.0 * b ** 3


def _round_dense_work(r, chi, D=1):
    """SURVEY.md section 8(d) per-site formulas for round(dense MPS with bonds r): (GEMM-shaped flops, QR flops, nominal
    SVD flops, algorithmic bytes = operand cores read once + rounded cores written once)."""
    n = len(r) - 1
    p = [1] * (n + 1)
    for k in range(1, n + 1):
        p[k] = min(4 * p[k - 1], r[k])
    out = [1] * (n + 1)
    for k in range(n - 1, 0, -1):
        out[k] = max(1, min(chi, p[k], 4 * out[k + 1]))
    g = q = sv = 0.0
    for l in range(1, n):                      # L->R: thin QR of (4 p_{l-1}) x r_l, carry R into the next core
        m, k = 4 * p[l - 1], r[l]
        if m > k:
            q += 4.0 * m * k * k - (4.0 / 3.0) * k ** 3
        if m > k or l > 1:
            g += 2.0 * p[l] * r[l] * 4 * r[l + 1] / D
    for l in range(n, 1, -1):                  # R->L: SVD of p_{l-1} x (4 r'_l), absorb U S into the left neighbour
        sv += _svd_nominal(p[l - 1], 4 * out[l])
        g += 2.0 * 4 * p[l - 2] * p[l - 1] * out[l - 1]
    byts = 8.0 * (sum(r[k] * 4 * r[k + 1] for k in range(n)) / (D * D if D > 1 else 1) * (1 + D * D if D > 1 else 1)
                  + sum(out[k] * 4 * out[k + 1] for k in range(n)))
    return g, q, sv, byts


def _zip_work(ra, rb, chi, cw):
    """The same for the fused Hadamard + round (zip-up with working bond cw)."""
    n = len(ra) - 1
    rw = [1] * (n + 1)
    for k in range(1, n):
        rw[k] = min(4 * rw[k - 1], ra[k] * rb[k], cw)
    out = [1] * (n + 1)
    for k in range(n - 1, 0, -1):
        out[k] = max(1, min(chi, rw[k], 4 * out[k + 1]))
    g = q = sv = 0.0
    byts = 8.0 * (sum(ra[k] * 4 * ra[k + 1] + rb[k] * 4 * rb[k + 1] for k in range(n))
                  + sum(out[k] * 4 * out[k + 1] for k in range(n)))
    for l in range(1, n + 1):
        r, pa, pb, qa, qb = rw[l - 1], ra[l - 1], rb[l - 1], ra[l], rb[l]
        g += 8.0 * r * pa * pb * qa + 8.0 * r * qa * pb * qb        # row a2, two GEMM passes
        byts += 2 * 8.0 * 4 * r * qa * qb                            # T written once, read once
        if l == n:
            break
        m, k = 4 * r, qa * qb
        if m <= min(k, cw):
            continue
        keep = min(m, k, cw)
        q += float(m) * m * k                                        # Gram-equivalent count of the (4r) x (ab) factorisation
        sv += _svd_nominal(m, min(m, k))
        g += 2.0 * keep * m * k                                      # carry R' = Q^T T
    for l in range(n, 1, -1):
        sv += _svd_nominal(rw[l - 1], 4 * out[l])
        g += 2.0 * 4 * rw[l - 2] * rw[l - 1] * out[l - 1]
    return g, q, sv, byts


def step_work_model(n, chi, cw=None, skew=False):
    """Algorithmic work of ONE qtt_rk4_step from SURVEY.md section 8(d)'s per-site formulas:
    per rhs 4 apply(D=3)+round, 2 apply(D=5)+round, 4 zip-ups, 2 three-term sums (skew: 7 zip-ups, 8 applies(D=3),
    2 five-term sums); 3 two-term stage sums x2 and one five-term sum x2.  Returns flops split and bytes."""
    cw = cw or 2 * chi
    r = _bond_profile(n, chi)
    mul = lambda D: [D * x if 0 < i < n else x for i, x in enumerate(r)]
    parts = {"apply3": _round_dense_work(mul(3), chi, 3), "apply5": _round_dense_work(mul(5), chi, 5),
             "had": _zip_work(r, r, chi, cw), "sum2": _round_dense_work(mul(2), chi),
             "sum3": _round_dense_work(mul(3), chi), "sum5": _round_dense_work(mul(5), chi)}
    if skew:
        counts = {"apply3": 32, "apply5": 8, "had": 28, "sum2": 6, "sum3": 0, "sum5": 8 + 2}
    else:
        counts = {"apply3": 16, "apply5": 8, "had": 16, "sum2": 6, "sum3": 8, "sum5": 2}
    G = sum(parts[k][0] * counts[k] for k in parts)
    Qf = sum(parts[k][1] * counts[k] for k in parts)
    S = sum(parts[k][2] * counts[k] for k in parts)
    B = sum(parts[k][3] * counts[k] for k in parts)
    return {"flops": G + Qf + S, "gemm_shaped_flops": G, "qr_flops": Qf, "svd_nominal_flops": S,
            "rounding_sweep_bytes": B,
            "per_primitive_gflop": {k: sum(v[:3]) * 1e-9 for k, v in parts.items()}, "counts": counts}


# ------------------------------------------------------------------------------------------- our arm
def fp64_peaks(Q, ctx):
    """Measured fp64 issue rates of this GPU (TFLOP/s): the DMMA.8x8x4 tensor pipe and the DFMA pipe."""
    import ctypes as C
    out = {}
    for kind, name in ((0, "dmma"), (1, "dfma")):
        t = C.c_double()
        rc = ctx.lib.qtt_diag_fp64_probe(C.c_void_p(ctx.stream.cuda_stream), kind, 148 * 8, 2000, C.byref(t))
        out[name] = t.value if rc == 0 else None
    return out


def run_ours(args):
    import torch
    import torch.distributed as dist
    import paper_2406_17823_b200 as Q

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    c, desc = workload(args.config)
    n, chi = c["n"], c["chi"]
    ctx = Q.Context(device=local, workspace_bytes=int(args.workspace_gib * (1 << 30)))
    Q.qtt_ctx_set_convection(ctx, SKEW)
    dx = 1.0 / (1 << n)
    Dx, Dy = Q.qtt_mpo_central_difference(ctx, n, 1, dx), Q.qtt_mpo_central_difference(ctx, n, 2, dx)
    Lap = Q.qtt_mpo_laplacian(ctx, n, dx)
    ux, uy = I.config_fields(args.config, seed=replica_seed(rank))
    u = [Q.qtt_mps_from_dense(ctx, torch.from_numpy(f).cuda(), chi) for f in (ux, uy)]
    ctx.synchronize()
    sketch_record = None
    if SKETCH is not None:
        # what the cheaper compression costs in accuracy: one step from the same state in both modes, and the
        # deterministic step's own distance to a step at twice the bond (its truncation error), for scale
        def one_step(mode, bond):
            Q.qtt_ctx_set_product_compression(ctx, mode, SKETCH or 0)
            w = [Q.qtt_mps_from_dense(ctx, torch.from_numpy(f).cuda(), chi) for f in (ux, uy)]
            Q.qtt_rk4_step(ctx, w, Dx, Dy, Lap, c["Re"], c["dt"], bond, EPS)
            d = [Q.qtt_to_dense(ctx, x) for x in w]
            ctx.synchronize()
            return d
        det, ske, fine = one_step(False, chi), one_step(True, chi), one_step(False, 2 * chi)
        nrm = lambda a, b: float(sum(torch.linalg.norm(x - y) ** 2 for x, y in zip(a, b)) ** 0.5
                                 / sum(torch.linalg.norm(y) ** 2 for y in b) ** 0.5)
        sketch_record = {"seed": SKETCH, "rel_diff_sketch_vs_svd_one_step": nrm(ske, det),
                         "rel_diff_svd_chi_vs_2chi_one_step": nrm(det, fine),
                         "rel_diff_sketch_chi_vs_svd_2chi_one_step": nrm(ske, fine)}
        del det, ske, fine
        Q.qtt_ctx_set_product_compression(ctx, True, SKETCH)
        Q.qtt_ctx_jacobi_stats(ctx)  # the validation record below is about the timed steps, not the 2 chi yardstick step
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")  # > 126 MB L2

    def step():
        Q.qtt_rk4_step(ctx, u, Dx, Dy, Lap, c["Re"], c["dt"], chi, EPS)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    launches0 = Q.qtt_ctx_launch_count(ctx)
    sampler = ClockSampler(local)
    sampler.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    barrier()
    with torch.cuda.stream(ctx.stream):
        for e0, e1 in ev:
            flush.zero_()  # L2 flush between timed iterations, outside the per-step event pair
            e0.record(ctx.stream)
            step()
            e1.record(ctx.stream)
    barrier()
    clocks = sampler.stop()
    # what was timed must be a converged, finite computation: no Jacobi SVD hit its sweep limit, norms are finite
    max_sweeps, limit_hits = Q.qtt_ctx_jacobi_stats(ctx)
    norms = [Q.qtt_mps_norm(ctx, x) for x in u]
    if limit_hits != 0 or not all(np.isfinite(v) and v > 0 for v in norms):
        raise RuntimeError(f"timed steps are invalid: jacobi limit hits {limit_hits}, norms {norms}")
    validation = {"jacobi_max_sweeps": int(max_sweeps), "jacobi_limit_hits": int(limit_hits),
                  "norms_after_timed_steps": [float(v) for v in norms],
                  "parity": "tests/test_gpu_parity.py compares this launch configuration with the oracle (config 3: "
                            "steps 1-3; config 4: one full step against tests/golden/cfg4_step1.npz)"}
    ms = sum(e0.elapsed_time(e1) for e0, e1 in ev)
    launches = Q.qtt_ctx_launch_count(ctx) - launches0
    ms = max_over_ranks(ms, world)
    ms_per_step = ms / args.steps
    value = whole_job_value(world, args.steps, ms)

    # ---- end to end through the C ABI with HOST buffers: cores in pinned host memory -> device, step, cores back
    host = [Q.qtt_mps_get_cores(ctx, x, pinned=True) for x in u]
    h2d = sum(a.nbytes for cs in host for a in cs)
    e2e_steps = max(1, min(args.steps, 5))
    barrier()
    t0 = time.perf_counter()
    d2h = 0
    for _ in range(e2e_steps):
        v = [Q.qtt_mps_from_cores(ctx, cs) for cs in host]
        Q.qtt_rk4_step(ctx, v, Dx, Dy, Lap, c["Re"], c["dt"], chi, EPS)
        host = [Q.qtt_mps_get_cores(ctx, x, pinned=True) for x in v]
        d2h = sum(a.nbytes for cs in host for a in cs)
    torch.cuda.synchronize()
    e2e_sec = (time.perf_counter() - t0) / e2e_steps
    e2e_sec = max_over_ranks(e2e_sec, world)
    e2e = {"value": world / e2e_sec, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
           "steps": e2e_steps}

    line = {
        "metric": METRICS[args.config], "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": desc, "l2": "256 MiB buffer zeroed between timed steps, outside the per-step CUDA "
                   "event pairs; ms_per_step = sum of the per-step event times / steps",
                   "graph": "whole RK4 step replayed as one CUDA graph" if EPS == 0.0 else
                   "eps > 0: ranks are data dependent, the step runs eagerly with one stream synchronisation per bond and batch",
                   "parallelism": "replicas only"},
        "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "validation": validation,
    }
    if sketch_record:
        line["product_compression"] = sketch_record
    if rank == 0:
        line.update(roofline_and_baseline(Q, ctx, u, (Dx, Dy, Lap), c, chi, args, ms_per_step))
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return 0


def ncu_traffic_table():
    """dram bytes (read + write) per launch from the committed ncu --set full captures: profiles/ncu_traffic.csv, lines
    `family,d0,d1,d2,d3,dram_bytes_per_launch,source` keyed by the launch shape tag of qtt_diag_profile_dump."""
    out = {}
    try:
        for ln in open(os.path.join(ROOT, "profiles", "ncu_traffic.csv")).read().splitlines()[1:]:
            f = [x.strip() for x in ln.split(",")]
            if len(f) >= 7 and f[0] and not f[0].startswith("#"):
                out[(f[0], tuple(int(x) for x in f[1:5]))] = (float(f[5]), f[6])
    except (OSError, ValueError):
        pass
    return out


KERNEL_NAMES = {"rowjacobi": "qtt_bj2_kernel (q <= 512) / qtt_sbj_round_kernel (q <= 2048)", "qrcp": "qtt_qrcp_reg_kernel",
                "gemm": "qtt_gemm_dmma_kernel",
                "lq_panel": "qtt_lq_panel_kernel / qtt_qrcp_kernel", "lq_update": "qtt_gemm_dmma_kernel",
                "select": "qtt_select_kernel", "move": "movement kernels"}


def launch_records(ctx):
    """Per-launch (family, shape tag, ms, work) of the event-bracketed launches since the last report."""
    import tempfile
    fd, path = tempfile.mkstemp(suffix=".csv")
    os.close(fd)
    out = []
    try:
        if ctx.lib.qtt_diag_profile_dump(path.encode()) != 0:
            return out
        for ln in open(path).read().splitlines()[1:]:
            f = ln.split(",")
            out.append({"family": f[0], "shape": tuple(int(x) for x in f[1:5]), "ms": float(f[5]), "work": float(f[6])})
    finally:
        os.unlink(path)
    return out


def contraction_probe(ctx, chi, peak):
    """The two GEMM passes of the row-a2 site contraction at the bulk-site shapes of bond chi (working bond 2 chi,
    4 operands per launch, as in qtt_rk4_step), run through the same grouped DMMA kernel (qtt_diag_gemm) on random
    operands: X[r,b,(w,a')] = sum_a R[r,a,b] A[a,(w,a')] and T[(r,a'),b'] = sum_b X[(r,a'),b] B[b,b'] per omega."""
    import ctypes as C
    import torch
    r = 2 * chi
    st = C.c_void_p(ctx.stream.cuda_stream)
    shapes = [(4 * chi, chi, chi, 4 * r, 1), (r * chi, chi, chi, 16, 0)]  # (M, N, K, nbatch, transA)
    tot_ms, tot_fl = 0.0, 0.0
    with torch.cuda.stream(ctx.stream):
        for (M, N, K, nb, ta) in shapes:
            A = torch.randn(nb * M * K, dtype=torch.float64, device="cuda")
            B = torch.randn(nb * K * N, dtype=torch.float64, device="cuda")
            Cm = torch.empty(nb * M * N, dtype=torch.float64, device="cuda")
            def go():
                return ctx.lib.qtt_diag_gemm(st, C.c_void_p(A.data_ptr()), C.c_void_p(B.data_ptr()), C.c_void_p(Cm.data_ptr()),
                                             M, N, K, ta, 0, M if ta else K, N, N, 1.0, 0.0, nb, M * K, K * N, M * N)
            for _ in range(3):
                assert go() == 0
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(ctx.stream)
            for _ in range(5):
                go()
            e1.record(ctx.stream)
            e1.synchronize()
            tot_ms += e0.elapsed_time(e1) / 5
            tot_fl += 2.0 * M * N * K * nb
    tf = tot_fl / (tot_ms * 1e-3) * 1e-12
    return {"tflops": tf, "peak_tflops": peak, "frac": tf / peak if peak else None, "chi": chi,
            "what": "both GEMM passes of the row-a2 site contraction at the chi=128 bulk-site shapes (config 4 / config 5), "
                    "4 operands per launch, operands larger than L2 in total (0.5 GiB), CUDA events on the launching stream"}


def primitive_sweep(args):
    """BASELINE.json configs[4]: 2^12 x 2^12 (12 sites), random N(0,1) site tensors with the full bond profile, batch of
    6 operands per launch; per chi: one apply (d/dx, d/dy or Laplacian MPO) + round(chi) and one Hadamard with the next
    operand + round(chi), each timed with CUDA events on the context's stream (median of `steps` repetitions after
    `warmup`), plus the kernel-family split of one profiled repetition.  Prints ONE JSON line."""
    import torch
    import paper_2406_17823_b200 as Q
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: there is no CPU fallback")
    n = 12
    ctx = Q.Context(device=0, workspace_bytes=int(max(args.workspace_gib, 64.0) * (1 << 30)))
    dx = 1.0 / (1 << n)
    mpos = [Q.qtt_mpo_central_difference(ctx, n, 1, dx), Q.qtt_mpo_central_difference(ctx, n, 2, dx),
            Q.qtt_mpo_laplacian(ctx, n, dx)]
    peaks = fp64_peaks(Q, ctx)
    out = {}
    r = lambda chi: _bond_profile(n, chi)
    for chi in (16, 32, 64, 128, 256):
        xs = [Q.qtt_mps_from_cores(ctx, I.random_cores(n, chi, seed=s)) for s in range(6)]
        # algorithmic work of the two primitives on the batch of 6 (SURVEY.md section 8(d) per-site formulas)
        mul = lambda D: [D * x if 0 < i < n else x for i, x in enumerate(r(chi))]
        w3, w5, wz = _round_dense_work(mul(3), chi, 3), _round_dense_work(mul(5), chi, 5), _zip_work(r(chi), r(chi), chi, 2 * chi)
        alg = {"apply_round": 4 * sum(w3[:3]) + 2 * sum(w5[:3]), "hadamard_round": 6 * sum(wz[:3])}
        alg_gemm = {"apply_round": 4 * w3[0] + 2 * w5[0], "hadamard_round": 6 * wz[0]}

        def apply_round():
            ys = [Q.qtt_apply_mpo(ctx, mpos[i % 3], xs[i]) for i in range(6)]
            Q.qtt_round_batch(ctx, ys, chi)

        def hadamard_round():
            hs = [Q.qtt_hadamard(ctx, xs[i], xs[(i + 1) % 6]) for i in range(6)]
            Q.qtt_round_batch(ctx, hs, chi)

        res = {}
        for name, fn in (("apply_round", apply_round), ("hadamard_round", hadamard_round)):
            for _ in range(max(args.warmup, 1)):
                fn()
            ctx.synchronize()
            times = []
            with torch.cuda.stream(ctx.stream):
                for _ in range(max(args.steps, 1)):
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    e0.record(ctx.stream)
                    fn()
                    e1.record(ctx.stream)
                    e1.synchronize()
                    times.append(e0.elapsed_time(e1))
            Q.qtt_ctx_profile(ctx, True)
            Q.qtt_ctx_profile_report(ctx)
            fn()
            rep = Q.qtt_ctx_profile_report(ctx)
            Q.qtt_ctx_profile(ctx, False)
            g = rep["gemm"]
            ms = float(np.median(times))
            tf = alg[name] / (ms * 1e-3) * 1e-12
            stats = Q.qtt_ctx_jacobi_stats(ctx)
            res[name] = {"ms_per_batch_of_6": ms,
                         "algorithmic_gflop": alg[name] * 1e-9, "gemm_shaped_share": alg_gemm[name] / alg[name],
                         "roofline": {"bound": "tensor", "achieved": tf, "peak": peaks["dmma"], "unit": "TFLOP/s",
                                      "frac": tf / peaks["dmma"]},
                         "family_ms": {k: round(v["ms"], 3) for k, v in rep.items()},
                         "gemm_tflops": g["work"] / max(g["ms"] * 1e-3, 1e-12) * 1e-12,
                         "gemm_frac_of_dmma_peak": (g["work"] / max(g["ms"] * 1e-3, 1e-12) * 1e-12) / peaks["dmma"],
                         "jacobi_max_sweeps": int(stats[0]), "jacobi_limit_hits": int(stats[1])}
        out[str(chi)] = res
        del xs
    line = {"metric": "primitive sweep at 2^12x2^12, batch 6 (BASELINE.json configs[4])", "unit": "ms per batch of 6",
            "dtype": "f64", "data": "synthetic", "n_gpus": 1, "steps": args.steps, "warmup": args.warmup,
            "chi": out, "fp64_peaks_tflops": peaks,
            "roofline_note": "per primitive: SURVEY.md section 8(d) algorithmic flops of the batch of 6 / median CUDA-event "
                             "time / measured DMMA issue rate (fp64 tensor peak == fp64 FMA peak on B200)"}
    print(json.dumps(line), flush=True)
    return 0


def variational_bench(args):
    """one stage of the paper's variational solver (Sec. II.C, App. B) at the bench
    workload's shape (config 3: 2^10 x 2^10, chi = 64) with the paper's settings (mu = 25e4, <= 20 sweeps, CG <= 100
    iterations / 1e-5): a = the initial state, B = the convective right-hand side formed by the hot-path primitives,
    v0 = a (plus a 2 % compressible disturbance of u_y).  The stage is host-driven (scalar read-backs inside CG), so it is timed by wall clock around the synchronous
    call, after one warm-up stage.  Prints ONE JSON line."""
    import torch
    import paper_2406_17823_b200 as Q
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: there is no CPU fallback")
    c, desc = workload(args.config)
    n, chi = c["n"], c["chi"]
    ctx = Q.Context(device=0, workspace_bytes=int(args.workspace_gib * (1 << 30)))
    dx = 1.0 / (1 << n)
    Dx, Dy = Q.qtt_mpo_central_difference(ctx, n, 1, dx), Q.qtt_mpo_central_difference(ctx, n, 2, dx)
    ux, uy = I.config_fields(args.config)
    # the bench state is divergence-free by construction (the penalty would have nothing to do: zero CG iterations at the
    # paper's tolerance); a compressible disturbance of 2 % gives the stage the work it has inside a real time step
    X, Y = I.grid(n)
    uy = uy + 0.02 * np.sin(2 * np.pi * X) * np.cos(4 * np.pi * Y)
    a = [Q.qtt_mps_from_dense(ctx, torch.from_numpy(f).cuda(), chi) for f in (ux, uy)]
    # B_i = sum_j u_j (.) D_j u_i, rounded to chi (the nonlinear part of Eq. B21 in convective form)
    B = []
    for i in range(2):
        terms = []
        for j, D in enumerate((Dx, Dy)):
            g = Q.qtt_apply_mpo(ctx, D, a[i])
            Q.qtt_round(ctx, g, chi)
            prod = Q.qtt_hadamard(ctx, a[j], g)
            Q.qtt_round(ctx, prod, chi)
            terms.append(prod)
        Q.qtt_axpy(ctx, 1.0, terms[0], terms[1])
        Q.qtt_round(ctx, terms[1], chi)
        B.append(terms[1])
    mu, h = 25e4, c["dt"]
    peaks = fp64_peaks(Q, ctx)
    times, infos = [], []
    th0 = Q.qtt_variational_cost(ctx, a, a, B, Dx, Dy, h, mu)
    for rep in range(3 + max(args.steps, 1)):  # 0: warm-up, 1: profiled (event pair per launch), 2: warm-up again, 3..: timed
        v = [Q.qtt_mps_clone(ctx, x) for x in a]
        if rep == 1:
            Q.qtt_ctx_profile(ctx, True)
            Q.qtt_ctx_profile_report(ctx)
        ctx.synchronize()
        t0 = time.perf_counter()
        info = Q.qtt_variational_stage(ctx, v, a, B, Dx, Dy, h, mu)
        ctx.synchronize()
        if rep >= 3:
            times.append(time.perf_counter() - t0)
            infos.append(info)
        if rep == 1:
            rep1 = Q.qtt_ctx_profile_report(ctx)
            Q.qtt_ctx_profile(ctx, False)
            th1 = Q.qtt_variational_cost(ctx, v, a, B, Dx, Dy, h, mu)
    sec = float(np.median(times))
    g = rep1["gemm"]
    line = {"metric": "variational stage (PAPER.md Sec. II.C) at 2^%d x 2^%d, chi=%d fp64" % (n, n, chi), "value": 1.0 / sec,
            "unit": "stages/s", "ms_per_stage": sec * 1e3, "n_gpus": 1, "steps": len(times), "dtype": "f64", "data": "synthetic",
            "config": {"workload": desc, "mu": mu, "h": h, "max_sweeps": 20, "sweep_tol": 1e-5, "cg_maxit": 100, "cg_tol": 1e-5,
                       "timing": "wall clock around the synchronous call, median over the timed repetitions; the repetition with "
                                 "an event pair per launch (family_ms) is separate and not timed"},
            "solver": infos[-1], "theta_before": th0, "theta_after": th1,
            "family_ms": {k: round(vv["ms"], 3) for k, vv in rep1.items()},
            "gemm_tflops": g["work"] / max(g["ms"] * 1e-3, 1e-12) * 1e-12,
            "gemm_frac_of_dmma_peak": (g["work"] / max(g["ms"] * 1e-3, 1e-12) * 1e-12) / peaks["dmma"],
            "launches_per_stage": int(sum(vv["launches"] for vv in rep1.values())), "fp64_peaks_tflops": peaks}
    print(json.dumps(line), flush=True)
    return 0


def three_d_bench(args):
    """SURVEY.md section 8f next-4 (reading 26): one right-hand side of the 3D Burgers equations in the d = 8
    encoding, composed from the batched C-ABI primitives as a caller would -- f_i = -sum_j u_j (.) D_j u_i + (1/Re) Lap u_i,
    i = 1..3: one batch of 12 apply + round, one of 9 zip-ups, one of 3 four-term sums -- on the Taylor-Green vortex plus seeded
    noise (qtt_inputs.taylor_green_3d) at 2^n points per direction.  Device-timed with CUDA events on the context's stream
    (eager launches: no graph for the composed path).  Prints ONE JSON line."""
    import torch
    import paper_2406_17823_b200 as Q
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: there is no CPU fallback")
    n, chi, Re = args.three_d, args.three_d_chi, 1600.0
    ctx = Q.Context(device=0, workspace_bytes=int(args.workspace_gib * (1 << 30)))
    Q.qtt_ctx_set_phys_dim(ctx, 8)
    dx = 1.0 / (1 << n)
    Dj = [Q.qtt_mpo_central_difference(ctx, n, j, dx) for j in (1, 2, 3)]
    Lap = Q.qtt_mpo_laplacian(ctx, n, dx)
    u = [Q.qtt_mps_from_dense(ctx, torch.from_numpy(f).cuda(), chi) for f in I.taylor_green_3d(n, seed=0, noise=1e-3)]

    def rhs():
        g = [[Q.qtt_apply_mpo(ctx, Dj[j], u[i]) for j in range(3)] for i in range(3)]
        lap = [Q.qtt_apply_mpo(ctx, Lap, u[i]) for i in range(3)]
        Q.qtt_round_batch(ctx, [x for row in g for x in row] + lap, chi)
        c = [[Q.qtt_hadamard(ctx, u[j], g[i][j]) for j in range(3)] for i in range(3)]
        Q.qtt_round_batch(ctx, [x for row in c for x in row], chi)
        for i in range(3):  # Re * f_i = lap - Re (c_i1 + c_i2 + c_i3): qtt_axpy weights the term it adds
            for j in (2, 1, 0):
                Q.qtt_axpy(ctx, -Re, c[i][j], lap[i])
        Q.qtt_round_batch(ctx, lap, chi)
        return lap

    peaks = fp64_peaks(Q, ctx)
    times = []
    for rep in range(args.warmup + max(args.steps, 1)):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ctx.synchronize()
        l0 = Q.qtt_ctx_launch_count(ctx)
        e0.record(ctx.stream)
        f = rhs()
        e1.record(ctx.stream)
        ctx.synchronize()
        if rep >= args.warmup:
            times.append(e0.elapsed_time(e1))
        launches = Q.qtt_ctx_launch_count(ctx) - l0
    Q.qtt_ctx_profile(ctx, True)
    Q.qtt_ctx_profile_report(ctx)
    f = rhs()
    fam = Q.qtt_ctx_profile_report(ctx)
    Q.qtt_ctx_profile(ctx, False)
    # whole RK4 steps through the library's own 3D step (qtt_rk4_step3: four right-hand sides, stage and final sums)
    dt = 0.1 * dx
    v = [Q.qtt_mps_clone(ctx, x) for x in u]
    step_ms = []
    for rep in range(args.warmup + max(args.steps, 1)):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ctx.synchronize()
        l0 = Q.qtt_ctx_launch_count(ctx)
        e0.record(ctx.stream)
        Q.qtt_rk4_step3(ctx, v, Dj, Lap, Re, dt, chi)
        e1.record(ctx.stream)
        ctx.synchronize()
        if rep >= args.warmup:
            step_ms.append(e0.elapsed_time(e1))
        step_launches = Q.qtt_ctx_launch_count(ctx) - l0
    sweeps, hits = Q.qtt_ctx_jacobi_stats(ctx)
    ms = float(np.median(times))
    g = fam["gemm"]
    line = {"metric": "3D Burgers right-hand sides/s at 2^%d^3, d=8, chi=%d fp64" % (n, chi), "value": 1e3 / ms, "unit": "rhs/s",
            "ms_per_rhs": ms, "rk4_step3": {"ms_per_step": float(np.median(step_ms)), "steps_per_s": 1e3 / float(np.median(step_ms)),
                                            "dt": dt, "gpu_launches_per_step": int(step_launches),
                                            "norms_after": [Q.qtt_mps_norm(ctx, x) for x in v]}, "n_gpus": 1, "steps": len(times), "warmup": args.warmup, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "Taylor-Green vortex + 1e-3 N(0,1) on a 2^%d cube (%d sites, d=8), chi_max=%d, chi_work=%d, "
                                   "Re=%g: 12 apply+round, 9 zip-ups, 3 four-term sums, batched per level" % (n, n, chi, 2 * chi, Re),
                       "timing": "CUDA events on the context's stream around the eagerly launched composition, median"},
            "bonds": Q.qtt_mps_bonds(f[0]), "norms": [Q.qtt_mps_norm(ctx, x) for x in f],
            "gpu_launches": int(launches), "jacobi_max_sweeps": sweeps, "jacobi_limit_hits": hits,
            "family_ms": {k: round(v["ms"], 3) for k, v in fam.items()},
            "gemm_tflops": g["work"] / max(g["ms"] * 1e-3, 1e-12) * 1e-12,
            "gemm_frac_of_dmma_peak": (g["work"] / max(g["ms"] * 1e-3, 1e-12) * 1e-12) / peaks["dmma"], "fp64_peaks_tflops": peaks}
    # roofline of the dominant family and of the whole right-hand side: algorithmic flops as counted per launch by the library
    # (the formulas of DESIGN.md section 6: nominal SVD / Householder / GEMM counts) over the measured times
    flop_fams = ("gemm", "lq_panel", "lq_update", "rowjacobi", "qrcp")
    dom = max(flop_fams, key=lambda k: fam[k]["ms"])
    dpeak = peaks["dmma"] if dom in ("gemm", "lq_update") else peaks["dfma"]
    dach = fam[dom]["work"] / max(fam[dom]["ms"] * 1e-3, 1e-12) * 1e-12
    flops = float(sum(fam[k]["work"] for k in flop_fams))
    line["roofline"] = {"kernel": dom + " family, summed over one right-hand side", "bound": "tensor" if dpeak == peaks["dmma"] else "alu",
                        "achieved": dach, "peak": dpeak, "unit": "TFLOP/s", "frac": dach / dpeak, "traffic": None}
    line["roofline_rhs"] = {"flops": flops, "achieved": flops / (ms * 1e-3) * 1e-12, "peak": peaks["dmma"], "unit": "TFLOP/s",
                            "frac": flops / (ms * 1e-3) * 1e-12 / peaks["dmma"]}
    print(json.dumps(line), flush=True)
    return 0


def roofline_and_baseline(Q, ctx, u, ops, c, chi, args, ms_per_step):
    """Per-kernel-family device times of one more (eagerly launched, event-bracketed) step -> roofline of the
    dominant family; the site-contraction TFLOP/s; and the CPU oracle timed on a bounded sample."""
    Dx, Dy, Lap = ops
    peaks = fp64_peaks(Q, ctx)
    Q.qtt_ctx_profile(ctx, True)
    Q.qtt_ctx_profile_report(ctx)  # clear
    nprof = 2
    for _ in range(nprof):
        Q.qtt_rk4_step(ctx, u, Dx, Dy, Lap, c["Re"], c["dt"], chi, EPS)
    per_launch = launch_records(ctx)  # before the report clears them
    rep = Q.qtt_ctx_profile_report(ctx)
    Q.qtt_ctx_profile(ctx, False)
    tot_ms = sum(v["ms"] for v in rep.values()) or 1.0
    fams = {}
    for k, v in rep.items():
        fams[k] = {"ms_per_step": v["ms"] / nprof, "launches_per_step": v["launches"] // nprof,
                   "share": v["ms"] / tot_ms,
                   "work_per_step": v["work"] / nprof}
    dom = max(rep, key=lambda k: rep[k]["ms"])
    d = rep[dom]
    bound = {"gemm": "tensor", "lq_panel": "alu", "lq_update": "tensor", "rowjacobi": "alu", "select": "hbm",
             "move": "hbm", "qrcp": "alu"}[dom]
    # the dominant KERNEL: the launch shape of the dominant family with the largest summed time
    shapes = {}
    for r in per_launch:
        if r["family"] == dom:
            a = shapes.setdefault(r["shape"], {"ms": 0.0, "work": 0.0, "n": 0})
            a["ms"] += r["ms"]; a["work"] += r["work"]; a["n"] += 1
    shape = max(shapes, key=lambda k: shapes[k]["ms"]) if shapes else None
    k = shapes[shape] if shape else {"ms": d["ms"], "work": d["work"], "n": max(d["launches"], 1)}
    if bound == "hbm":
        try:
            peak = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]
            src = "MEASURED_PEAKS.json hbm_gbs (of measured)"
        except Exception:
            peak, src = 6650.0, "B200_PROFILING.md fallback (of fallback)"
        achieved = k["work"] / (k["ms"] * 1e-3) * 1e-9
        unit = "GB/s"
    else:
        peak = peaks["dmma"] if bound == "tensor" else peaks["dfma"]
        src = ("qtt_diag_fp64_probe, measured in this run: register-only " +
               ("DMMA.8x8x4" if bound == "tensor" else "DFMA") + " issue rate on all 148 SMs (MEASURED_PEAKS.json has "
               "no fp64 figure; nominal 148 SM x 64 DFMA/clk x 2 x 1.965 GHz = 37.2 TFLOP/s, DESIGN.md section 6)")
        achieved = k["work"] / (k["ms"] * 1e-3) * 1e-12
        unit = "TFLOP/s"
    traffic, traffic_src = ncu_traffic_table().get((dom, shape), (None, None))
    roof = {"kernel": KERNEL_NAMES.get(dom, dom) + (f" launch shape (d0,d1,d2,d3)={shape}" if shape else ""),
            "bound": bound, "achieved": achieved, "peak": peak, "unit": unit,
            "frac": achieved / peak if peak else None, "traffic": traffic, "peak_source": src,
            "launches_per_step": k["n"] // nprof, "avg_launch_ms": k["ms"] / max(k["n"], 1),
            "share_of_step_kernel_time": k["ms"] / tot_ms, "family_share_of_step_kernel_time": d["ms"] / tot_ms,
            "algorithmic_work": "nominal SVD count 6ab^2+20b^3 per matrix (DESIGN.md section 6)" if dom == "rowjacobi"
            else "DESIGN.md section 6 per-family formulas",
            "traffic_source": ("dram__bytes_read.sum + dram__bytes_write.sum of one ncu --set full capture of this "
                               "launch shape (profiles/ncu_traffic.csv: " + traffic_src + ")") if traffic else None}
    try:
        hbm_peak = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]
        hbm_src = "MEASURED_PEAKS.json hbm_gbs (of measured)"
    except Exception:
        hbm_peak, hbm_src = 6650.0, "B200_PROFILING.md fallback (of fallback)"
    fam_bound = {"gemm": "tensor", "lq_panel": "alu", "lq_update": "tensor", "rowjacobi": "alu", "select": "hbm",
                 "move": "hbm", "qrcp": "alu"}
    for kf, v in fams.items():
        sec = max(v["ms_per_step"] * 1e-3, 1e-12)
        if fam_bound[kf] == "hbm":
            v.update(bound="hbm", achieved=v["work_per_step"] / sec * 1e-9, peak=hbm_peak, unit="GB/s")
        else:
            pk = peaks["dmma"] if fam_bound[kf] == "tensor" else peaks["dfma"]
            v.update(bound=fam_bound[kf], achieved=v["work_per_step"] / sec * 1e-12, peak=pk, unit="TFLOP/s")
        v["frac"] = v["achieved"] / v["peak"] if v["peak"] else None
    model = step_work_model(c["n"], chi, skew=SKEW)
    step_sec = ms_per_step * 1e-3
    sweep_fams = ("lq_panel", "lq_update", "rowjacobi", "select", "move", "qrcp")
    sweep_sec = sum(fams[kf]["ms_per_step"] for kf in sweep_fams) * 1e-3
    roofline_step = {
        "bound": "tensor", "achieved": model["flops"] / step_sec * 1e-12, "peak": peaks["dmma"], "unit": "TFLOP/s",
        "frac": (model["flops"] / step_sec * 1e-12) / peaks["dmma"] if peaks["dmma"] else None,
        "algorithmic_gflop_per_step": model["flops"] * 1e-9, "gemm_shaped_share": model["gemm_shaped_flops"] / model["flops"],
        "qr_gflop": model["qr_flops"] * 1e-9, "svd_nominal_gflop": model["svd_nominal_flops"] * 1e-9,
        "per_primitive_gflop": model["per_primitive_gflop"], "primitive_counts_per_step": model["counts"],
        "ms_per_step": ms_per_step,
        "what": "SURVEY.md section 8(d) per-site formulas (contraction + carry + absorb GEMMs, QR 4mk^2-4k^3/3, Gram-equivalent "
                "m^2 k of the zip-up factorisation, nominal SVD 6ab^2+20b^3) summed over one step / graph-replayed step time "
                "/ measured DMMA issue rate (fp64 tensor peak == fp64 FMA peak on this part)",
        "rounding_sweep": {"bound": "hbm", "achieved": model["rounding_sweep_bytes"] / max(sweep_sec, 1e-12) * 1e-9,
                           "peak": hbm_peak, "unit": "GB/s",
                           "frac": model["rounding_sweep_bytes"] / max(sweep_sec, 1e-12) * 1e-9 / hbm_peak,
                           "algorithmic_mbytes_per_step": model["rounding_sweep_bytes"] * 1e-6,
                           "kernel_ms_per_step": sweep_sec * 1e3, "peak_source": hbm_src,
                           "what": "operand cores read once + rounded cores written once (+ zip-up T written and read once) "
                                   "over the summed kernel time of the non-GEMM families; the working set of this config is "
                                   "L2-resident, so the HBM fraction is low by construction (SURVEY.md section 8d)"}}
    g = rep["gemm"]
    # the Hadamard site contractions proper at the bulk sites of this workload:
    # pass 1 (4 chi x chi x chi, batched over the working bond) and pass 2 (2 chi^2 x chi x chi, batched over omega)
    a2 = [r for r in per_launch if r["family"] == "gemm" and r["shape"][1] == chi and r["shape"][2] == chi
          and r["shape"][0] in (4 * chi, 2 * chi * chi)]
    a2_ms, a2_work = sum(r["ms"] for r in a2), sum(r["work"] for r in a2)
    if SKETCH is not None:
        roofline_step["note"] = ("flop model of the DETERMINISTIC step (SURVEY.md section 8d) over the sketched step's time: the sketched "
                                 "zip-up does less work than that, so this fraction overstates what the kernels achieve")
    out = {"roofline": roof, "roofline_step": roofline_step, "families": fams,
           "contraction_a2": {"tflops": a2_work / max(a2_ms * 1e-3, 1e-12) * 1e-12, "peak_tflops": peaks["dmma"],
                              "frac": (a2_work / max(a2_ms * 1e-3, 1e-12) * 1e-12) / peaks["dmma"] if peaks["dmma"] else None,
                              "launches_per_step": len(a2) // nprof,
                              "what": f"row a2 only: the two DMMA GEMM passes of the Hadamard site contraction at the bulk "
                                      f"sites (chi={chi}, working bond {2 * chi}), inside the profiled steps"},
           "contraction_chi128": contraction_probe(ctx, 128, peaks["dmma"]),
           "contraction": {"tflops": g["work"] / max(g["ms"] * 1e-3, 1e-12) * 1e-12, "peak_tflops": peaks["dmma"],
                           "frac": (g["work"] / max(g["ms"] * 1e-3, 1e-12) * 1e-12) / peaks["dmma"] if peaks["dmma"] else None,
                           "what": "sum 2MNK of all DMMA site-contraction GEMMs of a step / their summed kernel time"},
           "fp64_peaks_tflops": peaks,
           "step_flop_model": {"kernel_time_sum_ms": tot_ms / nprof, "graph_ms_per_step": ms_per_step}}
    if int(os.environ.get("WORLD_SIZE", "1")) == 1 and not args.no_cpu_baseline:
        sec, sample, _ = oracle_step_seconds(args.config)
        out["cpu_baseline"] = {"value": 1.0 / sec, "unit": UNIT, "cores": blas_threads(), "kind": "oracle",
                               "sample": "ONE whole oracle RK4 step of this workload from the initial state ("
                               + sample + ")", "seconds_per_step": sec}
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3, choices=(2, 3, 4))
    ap.add_argument("--impl", default="ours", choices=("ours", "reference"))
    ap.add_argument("--workspace-gib", type=float, default=8.0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--primitive-sweep", action="store_true",
                    help="BASELINE.json configs[4]: time apply+round and hadamard+round at 2^12 x 2^12, chi = 16..256, "
                         "batch 6, with each primitive's roofline fraction, instead of the RK4 step")
    ap.add_argument("--convection", default="convective", choices=("convective", "skew"),
                    help="convective (BASELINE.json's configs, default) or the paper's skew-symmetric form (Eq. B2)")
    ap.add_argument("--eps", type=float, default=0.0,
                    help="truncation tolerance of every rounding (PAPER.md Eq. 16-17) on top of the chi_max cap; 0 (default) = the "
                         "BASELINE configs.  eps > 0 runs eagerly (data-dependent ranks: one stream synchronisation per bond)")
    ap.add_argument("--product-compression", default="svd", choices=("svd", "sketch"),
                    help="svd (default): the deterministic zip-up of the BASELINE configs; sketch: the randomised range finder of "
                         "SURVEY.md section 8f next-4 (DESIGN.md reading 25) at the sites its rule admits -- another method, "
                         "reported with its one-step distance to the deterministic result")
    ap.add_argument("--sketch-seed", type=int, default=1)
    ap.add_argument("--three-d", type=int, default=0, metavar="NBITS",
                    help="time one 3D Burgers right-hand side in the d = 8 encoding on a 2^NBITS cube (SURVEY.md section 8f next-4)")
    ap.add_argument("--three-d-chi", type=int, default=32)
    ap.add_argument("--variational", action="store_true",
                    help="time one stage of the paper's variational solver (SURVEY.md section 8f next-1) at the workload's shape")
    ap.add_argument("--probe-contraction", type=int, default=0, metavar="CHI",
                    help="only run the row-a2 site-contraction GEMM passes at the bulk-site shapes of bond CHI and "
                         "print their TFLOP/s (the command the ncu capture in profiles/ is taken on)")
    args = ap.parse_args()
    global SKEW, EPS, SKETCH
    SKEW = args.convection == "skew"
    SKETCH = args.sketch_seed if args.product_compression == "sketch" else None
    EPS = args.eps
    if args.impl == "reference":
        return run_reference(args)
    if args.primitive_sweep:
        return primitive_sweep(args)
    if args.three_d:
        return three_d_bench(args)
    if args.variational:
        return variational_bench(args)
    if args.probe_contraction:
        import torch
        import paper_2406_17823_b200 as Q
        if not torch.cuda.is_available():
            raise RuntimeError("bench.py needs a CUDA device: there is no CPU fallback")
        ctx = Q.Context(device=0, workspace_bytes=1 << 28)
        peaks = fp64_peaks(Q, ctx)
        print(json.dumps({"contraction": contraction_probe(ctx, args.probe_contraction, peaks["dmma"]),
                          "fp64_peaks_tflops": peaks}), flush=True)
        return 0
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())

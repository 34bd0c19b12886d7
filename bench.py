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


SKEW = False  # --convection skew: the paper's skew-symmetric convection (PAPER.md Eq. B2) instead of the convective form


def workload(cfg: int):
    c = I.CONFIGS[cfg]
    name = {2: "config2 double shear layer", 3: "config3 decaying jet", 4: "config4 decaying turbulence"}[cfg]
    desc = (f"{name}: 2^{c['n']}x2^{c['n']} grid ({c['n']} sites, d=4), chi_max={c['chi']}, chi_work={2 * c['chi']}, "
            f"Re={c['Re']:g}, dt={c['dt']:g}, eps=0, "
            f"{'skew-symmetric convection (PAPER.md Eq. B2)' if SKEW else 'convective form'}, one qtt_rk4_step per step")
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
def oracle_sample_seconds(cfg: int, state=None):
    """Times a bounded sample of one RK4 step with the oracle as it stands: ONE of the four rhs evaluations
    (6 apply+round, 4 hadamard+round, 2 three-term sums) plus ONE of the four stage combinations, and
    extrapolates one step as 4 x that sample.  Returns (seconds per extrapolated step, description, state)."""
    from oracle import qtt_oracle as O
    c, _ = workload(cfg)
    n, chi = c["n"], c["chi"]
    if state is None:
        ux, uy = I.config_fields(cfg)
        dx = 1.0 / (1 << n)
        state = dict(U=[O.from_dense(ux, chi), O.from_dense(uy, chi)], Dx=O.mpo_d1(n, dx), Dy=O.mpo_d2(n, dx),
                     Lap=O.mpo_laplacian(n, dx))
    U = state["U"]
    t0 = time.perf_counter()
    k1 = O.rhs(U, state["Dx"], state["Dy"], state["Lap"], c["Re"], chi, skew=SKEW)
    U2 = [O.round_mps(O.lincomb([(1.0, U[i]), (c["dt"] / 2, k1[i])]), chi) for i in range(2)]
    t = time.perf_counter() - t0
    state["U"] = U2  # the next sample continues from the half-step state
    return 4.0 * t, "1 of the 4 rhs evaluations + 1 of the 4 stage combinations of one RK4 step, x4", state


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
    for _ in range(args.warmup):
        _, _, state = oracle_sample_seconds(args.config, state)
    tot, sample = 0.0, ""
    for _ in range(args.steps):
        s, sample, state = oracle_sample_seconds(args.config, state)
        tot += s
    sec = tot / max(args.steps, 1)
    val = 1.0 / sec
    cores = blas_threads()
    line = {
        "impl": "reference", "metric": METRICS[args.config], "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": desc, "note": "CPU oracle (NumPy fp64 + LAPACK) on the host cores; each step is a "
                   "bounded sample extrapolated to one RK4 step"},
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
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")  # > 126 MB L2

    def step():
        Q.qtt_rk4_step(ctx, u, Dx, Dy, Lap, c["Re"], c["dt"], chi)

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
        Q.qtt_rk4_step(ctx, v, Dx, Dy, Lap, c["Re"], c["dt"], chi)
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
                   "graph": "whole RK4 step replayed as one CUDA graph", "parallelism": "replicas only"},
        "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches),
    }
    if rank == 0:
        line.update(roofline_and_baseline(Q, ctx, u, (Dx, Dy, Lap), c, chi, args, ms_per_step))
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return 0


# dram bytes (read + write) per launch from the committed ncu --set full captures (profiles/), keyed by
# (family, launch shape tag of qtt_diag_profile_dump)
NCU_TRAFFIC_BYTES = {("rowjacobi", (512, 512, 4, 16)): 8.43e6}
KERNEL_NAMES = {"rowjacobi": "qtt_blockjacobi_kernel", "qrcp": "qtt_qrcp_reg_kernel", "gemm": "qtt_gemm_dmma_kernel",
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
    ctx = Q.Context(device=0, workspace_bytes=int(max(args.workspace_gib, 24.0) * (1 << 30)))
    dx = 1.0 / (1 << n)
    mpos = [Q.qtt_mpo_central_difference(ctx, n, 1, dx), Q.qtt_mpo_central_difference(ctx, n, 2, dx),
            Q.qtt_mpo_laplacian(ctx, n, dx)]
    peaks = fp64_peaks(Q, ctx)
    out = {}
    for chi in (16, 32, 64, 128):
        xs = [Q.qtt_mps_from_cores(ctx, I.random_cores(n, chi, seed=s)) for s in range(6)]

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
            res[name] = {"ms_per_batch_of_6": float(np.median(times)),
                         "family_ms": {k: round(v["ms"], 3) for k, v in rep.items()},
                         "gemm_tflops": g["work"] / max(g["ms"] * 1e-3, 1e-12) * 1e-12,
                         "gemm_frac_of_dmma_peak": (g["work"] / max(g["ms"] * 1e-3, 1e-12) * 1e-12) / peaks["dmma"]}
        out[str(chi)] = res
        del xs
    line = {"metric": "primitive sweep at 2^12x2^12, batch 6 (BASELINE.json configs[4])", "unit": "ms per batch of 6",
            "dtype": "f64", "data": "synthetic", "n_gpus": 1, "steps": args.steps, "warmup": args.warmup,
            "chi": out, "fp64_peaks_tflops": peaks,
            "not_run": {"256": "the zip-up SVD at chi = 256 has 2048 columns: beyond the streamed Jacobi kernel (<= 1024), "
                               "see DESIGN.md known limits"}}
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
        Q.qtt_rk4_step(ctx, u, Dx, Dy, Lap, c["Re"], c["dt"], chi)
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
    traffic = NCU_TRAFFIC_BYTES.get((dom, shape))
    roof = {"kernel": KERNEL_NAMES.get(dom, dom) + (f" launch shape (d0,d1,d2,d3)={shape}" if shape else ""),
            "bound": bound, "achieved": achieved, "peak": peak, "unit": unit,
            "frac": achieved / peak if peak else None, "traffic": traffic, "peak_source": src,
            "launches_per_step": k["n"] // nprof, "avg_launch_ms": k["ms"] / max(k["n"], 1),
            "share_of_step_kernel_time": k["ms"] / tot_ms, "family_share_of_step_kernel_time": d["ms"] / tot_ms,
            "algorithmic_work": "nominal SVD count 6ab^2+20b^3 per matrix (DESIGN.md section 6)" if dom == "rowjacobi"
            else "DESIGN.md section 6 per-family formulas",
            "traffic_source": "dram__bytes_read.sum + dram__bytes_write.sum of one ncu --set full capture of this "
            "launch shape (profiles/r1_blockjacobi_full.md)" if traffic else None}
    g = rep["gemm"]
    # the Hadamard site contractions proper at the bulk sites of this workload:
    # pass 1 (4 chi x chi x chi, batched over the working bond) and pass 2 (2 chi^2 x chi x chi, batched over omega)
    a2 = [r for r in per_launch if r["family"] == "gemm" and r["shape"][1] == chi and r["shape"][2] == chi
          and r["shape"][0] in (4 * chi, 2 * chi * chi)]
    a2_ms, a2_work = sum(r["ms"] for r in a2), sum(r["work"] for r in a2)
    out = {"roofline": roof, "families": fams,
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
        sec, sample, _ = oracle_sample_seconds(args.config)
        out["cpu_baseline"] = {"value": 1.0 / sec, "unit": UNIT, "cores": blas_threads(), "kind": "oracle",
                               "sample": sample, "seconds_per_step_extrapolated": sec}
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
                    help="BASELINE.json configs[4]: time apply+round and hadamard+round at 2^12 x 2^12, chi = 16..128, "
                         "batch 6, instead of the RK4 step")
    ap.add_argument("--convection", default="convective", choices=("convective", "skew"),
                    help="convective (BASELINE.json's configs, default) or the paper's skew-symmetric form (Eq. B2)")
    ap.add_argument("--probe-contraction", type=int, default=0, metavar="CHI",
                    help="only run the row-a2 site-contraction GEMM passes at the bulk-site shapes of bond CHI and "
                         "print their TFLOP/s (the command the ncu capture in profiles/ is taken on)")
    args = ap.parse_args()
    global SKEW
    SKEW = args.convection == "skew"
    if args.impl == "reference":
        return run_reference(args)
    if args.primitive_sweep:
        return primitive_sweep(args)
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

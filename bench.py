#!/usr/bin/env python
"""bench.py -- measures BASELINE.json's metric ("multi-RHS clover Dslash HBM GB/s & % of peak; batched CG sec/RHS").

One "step" is one pass of the whole hot path over one batch of synthetic sources: a batched
mixed-precision even-odd CG solve M x = b for N_rhs LapH-diluted sources.  Default workload: BASELINE.json configs[3]
(48^3 x 96, 12 RHS, int16+norm inner CG with fp32 clover, fp64 defect correction to 1e-9), the largest solver configuration
that fits one GPU; `--workload cfg1` is configs[1] (16^3 x 32, 8 RHS, fp32 inner CG).  `--steps K --warmup W` are honoured
exactly (W >= 3).
  value    = seconds per RHS, sources resident in HBM in the native layout (K timed solves between CUDA events)
  e2e      = the same through the C ABI with HOST buffers (pinned canonical arrays in and out: H2D, reorder, solve, reorder, D2H)
  roofline = the Dslash half of the metric: fused kernel A (A^-1 D, fp32, 18-real links) at N_rhs = 8 on configs[2] (32^3 x 64),
             timed alone with rotating buffer sets larger than L2, as algorithmic GB/s against the measured HBM peak, with the
             ALU fraction against an FP32 FMA peak measured in the same run ("report both fractions")
  rooflines = the same for N = 12 and 16, kernel B, configs[4] (64^3 x 128, N = 4, 12-real links) and the int16 kernels of configs[3]
  dslash_sweep = the configs[2] sweep over N_rhs in {1, 2, 4, 8, 16} (the paper's batching claim)
  cpu_baseline = the fp64 oracle on the host cores, bounded sample.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload cfg3|cfg1] [--no-extras]
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
sys.path.insert(0, ROOT)

from paper_2510_26313_b200 import inputs  # noqa: E402

L2_BYTES = 126e6
FLOP_A, FLOP_B, FLOP_HOP = 1824.0, 1872.0, 1320.0      # per output site per RHS (BASELINE.json north_star)


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured", float(d.get("sm_max_mhz", 1965.0))
    return 6650.0, "fallback", 1965.0


def bytes_per_site_rhs(kind: str, prec: str, nrhs: int, recon: int) -> float:
    """Compulsory (algorithmic) bytes per output site per RHS: every input site read once, output written once,
    8 links + 72 clover reals shared by the batch."""
    s = {"fp64": 8.0, "fp32": 4.0, "half": 2.0}[prec]
    g = 8.0 if prec == "fp64" else 4.0
    spinor = 24 * s + (4.0 if prec == "half" else 0.0)
    per_batch = 8 * recon * g + (0.0 if kind == "hop" else 72 * g)      # "probe" moves kernel A's bytes
    streams = 3 if kind == "B" else 2
    return streams * spinor + per_batch / nrhs


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, device: int):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(device), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits", "-lms", "100"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush(); self.f.seek(0)
        sm, mx, power, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            v = [q.strip() for q in line.split(",")]
            if len(v) < 7:
                continue
            try:
                sm.append(float(v[0])); mx.append(float(v[1])); power.append(float(v[2]))
            except ValueError:
                continue
            for n, q in zip(names, v[3:7]):
                if q.lower().startswith("active"):
                    reasons.add(n)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), power_w_max=float(max(power)), reasons=sorted(reasons), samples=len(sm))
        return out


# ------------------------------------------------------------------------------------------------ operator timing
def time_dslash(ctx, B, kind: str, prec: str, nrhs: int, recon: int, iters: int = 20, warmup: int = 3):
    """Average device time of one single-parity stencil launch (kernel A, kernel B or the bare hop), native layout,
    rotating buffer sets so that no launch starts with its operands in L2.  Returns a dict of seconds / GB/s / GFLOP/s."""
    import torch
    # fresh device allocations for every measurement: the same kernel on buffers carved out of the torch caching
    # allocator's older segments measured up to 8 % slower (placement-dependent), which made the sweep order matter
    torch.cuda.empty_cache()
    P = B.PREC[prec]
    pbytes = ctx.native_bytes(nrhs, P, True)
    per_set = pbytes * (3 if kind == "B" else 2)
    nsets = max(3, int(np.ceil(2.5 * L2_BYTES / per_set)) + 1)
    nsets = min(nsets, 64)
    sets = []
    for i in range(nsets):
        bufs = [ctx.native_empty(nrhs, P, True) for _ in range(3 if kind == "B" else 2)]
        for j, b in enumerate(bufs[1:]):
            ctx.fill_spinor_random(b, nrhs, P, 7000 + 10 * i + j, parity_only=True, parity=(0 if (kind == "B" and j == 0) else (0 if kind != "B" else 1)))
        sets.append(bufs)
    op = {"A": B.LQ_OP_KERNEL_A, "B": B.LQ_OP_KERNEL_B, "hop": B.LQ_OP_HOP_OE, "probe": B.LQ_OP_PROBE_LOADS}[kind]

    def launch(i):
        s = sets[i % nsets]
        if kind == "B":
            ctx.apply_native(op, s[0], s[1], nrhs, P, in2=s[2])
        else:
            ctx.apply_native(op, s[0], s[1], nrhs, P)

    for i in range(warmup):
        launch(i)
    ctx.stream.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(ctx.stream)
    for i in range(iters):
        launch(warmup + i)
    e1.record(ctx.stream)
    e1.synchronize()
    sec = e0.elapsed_time(e1) * 1e-3 / iters
    Vh = ctx.V // 2
    bps = bytes_per_site_rhs(kind, prec, nrhs, recon)
    flop = {"A": FLOP_A, "B": FLOP_B, "hop": FLOP_HOP, "probe": 0.0}[kind]
    del sets
    return dict(kind=kind, prec=prec, nrhs=nrhs, recon=recon, seconds=sec, bytes_per_site_rhs=bps,
                gbs=bps * Vh * nrhs / sec * 1e-9, gflops=flop * Vh * nrhs / sec * 1e-9, nsets=nsets)


def ncu_traffic(lattice, r):
    """DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum) of this kernel from the committed ncu --set full
    capture, if one exists for this lattice / kernel / batch (profiles/traffic.json, written by hand from the ncu report)."""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    if not os.path.exists(p):
        return None
    with open(p) as f:
        d = json.load(f)
    return d.get("%s:%s:%s:%d" % (lattice, r["kind"], r["prec"], r["nrhs"]))


def time_laplacian(ctx, B, nvec, prec="fp32", iters=20, warmup=3):
    """Batched 3-d covariant Laplacian on native colour-vector fields, rotating buffer sets.
    Algorithmic bytes per site per vector: 6 reals in + 6 reals out + 3 links of 18 reals shared by the batch."""
    import torch
    torch.cuda.empty_cache()
    P = B.PREC[prec]
    s = 8.0 if prec == "fp64" else 4.0
    nb = int(ctx.lib.lq_cv_native_bytes(ctx.h, nvec, P))
    nsets = min(64, max(3, int(np.ceil(2.5 * L2_BYTES / (2 * nb))) + 1))
    sets = []
    for i in range(nsets):
        a, b = ctx.cv_native_empty(nvec, P), ctx.cv_native_empty(nvec, P)
        ctx.cv_fill_random(b, nvec, P, 9000 + i)
        sets.append((a, b))
    for i in range(warmup):
        ctx.laplacian_native(sets[i % nsets][0], sets[i % nsets][1], nvec, P)
    ctx.stream.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(ctx.stream)
    for i in range(iters):
        ctx.laplacian_native(sets[(warmup + i) % nsets][0], sets[(warmup + i) % nsets][1], nvec, P)
    e1.record(ctx.stream)
    e1.synchronize()
    sec = e0.elapsed_time(e1) * 1e-3 / iters
    bps = 12 * s + 3 * 18 * s / nvec
    del sets
    return {"nvec": nvec, "prec": prec, "us": round(sec * 1e6, 1), "bytes_per_site_vec": bps, "gbs": round(bps * ctx.V * nvec / sec * 1e-9, 1),
            "gflops": round(6 * 72.0 * ctx.V * nvec / sec * 1e-9, 1)}


# FP32 instruction slots (one FMA, multiply or add each) per output site per RHS when every complex product is written as fused
# multiply-adds: hop 8 x (12 project + 72 SU(3) + 24 accumulate) = 864, clover 2 x 6 x 22 = 264
FP_SLOTS = {"A": 1128.0, "B": 1128.0, "hop": 864.0, "probe": 0.0}


def roofline_entry(r, peak, peak_src, traffic=None, fma=None, lattice=None):
    """HBM fraction (algorithmic bytes / CUDA-event time / measured copy bandwidth) and, when the FP32 FMA peak was measured in
    this run, the ALU fractions: `alu_frac` = counted flops (1320 + 504 per site per RHS) / peak, `alu_issue_frac` = FP32
    instruction slots x 2 / peak (what the FMA pipes must issue: adds and multiplies occupy a slot like an FMA)."""
    e = {"bound": "hbm", "kernel": "dslash_kernel<%s,N=%d,recon=%d,form=%s>" % (r["prec"], r["nrhs"], r["recon"], r["kind"]),
         "achieved": round(r["gbs"], 1), "peak": peak, "peak_source": peak_src, "unit": "GB/s",
         "frac": round(r["gbs"] / peak, 4), "frac_of_8TBs": round(r["gbs"] / 8000.0, 4), "traffic": traffic,
         "us_per_launch": round(r["seconds"] * 1e6, 2), "gflops": round(r["gflops"], 1),
         "algorithmic_bytes_per_site_rhs": r["bytes_per_site_rhs"]}
    if lattice:
        e["lattice"] = lattice
    if fma:
        flop = {"A": FLOP_A, "B": FLOP_B, "hop": FLOP_HOP, "probe": 1.0}[r["kind"]]
        e["alu_peak_tflops"] = fma["scalar_ffma"]
        e["alu_frac"] = round(r["gflops"] * 1e-3 / fma["scalar_ffma"], 4)
        e["alu_issue_frac"] = round(r["gflops"] * 1e-3 * (2.0 * FP_SLOTS[r["kind"]] / flop) / fma["scalar_ffma"], 4)
        e["alu_issue_frac_of_ffma2_shared"] = round(r["gflops"] * 1e-3 * (2.0 * FP_SLOTS[r["kind"]] / flop) / fma["ffma2_shared_operand"], 4)
    return e


def measure_fma_peak(ctx):
    """FP32 FMA peak through the C ABI (lq_fma_peak): scalar FFMA, packed FFMA2 with three distinct operands, packed FFMA2 with
    one operand shared by 4 consecutive instructions (the stencil's pattern).  TFLOP/s, 2 flops per FMA lane."""
    return {"scalar_ffma": round(ctx.fma_peak(0, 150.0), 2), "ffma2_distinct_operands": round(ctx.fma_peak(1, 150.0), 2),
            "ffma2_shared_operand": round(ctx.fma_peak(2, 150.0), 2), "ffma2_register_scalar_operand": round(ctx.fma_peak(3, 150.0), 2),
            "unit": "TFLOP/s", "nominal_1965MHz": 74.4,
            "how": "register-only FMA loops, 16 chains per thread, 8 CTAs x 256 threads per SM, ~150 ms each (csrc/fmapeak.cu)"}


# ------------------------------------------------------------------------------------------------ workloads
SOLVER_WORKLOADS = {
    "cfg1": dict(cfg=1, inner="fp32", delta=1e-4, desc="configs[1]: 16^3x32, 8 RHS LapH time/spin-diluted, fp32 inner CG + fp64 defect correction, tol 1e-8"),
    "cfg3": dict(cfg=3, inner="half", delta=1e-3, desc="configs[3]: 48^3x96, 12 RHS LapH-diluted, int16+norm inner CG, fp32 clover, fp64 outer, tol 1e-9"),
}


def solve_kwargs(B, wl, c, algorithm="cg", check_every=4, delta=0.0, use_graph=True):
    """The launch configuration of the timed step (tests/test_gpu_fullsize.py checks the configs[3] solve with exactly these)."""
    return dict(tol=c["tol"], inner_prec=B.PREC[wl["inner"]], delta=delta or wl["delta"], check_every=2 if algorithm == "bicgstab" else check_every,
                use_graph=use_graph, algorithm=1 if algorithm == "bicgstab" else 0)


def make_sources_host(cfg, out=None):
    c = inputs.CONFIGS[cfg]
    return inputs.laph_sources(c["dims"], c["nrhs"], c["n_t"], c["source_seed"], out=out)


ORACLE_SAMPLE_DIMS = (16, 16, 16, 32)


def oracle_sample_solve(cfg_id: int, k: int = 0):
    """One bounded sample of the workload for the CPU oracle: RHS k solved by oracle.solve_eo (fp64 CGNR, true residual
    recomputed every iteration) on the workload's lattice if that is 16^3 x 32 or smaller, else on a 16^3 x 32 lattice of the
    same recipe (links, kappa, c_sw, source structure, tolerance): a full 48^3 x 96 oracle solve takes hours.  Returns
    (seconds, iterations, lattice, volume ratio workload / sample)."""
    import oracle
    c = inputs.CONFIGS[cfg_id]
    dims = c["dims"] if inputs.volume(c["dims"]) <= inputs.volume(ORACLE_SAMPLE_DIMS) else ORACLE_SAMPLE_DIMS
    key = (cfg_id, dims)
    if oracle_sample_solve.cache.get("key") != key:
        U = inputs.make_links(dims, c["gauge_seed"], c["eps"])
        A = oracle.clover(dims, U, c["kappa"], c["csw"])
        oracle_sample_solve.cache = {"key": key, "U": U, "A": A, "Ainv": oracle.clover_inverse(A),
                                     "b": inputs.laph_sources(dims, 4, c["n_t"], c["source_seed"])}
    q = oracle_sample_solve.cache
    t0 = time.perf_counter()
    _, it, _ = oracle.solve_eo(dims, q["U"], q["A"], q["Ainv"], c["kappa"], q["b"][k % 4], c["tol"])
    return time.perf_counter() - t0, it, dims, inputs.volume(c["dims"]) / inputs.volume(dims)


oracle_sample_solve.cache = {}


def cpu_baseline(cfg_id: int, budget_s: float = 25.0):
    """The oracle as it stands on the host cores: single-RHS even-odd CG solves (bounded sample, see oracle_sample_solve), as
    many as fit the time budget (at least one).  `value` is seconds per RHS of the workload: the sample time scaled by the
    volume ratio when the sample lattice is smaller than the workload's (CG cost per iteration is linear in the volume; the
    iteration count of these well-conditioned random links does not grow with it)."""
    import oracle
    t0 = time.perf_counter()
    secs, its = [], []
    dims, ratio = None, 1.0
    while len(secs) < 4:
        dt, it, dims, ratio = oracle_sample_solve(cfg_id, len(secs))
        secs.append(dt); its.append(it)
        if time.perf_counter() - t0 > budget_s * 0.5:
            break
    return {"value": float(np.mean(secs)) * ratio, "unit": "s/RHS", "cores": oracle.num_threads(), "kind": "oracle",
            "measured_seconds_per_sample_solve": float(np.mean(secs)), "volume_scale": ratio,
            "sample": "%d single-RHS oracle.solve_eo solves (fp64 CGNR, true residual recomputed every iteration) on %s, tol %g, iterations %s%s"
                      % (len(secs), "x".join(map(str, dims)), inputs.CONFIGS[cfg_id]["tol"], its,
                         "" if ratio == 1.0 else "; value = measured seconds x %.0f (volume of the workload / volume of the sample lattice)" % ratio)}


def cpu_dslash_baseline():
    """The oracle's full operator M and its site-local kernel A on the host cores, ns per site per RHS (SURVEY 8(d) CPU
    baseline; lattice capped at 16^3x32: per-site cost is volume-independent beyond cache)."""
    import oracle
    c = inputs.CONFIGS[1]
    dims = c["dims"]
    V = inputs.volume(dims)
    U = inputs.make_links(dims, c["gauge_seed"], c["eps"])
    A = oracle.clover(dims, U, c["kappa"], c["csw"])
    psi = inputs.gaussian_spinors(dims, 1, 4242)[0]
    oracle.M(dims, U, A, c["kappa"], psi)
    t0 = time.perf_counter(); n = 0
    while time.perf_counter() - t0 < 3.0:
        oracle.M(dims, U, A, c["kappa"], psi); n += 1
    dt_M = (time.perf_counter() - t0) / n
    rng = np.random.default_rng(5)
    sites = np.stack([rng.integers(0, d, 20000) for d in dims], axis=1)
    sites = sites[(sites.sum(axis=1) % 2) == 1].astype(np.int32)
    t0 = time.perf_counter()
    oracle.site_eval(dims, 1, sites, c["kappa"], c["csw"], U=U, psi=psi.reshape(-1, 12))
    dt_A = time.perf_counter() - t0
    return {"kind": "oracle", "cores": oracle.num_threads(), "lattice": "x".join(map(str, dims)),
            "full_M_ns_per_site_rhs": round(dt_M / V * 1e9, 1), "full_M_gflops_1824": round(1824.0 * V / dt_M * 1e-9, 2),
            "site_local_kernel_A_ns_per_site_rhs": round(dt_A / len(sites) * 1e9, 1),
            "note": "kernel A by the site-local evaluator rebuilds F_mu_nu, A and A^-1 at every site (that is its definition), so it is not comparable with a stored-clover kernel"}


def time_eigensolve(B, device):
    """Time-batched Lanczos on the configs[1] lattice: lowest 16 / 64 / 128 eigenpairs of -Laplacian on each of
    the 32 slices (Chebyshev cut just above the wanted part of the spectrum)."""
    c = inputs.CONFIGS[1]
    ctx = B.Context(c["dims"], device=device)
    ctx.fill_gauge_random(c["gauge_seed"], c["eps"], recon=18)
    out = {"lattice": "x".join(map(str, c["dims"])), "cases": []}
    # (n_ev, Krylov space, cut, filter degree): the 128-eigenpair case from a sweep over m in 176..288 and degree 16 / 24 / 32
    for n_ev, m, cut, deg in ((16, 48, 0.5, 24), (64, 144, 1.0, 24), (128, 224, 1.6, 32)):
        kw = dict(n_ev=n_ev, m=m, cheb_degree=deg, cheb_a=cut, cheb_b=12.5, tol=1e-9, max_restarts=50, want_vectors=False)
        ctx.laph_eigensolve(**kw)
        ev, _, info = ctx.laph_eigensolve(**kw)
        out["cases"].append({"n_ev": n_ev, "krylov": m, "cheb_degree": deg, "seconds": round(info["seconds"], 4), "seconds_ritz": round(info["seconds_ritz"], 4), "seconds_ortho": round(info["seconds_ortho"], 4), "restarts": info["restarts"],
                             "laplacian_applies": info["lap_applies"], "converged": info["converged"],
                             "max_true_residual": info["max_true_residual"], "eigenvalue_range": [float(ev.min()), float(ev.max())]})
    ctx.close()
    return out


def time_projection(B, device, peak, shapes=((32, 8), (128, 32)), precs=("f64_fma", "tcgen05_3xtf32"), iters=10):
    """Eigenvector projection on the configs[1] lattice: n_ev eigenvector fields x n_sol solutions, device
    arrays; fp64 FMA kernel and the tcgen05 3xTF32 kernel."""
    import torch
    c = inputs.CONFIGS[1]
    Lx, Ly, Lz, Lt = c["dims"]
    ctx = B.Context(c["dims"], device=device)
    out = {"lattice": "x".join(map(str, c["dims"])), "shapes": [],
           "note": "wall clock around the synchronous C-ABI call (device arrays; includes its scratch allocation and the final device "
                   "synchronisation); compulsory bytes = the fp64 fields read once"}
    g = torch.Generator(device="cuda").manual_seed(7)
    for n_ev, n_sol in shapes:
        vc = torch.view_as_complex(torch.randn((n_ev, Lt, Lz, Ly, Lx, 3, 2), generator=g, device="cuda", dtype=torch.float64))
        xc = torch.view_as_complex(torch.randn((n_sol, Lt, Lz, Ly, Lx, 4, 3, 2), generator=g, device="cuda", dtype=torch.float64))
        nbytes = (vc.numel() + xc.numel()) * 16
        flops = 8.0 * n_ev * 4 * n_sol * 3 * Lx * Ly * Lz * Lt
        e = {"n_ev": n_ev, "n_sol": n_sol, "input_mb": round(nbytes / 1e6, 1)}
        ref = None
        for name in precs:
            prec = B.LQ_FP64 if name == "f64_fma" else B.LQ_FP32
            for _ in range(3):
                got = ctx.project(vc, xc, prec)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            for _ in range(iters):
                ctx.project(vc, xc, prec)
            torch.cuda.synchronize()
            sec = (time.perf_counter() - t0) / iters
            e[name] = {"us": round(sec * 1e6, 1), "compulsory_gbs": round(nbytes / sec * 1e-9, 1), "frac_measured_hbm": round(nbytes / sec * 1e-9 / peak, 4),
                       "gflops": round(flops / sec * 1e-9, 1)}
            if name == "f64_fma":
                ref = got
            elif ref is not None:
                e[name]["max_rel_diff_vs_f64"] = float((got - ref).abs().max() / ref.abs().max())
        if "tcgen05_3xtf32" in precs:      # the same kernel fed with complex64 fields (lq_project_c64): half the compulsory bytes
            v32, x32 = vc.to(torch.complex64), xc.to(torch.complex64)
            for _ in range(3):
                got = ctx.project_c64(v32, x32)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            for _ in range(iters):
                ctx.project_c64(v32, x32)
            torch.cuda.synchronize()
            sec = (time.perf_counter() - t0) / iters
            e["tcgen05_3xtf32_c64_fields"] = {"us": round(sec * 1e6, 1), "compulsory_gbs": round(nbytes / 2 / sec * 1e-9, 1), "frac_measured_hbm": round(nbytes / 2 / sec * 1e-9 / peak, 4),
                                              "gflops": round(flops / sec * 1e-9, 1)}
            if ref is not None:
                e["tcgen05_3xtf32_c64_fields"]["max_rel_diff_vs_f64_of_unrounded_fields"] = float((got - ref).abs().max() / ref.abs().max())
            del v32, x32
        out["shapes"].append(e)
        del vc, xc
    ctx.close()
    return out


def time_multigrid(B, device):
    """Two-level adaptive multigrid on the configs[1] lattice, 8 Gaussian right-hand sides, next to the
    library's CG on the same system: once on the configs[1] links (well conditioned) and once on smooth links with periodic
    boundaries at kappa near critical, where the CG iteration count grows."""
    import torch
    c = inputs.CONFIGS[1]
    Lx, Ly, Lz, Lt = c["dims"]
    out = {"lattice": "x".join(map(str, c["dims"])), "nrhs": 8, "tol": 1e-8, "hierarchy": "4^4 aggregates x 2 chiralities x 24 vectors, setup_tol 1e-4, one refinement pass",
           "cycle": "3 + 3 even-odd minimal-residual steps, 8 coarse GCR iterations, FGCR(8) in fp32 inside fp64 defect correction", "cases": []}
    g = torch.Generator(device="cuda").manual_seed(5)
    b = torch.view_as_complex(torch.randn((8, Lt, Lz, Ly, Lx, 4, 3, 2), generator=g, device="cuda", dtype=torch.float64))
    for name, eps, kappa, csw, t_bc in (("configs[1] links", c["eps"], c["kappa"], c["csw"], -1), ("smooth links, periodic, near-critical kappa", 0.05, 0.1252, 1.0, 1)):
        ctx = B.Context(c["dims"], device=device)
        ctx.fill_gauge_random(c["gauge_seed"], eps, recon=18, t_bc=t_bc)
        ctx.build_clover(kappa, csw)
        kw = dict(tol=1e-8, use_graph=True, max_inner=20000, max_outer=100)
        ctx.solve(b, **kw)
        xc, ci = ctx.solve(b, **kw)
        ms = ctx.mg_setup((4, 4, 4, 4), 24, nu_pre=3, nu_post=3, coarse_iters=8, restart=8, setup_tol=1e-4, seed=7, smoother=B.LQ_MG_SMOOTH_EO, refine=1)
        ctx.mg_solve(b, tol=1e-8, max_iter=300)
        x, si = ctx.mg_solve(b, tol=1e-8, max_iter=300)
        out["cases"].append({"links": name, "eps": eps, "kappa": kappa, "csw": csw, "t_bc": t_bc,
                             "cg": {"seconds": round(ci["seconds"], 4), "inner_iters": ci["inner_iters"], "converged": ci["converged"]},
                             "mg": {"seconds": round(si["seconds"], 4), "cycles": si["iters"], "m_applies": si["m_applies"], "converged": si["converged"],
                                    "true_rel_residual_max": max(si["true_rel_residual"]),
                                    "setup_seconds": round(ms["seconds_vectors"] + ms["seconds_prolongator"] + ms["seconds_coarse_op"], 4),
                                    "probes": ms["probes"], "hierarchy_mb": round(ms["bytes"] / 1e6, 1)},
                             "rel_diff_mg_vs_cg": float(torch.linalg.vector_norm(x - xc) / torch.linalg.vector_norm(xc))})
        ctx.close()
    return out


def dslash_report(B, device, peak, peak_src, quick=False):
    """The Dslash half of the metric.  configs[2] (32^3 x 64, fp32, 18-real links): kernel A / kernel B / bare hop over
    N_rhs in {1, 2, 4, 8, 12, 16}; configs[4] (64^3 x 128, N = 4, 12-real links); the int16+norm kernels of configs[3] come from
    the solver context (caller).  Returns (headline roofline entry, list of further roofline entries, sweep table, fma peaks)."""
    import torch
    rooflines, sweep, head, fma = [], [], None, None
    for cfg_id in (2, 4):
        c = inputs.CONFIGS[cfg_id]
        lat = "x".join(map(str, c["dims"]))
        ctx = B.Context(c["dims"], device=device)
        if fma is None:
            fma = measure_fma_peak(ctx)
        ctx.fill_gauge_random(c["gauge_seed"], c["eps"], recon=c["recon"])
        ctx.build_clover(c["kappa"], c["csw"])
        ns = (1, 2, 4, 8, 12, 16, 32) if cfg_id == 2 else (c["nrhs"],)
        for n in ns:
            for kind in ("A", "B", "hop"):
                if quick and (kind == "hop" or n in (1, 2)):
                    continue
                r = time_dslash(ctx, B, kind, "fp32", n, c["recon"], iters=20)
                e = roofline_entry(r, peak, peak_src, ncu_traffic(lat, r), fma, lat)
                sweep.append({"lattice": lat, "kernel": kind, "nrhs": n, "recon": c["recon"], "us": e["us_per_launch"], "gbs": e["achieved"], "gflops": e["gflops"],
                              "frac_measured_hbm": e["frac"], "frac_8TBs": e["frac_of_8TBs"], "alu_frac": e["alu_frac"], "alu_issue_frac": e["alu_issue_frac"]})
                if cfg_id == 2 and kind == "A" and n == 8:
                    head = e
                elif kind != "hop" and (n >= 8 or cfg_id == 4):
                    rooflines.append(e)
        if cfg_id == 2 and not quick:
            lap = []
            for n in (1, 4, 8, 16):
                r = time_laplacian(ctx, B, n)
                r["frac_measured_hbm"] = round(r["gbs"] / peak, 4)
                lap.append(r)
            sweep.append({"laplacian_32x32x32x64_fp32": lap})
        ctx.close()
        torch.cuda.empty_cache()
    return head, rooflines, sweep, fma


# ------------------------------------------------------------------------------------------------ reference arm
def run_reference(args, rank, world):
    """`--impl reference`: this tier has no reference implementation to install; the arm times the CPU oracle as it stands
    on the host cores (rank 0 only).  Each step is ONE bounded sample of the workload (oracle_sample_solve: a single-RHS
    oracle CG solve, on a 16^3 x 32 lattice of the same recipe when the workload's lattice is larger); `ms_per_step` is the
    measured wall time of such a step, so steps x ms_per_step is what this process really spent; `value` (seconds per RHS of
    the workload) is that time scaled by the volume ratio and is named as an extrapolation when the ratio is not 1."""
    if rank != 0:
        return
    import oracle
    wl = SOLVER_WORKLOADS[args.workload]
    c = inputs.CONFIGS[wl["cfg"]]
    for i in range(args.warmup):
        oracle_sample_solve(wl["cfg"], i)
    secs, its, dims, ratio = [], [], None, 1.0
    for i in range(max(1, args.steps)):
        dt, it, dims, ratio = oracle_sample_solve(wl["cfg"], i)
        secs.append(dt); its.append(it)
    per = float(np.mean(secs))
    v = per * ratio
    sample = ("each step = 1 single-RHS oracle.solve_eo solve (fp64 CGNR) on %s, tol %g; iterations %s" % ("x".join(map(str, dims)), c["tol"], its))
    line = {"impl": "reference", "metric": "batched CG sec/RHS", "value": v, "unit": "s/RHS", "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": per * 1e3, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": wl["desc"], "note": "CPU oracle; a step is a bounded sample of the workload: " + sample},
            "value_is_extrapolated": ratio != 1.0,
            "extrapolation": None if ratio == 1.0 else {"measured_seconds_per_step": per, "rhs_per_step": 1, "sample_lattice": "x".join(map(str, dims)),
                                                        "volume_scale": ratio, "rule": "value = measured seconds per step x volume_scale (cost per CG iteration is linear in the volume)"},
            "cpu_baseline": {"value": v, "unit": "s/RHS", "cores": oracle.num_threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": v, "unit": "s/RHS", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------------ multi-rank plumbing
def max_over_ranks(values, device=None):
    """Replicas-only scaling: every rank runs the same step on its own RHS batch; the job's time is the
    slowest rank's.  Works on whatever torch.distributed backend is initialised (nccl on GPUs, gloo in the CPU tests)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return [float(v) for v in values]
    t = torch.tensor(list(values), dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t]


def whole_job_seconds_per_rhs(seconds_total, steps, nrhs_per_rank, world):
    """metric value: seconds per RHS of the whole job = max-over-ranks step time / RHS solved by all ranks per step."""
    return seconds_total / steps / (nrhs_per_rank * world)


def rank_gauge_seed(base_seed, rank):
    """Each replica works on its own gauge configuration (independent tasks)."""
    return base_seed + rank


# ------------------------------------------------------------------------------------------------ single-operator mode
def run_op(args, B, device):
    f = args.op.split(":")
    cfg_id, kind, prec, n = int(f[0].replace("cfg", "")), f[1], f[2], int(f[3])
    variant = int(f[4]) if len(f) > 4 else 0
    rpt = int(f[5]) if len(f) > 5 else 0
    pfd = int(f[6]) if len(f) > 6 else -1
    c = inputs.CONFIGS[cfg_id]
    peak, peak_src, _ = measured_peaks()
    if kind == "proj":     # eigenvector projection: 128 eigenvectors x N solutions on the configs[1] lattice
        sampler = ClockSampler(device)
        r = time_projection(B, device, peak, shapes=((128, n),), precs=("tcgen05_3xtf32",) if prec == "fp32" else ("f64_fma",), iters=args.op_iters)
        r.update({"op": args.op, "clocks": sampler.stop()})
        print(json.dumps(r))
        return
    if kind == "mg":       # two-level multigrid: setup + ONE solve of N right-hand sides, near-critical smooth links
        import torch
        Lx, Ly, Lz, Lt = c["dims"]
        ctx = B.Context(c["dims"], device=device)
        ctx.fill_gauge_random(c["gauge_seed"], 0.05, recon=18, t_bc=1)
        ctx.build_clover(0.1252, 1.0)
        g = torch.Generator(device="cuda").manual_seed(5)
        b = torch.view_as_complex(torch.randn((n, Lt, Lz, Ly, Lx, 4, 3, 2), generator=g, device="cuda", dtype=torch.float64))
        ms = ctx.mg_setup((4, 4, 4, 4), 24, nu_pre=3, nu_post=3, coarse_iters=8, restart=8, setup_tol=1e-4, seed=7, smoother=B.LQ_MG_SMOOTH_EO, refine=1)
        x, si = ctx.mg_solve(b, tol=1e-8, max_iter=args.op_iters)
        ctx.close()
        print(json.dumps({"op": args.op, "lattice": "x".join(map(str, c["dims"])), "setup": ms, "solve": si}))
        return
    ctx = B.Context(c["dims"], device=device)
    ctx.fill_gauge_random(c["gauge_seed"], c["eps"], recon=c["recon"])
    ctx.build_clover(c["kappa"], c["csw"])
    if variant or rpt or pfd >= 0:
        ctx.set_tuning(variant, rpt, pfd)
    sampler = ClockSampler(device)
    if kind == "lap":      # batched 3-d covariant Laplacian
        r = time_laplacian(ctx, B, n, prec, iters=args.op_iters, warmup=max(args.warmup, 3))
        clocks = sampler.stop()
        ctx.close()
        r.update({"op": args.op, "lattice": "x".join(map(str, c["dims"])), "frac_measured_hbm": round(r["gbs"] / peak, 4), "clocks": clocks})
        print(json.dumps(r))
        return
    r = time_dslash(ctx, B, kind, prec, n, c["recon"], iters=args.op_iters, warmup=max(args.warmup, 3))
    clocks = sampler.stop()
    ctx.close()
    e = roofline_entry(r, peak, peak_src, ncu_traffic("x".join(map(str, c["dims"])), r))
    e.update({"op": args.op, "lattice": "x".join(map(str, c["dims"])), "iters": args.op_iters, "clocks": clocks})
    print(json.dumps(e))


# ------------------------------------------------------------------------------------------------ main
def pinned_complex(shape):
    """Pinned host array (torch owns the memory; numpy view for filling)."""
    import torch
    try:
        t = torch.empty(tuple(shape), dtype=torch.complex128, pin_memory=True)
        pinned = True
    except Exception:
        t = torch.empty(tuple(shape), dtype=torch.complex128)
        pinned = False
    return t, pinned


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg3", choices=sorted(SOLVER_WORKLOADS))
    ap.add_argument("--no-extras", action="store_true", help="skip the extras (configs[1] solve, BiCGStab variant, Lanczos, projection, multigrid, CPU Dslash baseline)")
    ap.add_argument("--no-dslash", action="store_true", help="skip the Dslash report (roofline of the configs[2]/[4] kernels) as well")
    ap.add_argument("--no-graph", action="store_true")
    ap.add_argument("--check-every", type=int, default=4, help="inner iterations between convergence tests")
    ap.add_argument("--delta", type=float, default=0.0, help="inner CG reduction per cycle (0 = the workload default)")
    ap.add_argument("--algorithm", choices=("cg", "bicgstab"), default="cg", help="inner solver of the timed step (default cg = the metric of BASELINE.json; bicgstab = the solver variant)")
    ap.add_argument("--op", default=None, metavar="CFG:KIND:PREC:N",
                    help="time ONE stencil kernel only, e.g. cfg2:A:fp32:8 (lattice and links of configs[CFG]; KIND A|B|hop|probe|lap|proj; "
                         "PREC fp64|fp32|half); optional :variant:rpt:pfd tuning suffix.  Prints its own JSON line (used for ncu captures)")
    ap.add_argument("--op-iters", type=int, default=20)
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1")); local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        return run_reference(args, rank, world)

    import torch
    import torch.distributed as dist
    from paper_2510_26313_b200 import binding as B
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if args.op:
        return run_op(args, B, local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    args.warmup = max(args.warmup, 3)

    wl = SOLVER_WORKLOADS[args.workload]
    c = inputs.CONFIGS[wl["cfg"]]
    dims, nrhs = c["dims"], c["nrhs"]
    Lx, Ly, Lz, Lt = dims
    peak, peak_src, _ = measured_peaks()
    # ---- the Dslash half of the metric first (configs[2], configs[4]), on a GPU that the long solver steps have not yet heated
    # into the power cap: these kernels are timed alone, as MEASURED_PEAKS.json's copy bandwidth was
    head, rooflines, sweep, fma = (None, [], [], None)
    if not args.no_dslash and world == 1:
        head, rooflines, sweep, fma = dslash_report(B, local, peak, peak_src, quick=args.no_extras)
    ctx = B.Context(dims, device=local)
    ctx.fill_gauge_random(rank_gauge_seed(c["gauge_seed"], rank), c["eps"], recon=c["recon"])
    ctx.build_clover(c["kappa"], c["csw"])
    b_host, pinned = pinned_complex((nrhs, Lt, Lz, Ly, Lx, 4, 3))
    x_host, _ = pinned_complex((nrhs, Lt, Lz, Ly, Lx, 4, 3))
    make_sources_host(wl["cfg"], out=b_host.numpy())
    kw = solve_kwargs(B, wl, c, args.algorithm, args.check_every, args.delta, not args.no_graph)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident steps: the sources sit in HBM in the native layout before the timed region starts
    nb = ctx.pack(b_host, nrhs, B.LQ_FP64)
    nx = ctx.native_empty(nrhs, B.LQ_FP64)
    info = None
    for _ in range(args.warmup):
        _, info = ctx.solve(nb, x_out=nx, native=True, nrhs=nrhs, **kw)
    assert info["converged"], info
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    l0 = ctx.launches
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(ctx.stream)
    for _ in range(args.steps):
        _, info = ctx.solve(nb, x_out=nx, native=True, nrhs=nrhs, **kw)
    e1.record(ctx.stream)
    barrier()
    launches = ctx.launches - l0
    t_dev = e0.elapsed_time(e1) * 1e-3
    del nb, nx
    torch.cuda.empty_cache()
    # ---- end to end: host buffers in, host buffers out, through the C ABI (lq_solve stages them a few RHS at a time)
    ctx.solve(b_host, x_out=x_host, **kw)
    barrier()
    w0 = time.perf_counter()
    for _ in range(args.steps):
        ctx.solve(b_host, x_out=x_host, **kw)
    torch.cuda.synchronize()
    t_e2e = time.perf_counter() - w0
    clocks = sampler.stop() if sampler else None
    t_dev, t_e2e = max_over_ranks([t_dev, t_e2e], device="cuda")
    h2d, d2h = b_host.numel() * 16, x_host.numel() * 16
    del x_host
    inner = wl["inner"]
    variant, variant_hl = None, None
    if not args.no_extras and world == 1 and args.algorithm == "cg":
        # solver variant, same sources, device resident: batched BiCGStab instead of CGNR (not the headline metric)
        kb = solve_kwargs(B, wl, c, "bicgstab", use_graph=not args.no_graph)
        nb = ctx.pack(b_host, nrhs, B.LQ_FP64)
        nx = ctx.native_empty(nrhs, B.LQ_FP64)
        ctx.solve(nb, x_out=nx, native=True, nrhs=nrhs, **kb)
        _, ib = ctx.solve(nb, x_out=nx, native=True, nrhs=nrhs, **kb)
        variant = {"algorithm": "batched BiCGStab on Mhat, complex per-RHS scalars, same defect correction", "seconds_per_rhs": ib["seconds"] / nrhs,
                   "ms_per_step": ib["seconds"] * 1e3, "inner_iters": ib["inner_iters"], "outer_cycles": ib["outer_cycles"],
                   "dslash_applies_per_step": ib["dslash_applies"], "true_rel_residual_max": max(ib["true_rel_residual"]), "converged": ib["converged"]}
        # solver variant: int16 fixed-point links in the half-storage kernels (reading #13), CG as in the headline step
        if inner == "half":
            ctx.set_half_links(True)
            ctx.solve(nb, x_out=nx, native=True, nrhs=nrhs, **kw)
            _, ih = ctx.solve(nb, x_out=nx, native=True, nrhs=nrhs, **kw)
            ctx.set_half_links(False)
            variant_hl = {"variant": "int16 links (36 instead of 72 bytes per link) in the int16+norm kernels", "seconds_per_rhs": ih["seconds"] / nrhs,
                          "ms_per_step": ih["seconds"] * 1e3, "inner_iters": ih["inner_iters"], "outer_cycles": ih["outer_cycles"],
                          "true_rel_residual_max": max(ih["true_rel_residual"]), "converged": ih["converged"]}
        del nb, nx
    del b_host
    torch.cuda.empty_cache()

    # ---- the kernels of this step alone, same lattice and batch (rotating buffers)
    inner = wl["inner"]
    fma0 = fma if fma is not None else (measure_fma_peak(ctx) if rank == 0 else None)
    rA = time_dslash(ctx, B, "A", inner, nrhs, c["recon"], iters=20)
    rB = time_dslash(ctx, B, "B", inner, nrhs, c["recon"], iters=20)
    lat = "x".join(map(str, dims))
    step_kernels = [roofline_entry(rA, peak, peak_src, ncu_traffic(lat, rA), fma0, lat), roofline_entry(rB, peak, peak_src, ncu_traffic(lat, rB), fma0, lat)]
    ctx.close()
    torch.cuda.empty_cache()
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    fma = fma0
    extras = {}
    if not args.no_extras and world == 1:
        extras["cpu_dslash_baseline"] = cpu_dslash_baseline()
        if variant is not None:
            extras["solver_variant_bicgstab"] = variant
        if variant_hl is not None:
            extras["solver_variant_int16_links"] = variant_hl
        extras["laph_eigensolve"] = time_eigensolve(B, local)
        extras["projection"] = time_projection(B, local, peak)
        extras["multigrid"] = time_multigrid(B, local)
    t_step = t_dev / args.steps
    line = {
        "metric": "batched CG sec/RHS", "value": whole_job_seconds_per_rhs(t_dev, args.steps, nrhs, world), "unit": "s/RHS", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": t_step * 1e3, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32" if inner == "fp32" else ("i16+f32" if inner == "half" else "f64"), "data": "synthetic",
        "config": {"workload": wl["desc"], "lattice": lat, "nrhs_per_gpu": nrhs, "parallelism": "replicas only (RHS-independent)",
                   "l2": "every vector of the iteration (%.0f MB) %s the 126 MB L2; the kernel timings rotate buffer sets larger than L2"
                         % (ctx.V // 2 * nrhs * (52 if inner == "half" else 96) / 1e6, "exceeds" if ctx.V // 2 * nrhs * 52 > 126e6 else "is comparable to"),
                   "cuda_graph": not args.no_graph, "algorithm": args.algorithm, "check_every": kw["check_every"], "delta": kw["delta"],
                   "kappa": c["kappa"], "csw": c["csw"], "tol": c["tol"], "links": "SU(3) projection of 1 + %.1f G, seed %d (device generator)" % (c["eps"], c["gauge_seed"])},
        "solver": {"converged": info["converged"], "outer_cycles": info["outer_cycles"], "inner_iters": info["inner_iters"],
                   "true_rel_residual_max": max(info["true_rel_residual"]), "dslash_applies_per_step": info["dslash_applies"],
                   "model_bytes_per_step": info["model_bytes"], "model_flops_per_step": info["model_flops"],
                   "model_gbs": round(info["model_bytes"] / t_step * 1e-9, 1), "model_frac_measured_hbm": round(info["model_bytes"] / t_step * 1e-9 / peak, 4),
                   "model_tflops": round(info["model_flops"] / t_step * 1e-12, 2)},
        "e2e": {"value": whole_job_seconds_per_rhs(t_e2e, args.steps, nrhs, world), "unit": "s/RHS", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "host_memory": "pinned" if pinned else "pageable"},
        "gpu_launches": int(launches),
        "clocks": clocks,
        # the Dslash half of the metric: fused kernel A, fp32, N_rhs = 8 on configs[2]; without the Dslash report the dominant kernel of the step
        "roofline": head if head is not None else step_kernels[1],
        "rooflines": step_kernels + rooflines,
        "fma_peak": fma,
        "dslash_sweep": sweep,
        "cpu_baseline": cpu_baseline(wl["cfg"]),
    }
    line.update(extras)
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

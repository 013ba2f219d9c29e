#!/usr/bin/env python
"""Benchmark of the COLA hot path on B200 (contract: see the task statement).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2] [--impl reference]

One STEP = one pass of the whole hot path over one source: a mixed-precision (fp32 inner, fp64 reliable
updates) even-odd CGNR solve of M x = b to |r| <= 1e-10 |b|, i.e. source preparation, ~2 Schur-operator
applications (4 fused dslash+clover kernels) and 2 fused BLAS-1 kernels per iteration, reliable updates in
fp64, reconstruction of the odd sites and the fp64 true residual -- SURVEY.md 8(a) H3-H12.  The gauge upload
+ clover build/inversion (H0-H2) is setup and is timed separately ("setup_s").

metric  = Dirac-operator GFLOP/s sustained over the solve, counted flops (1320/site hopping term, 504/site
          clover, 48/site xpay) / device time, whole job over all ranks (BASELINE.json "metric").
e2e     = the same through cola_cg_solve_host: b in pinned HOST memory, x returned to pinned HOST memory.
roofline= the dominant kernel (fused dslash + clover + xpay, fp32 with 12-real links) timed alone with CUDA
          events: algorithmic bytes per launch / average launch time, against MEASURED_PEAKS.json hbm_gbs;
          roofline.in_solve = the same kernel inside a solve (CUDA-event pair around each of its launches in one extra
          step; cola_profile_kernel).
extras  : (N = 1 only) solve_h16 / solve_r8 = the same step with 16-bit links + fp16 clover (mixed = 2) or 8-real links
          (mixed = 3) in the inner iteration; solve_bicgstab = the same step by BiCGStab on the Schur
          system and low_modes = the lowest modes of S^+S + the deflated step (NEXT-4); batched (config 3) = its 12 sources
          as one multi-rhs solve, CGNR and BiCGStab (NEXT-1); operators = every operator x {fp32 x12, fp64 x18, 16-bit,
          8-real, fp32 x12 with the 72-real A, fp32 x18 on a second context}, each the median of 10 bursts;
          compression_x12_vs_x18 = the 12-real and 18-real fp32 operators interleaved (what the compression buys).  --operators-only [--nrhs N] [--lattice X,Y,Z,T] [--staging 1] is the short
          launch sequence the ncu captures and the volume sweep in profiles/ come from; --ab-formats the interleaved
          comparison of the storage formats.
N > 1   : replicas only (the path has no inter-GPU exchange): every rank solves its own
          source on its own GPU; value = all ranks' flops / max-over-ranks time ("weak").
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import torch  # noqa: E402

from paper_2302_00850_b200 import inputs  # noqa: E402

# algorithmic bytes per output site, fp32 with 12-real links; fp64 x18 in the second column
BYTES = {
    # f32h16 = COLA_F32_H16: fp32 spinors, links as 12 x int16, clover as 72 x fp16
    # The fp32 kernels read A in its 48-real field-strength form (192 B), A^-1 as 72 reals (288 B).
    # f32x12_a72 = the same kernels reading the 72-real packed A (cola_set_compact(1)); f32r8 = COLA_F32_R8: links as 8 fp32 reals
    "dslash": {"f32x12": 576, "f32x18": 768, "f64x18": 1536, "f32h16": 384, "f32r8": 448, "f32x12_a72": 576},   # 8 links + 1 spinor in + 1 out
    "dslash_clover_inv": {"f32x12": 864, "f32x18": 1056, "f64x18": 2112, "f32h16": 528, "f32r8": 736, "f32x12_a72": 864},   # + 72 reals clover (A^-1)
    "dslash_clover_xpay": {"f32x12": 864, "f32x18": 1056, "f64x18": 2304, "f32h16": 624, "f32r8": 736, "f32x12_a72": 960},  # + A (48 or 72 reals) + 24 (x)
}
R8_MASK = {"f32r8": 3, "f32x12_a72": 1}
FLOPS = {"dslash": 1320, "dslash_clover_inv": 1824, "dslash_clover_xpay": 1872}
# dram__bytes_read.sum + dram__bytes_write.sum per launch of dslash_kernel<F32x12, XPAY=2> is read from
# profiles/ncu_traffic.json, which records the commit and the hash of csrc/ it was captured at: when the kernels have
# changed since, `traffic` is reported as null rather than a stale number.
def csrc_hash():
    import hashlib

    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2302_00850_b200", "csrc")
    for f in sorted(os.listdir(d)):
        if f.endswith((".cu", ".cuh", ".h")):
            h.update(f.encode())
            h.update(open(os.path.join(d, f), "rb").read())
    return h.hexdigest()[:16]


def ncu_traffic(dims):
    path = os.path.join(ROOT, "profiles", "ncu_traffic.json")
    if not os.path.exists(path):
        return None, "profiles/ncu_traffic.json absent"
    rec = json.load(open(path))
    ent = rec.get("entries", {}).get("x".join(str(d) for d in dims))
    if ent is None:
        return None, "no ncu capture for this lattice"
    if rec.get("csrc_sha16") != csrc_hash():
        return None, f"csrc/ changed since the capture at {rec.get('commit')}: stale, not reported"
    return int(ent["bytes_per_launch"]), f"{ent['source']} (commit {rec.get('commit')})"


CPU_SAMPLE_MAX_SITES = 1 << 22   # largest lattice the oracle's full fields are built for inside bench.py
NOMINAL_HBM_GBS = 8000.0   # BASELINE.json north_star's denominator, reported beside the measured one


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        d = json.load(open(path))
        return float(d["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (torch copy, read+write)"
    return 6650.0, "fallback 6.65 TB/s (B200_PROFILING.md; MEASURED_PEAKS.json absent)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100",
                                          "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([f.strip() for f in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm = [float(r[0]) for r in self.rows if len(r) >= 7 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 7 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({names[i] for r in self.rows if len(r) >= 7 for i in range(4) if r[3 + i].lower().startswith("active")})
        pw = [float(r[2]) for r in self.rows if len(r) >= 7 and r[2].replace(".", "").isdigit()]
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": reasons}


def aggregate_over_ranks(local_ms: float, local_units: float, device=None):
    """(max-over-ranks time, sum-over-ranks units).  Works on any initialised process group (nccl or gloo)."""
    import torch.distributed as dist

    if not (dist.is_available() and dist.is_initialized()):
        return local_ms, local_units
    t = torch.tensor([local_ms], dtype=torch.float64, device=device)
    u = torch.tensor([local_units], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def time_launches(fn, n_warm, n_timed, bursts=10):
    """Device time (ms) of one fn() call: the MEDIAN over `bursts` back-to-back bursts of n_timed / bursts calls each
    (n_timed calls in all, SURVEY 8(d) "median of >= 200 timed launches"), each burst bracketed by CUDA events on the
    current stream.  A median of bursts rather than a mean of everything: under the power cap the SM clock moves by ~10 %
    within a run, and a mean folds that drift into whichever row happens to be measured at the time."""
    for _ in range(n_warm):
        fn()
    bursts = max(1, min(bursts, n_timed))
    per = max(1, n_timed // bursts)
    evs = [torch.cuda.Event(enable_timing=True) for _ in range(bursts + 1)]
    torch.cuda.synchronize()
    evs[0].record()
    for k in range(bursts):
        for _ in range(per):
            fn()
        evs[k + 1].record()
    torch.cuda.synchronize()
    return statistics.median(evs[k].elapsed_time(evs[k + 1]) / per for k in range(bursts))


def operator_table(ctx, fmt32, n_warm=20, n_timed=200, nrhs=0, only_fmt32=False):
    """Per-kernel throughput of the operator family, each timed alone (inputs larger than L2).
    nrhs > 1 adds the multi-right-hand-side Schur operator over nrhs vectors.
    only_fmt32: just the rows of the context's own fp32 link format (the second, 18-real context of the x12 / x18 comparison)."""
    peak, _ = measured_peaks()
    out = {}
    Vh = ctx.Vh
    fmts = [(torch.float32, fmt32), (torch.float64, "f64x18"), (torch.float32, "f32h16")]
    if fmt32 == "f32x12":   # the compact fields are measured against the 12-real links they replace
        fmts += [(torch.float32, "f32r8"), (torch.float32, "f32x12_a72")]
    if only_fmt32:
        fmts = fmts[:1]
    for prec, fmt in fmts:
        full = ctx.empty_internal(prec, full=True).normal_()
        dst = ctx.empty_internal(prec, full=True)
        h = fmt == "f32h16"
        of = "h16" if h else ("r8" if fmt == "f32r8" else None)
        ctx.set_compact(R8_MASK.get(fmt, 3))
        rows = {
            "dslash_even": ("dslash", 1, lambda: ctx.dslash_apply(0, full[1], out=dst[0], fmt=of)),
            "dslash_odd": ("dslash", 1, lambda: ctx.dslash_apply(1, full[0], out=dst[1], fmt=of)),
            "fermion_matrix": ("dslash_clover_xpay", 2, lambda: ctx.fermion_matrix_apply(full, out=dst, fmt=of)),
            "schur": (None, 2, lambda: ctx.schur_apply(full[0], out=dst[0], fmt=of)),
        }
        for name, (kind, launches, fn) in rows.items():
            ms = time_launches(fn, n_warm, n_timed)
            if kind is None:   # Schur = dslash+A^-1 then dslash+A+xpay
                nbytes = (BYTES["dslash_clover_inv"][fmt] + BYTES["dslash_clover_xpay"][fmt]) * Vh
                flops = (FLOPS["dslash_clover_inv"] + FLOPS["dslash_clover_xpay"]) * Vh
            else:
                nbytes = BYTES[kind][fmt] * Vh * launches
                flops = FLOPS[kind] * Vh * launches
            gbs = nbytes / (ms * 1e-3) / 1e9
            out[f"{name}_{fmt}"] = {"ms": round(ms, 5), "launches": launches, "GB/s": round(gbs, 1), "GFLOP/s": round(flops / (ms * 1e-3) / 1e9, 1),
                                    "frac_measured": round(gbs / peak, 4), "frac_nominal_8TBs": round(gbs / NOMINAL_HBM_GBS, 4)}
        del full, dst
        if nrhs > 1 and fmt in ("f32x12", "f32x18", "f64x18"):
            ctx.set_mrhs_workspace(nrhs)
            vin = ctx.empty_internal_mrhs(nrhs, prec, full=False).normal_()
            vout = torch.empty_like(vin)
            ms = time_launches(lambda: ctx.schur_apply_mrhs(vin, out=vout), max(n_warm // 4, 1), max(n_timed // 4, 1))
            w = 4 if prec == torch.float32 else 8
            G = {"f32x12": 12, "f32x18": 18, "f64x18": 18}[fmt]
            # per site and vector: links and clover of both kernels shared by nrhs vectors + 5 spinor passes
            clov = 72 + (48 if prec == torch.float32 else 72)   # A^-1 (72 reals) + A (fp32: its 48-real form)
            nbytes = ((2 * 8 * G + clov) * w / nrhs + 5 * 24 * w) * Vh * nrhs
            flops = (FLOPS["dslash_clover_inv"] + FLOPS["dslash_clover_xpay"]) * Vh * nrhs
            single = out[f"schur_{fmt}"]["ms"]
            out[f"schur_mrhs{nrhs}_{fmt}"] = {"ms": round(ms, 5), "launches": 2, "ms_per_rhs": round(ms / nrhs, 5), "speedup_vs_single": round(single / (ms / nrhs), 3),
                                              "GB/s": round(nbytes / (ms * 1e-3) / 1e9, 1), "GFLOP/s": round(flops / (ms * 1e-3) / 1e9, 1)}
            del vin, vout
            ctx.release_mrhs_workspace()
            torch.cuda.empty_cache()
    ctx.set_compact(3)
    return out


def x12_vs_x18(ctx12, ctx18, rounds=10, burst=20):
    """What the 12-real link compression of BJ:ns buys on B200 ("additional computation in order to reduce traffic"):
    the same fp32 operators on a 12-real and an 18-real context over the same links, interleaved in short bursts, medians."""
    out = {}
    bufs = {}
    for key, c in (("x12", ctx12), ("x18", ctx18)):
        bufs[key] = (c, c.empty_internal(torch.float32, full=True).normal_(), c.empty_internal(torch.float32, full=True))
    ops = {"dslash": lambda c, a, d: c.dslash_apply(0, a[1], out=d[0]),
           "fermion_matrix": lambda c, a, d: c.fermion_matrix_apply(a, out=d),
           "schur": lambda c, a, d: c.schur_apply(a[0], out=d[0])}
    kinds = {"dslash": ("dslash", 1), "fermion_matrix": ("dslash_clover_xpay", 2), "schur": (None, 2)}
    res = {(o, k): [] for o in ops for k in bufs}
    for _ in range(rounds):
        for o, fn in ops.items():
            for k, (c, a, d) in bufs.items():
                res[(o, k)].append(time_launches(lambda: fn(c, a, d), 3, burst, bursts=1))
    peak, _ = measured_peaks()
    for o in ops:
        row = {}
        for k in bufs:
            ms = statistics.median(res[(o, k)][2:])
            fmt = "f32" + k
            kind, launches = kinds[o]
            nb = (BYTES["dslash_clover_inv"][fmt] + BYTES["dslash_clover_xpay"][fmt]) if kind is None else BYTES[kind][fmt] * launches
            row[k] = {"ms": round(ms, 5), "GB/s": round(nb * ctx12.Vh / (ms * 1e-3) / 1e9, 1), "frac_measured": round(nb * ctx12.Vh / (ms * 1e-3) / 1e9 / peak, 4)}
        row["time_x18_over_x12"] = round(row["x18"]["ms"] / row["x12"]["ms"], 3)
        fmt_b = lambda f: (BYTES["dslash_clover_inv"][f] + BYTES["dslash_clover_xpay"][f]) if kinds[o][0] is None else BYTES[kinds[o][0]][f] * kinds[o][1]
        row["bytes_x18_over_x12"] = round(fmt_b("f32x18") / fmt_b("f32x12"), 3)
        out[o] = row
    return out


def ab_formats(ctx, rounds=12, burst=40):
    """Interleaved A/B of the fp32 operator formats: short bursts of each format in turn, many rounds,
    medians -- the SM clock drifts by ~10 % under the power cap over a run, which a format-after-format table folds into the
    comparison.  Formats: x12 = 12-real links + 48-real A (the default); a72 = 12-real links + 72-real packed A;
    r8 = 8-real links + 48-real A; r8_a72 = 8-real links + 72-real A; h16 = 16-bit links + fp16 clover."""
    full = ctx.empty_internal(torch.float32, full=True).normal_()
    dst = ctx.empty_internal(torch.float32, full=True)
    fmts = {"x12": (None, 3), "a72": (None, 1), "r8": ("r8", 3), "r8_a72": ("r8", 1), "h16": ("h16", 3)}
    ops = {"dslash": lambda f: ctx.dslash_apply(0, full[1], out=dst[0], fmt=f),
           "fermion_matrix": lambda f: ctx.fermion_matrix_apply(full, out=dst, fmt=f),
           "schur": lambda f: ctx.schur_apply(full[0], out=dst[0], fmt=f)}
    res = {(o, k): [] for o in ops for k in fmts}
    for _ in range(rounds):
        for o, fn in ops.items():
            for k, (f, mask) in fmts.items():
                ctx.set_compact(mask)
                res[(o, k)].append(time_launches(lambda: fn(f), 5, burst))
    ctx.set_compact(3)
    out = {}
    for o in ops:
        base = statistics.median(res[(o, "x12")][2:])
        out[o] = {k: {"ms": round(statistics.median(res[(o, k)][2:]), 5), "vs_x12": round(statistics.median(res[(o, k)][2:]) / base, 3)} for k in fmts}
    return out


def timeline(ctx, b, first_iter=40, n_iter=3):
    """Device timestamps (CUPTI activity records through torch.profiler) of every kernel of `n_iter` consecutive CGLS
    iterations of one solve: start, duration and the gap to the end of the previous kernel.  Not a bench line."""
    from torch.profiler import ProfilerActivity, profile

    ctx.cg_solve(b, tol=1e-10, even_odd=True, mixed=True)     # warm
    torch.cuda.synchronize()
    with profile(activities=[ProfilerActivity.CUDA]) as prof:
        ctx.cg_solve(b, tol=1e-10, even_odd=True, mixed=True)
        torch.cuda.synchronize()
    evs = sorted((e for e in prof.events() if e.device_type == torch.autograd.DeviceType.CUDA and "Memcpy" not in e.name and "Memset" not in e.name),
                 key=lambda e: e.time_range.start)
    # an iteration ends with xp_update<float,1,1>; find the launches of iterations first_iter .. first_iter + n_iter - 1
    ends = [i for i, e in enumerate(evs) if "xp_update_kernel<float, true, true>" in e.name or "xp_update_kernel<float, 1, 1>" in e.name]
    # the first window of n_iter iterations from first_iter on without a reliable update (whose speculative launches return at once)
    while first_iter + n_iter < len(ends) and any((e.time_range.end - e.time_range.start) < 20.0
                                                   for e in evs[ends[first_iter - 1] + 1:ends[first_iter + n_iter - 1] + 1]):
        first_iter += 1
    lo, hi = ends[first_iter - 1] + 1, ends[first_iter + n_iter - 1] + 1
    rows, prev_end, t0 = [], None, evs[lo].time_range.start
    for e in evs[lo:hi]:
        st, en = e.time_range.start, e.time_range.end
        name = e.name.replace("void ", "").replace("cola::(anonymous namespace)::", "").split("(")[0]
        rows.append({"kernel": name, "start_us": round(st - t0, 2), "dur_us": round(en - st, 2), "gap_us": None if prev_end is None else round(st - prev_end, 2)})
        prev_end = en
    busy = sum(r["dur_us"] for r in rows)
    span = rows[-1]["start_us"] + rows[-1]["dur_us"]
    return {"iterations": [first_iter, first_iter + n_iter - 1], "kernels": rows, "span_us": round(span, 2), "kernel_sum_us": round(busy, 2),
            "gaps_us": round(span - busy, 2), "note": "gap < 0: the next kernel's blocks started under programmatic dependent launch before the previous grid had drained"}


def _set_oracle_threads(n):
    """OpenMP thread count of the oracle's site loops (the oracle itself is untouched: same library, same code)."""
    import ctypes

    try:
        ctypes.CDLL("libgomp.so.1").omp_set_num_threads(int(n))
        return True
    except OSError:
        return False


def cpu_baseline_sample(cfg, U_cpu, n_pairs=6, table=True):
    """The oracle as it stands on the host cores.  `value`: n_pairs x (S, S^dagger) applications on the configuration's
    lattice with all cores.  `table`: M and S, 16^3x32 and 32^3x64 extents of the same recipe, 1 core and all
    cores, one application each; the stored times of the oracle's full CGNR solves (tests/golden/solver_golden.json, with
    their thread count) and, labelled as such, the CPU time-to-solution extrapolated to configs 3 and 4 as (seconds per
    S, S^dagger pair per site) x (sites) x (GPU iteration count)."""
    import numpy as np

    import oracle

    dims, kappa, csw = cfg["dims"], cfg["kappa"], cfg["csw"]
    Un = U_cpu.numpy()
    A = oracle.clover(dims, Un, kappa, csw)
    Ainv = oracle.clover_inverse(A)
    x = (inputs.source_gaussian(dims, 77) * torch.from_numpy(oracle.parity_mask(dims) == 0)[..., None, None]).numpy()
    Vh = inputs.volume(dims) // 2
    cores = oracle.num_threads()
    t0 = time.time()
    for _ in range(n_pairs):
        y = oracle.schur(dims, inputs.BC, Un, A, Ainv, kappa, x)
        x = oracle.schur(dims, inputs.BC, Un, A, Ainv, kappa, y, dagger=True)
        x = x / np.linalg.norm(x.ravel())
    dt = time.time() - t0
    flops = n_pairs * 2 * 3696.0 * Vh
    out = {"value": round(flops / dt / 1e9, 3), "unit": "GFLOP/s", "cores": cores, "kind": "oracle",
           "sample": f"{n_pairs} x (S, S^dagger) oracle applications on the full {dims} lattice = the operator work of {n_pairs} CGLS iterations, {dt:.1f} s",
           "seconds": round(dt, 2)}
    if not table:
        return out
    rows = []
    pair_s_per_site = dt / n_pairs / Vh          # all cores, seconds per (S, S^dagger) pair and even site
    fields = {tuple(dims): (Un, A, Ainv)}
    for d in ((16, 16, 16, 32), (32, 32, 32, 64)):
        if inputs.volume(d) > inputs.volume(dims):
            continue
        if d not in fields:
            Ud = inputs.links_smooth(d, cfg["eps"], 20230200 + 99).numpy()
            Ad = oracle.clover(d, Ud, kappa, csw)
            fields[d] = (Ud, Ad, oracle.clover_inverse(Ad))
        Ud, Ad, Aid = fields[d]
        psi = inputs.source_gaussian(d, 78).numpy()
        psi_e = psi * (oracle.parity_mask(d) == 0)[..., None, None]
        V = inputs.volume(d)
        for nthr in (1, cores):
            if not _set_oracle_threads(nthr):
                continue
            for name, fl, fn in (("M", 1872.0 * V, lambda: oracle.M(d, inputs.BC, Ud, Ad, kappa, psi)),
                                 ("S", 3696.0 * V / 2, lambda: oracle.schur(d, inputs.BC, Ud, Ad, Aid, kappa, psi_e))):
                t1 = time.time()
                fn()
                el = time.time() - t1
                rows.append({"operator": name, "lattice": list(d), "cores": nthr, "seconds": round(el, 4), "GFLOP/s": round(fl / el / 1e9, 3)})
        _set_oracle_threads(cores)
    out["table"] = rows
    gold = os.path.join(ROOT, "tests", "golden", "solver_golden.json")
    if os.path.exists(gold):
        g = json.load(open(gold))
        out["oracle_cgnr_solves"] = [{"config": int(k), "lattice": v["dims"], "mode": m, "iters": v[m]["iters"], "seconds": round(v[m]["seconds"], 2),
                                      "threads": v.get("threads"), "source": "tests/golden/solver_golden.json (written by tests/golden/make_golden.py on the build box)"}
                                     for k, v in sorted(g.items()) for m in ("full", "eo") if m in v]
    # extrapolation, labelled: CPU seconds per iteration scale with the volume; iteration counts are the GPU's
    out["extrapolated_cpu_time_to_solution_s"] = {
        "note": "EXTRAPOLATED, not measured: (all-core seconds per (S, S^dagger) pair per even site, measured above) x even sites x the CUDA solver's iteration count",
        "config3_48^3x96_per_source_97_iters": round(pair_s_per_site * (48 ** 3 * 96 // 2) * 97, 1),
        "config4_64^3x128_136_iters": round(pair_s_per_site * (64 ** 3 * 128 // 2) * 136, 1)}
    return out


def reference_arm(args, cfg, workload):
    """--impl reference: the CPU oracle (this tier's reference arm) on the host cores, rank 0 only."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import numpy as np

    import oracle

    dims, kappa, csw = cfg["dims"], cfg["kappa"], cfg["csw"]
    note = ""
    if inputs.volume(dims) > CPU_SAMPLE_MAX_SITES:   # see main(): the oracle's fields for the big lattices exceed host memory
        note = f"; run on (32, 32, 32, 64) extents of the same link recipe because the oracle's fields for {tuple(dims)} exceed host memory"
        dims = (32, 32, 32, 64)
    dev = "cuda" if torch.cuda.is_available() else "cpu"
    U = inputs.make_links(args.config, dims=dims, device=dev).cpu()
    Un = U.numpy()
    A = oracle.clover(dims, Un, kappa, csw)
    Ainv = oracle.clover_inverse(A)
    x = (inputs.source_gaussian(dims, 77) * torch.from_numpy(oracle.parity_mask(dims) == 0)[..., None, None]).numpy()
    Vh = inputs.volume(dims) // 2

    def step(x):
        y = oracle.schur(dims, inputs.BC, Un, A, Ainv, kappa, x)
        x = oracle.schur(dims, inputs.BC, Un, A, Ainv, kappa, y, dagger=True)
        return x / np.linalg.norm(x.ravel())

    for _ in range(args.warmup):
        x = step(x)
    t0 = time.time()
    for _ in range(args.steps):
        x = step(x)
    dt = time.time() - t0
    val = args.steps * 2 * 3696.0 * Vh / dt / 1e9
    sample = f"each step = one (S, S^dagger) oracle application pair on the full {dims} lattice (operator work of one CGLS iteration)" + note
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": round(val, 3), "unit": "GFLOP/s", "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": round(dt / args.steps * 1e3, 2), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": workload,
        "cpu_baseline": {"value": round(val, 3), "unit": "GFLOP/s", "cores": oracle.num_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": round(val, 3), "unit": "GFLOP/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


METRIC = "Dirac-op GFLOP/s (counted flops) sustained over a mixed-precision even-odd CGNR solve to 1e-10"


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json configs[K] (default 2: 32^3x64, fp32 12-real links)")
    ap.add_argument("--impl", default="cola", choices=["cola", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-operator-table", action="store_true")
    ap.add_argument("--operators-only", action="store_true",
                    help="profiling aid: skip the solves, run only the operator table (few launches: --op-warm/--op-timed) and print it")
    ap.add_argument("--lattice", default="", help="test aid: run the config's recipe on other extents, e.g. 16,16,16,32")
    ap.add_argument("--no-x18", action="store_true", help="skip the 18-real fp32 operator rows and the interleaved 12-real / 18-real comparison")
    ap.add_argument("--no-h16", action="store_true", help="skip the extra solve with 16-bit links/clover in the inner iteration")
    ap.add_argument("--no-bicgstab", action="store_true", help="skip the extra solves by BiCGStab on the Schur system")
    ap.add_argument("--no-eig", action="store_true", help="skip the low-mode solve and the deflated step")
    ap.add_argument("--eig", action="store_true", help="run the low-mode solve also on lattices larger than 32^3x64 (48^3x96: 3 minutes)")
    ap.add_argument("--n-ev", type=int, default=8, help="eigenpairs of S^+S for the deflated step")
    ap.add_argument("--no-batched", action="store_true", help="config 3: skip the batched (multi-rhs) solve of the 12 sources")
    ap.add_argument("--nrhs", type=int, default=0, help="with --operators-only: also time the multi-rhs Schur operator over this many vectors")
    ap.add_argument("--staging", type=int, default=0, choices=[0, 1],
                    help="kernel family of the fp32 / 16-bit single-rhs operators: 0 direct global loads (default), 1 neighbour spinors staged in shared memory")
    ap.add_argument("--ab-formats", action="store_true", help="measurement aid: interleaved A/B of the fp32 link / clover storage formats, then exit")
    ap.add_argument("--bicgstab-only", action="store_true", help="measurement aid: one mixed-precision BiCGStab solve, then exit")
    ap.add_argument("--timeline", action="store_true", help="measurement aid: device timestamps of the kernels of three consecutive iterations, then exit")
    ap.add_argument("--op-warm", type=int, default=20)
    ap.add_argument("--op-timed", type=int, default=200)
    args = ap.parse_args()

    cfg = dict(inputs.CONFIGS[args.config])
    if args.lattice:   # test aid: the same recipe on other extents (the line's config.lattice says so; not a bench value)
        cfg["dims"] = tuple(int(v) for v in args.lattice.split(","))
    dims = cfg["dims"]
    workload = {
        "workload": f"BASELINE.json configs[{args.config}]: {dims[0]}x{dims[1]}x{dims[2]}x{dims[3]} lattice, links exp(i*{cfg['eps']}*H) seeded, "
                    f"kappa={cfg['kappa']}, csw={cfg['csw']}, bc=(+,+,+,-), "
                    + ("12 point sources at the origin (one per spin-colour component) solved one after the other"
                       if cfg["source"] == "point" else "Gaussian source")
                    + ", fp32 links stored as 12 reals; step = mixed-precision (fp32 inner / fp64 reliable updates, delta=0.1) "
                      "even-odd CGNR to 1e-10" + (" for each source" if cfg["source"] == "point" else ""),
        "lattice": list(dims), "kappa": cfg["kappa"], "csw": cfg["csw"], "tol": 1e-10, "parallelism": f"replicas x{args.gpus}",
        "l2": "inputs larger than L2 (fp32 gauge+clover alone are > 1 GB per operator application at 32^3x64)",
    }
    if args.impl == "reference":
        return reference_arm(args, cfg, workload)

    from paper_2302_00850_b200 import binding   # raises if libcola.so is missing: no CPU fallback

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (the COLA hot path has no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        import torch.distributed as dist

        dist.init_process_group("nccl", device_id=dev)

    # ---- setup (H0-H2), not part of a step
    U = inputs.make_links(args.config, dims=dims, device=dev)
    point = cfg["source"] == "point"    # BJ:c3: 12 point sources at the origin, one per spin-colour component
    if point:
        def source(n):
            return inputs.source_point(dims, n // 3, n % 3, device=dev)
        n_src = 12
    else:
        def source(n):
            return inputs.source_gaussian(dims, inputs.config_seed_source(args.config) + rank, device=dev)
        n_src = 1
    ctx = binding.Cola(dims, cfg["kappa"], cfg["csw"], bc=inputs.BC, compress12=True, device=local)
    ctx.set_staging(args.staging)
    torch.cuda.synchronize()
    t0 = time.time()
    ctx.gauge_upload(U)
    torch.cuda.synchronize()
    setup_s = time.time() - t0
    want_cpu = rank == 0 and world == 1 and not args.no_cpu_baseline
    cpu_dims = tuple(dims)
    if want_cpu and inputs.volume(dims) > CPU_SAMPLE_MAX_SITES:
        # the oracle's dense 12x12 clover field alone is 2.3 KB per site: on the big lattices the bounded CPU sample
        # runs the same recipe (links, kappa, csw) on 32^3x64 extents; the oracle's cost per site does not depend on V
        cpu_dims = (32, 32, 32, 64)
        U_cpu = inputs.make_links(args.config, dims=cpu_dims, device=dev).cpu()
    else:
        U_cpu = U.cpu() if want_cpu else None
    del U
    torch.cuda.empty_cache()

    def barrier():
        if world > 1:
            torch.distributed.barrier()
        torch.cuda.synchronize()

    if args.ab_formats:       # not a bench line: interleaved comparison of the link / clover storage formats
        print(json.dumps({"ab_formats": True, "lattice": list(dims), "operators": ab_formats(ctx)}))
        return
    if args.operators_only:   # not a bench line: a short launch sequence for ncu captures of each operator kernel
        print(json.dumps({"operators_only": True, "lattice": list(dims),
                          "operators": operator_table(ctx, "f32x12", n_warm=args.op_warm, n_timed=args.op_timed, nrhs=args.nrhs)}))
        return

    def one_step():
        """One pass of the hot path over the configuration's sources, solved one after the other."""
        fl, infos = 0.0, []
        for n in range(n_src):
            bn = b if n_src == 1 else source(n)
            xn, info = ctx.cg_solve(bn, tol=1e-10, even_odd=True, mixed=True)
            fl += info["op_flops"]
            infos.append(info)
            del xn
        return fl, infos

    b = source(0) if n_src == 1 else None
    if args.bicgstab_only:    # not a bench line: one BiCGStab solve, the launch sequence the ncu captures of its kernels come from
        x_, inf_ = ctx.cg_solve(b if b is not None else source(0), tol=1e-10, even_odd=True, mixed=1, method="bicgstab")
        print(json.dumps({"bicgstab_only": True, "lattice": list(dims), "iters": inf_["iters"], "true_residual": inf_["true_residual"]}))
        return
    if args.timeline:         # not a bench line: kernel start times of three consecutive iterations (profiles/r2_timeline.md)
        print(json.dumps({"timeline": True, "lattice": list(dims), **timeline(ctx, b if b is not None else source(0))}))
        return
    # ---- device-resident steps
    for _ in range(args.warmup):
        one_step()
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    l0 = ctx.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    flops = 0.0
    for _ in range(args.steps):
        fl, infos = one_step()
        flops += fl
    e1.record()
    barrier()
    launches = ctx.launch_count() - l0
    clocks = sampler.stop()
    info = infos[-1]
    ms_local = e0.elapsed_time(e1)
    ms, flops_all = aggregate_over_ranks(ms_local, flops, device=dev)
    value = flops_all / (ms * 1e-3) / 1e9

    # ---- one more step with CUDA-event pairs around every launch of the dominant kernel (in-solve duration for `roofline`)
    in_solve = None
    if rank == 0:
        ctx.profile_kernel(True)
        one_step()
        k_ms, k_n, k_skipped = ctx.profile_result()
        ctx.profile_kernel(False)
        in_solve = {"avg_launch_ms": round(k_ms, 5), "launches": k_n, "skipped_speculative_launches": k_skipped}

    # ---- end to end: host buffers through cola_cg_solve_host
    b_host = source(0).cpu().pin_memory()
    x_host = torch.empty_like(b_host).pin_memory()

    def host_step():
        fl = 0.0
        for n in range(n_src):
            if n_src > 1:
                b_host.zero_()
                b_host[0, 0, 0, 0, n // 3, n % 3] = 1.0
            _, info_e = ctx.cg_solve(b_host, tol=1e-10, even_odd=True, mixed=True, x=x_host)
            fl += info_e["op_flops"]
        return fl

    host_step()
    barrier()
    e0.record()
    flops_e = 0.0
    for _ in range(args.steps):
        flops_e += host_step()
    e1.record()
    barrier()
    ms_e, flops_e_all = aggregate_over_ranks(e0.elapsed_time(e1), flops_e, device=dev)
    nbytes = b_host.numel() * b_host.element_size() * n_src

    # ---- the same step with the inner operator reading 16-bit links and clover (mixed = 2) or the
    # 8-real links and the 48-real A (mixed = 3)
    def extra_solve(mode, delta=0.1):
        def one_step():
            fl, infs = 0.0, []
            for n in range(n_src):
                bn = b if n_src == 1 else source(n)
                xn, inf = ctx.cg_solve(bn, tol=1e-10, even_odd=True, mixed=mode, delta=delta)
                fl += inf["op_flops"]
                infs.append(inf)
                del xn
            return fl, infs

        for _ in range(min(args.warmup, 2)):
            one_step()
        torch.cuda.synchronize()
        e0.record()
        fl_h = 0.0
        for _ in range(args.steps):
            f1, infs_h = one_step()
            fl_h += f1
        e1.record()
        torch.cuda.synchronize()
        ms_h = e0.elapsed_time(e1) / args.steps
        return {"ms_per_step": round(ms_h, 3), "GFLOP/s": round(fl_h / args.steps / (ms_h * 1e-3) / 1e9, 1),
                "speedup_vs_fp32_inner": round(ms_local / args.steps / ms_h, 3), "iters": [i["iters"] for i in infs_h],
                "reliable_updates": [i["reliable_updates"] for i in infs_h],
                "max_true_residual": max(i["true_residual"] for i in infs_h), "converged": all(i["converged"] for i in infs_h)}

    solve_h16 = solve_r8 = solve_delta = None
    extras = rank == 0 and world == 1   # the extra modes are single-GPU context for the line, not part of the scaling runs
    if extras and not args.no_h16:
        solve_h16 = extra_solve(2)
        solve_r8 = extra_solve(3)
        # the headline step with the reliable-update threshold delta = 0.01 (an update every two decades instead of every decade;
        # the paper is silent on delta, reading A9 keeps 0.1 for the step): what the fp64 outer work costs
        solve_delta = extra_solve(1, delta=0.01)
        solve_delta["delta"] = 0.01

    # ---- the same step by BiCGStab on the Schur system (two S per pass instead of S and S^+)
    solve_bicgstab = None
    if extras and not args.no_bicgstab:
        solve_bicgstab = {}
        for key, mode in (("fp32_inner", 1), ("h16_inner", 2), ("r8_inner", 3)):
            def bi_step():
                fl, infs = 0.0, []
                for n in range(n_src):
                    bn = b if n_src == 1 else source(n)
                    xn, inf = ctx.cg_solve(bn, tol=1e-10, even_odd=True, mixed=mode, method="bicgstab")
                    fl += inf["op_flops"]
                    infs.append(inf)
                    del xn
                return fl, infs

            for _ in range(min(args.warmup, 2)):
                bi_step()
            torch.cuda.synchronize()
            e0.record()
            fl_b = 0.0
            for _ in range(args.steps):
                f1, infs_b = bi_step()
                fl_b += f1
            e1.record()
            torch.cuda.synchronize()
            ms_b = e0.elapsed_time(e1) / args.steps
            solve_bicgstab[key] = {"ms_per_step": round(ms_b, 3), "GFLOP/s": round(fl_b / args.steps / (ms_b * 1e-3) / 1e9, 1),
                                   "speedup_vs_cgnr_fp32_inner": round(ms_local / args.steps / ms_b, 3), "passes": [i["iters"] for i in infs_b],
                                   "reliable_updates": [i["reliable_updates"] for i in infs_b],
                                   "max_true_residual": max(i["true_residual"] for i in infs_b), "converged": all(i["converged"] for i in infs_b)}

    # ---- the lowest modes of S^+S and the same step started from the deflated guess
    low_modes = None
    if extras and not args.no_eig and (ctx.Vh <= (1 << 20) or args.eig):   # larger lattices: minutes of Lanczos for nothing
        try:
            torch.cuda.synchronize()
            t0 = time.time()
            ev, evecs, einfo = ctx.eig_lowest(args.n_ev, tol=1e-9)
            torch.cuda.synchronize()
            t_eig = time.time() - t0
            e0.record()
            infs_d = []
            for n in range(n_src):
                bn = b if n_src == 1 else source(n)
                xn, inf = ctx.cg_solve_deflated(bn, ev, evecs, tol=1e-10, mixed=1)
                infs_d.append(inf)
                del xn
            e1.record()
            torch.cuda.synchronize()
            ms_d = e0.elapsed_time(e1)
            low_modes = {"n_ev": args.n_ev, "eig_seconds": round(t_eig, 3), "eig_converged": einfo["converged"], "restarts": einfo["restarts"],
                         "op_applications": einfo["op_applications"], "lowest_eigenvalues_of_SdagS": [float(f"{v:.6e}") for v in ev[:4]],
                         "max_eig_residual": max(einfo["residuals"]), "deflated_solve_ms_per_step": round(ms_d, 3),
                         "deflated_iters": [i["iters"] for i in infs_d], "undeflated_iters": [i["iters"] for i in infos],
                         "max_true_residual": max(i["true_residual"] for i in infs_d),
                         "note": "heavy-quark configs: cond(S^+S) is small, so deflating a few modes saves few iterations; reported, not the headline"}
            del evecs
            torch.cuda.empty_cache()
        except (RuntimeError, binding.ColaError) as ex:
            low_modes = {"unavailable": str(ex)[:200]}

    # ---- the same sources as ONE batched solve (links and clover read once per pass for all)
    batched = None
    if n_src > 1 and extras and not args.no_batched:
        del b_host, x_host
        torch.cuda.empty_cache()
        try:
            bs = torch.stack([source(n) for n in range(n_src)])
            xs = torch.empty_like(bs)
            ctx.set_mrhs_workspace(n_src)
            batched = {"nrhs": n_src}
            for key, mode, meth in (("fp32_inner", 1, "cgnr"), ("h16_inner", 2, "cgnr"), ("r8_inner", 3, "cgnr"),
                                    ("bicgstab_fp32_inner", 1, "bicgstab"), ("bicgstab_h16_inner", 2, "bicgstab")):
                for _ in range(min(args.warmup, 1)):
                    ctx.cg_solve_mrhs(bs, tol=1e-10, x=xs, mixed=mode, method=meth)
                torch.cuda.synchronize()
                e0.record()
                fl_b = 0.0
                for _ in range(args.steps):
                    _, infos_b = ctx.cg_solve_mrhs(bs, tol=1e-10, x=xs, mixed=mode, method=meth)
                    fl_b += sum(i["op_flops"] for i in infos_b)
                e1.record()
                torch.cuda.synchronize()
                ms_b = e0.elapsed_time(e1) / args.steps
                batched[key] = {"ms_per_step": round(ms_b, 3), "GFLOP/s": round(fl_b / args.steps / (ms_b * 1e-3) / 1e9, 1),
                                "speedup_vs_sequential": round(ms / args.steps / ms_b, 3),
                                "iters": [i["iters"] for i in infos_b], "reliable_updates": [i["reliable_updates"] for i in infos_b],
                                "max_true_residual": max(i["true_residual"] for i in infos_b)}
            del bs, xs
        except (RuntimeError, binding.ColaError) as ex:   # e.g. out of memory for 12 systems at once
            batched = {"unavailable": str(ex)[:200]}
        torch.cuda.empty_cache()

    if rank != 0:
        if world > 1:
            torch.distributed.destroy_process_group()
        return

    # ---- roofline of the dominant kernel + operator table (rank 0, kernels timed alone)
    peak, peak_src = measured_peaks()
    table = {} if (args.no_operator_table or world > 1) else operator_table(ctx, "f32x12", n_warm=args.op_warm, n_timed=args.op_timed)
    # ---- the fp32 x18 column of SURVEY 8(d) and what 12-real compression buys (second context on the same links)
    compression = None
    if table and rank == 0 and not args.no_x18:
        try:
            c18 = binding.Cola(dims, cfg["kappa"], cfg["csw"], bc=inputs.BC, compress12=False, device=local, features=binding.COLA_FEAT_FULL_M)
            need = c18.workspace_bytes() + inputs.volume(dims) * (4 * 18 * 8 + 4 * 24 * 4) + (2 << 30)
            if torch.cuda.mem_get_info(dev)[0] > need:
                U18 = inputs.make_links(args.config, dims=dims, device=dev)
                c18.gauge_upload(U18)
                del U18
                torch.cuda.empty_cache()
                table.update(operator_table(c18, "f32x18", n_warm=args.op_warm, n_timed=args.op_timed, only_fmt32=True))
                compression = x12_vs_x18(ctx, c18)
            else:
                compression = {"unavailable": "a second (18-real) context does not fit beside the first on this lattice"}
            c18.close()
            del c18
            torch.cuda.empty_cache()
        except (RuntimeError, binding.ColaError) as ex:
            compression = {"unavailable": str(ex)[:200]}
    roof = None
    if table:
        k = table["fermion_matrix_f32x12"]   # two launches of the fused dslash + clover + xpay kernel
        per_launch_bytes = BYTES["dslash_clover_xpay"]["f32x12"] * ctx.Vh
        roof = {"kernel": "dslash_kernel<F32x12, XPAY=A*y+c*v> (Schur kernel 2 / M), timed alone through cola_fermion_matrix_apply (2 launches per call)",
                "bound": "hbm", "achieved": k["GB/s"], "peak": peak, "unit": "GB/s", "frac": round(k["GB/s"] / peak, 4),
                "frac_of_nominal_8TBs": round(k["GB/s"] / NOMINAL_HBM_GBS, 4), "peak_source": peak_src + " (burst figure; kernel timed alone)",
                "algorithmic_bytes_per_launch": per_launch_bytes, "avg_launch_ms": round(k["ms"] / 2, 5), "traffic": None}
        roof["traffic"], roof["traffic_source"] = ncu_traffic(dims)
        if roof["traffic"]:
            # `achieved` counts ALGORITHMIC bytes (the contract); the bytes ncu saw at the DRAM are ~3 % fewer (part of the
            # 100 MB y / in vectors survives in L2 between back-to-back launches), which is how frac can exceed 1 against a
            # peak that is itself a measured copy, not a physical limit
            roof["achieved_by_traffic"] = round(roof["traffic"] / (roof["avg_launch_ms"] * 1e-3) / 1e9, 1)
            roof["frac_by_traffic"] = round(roof["achieved_by_traffic"] / peak, 4)
    if in_solve and in_solve["launches"]:
        # the same kernel inside a solve step (event pair around each launch, speculative no-op launches excluded)
        per_launch_bytes = BYTES["dslash_clover_xpay"]["f32x12"] * ctx.Vh
        gbs = per_launch_bytes / (in_solve["avg_launch_ms"] * 1e-3) / 1e9
        in_solve.update({"achieved": round(gbs, 1), "frac": round(gbs / peak, 4), "frac_of_nominal_8TBs": round(gbs / NOMINAL_HBM_GBS, 4),
                         "note": "same peak (MEASURED_PEAKS.json has one HBM figure); measured in an extra step after the timed ones"})
        if roof is None:   # --no-operator-table: the in-solve measurement is the roofline entry
            roof = {"kernel": "dslash_kernel<F32x12, XPAY=A*y+c*v> (Schur kernel 2), CUDA-event pair around each launch inside a solve step",
                    "bound": "hbm", "achieved": in_solve["achieved"], "peak": peak, "unit": "GB/s", "frac": in_solve["frac"],
                    "frac_of_nominal_8TBs": in_solve["frac_of_nominal_8TBs"], "peak_source": peak_src,
                    "algorithmic_bytes_per_launch": per_launch_bytes, "avg_launch_ms": in_solve["avg_launch_ms"],
                    "traffic": ncu_traffic(dims)[0]}
        roof["in_solve"] = in_solve
        # the same three figures as flat keys (a record that keeps only the top level of `roofline` still has them)
        roof["in_solve_avg_launch_ms"] = in_solve["avg_launch_ms"]
        roof["in_solve_frac"] = in_solve["frac"]
        roof["in_solve_launches"] = in_solve["launches"]
    cpu = None
    if U_cpu is not None:
        cpu = cpu_baseline_sample(dict(cfg, dims=cpu_dims), U_cpu)
        if cpu_dims != tuple(dims):
            cpu["sample"] += f"; run on {cpu_dims} extents of the same link recipe because the oracle's fields for {tuple(dims)} exceed host memory"

    line = {
        "metric": METRIC, "value": round(value, 1), "unit": "GFLOP/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": round(ms / args.steps, 3), "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic", "config": workload,
        "solve": {"iters": info["iters"], "reliable_updates": info["reliable_updates"], "true_residual": info["true_residual"],
                  "time_to_solution_s": round(ms / args.steps * 1e-3, 5), "converged": info["converged"]},
        "setup_s": round(setup_s, 3),
        "e2e": {"value": round(flops_e_all / (ms_e * 1e-3) / 1e9, 1), "unit": "GFLOP/s", "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes,
                "ms_per_step": round(ms_e / args.steps, 3)},
        "gpu_launches": int(launches), "clocks": clocks, "roofline": roof, "cpu_baseline": cpu, "operators": table,
    }
    if n_src > 1:
        line["solve"]["sources"] = n_src
        line["solve"]["iters_per_source"] = [i["iters"] for i in infos]
        line["solve"]["max_true_residual"] = max(i["true_residual"] for i in infos)
        line["batched"] = batched
    line["compression_x12_vs_x18"] = compression
    line["solve_h16"] = solve_h16
    line["solve_r8"] = solve_r8
    line["solve_delta_0.01"] = solve_delta
    line["low_modes"] = low_modes
    line["solve_bicgstab"] = solve_bicgstab
    print(json.dumps(line))
    if world > 1:
        torch.distributed.destroy_process_group()


if __name__ == "__main__":
    main()

#!/usr/bin/env python
"""bench.py -- throughput of the sGW hot path on B200 (contract: DESIGN.md section 6 "Measurement").

A step = one pass of the whole hot path over one batch of the LARGEST single-GPU
config, BASELINE.json configs[4]: 384^3 grid (h = 0.6), Si8381H1620-shaped V_loc + 8381 Kleinman-Bylander spheres,
all 32 vectors in flight: +-1 vectors from the hash (a1), a slice of 16 of the 2047 Chebyshev applications (a2-a7)
and 4 of the 500 split-operator steps with the per-step Hartree rebuild (a8-a10) -- the config's 4:1 ratio.
value = grid-pt * vector * H-applies per second (1 TD step = 1 application, R-19), inputs resident in HBM.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]
"""
from __future__ import annotations

import argparse
import json
import math
import os
import socket
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2601_21005_b200 import shard, workloads as W  # noqa: E402

METRIC = "grid-pt*vector H-applies/s (Chebyshev filter + TD step)"
UNIT = "grid-pt*vec*H-applies/s"
WORKLOAD = "cfg4"
SLICE_APPLIES = 16          # of the 2047 Chebyshev applications per step
SLICE_TD = 4                # of the 500 TD-Hartree steps per step
TRAFFIC_JSON = os.path.join(ROOT, "profiles", "r02_traffic.json")
SUBCELL_N = 128             # oracle timing sample: central 128^3 sub-cell of the workload


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def ncu_traffic(kernel_key):
    """dram bytes per launch of a kernel from the ncu --set full capture summarised in profiles/ (or None)."""
    if not os.path.exists(TRAFFIC_JSON):
        return None, None
    d = json.load(open(TRAFFIC_JSON))
    e = d.get("kernels", {}).get(kernel_key)
    return (e["dram_bytes_per_unit"], d.get("source")) if e else (None, d.get("source"))


class ClockSampler:
    """nvidia-smi clocks/throttle reasons sampled during the timed region."""

    def __init__(self, index=0):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "200"], stdout=subprocess.PIPE, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except OSError:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.rows.append([x.strip() for x in ln.split(",")])

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
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx = float(r[1])
            except (ValueError, IndexError):
                continue
            for n, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm)}


# ------------------------------------------------------------------------------------------------------------
# the oracle arm (cpu_baseline and --impl reference): the only place bench.py executes oracle/
# ------------------------------------------------------------------------------------------------------------
_SUB = {}


def subcell_workload():
    if "w" not in _SUB:
        _SUB["w"] = W.make_workload(WORKLOAD, n=SUBCELL_N, nterms=2048, subcell=True)
    return _SUB["w"]


def oracle_sample(nvec, napplies, nsteps):
    """Time the oracle (double, OpenMP over vectors) on the central SUBCELL_N^3 sub-cell of the bench workload (same
    spacing, its atoms and KB spheres): nvec vectors x (napplies Chebyshev applications + nsteps TD-Hartree steps)."""
    from oracle import sgw_oracle as o
    o.build()
    w = subcell_workload()
    threads = o.max_threads()
    nvec = min(nvec, max(1, threads))
    psi = o.random_vectors(w.grid, W.SEED_VEC, 0, nvec)
    coeffs = np.ascontiguousarray(w.coeffs[:napplies + 1])
    t0 = time.perf_counter()
    psi = o.cheb_filter(w.grid, w.vloc, w.kb, psi, coeffs, w.emin, w.emax, ld=False)
    if nsteps:
        o.td_propagate(w.grid, w.vloc, w.kb, psi, w.dt, nsteps, 1, 2.0 / (nvec * w.grid.dV), ld=False)
    dt = time.perf_counter() - t0
    units = w.grid.ng * nvec * (napplies + nsteps)
    what = (f"central {SUBCELL_N}^3 sub-cell of {WORKLOAD} (h=0.6, {w.atoms}, {w.kb.nsphere} KB spheres): {nvec} vectors x "
            f"({napplies} Chebyshev applications + {nsteps} TD-Hartree steps)")
    return units / dt, dt, nvec, min(threads, nvec), what


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cores = os.cpu_count() or 1
    for _ in range(min(args.warmup, 1)):
        oracle_sample(cores, 1, 0)
    tot_units, tot_t, used, what = 0.0, 0.0, 1, ""
    for _ in range(args.steps):
        v, dt, nvec, used, what = oracle_sample(cores, 4, 1)
        tot_units += v * dt
        tot_t += dt
    val = tot_units / tot_t
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(32), "sample": what + " per step (4:1 as in the GPU arm's slice)"},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": used, "kind": "oracle", "sample": what + " per step"},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def workload_name(nvec):
    return (f"{WORKLOAD} (BASELINE.json configs[4], the largest single-GPU config): 384^3 grid h=0.6, Si8381H1620-shaped V_loc + "
            f"8381 KB spheres (4 projectors each), {nvec} +-1 vectors in flight per GPU; per step: {SLICE_APPLIES} of the 2047 "
            f"Chebyshev applications (sqrt-Fermi-Dirac coefficients 0..{SLICE_APPLIES}) + {SLICE_TD} of the 500 TD steps "
            f"(dt=0.05, Hartree rebuilt every step)")


# ------------------------------------------------------------------------------------------------------------
# the GPU arm
# ------------------------------------------------------------------------------------------------------------
AXES = {0: "x", 1: "y", 2: "z"}
KINDS = ["store", "acc", "hfin", "cheb", "td", "mul3d", "fwd", "inv", "kb_project", "kb_scatter", "density"]


def collect_passes(ctx):
    out = {}
    for a in range(3):
        for k in range(len(KINDS)):
            n, ms = ctx.sgw_profile_get(a, k)
            if n:
                name = f"{AXES[a]}_{KINDS[k]}" if k < 8 else (KINDS[k] if a == 0 else KINDS[k] + "_points")
                out[name] = {"launches": n, "ms_total": ms}
    return out


def pass_model(passes, nvec, n, kb_frac, uniq_frac=0.0):
    """Algorithmic bytes per grid-pt*vector of each profiled launch kind and a display name.
    Filter launches: 'y_acc' + 'z_cheb' = accumulate kernel in two launches (planes: w, x, y tiles; then z tiles),
    'y_acc' alone = accumulate kernel in one launch, 'x_store' present = three register-operand axis passes."""
    acc2 = "x_store" not in passes and "z_cheb" in passes
    acc1 = "x_store" not in passes and "z_cheb" not in passes
    plane_t = "x_td" not in passes
    tma_t = not plane_t and n >= 256
    m = {
        "x_store": (48.0 + 16.0 + 8.0 / nvec, f"axis_lean_kernel<{n},8,real,x> (x round trip, potential, recurrence, series every 2nd term)"),
        "y_acc": ((64.0 + 8.0 / nvec, f"acc_tma_kernel<{n}> (x and y tiles of whole planes: TMA loads, in-place round trips, bulk reduce-add; Clenshaw v read)") if acc2
                  else ((64.0 + 8.0 / nvec, f"acc_tma_kernel<{n}> (x, y and z tiles of whole vectors in one launch)") if acc1
                        else (48.0, f"axis_lean_kernel<{n},8,real,y> (y round trip, accumulate)"))),
        "z_cheb": (48.0, f"acc_tma_kernel<{n}> (z tiles: TMA tensor loads, bulk reduce-add)" if acc2 else f"axis_lean_kernel<{n},8,real,z> (z round trip, accumulate)"),
        "x_td": (32.0 + 16.0 / nvec, f"td_tma_kernel<{n},x> (x factor of exp(-iT dt), phases kept in registers across a block's vectors)" if tma_t
                 else f"axis_lean_kernel<{n},8,complex,x> (x factor of exp(-iT dt), phase on load)"),
        "y_td": ((32.0 + 16.0 / nvec, f"plane kernel<{n},8,complex> (x and y factors of exp(-iT dt), team- or CTA-owned planes)") if plane_t
                 else (32.0, f"td_tma_kernel<{n},y> (y factor of exp(-iT dt))" if tma_t else f"axis_lean_kernel<{n},8,complex,y> (y factor of exp(-iT dt))")),
        "z_td": (32.0 + 8.0 / nvec, f"td_tma_kernel<{n},z> (z factor, density summed in registers over a block's vectors)" if tma_t
                 else f"axis_lean_kernel<{n},8,complex,z> (z factor, phase / density on store)"),
        "kb_project": (16.0 * kb_frac + 32.0 * kb_frac / nvec, "kb_project_kernel<4> (gather-dot over sphere points)"),
        "kb_scatter": (32.0 * kb_frac + 32.0 * kb_frac / nvec, "kb_scatter_kernel<4> (FP64 atomics where spheres overlap)"),
        "density": (16.0, "density_kernel (rho from all vectors; first step of a call only)"),
        "density_points": (16.0 * uniq_frac + 16.0 * uniq_frac / nvec, "density_points_kernel (rho corrected at the distinct sphere points around the closing nonlocal factor)"),
    }
    return m


def bound_fraction(bytes_per_unit, flops_per_unit, units, seconds, hbm_gbs, fp64_flops):
    """achieved fraction of the roofline = W * max(B_c / BW, F_c / P64) / t."""
    t_hbm = bytes_per_unit / (hbm_gbs * 1e9)
    t_f64 = flops_per_unit / fp64_flops if fp64_flops else 0.0
    lim = max(t_hbm, t_f64)
    return {"bytes_per_unit": bytes_per_unit, "flops_per_unit": flops_per_unit,
            "bound": "hbm" if t_hbm >= t_f64 else "fp64",
            "achieved": bytes_per_unit * units / seconds / 1e9, "unit": "GB/s", "frac": lim * units / seconds,
            "frac_hbm": t_hbm * units / seconds, "frac_fp64": t_f64 * units / seconds}


def run_gpu(args):
    import torch
    import torch.distributed as dist
    from paper_2601_21005_b200 import api

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    w = W.make_workload(WORKLOAD, nvec=args.nvec)
    g = w.grid
    nvec = w.nvec
    coeffs = np.ascontiguousarray(w.coeffs[:SLICE_APPLIES + 1])
    units_f, units_t = g.ng * nvec * SLICE_APPLIES, g.ng * nvec * SLICE_TD
    units_rank = units_f + units_t
    stream = torch.cuda.current_stream(dev)
    ctx = api.context_for(w, max_nvec=nvec, stream=stream, device=f"cuda:{local}")
    first = shard.first_vector(rank, nvec)                   # each rank owns its own vectors (replicas, weak scaling)
    psi = torch.empty((nvec,) + g.shape, dtype=torch.complex128, device=dev)
    ctx.sgw_set_td(1, w.rho_scale)

    def barrier():
        torch.cuda.synchronize(dev)
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(args.steps)]

    def step(e=None):
        ctx.sgw_random_vectors(W.SEED_VEC, first, nvec, psi)                 # a1
        if e:
            e[0].record(stream)
        ctx.sgw_cheb_filter(psi, coeffs, w.emin, w.emax)                      # a2-a7
        if e:
            e[1].record(stream)
        ctx.sgw_td_propagate(psi, w.dt, SLICE_TD)                             # a8-a10
        if e:
            e[2].record(stream)

    for _ in range(args.warmup):
        step()
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    l0 = ctx.sgw_launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(stream)
    for k in range(args.steps):
        step(ev[k])
    e1.record(stream)
    barrier()
    ms = e0.elapsed_time(e1)
    launches = ctx.sgw_launch_count() - l0
    clocks = sampler.stop() if rank == 0 else None
    ms_f = sum(e[0].elapsed_time(e[1]) for e in ev)
    ms_t = sum(e[1].elapsed_time(e[2]) for e in ev)
    ms = shard.max_over_ranks(ms, dev)
    value = shard.whole_job_rate(units_rank, world, args.steps, ms)
    fp64_flops = ctx.sgw_probe_fp64()                                         # at the clocks the run leaves the device at

    # ---- per-pass breakdown: one separate step with an event pair around every launch (not the headline loop)
    ctx.sgw_profile_reset()
    ctx.sgw_profile_enable(1)
    ctx.sgw_random_vectors(W.SEED_VEC, first, nvec, psi)
    ctx.sgw_cheb_filter(psi, coeffs, w.emin, w.emax)
    passes_f = collect_passes(ctx)
    ctx.sgw_profile_reset()
    ctx.sgw_td_propagate(psi, w.dt, SLICE_TD)
    passes_t = collect_passes(ctx)
    ctx.sgw_profile_enable(0)
    norms = ctx.sgw_norms(psi)
    finite = bool(torch.isfinite(norms).all())

    # ---- end to end: host buffers, H2D of the start vectors and D2H of the result inside the timed region
    e2e = None
    if not args.no_e2e:
        e2e = run_e2e(torch, ctx, w, psi, coeffs, stream, dev, first, barrier, min(args.steps, 3), world, units_rank)

    others = None
    if world == 1 and not args.no_others:
        del psi
        ctx.close()
        torch.cuda.empty_cache()
        others = run_other_configs(torch, api, dev, stream, args, fp64_flops)

    if rank == 0:
        peak, peak_src = measured_peaks()
        kb_frac = float(w.kb.sph_idx.size) / g.ng
        uniq_frac = float(np.unique(w.kb.sph_idx).size) / g.ng if w.kb.sph_idx.size else 0.0
        model = pass_model({**passes_f, **passes_t}, nvec, g.nx, kb_frac, uniq_frac)
        allp = {k: dict(v, stage="filter") for k, v in passes_f.items()}
        allp.update({k: dict(v, stage="td") for k, v in passes_t.items()})
        dn, dv = max(allp.items(), key=lambda kv: kv[1]["ms_total"])
        bpu, kname = model.get(dn, (32.0, dn))
        units_launch = g.ng * nvec
        avg_ms = dv["ms_total"] / dv["launches"]
        ach = bpu * units_launch / (avg_ms * 1e-3) / 1e9
        traffic_pu, traffic_src = ncu_traffic(dn)          # ncu capture at fewer vectors: scaled per grid-pt*vector
        traffic = traffic_pu * units_launch if traffic_pu else None
        lg = math.log2(g.ng)
        cheb = bound_fraction(80.0 + 8.0 / nvec, 10.0 * lg + 20.0, units_f * args.steps, ms_f * 1e-3, peak, fp64_flops)
        td = bound_fraction(32.0 + 40.0 / nvec, 10.0 * lg + 30.0, units_t * args.steps, ms_t * 1e-3, peak, fp64_flops)
        for name, ps in (("filter", passes_f), ("td", passes_t)):
            for k_, v_ in ps.items():
                b_ = model.get(k_, (None, None))[0]
                v_["avg_ms"] = v_["ms_total"] / v_["launches"]
                if b_:
                    v_["bytes_per_unit"] = b_
                    v_["algorithmic_gbs"] = b_ * units_launch / (v_["avg_ms"] * 1e-3) / 1e9
                    v_["frac_of_hbm_peak"] = v_["algorithmic_gbs"] / peak
        cpu_val, cpu_dt, cpu_nv, cpu_cores, cpu_what = oracle_sample(os.cpu_count() or 1, 4, 1)
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(nvec),
                       "l2": f"inputs larger than L2 (each vector array {g.ng * nvec * 16 / 1e9:.1f} GB per GPU)",
                       "timing": "headline loop without per-launch events; pass breakdown from one separate profiled step",
                       "kinetic_operator": "full 1/2 k^2 (the paper's E_cut = 28 Ha cap is reading R-14: see sgw_set_kinetic_cutoff / other_configs)"},
            "clocks": clocks,
            "e2e": e2e,
            "gpu_launches": int(launches),
            "stage_rates": {"filter_units_per_s": units_f * args.steps / (ms_f * 1e-3), "filter_ms_per_application": ms_f / args.steps / SLICE_APPLIES,
                            "td_units_per_s": units_t * args.steps / (ms_t * 1e-3), "td_ms_per_step": ms_t / args.steps / SLICE_TD},
            "roofline": {"bound": "hbm", "kernel": kname, "stage": dv["stage"], "achieved": ach, "peak": peak, "unit": "GB/s",
                         "frac": ach / peak, "traffic": traffic, "traffic_source": traffic_src,
                         "algorithmic_bytes_per_launch": bpu * units_launch, "bytes_per_unit": bpu, "avg_launch_ms": avg_ms,
                         "peak_source": peak_src, "kernel_share_of_profiled_step": dv["ms_total"] / sum(v["ms_total"] for v in allp.values()),
                         "term_strict": cheb, "passes": passes_f},
            "roofline_td": dict(td, passes=passes_t, peak=peak),
            "fp64_peak_measured": {"flops_per_s": fp64_flops, "how": "sgw_probe_fp64: dependent-free DFMA loop right after the timed region",
                                   "nominal_flops_per_s": 148 * 64 * 2 * 1.965e9},
            "checks": {"finite": finite},
            "other_configs": others,
            "cpu_baseline": {"value": cpu_val, "unit": UNIT, "cores": cpu_cores, "kind": "oracle", "sample": f"{cpu_what} ({cpu_dt:.1f} s)"},
        }
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def run_e2e(torch, ctx, w, psi, coeffs, stream, dev, first, barrier, steps, world, units_rank):
    """The same step through the C-ABI with HOST buffers: start vectors copied host -> device and the result copied
    device -> host inside the timed region (one pinned buffer per vector, so a failed pin degrades per vector)."""
    nvec = w.nvec
    ctx.sgw_random_vectors(W.SEED_VEC, first, nvec, psi)
    pinned = True
    h_in, h_out = [], []
    for v in range(nvec):
        try:
            a = torch.empty(w.grid.shape, dtype=torch.complex128, pin_memory=True)
            b = torch.empty(w.grid.shape, dtype=torch.complex128, pin_memory=True)
        except RuntimeError:
            pinned = False
            a = torch.empty(w.grid.shape, dtype=torch.complex128)
            b = torch.empty(w.grid.shape, dtype=torch.complex128)
        a.copy_(psi[v])
        h_in.append(a)
        h_out.append(b)
    nbytes = nvec * w.grid.ng * 16
    # Pipelined: the start vectors arrive in chunks on a copy stream and the filter of a chunk starts when its chunk
    # has landed (the filter shards over vectors; the TD-Hartree steps couple all vectors through rho and wait for the
    # last chunk); results leave on a second copy stream from one of two device buffers while the next step computes
    # in the other.  Every byte of every step crosses inside the timed region.
    chunk = 8 if nvec % 8 == 0 else nvec
    try:
        bufs = [psi, torch.empty_like(psi)]
    except RuntimeError:                                   # not enough device memory for a second buffer: one buffer, serial steps
        bufs = [psi]
    cs_in, cs_out = torch.cuda.Stream(dev), torch.cuda.Stream(dev)
    ev_out = [None] * len(bufs)

    def step(i):
        b = i % len(bufs)
        buf = bufs[b]
        ev_in = []
        with torch.cuda.stream(cs_in):
            if ev_out[b] is not None:
                cs_in.wait_event(ev_out[b])                # the buffer's previous results have left
            else:
                cs_in.wait_stream(stream)
            for c0 in range(0, nvec, chunk):
                for v in range(c0, c0 + chunk):
                    buf[v].copy_(h_in[v], non_blocking=True)
                e = torch.cuda.Event()
                e.record(cs_in)
                ev_in.append(e)
        for k, c0 in enumerate(range(0, nvec, chunk)):
            stream.wait_event(ev_in[k])
            ctx.sgw_cheb_filter(buf[c0:c0 + chunk], coeffs, w.emin, w.emax)
        ctx.sgw_td_propagate(buf, w.dt, SLICE_TD)
        done = torch.cuda.Event()
        done.record(stream)
        with torch.cuda.stream(cs_out):
            cs_out.wait_event(done)
            for v in range(nvec):
                h_out[v].copy_(buf[v], non_blocking=True)
            ev_out[b] = torch.cuda.Event()
            ev_out[b].record(cs_out)

    def drain():
        for e in ev_out:
            if e is not None:
                stream.wait_event(e)

    step(0)
    drain()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(stream)
    for i in range(steps):
        step(i + 1)
    drain()                                                # the last results are on the host before the clock stops
    e1.record(stream)
    barrier()
    ms = shard.max_over_ranks(e0.elapsed_time(e1), dev)
    checksum = float(sum(float(torch.view_as_real(b[0]).abs().sum()) for b in h_out))
    return {"value": shard.whole_job_rate(units_rank, world, steps, ms), "unit": UNIT, "h2d_bytes_per_step": nbytes,
            "d2h_bytes_per_step": nbytes, "ms_per_step": ms / steps, "steps": steps, "pinned": pinned, "checksum_plane0": checksum,
            "pipeline": f"H2D in chunks of {chunk} vectors on a copy stream overlapping the filter of the previous chunk; D2H on a second "
                        f"copy stream overlapping the next step ({len(bufs)} device buffer(s))",
            "note": "the config uploads once per 2047 applications + 500 steps; this slice pays the same transfer for 16 + 4"}


def timed(torch, stream, dev, fn):
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize(dev)
    e0.record(stream)
    fn()
    e1.record(stream)
    torch.cuda.synchronize(dev)
    return e0.elapsed_time(e1)


def run_other_configs(torch, api, dev, stream, args, fp64_flops):
    """The other BASELINE.json configs, each with its own strict-roofline fraction: cfg1 and cfg2 at full vector count
    and (cfg1) full length, cfg3 as one 64-vector sub-batch, cfg0 (launch-latency bound)."""
    peak, _ = measured_peaks()
    out = {}
    # cfg1: the whole 512-term filter on 64 vectors (round 1's headline)
    w = W.make_workload("cfg1")
    ctx = api.context_for(w, max_nvec=w.nvec, stream=stream, device=str(dev))
    psi = ctx.sgw_random_vectors(W.SEED_VEC, 0, w.nvec)
    ctx.sgw_cheb_filter(psi, w.coeffs[:9], w.emin, w.emax)
    best = min(timed(torch, stream, dev, lambda: (ctx.sgw_random_vectors(W.SEED_VEC, 0, w.nvec, psi),
                                                   ctx.sgw_cheb_filter(psi, w.coeffs, w.emin, w.emax))) for _ in range(2))
    units = w.grid.ng * w.nvec * (w.nterms - 1)
    out["cfg1"] = {"what": "96^3, Si35H36 V_loc, 64 vectors, all 512 terms (511 applications), RNG included", "filter_ms": best,
                   "filter_units_per_s": units / (best * 1e-3),
                   "term_strict": bound_fraction(80.0 + 8.0 / w.nvec, 10.0 * math.log2(w.grid.ng) + 20.0, units, best * 1e-3, peak, fp64_flops)}
    # the cost of the paper's operator with its kinetic-energy cutoff (non-separable, five-pass route)
    if hasattr(ctx, "sgw_set_kinetic_cutoff"):
        ctx.sgw_set_kinetic_cutoff(28.0)
        emax_c = min(28.0, 1.5 * (math.pi / w.grid.hx) ** 2) + float(w.vloc.max())      # the narrower window the cutoff buys
        co = W.cheb_coeffs(W.sqrt_fermi, w.emin, emax_c, 65)
        ctx.sgw_random_vectors(W.SEED_VEC, 0, w.nvec, psi)
        msc = timed(torch, stream, dev, lambda: ctx.sgw_cheb_filter(psi, co, w.emin, emax_c))
        out["cfg1"]["with_kinetic_cutoff_28Ha"] = {"what": "same grid and vectors, kinetic operator min(1/2 k^2, 28 Ha) (P:142), 64 applications",
                                                    "filter_units_per_s": w.grid.ng * w.nvec * 64 / (msc * 1e-3)}
        ctx.sgw_set_kinetic_cutoff(0.0)
    ctx.close()
    del psi
    torch.cuda.empty_cache()
    # cfg2: TD steps with the Hartree rebuild
    w = W.make_workload("cfg2", nterms=129)
    ctx = api.context_for(w, max_nvec=w.nvec, stream=stream, device=str(dev))
    psi = ctx.sgw_random_vectors(W.SEED_VEC, 0, w.nvec)
    ctx.sgw_cheb_filter(psi, w.coeffs[:33], w.emin, w.emax)
    scratch = psi.clone()                                                      # the filter leg: 128 applications on a copy
    co = w.coeffs
    ctx.sgw_cheb_filter(scratch, co[:9], w.emin, w.emax)
    msf = timed(torch, stream, dev, lambda: ctx.sgw_cheb_filter(scratch, co, w.emin, w.emax))
    units_f = w.grid.ng * w.nvec * 128
    del scratch
    ctx.sgw_set_td(1, w.rho_scale)
    ctx.sgw_td_propagate(psi, w.dt, 10)
    n0 = ctx.sgw_norms(psi)
    nst = args.td_steps
    ms = timed(torch, stream, dev, lambda: ctx.sgw_td_propagate(psi, w.dt, nst))
    units = w.grid.ng * w.nvec * nst
    out["cfg2"] = {"what": f"128^3, Si87H76 V_loc, 16 filtered vectors, 128 filter applications (timing only), {nst} of the 2000 TD-Hartree steps",
                   "filter_units_per_s": units_f / (msf * 1e-3),
                   "term_strict": bound_fraction(80.0 + 8.0 / w.nvec, 10.0 * math.log2(w.grid.ng) + 20.0, units_f, msf * 1e-3, peak, fp64_flops),
                   "td_ms_per_step": ms / nst,
                   "td_units_per_s": units / (ms * 1e-3), "norm_drift": float((ctx.sgw_norms(psi) / n0 - 1.0).abs().max()),
                   "td_strict": bound_fraction(32.0 + 40.0 / w.nvec, 10.0 * math.log2(w.grid.ng) + 30.0, units, ms * 1e-3, peak, fp64_flops)}
    ctx.close()
    del psi
    torch.cuda.empty_cache()
    # cfg3: one 64-vector sub-batch of the 256
    w = W.make_workload("cfg3", nvec=64)
    ctx = api.context_for(w, max_nvec=64, stream=stream, device=str(dev))
    psi = ctx.sgw_random_vectors(W.SEED_VEC, 0, 64)
    ctx.sgw_cheb_filter(psi[:2].clone(), w.coeffs[:3], w.emin, w.emax)
    ms = timed(torch, stream, dev, lambda: ctx.sgw_cheb_filter(psi, w.coeffs[:17], w.emin, w.emax))
    units = w.grid.ng * 64 * 16
    ctx.sgw_set_td(1, w.rho_scale)
    ctx.sgw_td_propagate(psi, w.dt, 1)
    mst = timed(torch, stream, dev, lambda: ctx.sgw_td_propagate(psi, w.dt, 4))
    out["cfg3"] = {"what": "256^3, Si705H300 V_loc + 705 KB spheres, one 64-vector sub-batch of the 256, 16 of the 2047 applications; 4 TD-Hartree steps",
                   "filter_units_per_s": units / (ms * 1e-3),
                   "term_strict": bound_fraction(80.0 + 8.0 / 64, 10.0 * math.log2(w.grid.ng) + 20.0, units, ms * 1e-3, peak, fp64_flops),
                   "td_units_per_s": w.grid.ng * 64 * 4 / (mst * 1e-3)}
    ctx.close()
    del psi
    torch.cuda.empty_cache()
    # cfg0: launch-latency bound; the repeated call replays a cached CUDA graph
    w = W.make_workload("cfg0")
    ctx = api.context_for(w, max_nvec=w.nvec, stream=stream, device=str(dev))
    psi0 = ctx.sgw_random_vectors(W.SEED_VEC, 0, w.nvec)
    psi = psi0.clone()
    best = None
    for _ in range(4):
        psi.copy_(psi0)
        m_ = timed(torch, stream, dev, lambda: ctx.sgw_cheb_filter(psi, w.coeffs, w.emin, w.emax))
        best = m_ if best is None or m_ < best else best
    out["cfg0"] = {"what": "32^3, 4 vectors, all 128 terms (launch-latency bound: roofline fraction not meaningful)", "filter_ms": best,
                   "filter_units_per_s": w.grid.ng * w.nvec * 127 / (best * 1e-3)}
    ctx.close()
    return out


def write_traffic(csv_paths, source, units_per_launch):
    """Post-processing of ncu raw pages (ncu -i <rep> --page raw --csv > csv; several files separated by commas): dram
    bytes per launch and per grid-pt*vector for every kernel kind, written to profiles/r02_traffic.json, which the bench
    line's roofline.traffic reads (scaled to its own units per launch)."""
    import csv
    acc = {}
    nacc = 0
    for csv_path in csv_paths.split(","):
        nacc = _traffic_rows(csv, csv_path, acc, nacc)
    out = {"source": source, "units_per_launch_in_capture": units_per_launch,
           "kernels": {k: {"dram_bytes_per_launch": v["bytes"] / v["launches"], "dram_bytes_per_unit": v["bytes"] / v["launches"] / units_per_launch,
                           "avg_ms_under_ncu": v["ms"] / v["launches"], "launches": v["launches"], "kernel": v["kernel"]}
                       for k, v in acc.items()}}
    json.dump(out, open(TRAFFIC_JSON, "w"), indent=1)
    print(json.dumps(out, indent=1))


def _traffic_rows(csv, csv_path, acc, nacc):
    rows = list(csv.reader(open(csv_path)))
    hdr = rows[0]
    col = {n: i for i, n in enumerate(hdr)}
    rd, wr, nm, dur = col["dram__bytes_read.sum"], col["dram__bytes_write.sum"], col["Kernel Name"], col["gpu__time_duration.sum"]
    units = rows[1]
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}

    def key_of(name):
        if "acc_tma" in name:
            return "acc"
        if "td_tma" in name:                # td_tma_kernel<N, axis>
            ax = name.split("<")[1].split(">")[0].replace(" ", "").replace("(int)", "").split(",")
            return {"0": "x_td", "1": "y_td", "2": "z_td"}.get(ax[1] if len(ax) > 1 else "", "tdk")
        cplx = False
        if "<" in name:
            args_ = name.split("<")[1].split(">")[0].replace(" ", "").replace("(bool)", "").replace("(int)", "").split(",")
            cplx = len(args_) > 2 and args_[2] in ("true", "1")
        fam = "td" if cplx else None
        if "kb_project" in name:
            return "kb_project"
        if "kb_scatter" in name:
            return "kb_scatter"
        if "density_points" in name:
            return "density_points"
        if "density" in name:
            return "density"
        if "plane" in name:
            return "y_td" if fam else "y_acc"
        if "axis_lean" in name:
            axis = {"0": "x", "1": "y", "2": "z"}[args_[3]]
            if cplx:
                return f"{axis}_td"
            return {"x": "x_store", "y": "y_acc", "z": "z_cheb"}[axis]
        return None
    ntd = 0
    for r in rows[2:]:
        k = key_of(r[nm])
        if not k:
            continue
        if k == "acc":                      # two launches per term: planes (y_acc), then z columns (z_cheb)
            k = "y_acc" if nacc % 2 == 0 else "z_cheb"
            nacc += 1
        if k == "tdk":                      # three launches per step: x, y, z
            k = ("x_td", "y_td", "z_td")[ntd % 3]
            ntd += 1
        b = float(r[rd].replace(",", "")) * scale.get(units[rd], 1.0) + float(r[wr].replace(",", "")) * scale.get(units[wr], 1.0)
        tscale = {"ns": 1e-6, "us": 1e-3, "ms": 1.0, "s": 1e3}.get(units[dur], 1.0)
        e = acc.setdefault(k, {"launches": 0, "bytes": 0.0, "ms": 0.0, "kernel": r[nm][:120]})
        e["launches"] += 1
        e["bytes"] += b
        e["ms"] += float(r[dur].replace(",", "")) * tscale
    return nacc


def spawn_ranks(args):
    """python bench.py --gpus N outside torchrun: start the N ranks ourselves (one process per GPU)."""
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    raise SystemExit(subprocess.call(cmd))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="sgw", choices=["sgw", "reference"])
    ap.add_argument("--nvec", type=int, default=None, help="vectors in flight (profiling runs under ncu only; default: the config's 32)")
    ap.add_argument("--no-others", action="store_true", help="skip the other configs (cfg0-cfg3)")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer leg (profiling runs under ncu only)")
    ap.add_argument("--td-steps", type=int, default=100, help="timed steps of the cfg2 TD entry (default 100 of the 2000)")
    ap.add_argument("--write-traffic", default=None, metavar="NCU_RAW_CSV",
                    help="post-process an ncu raw page into profiles/r02_traffic.json and exit (no GPU needed)")
    ap.add_argument("--traffic-source", default="profiles/r02_cfg4_ncu.md")
    ap.add_argument("--traffic-units", type=float, default=8 * 384.0 ** 3, help="grid-pt*vectors per launch in the ncu capture")
    args = ap.parse_args()
    if args.write_traffic:
        write_traffic(args.write_traffic, args.traffic_source, args.traffic_units)
        return
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        spawn_ranks(args)
    if args.impl == "reference":
        run_reference(args)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()

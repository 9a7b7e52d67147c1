#!/usr/bin/env python
"""bench.py -- SHO project + add-back throughput on B200 (BASELINE.json metric), one JSON line.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--impl ours|reference]

A step is one pass of the whole hot path over one batch of synthetic input: c = sho_project(psi)
followed by psi' += sho_add(c).  ``value`` is psi-GB/s(box): the bytes of every atom's psi box
(read once by project, read + written once by add: 3 * sum_a |box_a| * nbands * sizeof(elem)) divided
by the device time of the step, inputs resident in HBM.  ``e2e`` is the same metric through the
HOST-buffer C-ABI call sho_apply_host (project -> D c -> add; psi crosses the link once each way), copies inside the
timed region, beside the link rates measured in the same run; ``e2e.project_host_plus_add_host`` keeps round 1's
definition (sho_project_host then sho_add_host).
``--impl reference`` times the CPU oracle (oracle/, test infrastructure) on a bounded sample.
See DESIGN.md "Measurement" for every definition used here.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1905_00480_b200 import workloads  # noqa: E402  (seeded inputs; no method arithmetic)

METRIC = "SHO project+add psi-GB/s(box) at 1 B200 (HBM-roofline metric of BASELINE.json); atom*band projections/s in detail"
ESZ = {"r64": 8, "c128": 16, "r32": 4, "c64": 8}
# FP64 pipe peak derived from the guide's unit counts: 148 SMs x 64 FP64 FMA
# lanes x 2 flop x 1.965 GHz (clocks.max.sm).  DMMA and DFMA share this pipe (measured: 37.1 TFLOP/s both).
FP64_PEAK_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12
FP32_PEAK_TFLOPS = 2 * FP64_PEAK_TFLOPS


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return json.load(f), "measured"
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0}, "fallback"


def committed_traffic(workload, dtype, kernel):
    """dram__bytes_read + dram__bytes_write of one launch of ``kernel``, read from the committed summary of the
    ncu --set full capture of this workload (profiles/r<N>_final_<workload>_ncu_full.txt, the latest round that has
    one; its first line names the element type, its second the command).  (None, None) if there is no capture."""
    import glob
    import re
    unit = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}
    for path in sorted(glob.glob(os.path.join(ROOT, "profiles", "r*_final_%s_ncu_full.txt" % workload)), reverse=True):
        with open(path) as f:
            lines = f.read().splitlines()
        if not lines or dtype not in lines[0]:
            continue
        cur, found = None, {}
        for ln in lines:
            if ln.startswith("kernel:"):
                cur = ln
            elif cur and re.search(r"\b%s\b" % re.escape(kernel), cur):
                m = re.match(r"\s*dram__bytes_(read|write)\.sum\s+(\w+)\s+([0-9.eE+-]+)\s*$", ln)
                if m and m.group(2) in unit and m.group(1) not in found:
                    found[m.group(1)] = float(m.group(3)) * unit[m.group(2)]
        if len(found) == 2:
            return found["read"] + found["write"], "%s (ncu --set full, one launch)" % os.path.relpath(path, ROOT)
    return None, None


def geometry(w, boxes=None):
    """Counts only (no method arithmetic): box points and algorithmic flops of one project (= one add)
    launch over all atoms and bands.  F = 2 P [ box M + n_z n_x pairs + n_z N_SHO ] per atom and band
    (first-, second- and third-axis contraction of the separable scheme)."""
    if boxes is None:
        import oracle  # only reached from the cpu_baseline / reference legs
        boxes = np.zeros((w.natoms, 3, 2), np.int64)
        for a in range(w.natoms):
            lo, hi, _ = oracle.box(w.ng, w.h, w.periodic, w.pos[a], w.sigma[a], w.rcut_sigma)
            boxes[a, :, 0], boxes[a, :, 1] = lo, hi
    n = np.maximum(boxes[:, :, 1].astype(np.int64) - boxes[:, :, 0] + 1, 0)
    box = n[:, 0] * n[:, 1] * n[:, 2]
    M = w.numax + 1
    pairs, nsho = M * (M + 1) // 2, M * (M + 1) * (M + 2) // 6
    P = 2 if w.is_complex else 1
    flops_atom = 2.0 * P * (box * M + n[:, 2] * n[:, 0] * pairs * (box > 0) + n[:, 2] * nsho * (box > 0))
    return {"box_points": box, "sum_box": int(box.sum()), "flops_per_band": float(flops_atom.sum()),
            "nsho": nsho, "P": P}


class ClockSampler:
    """nvidia-smi sampled DURING the timed region (B200_PROFILING.md clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "100"], stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            c = [x.strip() for x in line.split(",")]
            if len(c) < 7:
                continue
            try:
                sm.append(float(c[0])); mx.append(float(c[1])); pw.append(float(c[2]))
            except ValueError:
                continue
            for nm, v in zip(names, c[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), power_w_max=float(max(pw)),
                       samples=len(sm), reasons=sorted(reasons))
        return out


# --------------------------------------------------------------------------------------------------
# CPU oracle legs (cpu_baseline of our arm; the whole of --impl reference)


def oracle_sample_setup(w, cpu_seconds=20.0):
    """A bounded sample of the workload for the oracle: the first n_a atoms x n_b bands, sized for about
    ``cpu_seconds`` core-seconds (project + add).  The oracle's speed is calibrated on one atom first, so the
    sample runs at least 2 s of wall time on any host."""
    import oracle
    cores = oracle.num_threads()
    g = geometry(w)
    n_b = min(w.nbands, cores)
    psi = w.psi(range(n_b))
    if w.psi_dist == "zero":
        psi = workloads.Workload(**{**w.__dict__, "psi_dist": "normal"}).psi(range(n_b))
    wide = np.complex128 if w.is_complex else np.float64
    psi = psi.astype(wide)
    t_atom = 1e9
    for _ in range(2):                                             # the first call also loads the library and starts OpenMP
        t0 = time.perf_counter()
        c1 = oracle.project(w.ng, w.h, w.periodic, w.kfrac, w.pos[:1], w.sigma[:1], w.numax, psi, w.rcut_sigma)
        oracle.add(w.ng, w.h, w.periodic, w.kfrac, w.pos[:1], w.sigma[:1], w.numax, c1, psi, w.rcut_sigma)
        t_atom = min(t_atom, max(time.perf_counter() - t0, 1e-4))
    t_atom *= float(np.mean(g["box_points"])) / max(float(g["box_points"][0]), 1.0)
    wall = max(3.5, cpu_seconds / max(cores, 1))                   # seconds of wall time to aim for (>= 2 s)
    n_a = int(max(1, min(w.natoms, round(wall / t_atom))))
    # one atom over-estimates the time per atom (fixed costs): time the estimate and rescale it once
    t0 = time.perf_counter()
    c1 = oracle.project(w.ng, w.h, w.periodic, w.kfrac, w.pos[:n_a], w.sigma[:n_a], w.numax, psi, w.rcut_sigma)
    oracle.add(w.ng, w.h, w.periodic, w.kfrac, w.pos[:n_a], w.sigma[:n_a], w.numax, c1, psi, w.rcut_sigma)
    t_est = max(time.perf_counter() - t0, 1e-4)
    if t_est < 0.8 * wall:
        n_a = int(max(n_a, min(w.natoms, math.ceil(n_a * wall / t_est))))
    sub_box = int(g["box_points"][:n_a].sum()) * n_b
    return {"n_a": n_a, "n_b": n_b, "psi": psi, "cores": cores, "box_band_points": sub_box,
            "bytes": 3.0 * sub_box * ESZ[w.dtype], "pairs": n_a * n_b,
            "sample": "first %d atoms x %d bands of %s = %d (atom, band) pairs: oracle project (direct triple sum) then oracle add"
                      % (n_a, n_b, w.name, n_a * n_b)}


def oracle_sample_run(w, s):
    import oracle
    n_a = s["n_a"]
    t0 = time.perf_counter()
    c = oracle.project(w.ng, w.h, w.periodic, w.kfrac, w.pos[:n_a], w.sigma[:n_a], w.numax, s["psi"], w.rcut_sigma)
    oracle.add(w.ng, w.h, w.periodic, w.kfrac, w.pos[:n_a], w.sigma[:n_a], w.numax, c, s["psi"], w.rcut_sigma)
    return time.perf_counter() - t0


def run_reference(args, w):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    s = oracle_sample_setup(w, cpu_seconds=args.ref_cpu_seconds)
    for _ in range(args.warmup):
        oracle_sample_run(w, s)
    ts = [oracle_sample_run(w, s) for _ in range(args.steps)]
    t = float(np.sum(ts))
    value = s["bytes"] * args.steps / t / 1e9
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": "GB/s", "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * t / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": {"r64": "f64", "c128": "c128", "r32": "f32", "c64": "c64"}[w.dtype], "data": "synthetic",
        "config": {"workload": w.name, "note": "CPU oracle on a bounded sample of the workload"},
        "cpu_baseline": {"value": value, "unit": "GB/s", "cores": s["cores"], "kind": "oracle", "sample": s["sample"]},
        "e2e": {"value": value, "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "atom_band_per_s": s["n_a"] * s["n_b"] * args.steps / t,
    }
    print(json.dumps(line))
    return 0


# --------------------------------------------------------------------------------------------------


def stored_vs_on_the_fly(sho, torch, dev, w3, steps):
    """On-the-fly projection against the stored-projector baseline (a7) on one workload: median device times, table
    bytes, and the baseline's own bound max(table bytes / HBM, its flops / FP64 peak)."""
    plan = sho.plan_for(w3)
    g3 = geometry(w3, plan.boxes())
    tdt = {"r64": torch.float64, "c128": torch.complex128, "r32": torch.float32, "c64": torch.complex64}[w3.dtype]
    gen = torch.Generator(device=dev)
    gen.manual_seed(w3.seed)
    psi = torch.randn((w3.nbands, w3.ng[2], w3.ng[1], w3.ng[0]), dtype=tdt, device=dev, generator=gen)
    coeff = plan.new_coeff(w3.nbands, dev)
    stream = torch.cuda.current_stream()
    need = plan.tables_bytes()
    out = {"workload": w3.name, "table_bytes": need}
    if need > 0.8 * torch.cuda.mem_get_info(dev)[0]:
        out["status"] = "does not fit"
        plan.close()
        return out
    tb = plan.tables()

    def med(fn):
        for _ in range(2):
            fn()
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(max(steps, 3))]
        for a, b in evs:
            a.record(stream); fn(); b.record(stream)
        torch.cuda.synchronize()
        return float(np.median([a.elapsed_time(b) for a, b in evs])) * 1e-3

    t_fly = med(lambda: plan.project(psi, coeff, stream))
    t_sto = med(lambda: plan.project_stored(tb, psi, coeff, stream))
    tb.close()
    psi.zero_()
    t_add = med(lambda: plan.add(coeff, psi, stream))
    out["ms_add_on_the_fly"] = 1e3 * t_add
    plan.close()
    peaks, _ = measured_peaks()
    P = g3["P"]
    f_sto = 2.0 * P * g3["nsho"] * float(g3["sum_box"]) * w3.nbands       # non-separable: N_SHO MACs per box point and band
    bound = max(need / (peaks["hbm_gbs"] * 1e9), f_sto / (FP64_PEAK_TFLOPS * 1e12))
    out.update(status="ok", ms_project_on_the_fly=1e3 * t_fly, ms_project_stored=1e3 * t_sto, slowdown_vs_on_the_fly=t_sto / t_fly,
               table_gbs=need / t_sto / 1e9, stored_bound_ms=1e3 * bound, stored_frac_of_its_bound=bound / t_sto,
               on_the_fly_gain_if_stored_ran_at_its_bound=bound / t_fly)
    return out


def run_ours(args, w):
    import torch
    import torch.distributed as dist

    import paper_1905_00480_b200 as sho
    from paper_1905_00480_b200 import sharding

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    sho.lib()                                                        # fail loudly if libsho.so is missing

    plan = sho.plan_for(w)
    info = plan.info()
    g = geometry(w, plan.boxes())
    nb, esz, P = w.nbands, ESZ[w.dtype], g["P"]
    tdt = {"r64": torch.float64, "c128": torch.complex128, "r32": torch.float32, "c64": torch.complex64}[w.dtype]
    # weak scaling over bands: the job has world * nbands bands, rank r owns the contiguous
    # range sharding.band_range gives it and draws its psi from a seed of its own; no data-path collective
    band_lo, band_hi = sharding.band_range(world * nb, rank, world)
    assert band_hi - band_lo == nb
    gen = torch.Generator(device=dev)
    gen.manual_seed(w.seed * 1000 + band_lo)
    shape = (nb, w.ng[2], w.ng[1], w.ng[0])
    psi = torch.randn(shape, dtype=tdt, device=dev, generator=gen)   # read by project
    psi_out = torch.zeros(shape, dtype=tdt, device=dev)             # accumulated into by add (stays finite)
    coeff = plan.new_coeff(nb, dev)
    stream = torch.cuda.current_stream()

    bf = args.layout == "bf"
    if bf:
        psi = psi.permute(1, 2, 3, 0).contiguous()
        psi_out = psi_out.permute(1, 2, 3, 0).contiguous()
        work = torch.empty((min(nb, 64),) + shape[1:], dtype=tdt, device=dev)
    do_project = (lambda: plan.project_bf(psi, coeff, work, stream)) if bf else (lambda: plan.project(psi, coeff, stream))
    do_add = (lambda: plan.add_bf(coeff, psi_out, work, stream)) if bf else (lambda: plan.add(coeff, psi_out, stream))

    def step():
        do_project()
        do_add()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(args.steps)]
    sampler = ClockSampler(local) if rank == 0 else None
    barrier()
    for k in range(args.steps):
        ev[k][0].record(stream)
        do_project()
        ev[k][1].record(stream)
        do_add()
        ev[k][2].record(stream)
    barrier()
    clocks = sampler.stop() if sampler else None
    t_total = ev[0][0].elapsed_time(ev[-1][2]) * 1e-3
    # per-kernel times: median over the timed steps (the paper's protocol)
    t_prj = float(np.median([e[0].elapsed_time(e[1]) for e in ev])) * 1e-3
    t_add = float(np.median([e[1].elapsed_time(e[2]) for e in ev])) * 1e-3
    t_total, t_prj, t_add = sharding.max_over_ranks([t_total, t_prj, t_add], device=dev)

    box_bytes = float(g["sum_box"]) * nb * esz                        # B_box of one rank
    step_bytes = 3.0 * box_bytes * world
    value = step_bytes * args.steps / t_total / 1e9
    peaks, peak_kind = measured_peaks()
    F = g["flops_per_band"] * nb                                     # algorithmic flops of one project (= one add) launch
    dom, t_dom = ("sho_add_kernel", t_add) if t_add >= t_prj else ("sho_project_kernel", t_prj)
    alu_peak = FP64_PEAK_TFLOPS                                      # arithmetic is fp64 for all four dtypes
    traffic, traffic_src = committed_traffic(w.name, w.dtype, dom)
    roofline = {"bound": "alu", "kernel": dom, "achieved": F / t_dom / 1e12, "peak": alu_peak, "unit": "TFLOP/s",
                "frac": F / t_dom / 1e12 / alu_peak, "traffic": traffic, "traffic_source": traffic_src,
                "peak_source": "derived: 148 SM x 64 FP64 lanes x 2 x 1.965 GHz (DESIGN.md); DMMA/DFMA micro-benchmark in fp64_peak_measured_tflops",
                "flops_per_launch": F,
                "frac_project": F / t_prj / 1e12 / alu_peak, "frac_add": F / t_add / 1e12 / alu_peak}

    if bf:
        args.no_e2e = args.no_stored = True      # the remaining legs use the native layout
        psi_out = torch.zeros(shape, dtype=tdt, device=dev)
        psi = psi.permute(3, 0, 1, 2).contiguous()
    # ---- the three-step action project -> D -> add in one call (f2), device resident, outside the timed region ----
    dmat = torch.from_numpy(w.dmatrix(plan.nsho)).to(dev)
    plan.apply(dmat, psi_out, coeff, stream)
    ka = max(3, min(args.steps, 5))                                   # medians, like the per-kernel times above
    eva = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(ka)]
    for e0, e1, e2 in eva:
        psi_out.zero_()                                               # keeps psi finite over repeated applications
        e0.record(stream)
        plan.dmul(dmat, coeff, coeff, stream)
        e1.record(stream)
        plan.apply(dmat, psi_out, coeff, stream)
        e2.record(stream)
    torch.cuda.synchronize()
    t_dmul = float(np.median([e[0].elapsed_time(e[1]) for e in eva])) * 1e-3
    t_apply = float(np.median([e[1].elapsed_time(e[2]) for e in eva])) * 1e-3
    psi_out.zero_()

    # ---- end to end through the HOST-buffer C-ABI call sho_apply_host (pinned host memory): psi is uploaded once,
    # project -> D -> add run on the device, psi is downloaded once; the coefficients never leave the device ----
    e2e = None
    if not args.no_e2e:
        hp = torch.empty(shape, dtype=tdt, pin_memory=True)
        hd = torch.from_numpy(w.dmatrix(plan.nsho)).pin_memory()
        hp.copy_(psi)
        torch.cuda.synchronize()
        ke = max(1, min(args.steps, args.e2e_steps))
        plan.apply_host(hd, hp, stream)                                  # warm-up (allocates the plan workspace)
        hp.copy_(psi)
        barrier()
        t0 = time.perf_counter()
        for _ in range(ke):
            plan.apply_host(hd, hp, stream)
        torch.cuda.synchronize()
        te = time.perf_counter() - t0
        (te,) = sharding.max_over_ranks([te], device=dev)
        psi_b, d_b = int(np.prod(shape)) * esz, w.natoms * plan.nsho * plan.nsho * 8
        e2e = {"value": step_bytes * ke / te / 1e9, "unit": "GB/s", "h2d_bytes_per_step": psi_b + d_b,
               "d2h_bytes_per_step": psi_b, "steps": ke, "ms_per_step": 1e3 * te / ke,
               "call": "sho_apply_host (project -> D c -> add, one upload and one download of psi per step)"}
        # the host link measured in the same run: pinned H2D and D2H copies of up to 2 GB each, at the same time on two
        # streams (the pattern of the chunk pipeline); the step's link bound is the slower direction's bytes / rate
        nlink = min(psi_b, 2 << 30)
        src_h = hp.view(torch.uint8).reshape(-1)[:nlink]
        dst_h = torch.empty(nlink, dtype=torch.uint8, pin_memory=True)
        dev_a = torch.empty(nlink, dtype=torch.uint8, device=dev)
        dev_b = torch.empty(nlink, dtype=torch.uint8, device=dev)
        sa, sb = torch.cuda.Stream(dev), torch.cuda.Stream(dev)
        rates = []
        for _ in range(3):                                               # the first pass is a warm-up
            torch.cuda.synchronize()
            ea0, ea1, eb0, eb1 = (torch.cuda.Event(enable_timing=True) for _ in range(4))
            with torch.cuda.stream(sa):
                ea0.record(sa); dev_a.copy_(src_h, non_blocking=True); ea1.record(sa)
            with torch.cuda.stream(sb):
                eb0.record(sb); dst_h.copy_(dev_b, non_blocking=True); eb1.record(sb)
            torch.cuda.synchronize()
            rates.append((nlink / (ea0.elapsed_time(ea1) * 1e-3) / 1e9, nlink / (eb0.elapsed_time(eb1) * 1e-3) / 1e9))
        h2d_gbs, d2h_gbs = max(r[0] for r in rates[1:]), max(r[1] for r in rates[1:])
        link_bound = max((psi_b + d_b) / (h2d_gbs * 1e9), psi_b / (d2h_gbs * 1e9))
        e2e.update(pcie_h2d_gbs=h2d_gbs, pcie_d2h_gbs=d2h_gbs, link_bound_ms=1e3 * link_bound,
                   frac_of_link_bound=link_bound / (te / ke),
                   link_note="pinned H2D and D2H measured concurrently in this run; bound = max(h2d bytes / h2d rate, d2h bytes / d2h rate)")
        del src_h, dst_h, dev_a, dev_b
        # the round-1 end-to-end leg, kept so that the series stays comparable: sho_project_host (psi up, c down) followed
        # by sho_add_host (c and psi up, psi down)
        if w.natoms > 0:
            hc = torch.empty((w.natoms, nb, plan.nsho), dtype=tdt, pin_memory=True)
            hp.copy_(psi)
            plan.project_host(hp, hc, stream)
            hp.zero_()
            plan.add_host(hc, hp, stream)                                 # warm-up of both calls
            barrier()
            t0 = time.perf_counter()
            plan.project_host(hp, hc, stream)
            plan.add_host(hc, hp, stream)
            torch.cuda.synchronize()
            tpa = time.perf_counter() - t0
            (tpa,) = sharding.max_over_ranks([tpa], device=dev)
            c_b = w.natoms * nb * plan.nsho * esz
            e2e["project_host_plus_add_host"] = {"value": step_bytes / tpa / 1e9, "unit": "GB/s", "ms_per_step": 1e3 * tpa,
                                                 "h2d_bytes_per_step": 2 * psi_b + c_b, "d2h_bytes_per_step": psi_b + c_b,
                                                 "note": "the e2e definition of BENCH_r01 (two calls, psi crosses the link three times)"}
            del hc
        del hp, hd

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    fp64_meas = sho.measure_fp64_peak(20000) / 1e12
    # ---- stored-projector baseline (a7): the same projection from pre-sampled 3D tables in HBM;
    # outside the timed region of the step.  Tables that do not fit are reported with their size (the capacity wall).
    stored = None
    if not args.no_stored:
        need = plan.tables_bytes()
        free_b = torch.cuda.mem_get_info(dev)[0]
        stored = {"table_bytes": need}
        if need > 0.8 * free_b:
            stored.update(status="does not fit", free_bytes=int(free_b))
        else:
            tb = plan.tables()
            for _ in range(2):
                plan.project_stored(tb, psi, coeff, stream)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            ks = max(1, min(args.steps, 5))
            e0.record(stream)
            for _ in range(ks):
                plan.project_stored(tb, psi, coeff, stream)
            e1.record(stream)
            torch.cuda.synchronize()
            t_sto = e0.elapsed_time(e1) * 1e-3 / ks
            tb.close()
            stored.update(status="ok", ms_project_stored=1e3 * t_sto, table_gbs=need / t_sto / 1e9,
                          slowdown_vs_on_the_fly=t_sto / t_prj,
                          table_bytes_over_psi_box_bytes=need / box_bytes)
    # ---- stored-1D-table separable variant (f3): the same kernels reading the factor values
    # phi_n(u) of every atom from device memory instead of generating them; separates the gain of factorisation (both
    # variants have it) from the gain of on-the-fly sampling (the difference of the two times)
    sep1d = None
    if not args.no_stored and not bf:
        t1 = plan.tables1d()
        def med3(fn):
            for _ in range(2):
                fn()
            evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(max(3, min(args.steps, 5)))]
            for a, b in evs:
                a.record(stream); fn(); b.record(stream)
            torch.cuda.synchronize()
            return float(np.median([a.elapsed_time(b) for a, b in evs]))
        sep1d = {"table_bytes": plan.tables1d_bytes(),
                 "ms_project_stored1d": med3(lambda: plan.project_stored1d(t1, psi, coeff, stream)),
                 "ms_add_stored1d": med3(lambda: plan.add_stored1d(t1, coeff, psi_out, stream)),
                 "ms_project_on_the_fly": 1e3 * t_prj, "ms_add_on_the_fly": 1e3 * t_add}
        t1.close()
        psi_out.zero_()
    # cfg 3 is the config BASELINE.json states the on-the-fly vs stored comparison on; when the benched workload's tables do
    # not fit, run that comparison as a sub-leg (outside the timed region) so that it is observed in the default run too
    stored_cfg3 = None
    if not args.no_stored and w.name != "cfg3" and world == 1:
        del psi_out
        torch.cuda.empty_cache()
        stored_cfg3 = stored_vs_on_the_fly(sho, torch, dev, workloads.make(3), min(args.steps, 5))
    # the paper's own benchmark (sec. 6, tab. 1: 64^3, 665 atoms, 1024 bands, 56 coefficients, double) as a
    # sub-leg of the default run, outside the timed region: on-the-fly project / add and the stored-projector projection
    paper_nu5 = None
    if not args.no_stored and not w.name.startswith("paper") and world == 1:
        torch.cuda.empty_cache()
        paper_nu5 = stored_vs_on_the_fly(sho, torch, dev, workloads.make_paper(5, "r64"), min(args.steps, 5))
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        s = oracle_sample_setup(w, cpu_seconds=args.ref_cpu_seconds)
        tc = oracle_sample_run(w, s)
        cpu = {"value": s["bytes"] / tc / 1e9, "unit": "GB/s", "cores": s["cores"], "kind": "oracle", "sample": s["sample"],
               "seconds": tc, "atom_band_per_s": s["n_a"] * s["n_b"] / tc}
    line = {
        "metric": METRIC, "value": value, "unit": "GB/s", "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": 1e3 * t_total / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": {"r64": "f64", "c128": "c128", "r32": "f32", "c64": "c64"}[w.dtype], "data": "synthetic",
        "config": {"workload": w.name, "grid": list(w.ng), "h": w.h, "natoms": w.natoms, "numax": w.numax, "nbands_per_gpu": nb,
                   "elem": w.dtype, "layout": args.layout, "l2": "inputs larger than L2 (psi %.2f GB per GPU)" % (np.prod(shape) * esz / 1e9)
                   if np.prod(shape) * esz > 2.5e8 else "psi smaller than L2: L2-resident by design of the config",
                   "sharding": "bands (weak): each rank runs the config's nbands on its own psi, no collective"},
        "clocks": clocks, "e2e": e2e, "gpu_launches": 2 * args.steps, "roofline": roofline, "cpu_baseline": cpu,
        "detail": {
            "ms_project": 1e3 * t_prj, "ms_add": 1e3 * t_add,
            "psi_gbs_box_project": box_bytes / t_prj / 1e9, "psi_gbs_box_add": 2 * box_bytes / t_add / 1e9,
            "box_bytes_over_hbm_peak_project": box_bytes / t_prj / 1e9 / peaks["hbm_gbs"],
            "box_bytes_over_hbm_peak_add": 2 * box_bytes / t_add / 1e9 / peaks["hbm_gbs"],
            "box_bytes_over_hbm_peak_step": value / world / peaks["hbm_gbs"],
            "box_bytes_note": "psi-GB/s(box) counts every psi value once per box that holds it (the traffic of a kernel without reuse, "
                              "BASELINE.json's metric); these ratios exceed 1 when L2 / ownership tiling capture the overlap and are "
                              "NOT an HBM roofline -- see roofline (FP64 pipe) and roofline.traffic (real DRAM bytes)", "hbm_peak_gbs": peaks["hbm_gbs"], "hbm_peak_kind": peak_kind,
            "atom_band_per_s": world * info["atoms_nonempty"] * nb * args.steps / t_total,
            "tflops_project": F / t_prj / 1e12, "tflops_add": F / t_add / 1e12, "fp64_peak_measured_tflops": fp64_meas,
            "ms_dmul": 1e3 * t_dmul, "ms_apply_project_dmul_add": 1e3 * t_apply,
            "stored_baseline": stored, "stored_baseline_cfg3": stored_cfg3, "paper_nu5": paper_nu5, "pcie_gbs": ({"h2d": e2e["pcie_h2d_gbs"], "d2h": e2e["pcie_d2h_gbs"]} if e2e else None), "separable_stored1d": sep1d, "sum_box_points": g["sum_box"], "psi_bytes_unique": int(np.prod(shape)) * esz, "add_tile_pairs": info["add_pairs"],
        },
    }
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="5", help="BASELINE.json config 1..5 (default: the largest, cfg 5), or 'paper': "
                    "the paper's own benchmark (sec. 6: 64^3, fcc, 665 atoms, 1024 bands; --numax 0..5 = 1..56 coefficients)")
    ap.add_argument("--numax", type=int, default=5, help="numax of --config paper")
    ap.add_argument("--layout", default="xf", choices=["xf", "bf"], help="psi layout: x-fastest [b][z][y][x] (the ABI's native one) or "
                    "band-fastest [z][y][x][b] (the paper's, PAPER.md:371; converted in chunks of 64 bands by sho_project_bf / sho_add_bf)")
    ap.add_argument("--dtype", default=None, help="override the config's element type (cfg 4: r32 or r64)")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-stored", action="store_true", help="skip the stored-projector baseline leg")
    ap.add_argument("--ref-cpu-seconds", type=float, default=20.0)
    args = ap.parse_args()
    if args.config == "paper":
        w = workloads.make_paper(args.numax, args.dtype or "r64")
    else:
        w = workloads.make(int(args.config), dtype=args.dtype)
    if args.dtype in ("r32", "r64"):
        w.kfrac = None
    if args.impl == "reference":
        return run_reference(args, w)
    return run_ours(args, w)


if __name__ == "__main__":
    sys.exit(main())

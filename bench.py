#!/usr/bin/env python
"""bench.py -- throughput of the fused finite-volume step on B200 (contract in DESIGN.md section 8).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--extras]

A "step" is one explicit time step of the whole hot path (U, V and W updated together, eq. (3) of
arXiv 2006.01748) over BASELINE.json's headline workload: config 3, 8192 x 8192 cells, fp64,
layered discontinuous tensor, three tumour disks (synthetic, seeded: workloads.make(3)).

Prints ONE JSON line on stdout:
  value         cell-updates/s in GLUPS, whole job, inputs resident in HBM, K steps timed on the
                device (CUDA events recorded by libgg on its stream around the K launches)
  e2e           the same metric through the C ABI with HOST (pinned) buffers: upload tensor and
                state, K steps, download state, all inside the timed region
  roofline      compulsory bytes (72 B per cell-update in fp64) / measured launch time against the
                measured HBM copy peak (MEASURED_PEAKS.json); `traffic` (ncu DRAM bytes per launch)
                and `alu.instr_per_cell_step` come from profiles/ncu_traffic.json and are null
                unless that record was made for the kernel that ran AND for the csrc/ on disk
  configs       the other BASELINE.json configs (3 in fp32, 2, 4, 1, 0) on rank 0 at N = 1: GLUPS,
                us per step, the kernel AUTO resolved to, window parity against the oracle
  cpu_baseline  the CPU oracle, as it stands, on a bounded sample of the same workload
N > 1 (torchrun): the path does not shard without a halo exchange that north_star excludes, so
every rank runs an independent replica of the same workload ("replicas only", weak scaling);
value = all ranks' cell-updates / max-over-ranks device time.
`--impl reference` times the oracle (the reference arm of this tier) on rank 0 only.
`--record-traffic RAW.csv` (no GPU needed) turns `ncu -i X.ncu-rep --page raw --csv` output into
the profiles/ncu_traffic.json entries of the kernels it contains.
"""
from __future__ import annotations

import argparse
import csv
import glob
import hashlib
import json
import os
import re
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "cell-updates/s, explicit finite-volume step, fp64 8192^2 (BASELINE config 3)"   # --dtype f32: labelled fp32
UNIT = "GLUPS"
BYTES_PER_CELL = {"f64": 72.0, "f32": 36.0}   # 3 fields read + 3 written + 3 coefficients read
FALLBACK_HBM_GBS = 6650.0                      # /opt/skills/guides/B200_PROFILING.md
TRAFFIC_JSON = os.path.join(ROOT, "profiles", "ncu_traffic.json")
WORKLOAD3 = "BASELINE.json configs[3]: 8192x8192 {dtype}, 6-band discontinuous tensor, 3 tumour disks, h=1/64, d=10, alpha=1e-3"


def log(*a):
    print(*a, file=sys.stderr, flush=True)


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def csrc_sha16() -> str:
    """Hash of the kernel sources on disk: an ncu record made for other sources is stale."""
    h = hashlib.sha256()
    for f in sorted(glob.glob(os.path.join(ROOT, "paper_2006_01748_b200", "csrc", "*"))):
        h.update(os.path.basename(f).encode())
        h.update(open(f, "rb").read())
    return h.hexdigest()[:16]


def ncu_record(kernel_name):
    """The committed ncu record of `kernel_name` (per launch at 8192^2) if it was captured from
    the csrc/ now on disk, else None -- never a stale constant."""
    try:
        rec = json.load(open(TRAFFIC_JSON))
        if rec.get("csrc_sha16") != csrc_sha16():
            return None
        return rec["kernels"].get(kernel_name)
    except Exception:
        return None


def record_traffic(raw_csv):
    """profiles/ncu_traffic.json entries from an `ncu --page raw --csv` dump of 8192^2 launches."""
    rows = list(csv.reader(open(raw_csv)))
    hdr = rows[0]
    col = {h: i for i, h in enumerate(hdr)}

    def num(r, name):
        return float(r[col[name]].replace(",", "")) if name in col and r[col[name]] else None
    try:
        rec = json.load(open(TRAFFIC_JSON))
        if rec.get("csrc_sha16") != csrc_sha16():
            rec = {}
    except Exception:
        rec = {}
    rec = {"csrc_sha16": csrc_sha16(), "kernels": rec.get("kernels", {}),
           "source": "per launch at 8192x8192, from `ncu --set full` captures turned into CSV with "
                     "`ncu -i X.ncu-rep --page raw --csv` and recorded by `python bench.py "
                     "--record-traffic X.csv`; valid only for the csrc/ whose hash is csrc_sha16"}
    for r in rows[2:]:
        name = re.sub(r"\s+", "", r[col["Kernel Name"]])
        m = re.match(r"(?:void)?(?:gg::)?(gg_step_\w+<[^>]*>)", name)
        if not m:
            continue
        name = m.group(1)
        f64 = "<double" in name
        steps = 4 if "quad" in name else 2 if ("pair" in name or "stream2" in name) else 1
        scale_of = lambda m: {"Gbyte": 1e9, "Mbyte": 1e6, "Kbyte": 1e3, "byte": 1.0}.get(rows[1][col[m]], 1.0)
        rd = num(r, "dram__bytes_read.sum") * scale_of("dram__bytes_read.sum")
        wr = num(r, "dram__bytes_write.sum") * scale_of("dram__bytes_write.sum")
        scale = 1.0
        pipe = "smsp__inst_executed_pipe_fp64.sum" if f64 else "smsp__inst_executed_pipe_fma.sum"
        inst = num(r, pipe)
        if inst is None:
            # `--set full` has the pipe's utilisation but not its instruction count: warp
            # instructions = utilisation x peak rate (fp64: 1 per 2 cycles and SM sub-partition,
            # fma: 1 per cycle) x active cycles x 592 sub-partitions
            pct = num(r, ("sm__inst_executed_pipe_fp64" if f64 else "sm__inst_executed_pipe_fma") + ".avg.pct_of_peak_sustained_active")
            cyc = num(r, "smsp__cycles_active.avg")
            if pct is not None and cyc is not None:
                inst = pct / 100.0 * (0.5 if f64 else 1.0) * cyc * 592.0
                pipe += " (derived from the pipe's pct_of_peak_sustained_active)"
        entry = {"traffic_bytes_per_launch": (rd + wr) * scale, "steps_per_launch": steps,
                 "gpu_time_under_ncu": num(r, "gpu__time_duration.sum"),
                 "gpu_time_unit": rows[1][col["gpu__time_duration.sum"]]}
        if inst is not None:
            entry["pipe_instr_per_cell_step"] = inst * 32.0 / (8192.0 * 8192.0 * steps)
            entry["pipe_metric"] = pipe
        rec["kernels"][name] = entry
        log(f"recorded {name}: {entry}")
    json.dump(rec, open(TRAFFIC_JSON, "w"), indent=1)


class ClockSampler:
    """nvidia-smi clock / throttle-reason samples while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index, self.rows, self.proc = index, [], None

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                 "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def wait_first(self, timeout=5.0):
        """Block until nvidia-smi has delivered its first sample (it takes a few 100 ms to start),
        then drop what was sampled before the timed region."""
        t0 = time.perf_counter()
        while self.proc and not self.rows and time.perf_counter() - t0 < timeout:
            time.sleep(0.02)
        self.rows.clear()

    def __exit__(self, *exc):
        if self.proc:
            time.sleep(0.15)
            self.proc.terminate()
            self.t.join(timeout=2)

    def summary(self):
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
                for n, v in zip(names, r[2:6]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                pass
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": max(mx), "reasons": sorted(reasons),
                "samples": len(sm)}


# ---------------------------------------------------------------------------------------------
# CPU oracle leg (cpu_baseline / --impl reference): the oracle as it stands, bounded sample
# ---------------------------------------------------------------------------------------------
SAMPLE_ROWS = 2048


def oracle_sample(wl, steps, warmup=1, min_seconds=0.0, rows=SAMPLE_ROWS):
    """Time blocks of `steps` oracle steps on the first `rows` rows of the workload (full width,
    so the memory access pattern per row is the workload's), repeated until `min_seconds` have
    passed.  Returns (GLUPS, description, threads, seconds per step)."""
    import oracle
    rows = min(rows, wl.ny)
    sl = slice(0, rows)
    U, V, W = wl.U[0, sl], wl.V[0, sl], wl.W[0, sl]
    a, b, c = wl.a[sl], wl.b[sl], wl.c[sl]
    kw = dict(r=wl.r[0], d=wl.d[0], alpha=wl.alpha[0], c_r=wl.c_r[0], dt=wl.dt, dx=wl.h)
    oracle.step(U, V, W, a, b, c, n=max(warmup, 1), **kw)  # warm-up (page faults, library load)
    done, t = 0, 0.0
    while done == 0 or t < min_seconds:
        t0 = time.perf_counter()
        oracle.step(U, V, W, a, b, c, n=steps, **kw)
        t += time.perf_counter() - t0
        done += steps
    glups = rows * wl.nx * done / t / 1e9
    desc = (f"oracle/gg_oracle.cpp (fp64, OpenMP over rows), {done} steps ({done // steps} x {steps}) on rows "
            f"0..{rows - 1} x all {wl.nx} columns of {wl.name}, {t:.2f} s")
    return glups, desc, oracle.max_threads(), t / done


def run_reference(args, wl):
    """Reference arm of this tier = the CPU oracle.  A 'step' is one oracle step on the bounded
    sample (rows 0..2047 x all columns of the 8192^2 workload); W warm-up steps, then blocks of K
    timed steps until at least 2 s have passed."""
    glups, desc, cores, s_per_step = oracle_sample(wl, args.steps, warmup=args.warmup, min_seconds=2.0)
    return {
        "impl": "reference", "metric": METRIC, "value": glups, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": s_per_step * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": WORKLOAD3.format(dtype="f64"), "sample": desc},
        "cpu_baseline": {"value": glups, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
        "e2e": {"value": glups, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }


# ---------------------------------------------------------------------------------------------
# multi-rank aggregation ("replicas only": ranks never exchange field data)
# ---------------------------------------------------------------------------------------------
def max_over_ranks(x, world, device):
    """MAX of a per-rank scalar over all ranks (identity for world == 1)."""
    if world <= 1:
        return float(x)
    import torch
    import torch.distributed as td
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    td.all_reduce(t, op=td.ReduceOp.MAX)
    return float(t.item())


def job_glups(cells_per_rank, steps, ms_local, world, device):
    """Whole-job throughput: every rank advanced `cells_per_rank` cells by `steps` steps; the job
    took the slowest rank's device time.  Returns (GLUPS, ms_max)."""
    ms = max_over_ranks(ms_local, world, device)
    return cells_per_rank * world * steps / (ms * 1e-3) / 1e9, ms


# ---------------------------------------------------------------------------------------------
# GPU leg
# ---------------------------------------------------------------------------------------------
KERNEL_IDS = ("generic", "stream", "stream2", "pair", "quad")


def run_ours(args, wl, rank, world, device):
    import torch
    from paper_2006_01748_b200 import binding

    dtype = args.dtype
    npd = np.float64 if dtype == "f64" else np.float32
    K, Wm = args.steps, max(args.warmup, 3)
    cells = wl.nx * wl.ny * wl.batch
    dist = world > 1
    if dist:
        import torch.distributed as td

    def barrier():
        if dist:
            td.barrier()
        torch.cuda.synchronize(device)

    sim = binding.Simulation(wl.nx, wl.ny, wl.h, wl.r, wl.d, wl.alpha, wl.c_r, dtype=dtype,
                             batch=wl.batch, device=str(device))
    if args.kernel:
        sim.set_option(binding.GG_OPT_KERNEL, getattr(binding, "GG_KERNEL_" + args.kernel.upper()))
    for o, v in (("warps", binding.GG_OPT_STREAM_WARPS), ("variant", binding.GG_OPT_PAIR_VARIANT),
                 ("quad_variant", binding.GG_OPT_QUAD_VARIANT)):
        if getattr(args, o) is not None:
            sim.set_option(v, getattr(args, o))
    # pinned host copies of the inputs (what a host-side caller holds)
    host = {k: torch.from_numpy(np.ascontiguousarray(getattr(wl, k), dtype=npd)).pin_memory()
            for k in ("a", "b", "c", "U", "V", "W")}
    out = {k: torch.empty_like(host[k]).pin_memory() for k in ("U", "V", "W")}
    ptr = lambda t: t.data_ptr()
    binding.gg_set_tensor_host(sim.ctx, ptr(host["a"]), ptr(host["b"]), ptr(host["c"]))
    binding.gg_set_state_host(sim.ctx, ptr(host["U"]), ptr(host["V"]), ptr(host["W"]))

    # ---- device-resident timing: W warm-up steps, then exactly K steps -----------------------
    sim.step(Wm, wl.dt)
    sim.step(K, wl.dt)          # builds and caches the K-step graphs (untimed)
    # enough repetitions of the K timed steps for nvidia-smi (100 ms period) to see the load
    est_ms = max(sim.last_step_ms(), 1e-3)
    nreps = max(args.reps, int(np.ceil(600.0 / est_ms)) if est_ms < 600.0 else args.reps)
    nreps = min(nreps, 200)
    binding.gg_set_state_host(sim.ctx, ptr(host["U"]), ptr(host["V"]), ptr(host["W"]))
    l0 = sim.launches
    barrier()
    with ClockSampler(device.index or 0) as clk:
        clk.wait_first()
        reps = []
        for _ in range(nreps):
            barrier()
            sim.step(K, wl.dt)
            reps.append(sim.last_step_ms())   # CUDA events on libgg's stream around the K launches
            barrier()
    launches = (sim.launches - l0) // nreps
    value, ms = job_glups(cells, K, float(np.median(reps)), world, device)

    # ---- end to end through the C ABI with host buffers --------------------------------------
    barrier()
    t0 = time.perf_counter()
    binding.gg_set_tensor_host(sim.ctx, ptr(host["a"]), ptr(host["b"]), ptr(host["c"]))
    binding.gg_set_state_host(sim.ctx, ptr(host["U"]), ptr(host["V"]), ptr(host["W"]))
    sim.step(K, wl.dt)
    binding.gg_get_state_host(sim.ctx, ptr(out["U"]), ptr(out["V"]), ptr(out["W"]))
    torch.cuda.synchronize(device)
    e2e_s = max_over_ranks(time.perf_counter() - t0, world, device)
    es = 8 if dtype == "f64" else 4
    h2d = (3 * wl.nx * wl.ny + 3 * cells) * es
    d2h = 3 * cells * es
    e2e = {"value": cells * world * K / e2e_s / 1e9, "unit": UNIT,
           "h2d_bytes_per_step": h2d / K, "d2h_bytes_per_step": d2h / K,
           "what": f"gg_set_tensor_host + gg_set_state_host + gg_step({K}) + gg_get_state_host, "
                   f"pinned host buffers, {h2d / 1e9:.2f} GB up and {d2h / 1e9:.2f} GB down per job",
           "seconds": e2e_s}
    final = tuple(out[k].numpy() for k in ("U", "V", "W"))
    kernel, kernel_name = sim.kernel, sim.kernel_name
    reductions = None
    if not args.no_extras:
        # the device-side reductions next to the step: one pass over
        # U, V, W; wall clock around the synchronising C-ABI call (includes the launch and the
        # result copy), median of 7.  And the adaptive step loop: dt_k re-evaluated on the device
        # every 4 steps (one four-step launch per dt_k), against the fixed-dt loop above.
        def timed(fn):
            ts = []
            for _ in range(7):
                torch.cuda.synchronize(device)
                t0 = time.perf_counter()
                fn()
                ts.append(time.perf_counter() - t0)
            return float(np.median(ts))
        t_diag = timed(lambda: sim.diagnostics(1e-2))
        t_dtmax = timed(lambda: sim.max_stable_dt(0.2))
        # gg_diagnostics_noalloc on caller-held copies of the fields: device time of the ONE kernel
        # (plus its counter memset) by CUDA events on torch's current stream, which is the stream
        # the call is given; median of 7
        Ud, Vd, Wd = sim.get_state()
        dout = torch.empty((wl.batch, binding.GG_DIAG_COUNT), dtype=torch.float64, device=device)
        cur = torch.cuda.current_stream(device)
        na = []
        for _ in range(8):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(cur)
            binding.gg_diagnostics_noalloc(Ud.data_ptr(), Vd.data_ptr(), Wd.data_ptr(), wl.batch, wl.nx, wl.ny,
                                           sim.dtype, 1e-2, dout.data_ptr(), int(cur.cuda_stream))
            e1.record(cur)
            e1.synchronize()
            na.append(e0.elapsed_time(e1))
        t_na = float(np.median(na[1:])) * 1e-3
        na_same = bool(np.allclose(dout.cpu().numpy(), sim.diagnostics(1e-2), rtol=1e-12, atol=1e-12))
        del Ud, Vd, Wd
        sim.step_adaptive(K, 0.2, 4)
        ad = []
        for _ in range(5):
            sim.step_adaptive(K, 0.2, 4)
            ad.append(sim.last_step_ms())
        peak_gbs, _ = measured_peak()
        gbs = lambda t: 3 * cells * es / t / 1e9
        reductions = {"bound": "hbm", "bytes": "3 arrays read once, 24 B (fp64) / 12 B (fp32) per cell",
                      "timing": "gg_diagnostics / gg_max_stable_dt: wall clock around the synchronising C-ABI call "
                                "(launches + result copy included), median of 7; gg_diagnostics_noalloc: CUDA events "
                                "around the enqueue-only call, median of 7",
                      "gg_diagnostics_ms": t_diag * 1e3, "gg_diagnostics_gbs": gbs(t_diag),
                      "gg_diagnostics_frac": gbs(t_diag) / peak_gbs,
                      "gg_diagnostics_noalloc_ms": t_na * 1e3, "gg_diagnostics_noalloc_gbs": gbs(t_na),
                      "gg_diagnostics_noalloc_frac": gbs(t_na) / peak_gbs,
                      "gg_diagnostics_noalloc_matches_gg_diagnostics": na_same,
                      "gg_max_stable_dt_ms": t_dtmax * 1e3,
                      "gg_max_stable_dt_note": "lambda_max(A) is reduced once by gg_set_tensor and cached on the device: "
                                               "this call is one 64-byte read-back",
                      "gg_step_adaptive_every_4_glups": cells * K / (float(np.median(ad)) * 1e-3) / 1e9,
                      "gg_step_adaptive_every_4_vs_fixed": cells * K / (float(np.median(ad)) * 1e-3) / 1e9 / value}
    sim.close()
    return dict(value=value, ms=ms / K, reps_ms=reps, launches=launches, e2e=e2e,
                clocks=clk.summary(), kernel=kernel, kernel_name=kernel_name, final=final,
                reductions=reductions)


def window_parity(wl, final, K, s=0, size=48):
    """Oracle check of an end state on two windows the oracle can afford: the domain corner (true
    Neumann faces on two sides) and a window on the rim of the first tumour disk.  A window is cut
    with a margin of K cells on its interior sides (the stencil moves information one cell per
    step), the oracle runs K steps on the cut, and only the uncontaminated core is compared."""
    import oracle
    inside = wl.V[s] > 0.5
    jj, ii = np.nonzero(inside)
    k = np.argmin(ii)  # leftmost cell of a disk: a front
    size = min(size, wl.nx, wl.ny)
    spots = {"corner": (0, 0), "front": (min(max(int(ii[k]) - size // 2, 0), wl.nx - size),
                                          min(max(int(jj[k]) - size // 2, 0), wl.ny - size))}
    worst = 0.0
    for name, (i0, j0) in spots.items():
        ia, ja = max(i0 - K, 0), max(j0 - K, 0)
        ib, jb = min(i0 + size + K, wl.nx), min(j0 + size + K, wl.ny)
        cut = (slice(ja, jb), slice(ia, ib))
        ref = oracle.step(wl.U[s][cut], wl.V[s][cut], wl.W[s][cut], wl.a[cut], wl.b[cut], wl.c[cut],
                          r=wl.r[s], d=wl.d[s], alpha=wl.alpha[s], c_r=wl.c_r[s], n=K, dt=wl.dt,
                          dx=wl.h)
        core = (slice(j0 - ja, j0 - ja + size), slice(i0 - ia, i0 - ia + size))
        full = (slice(j0, j0 + size), slice(i0, i0 + size))
        for f in range(3):
            worst = max(worst, float(np.max(np.abs(final[f][s][full].astype(np.float64) - ref[f][core]))))
    return worst


def other_configs(device, wl3, only=None):
    """The other BASELINE.json configs with AUTO kernel selection, inputs resident in HBM: median
    device time of 5 repetitions of K steps (K scaled to the config), and window parity of the end
    state of ONE K-step run against the oracle.  Builder-side numbers become driver-side ones."""
    import torch
    from paper_2006_01748_b200 import binding, workloads
    out = {}
    peak, _ = measured_peak()
    plan = [("cfg3_f32", lambda: wl3, "f32", 40), ("cfg2_d10", lambda: workloads.make(2, d=10.0), "f64", 200),
            ("cfg4_batch64", lambda: workloads.make(4), "f64", 40), ("cfg1", lambda: workloads.make(1), "f64", 400),
            ("cfg0", lambda: workloads.make(0), "f64", 200)]
    for name, mk, dtype, K in plan:
        if only and name != only:
            continue
        wl = mk()
        with binding.from_workload(wl, dtype=dtype, device=str(device)) as sim:
            sim.step(K, wl.dt)
            final = sim.get_state_numpy()
            err = max(window_parity(wl, final, K, s) for s in sorted({0, wl.batch - 1}))
            ms = []
            for _ in range(5):
                sim.step(K, wl.dt)
                ms.append(sim.last_step_ms())
            torch.cuda.synchronize(device)
            t = float(np.median(ms))
            glups = wl.cells * K / (t * 1e-3) / 1e9
            # algorithmic bytes per cell-step: U, V, W read and written, the three tensor fields read
            # once per step and shared by the whole batch
            es = 8 if dtype == "f64" else 4
            bpc = (6.0 + 3.0 / wl.batch) * es
            out[name] = {"workload": wl.name, "dtype": dtype, "steps": K, "kernel": sim.kernel,
                         "kernel_name": sim.kernel_name, "glups": glups,
                         "us_per_step": t * 1e3 / K,
                         "roofline": {"bound": "hbm", "achieved": glups * bpc, "peak": peak, "unit": "GB/s",
                                      "frac": glups * bpc / peak, "algorithmic_bytes_per_cell_step": bpc,
                                      "traffic": None,
                                      "note": "k-step kernels cross HBM once per k steps, so frac may exceed 1; "
                                              "grids that stay on chip (cfg0, cfg1) are latency-bound, not HBM-bound"},
                         "parity_window_max_abs_err": err,
                         "tolerance": 1e-10 if dtype == "f64" else 2e-4}
        log(f"config {name}: {out[name]}")
        del wl
    if not only or only.startswith("ext3d"):
        out.update(extension_3d(device, only))
    return out


def extension_3d(device, only=None):
    """The three-dimensional extension (include/gg3.h): 256 x 256 x 256 cells of
    the seeded 3-D recipe, AUTO kernel, fp64 and fp32; median device time of 5 repetitions of 10
    steps; parity of a 40^3 corner window (three Neumann faces) of a separate 4-step run against
    the 3-D oracle, recomputed from the initial data with a 4-cell margin."""
    import torch
    import oracle
    from paper_2006_01748_b200 import binding3, workloads
    peak, _ = measured_peak()
    wl = workloads.make3d(256, 256, 256)
    out = {}
    for dtype, tol in (("f64", 1e-10), ("f32", 2e-4)):
        if only and only != "ext3d_" + dtype:
            continue
        es = 8 if dtype == "f64" else 4
        with binding3.from_workload(wl, dtype=dtype, device=str(device)) as sim:
            n, win = 4, 40
            sim.step(n, wl.dt)
            got = sim.get_state_numpy()
            m = win + n
            cut = lambda P: np.ascontiguousarray(P[:m, :m, :m])
            ref = oracle.step3d(cut(wl.U), cut(wl.V), cut(wl.W), [cut(t) for t in wl.tensor], r=wl.r, d=wl.d,
                                alpha=wl.alpha, c_r=wl.c_r, n=n, dt=wl.dt, dx=wl.dx, dy=wl.dy, dz=wl.dz)
            err = max(float(np.max(np.abs(g[:win, :win, :win].astype(np.float64) - r[:win, :win, :win]))) for g, r in zip(got, ref))
            K, ms = 10, []
            sim.step(K, wl.dt)
            for _ in range(5):
                sim.step(K, wl.dt)
                ms.append(sim.last_step_ms())
            torch.cuda.synchronize(device)
            t = float(np.median(ms))
            glups = wl.cells * K / (t * 1e-3) / 1e9
            out["ext3d_" + dtype] = {"workload": wl.name, "dtype": dtype, "steps": K, "kernel": "gg3_step_" + sim.kernel,
                                     "glups": glups, "us_per_step": t * 1e3 / K,
                                     "roofline": {"bound": "hbm", "achieved": glups * 12 * es, "peak": peak, "unit": "GB/s",
                                                  "frac": glups * 12 * es / peak,
                                                  "algorithmic_bytes_per_cell_step": 12 * es},
                                     "parity_window_max_abs_err": err, "tolerance": tol}
        log(f"config ext3d_{dtype}: {out['ext3d_' + dtype]}")
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--dtype", default="f64", choices=["f64", "f32"])
    ap.add_argument("--kernel", default=None, choices=[None, *KERNEL_IDS])
    ap.add_argument("--warps", type=int, default=None, help="tuning: GG_OPT_STREAM_WARPS")
    ap.add_argument("--variant", type=int, default=None, help="tuning: GG_OPT_PAIR_VARIANT")
    ap.add_argument("--quad-variant", dest="quad_variant", type=int, default=None, help="tuning: GG_OPT_QUAD_VARIANT")
    ap.add_argument("--reps", type=int, default=3)
    ap.add_argument("--n", type=int, default=8192, help="grid edge (8192 = the headline config)")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--no-configs", action="store_true", help="skip the `configs` object (other BASELINE configs)")
    ap.add_argument("--only-config", dest="only_config", default=None, metavar="NAME",
                    help="run ONE entry of the `configs` object (cfg3_f32, cfg2_d10, cfg4_batch64, cfg1, cfg0, "
                         "ext3d_f64, ext3d_f32), print it as a JSON line and exit: the short command the ncu "
                         "captures of those kernels are taken with")
    ap.add_argument("--extras", action="store_true", help="(default since round 3; kept so that old commands still parse)")
    ap.add_argument("--no-extras", dest="no_extras", action="store_true",
                    help="skip the `reductions` object (gg_diagnostics, gg_diagnostics_noalloc, gg_max_stable_dt and "
                         "gg_step_adaptive timed next to the step; costs about a second)")
    ap.add_argument("--record-traffic", default=None, metavar="RAW.csv",
                    help="update profiles/ncu_traffic.json from an `ncu --page raw --csv` dump and exit")
    args = ap.parse_args()
    if args.record_traffic:
        record_traffic(args.record_traffic)
        return 0

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    from paper_2006_01748_b200 import workloads

    if args.impl == "reference":
        if rank != 0:
            return 0
        wl = workloads.make(3, nx=args.n, ny=args.n)
        print(json.dumps(run_reference(args, wl)), flush=True)
        return 0

    import torch
    if not torch.cuda.is_available():
        log("bench.py: no CUDA device; the product has no CPU fallback")
        return 2
    device = torch.device("cuda", local)
    torch.cuda.set_device(device)
    if world > 1:
        import torch.distributed as td
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        td.init_process_group("nccl", device_id=device)
    if args.only_config:
        wl3 = workloads.make(3) if args.only_config == "cfg3_f32" else None
        print(json.dumps({"configs": other_configs(device, wl3, args.only_config)}), flush=True)
        return 0
    wl = workloads.make(3, nx=args.n, ny=args.n)
    log(f"[rank {rank}] workload {wl.name}, dt={wl.dt:.6e}")
    res = run_ours(args, wl, rank, world, device)
    if rank == 0:
        peak, peak_src = measured_peak()
        cells = wl.nx * wl.ny
        bpc = BYTES_PER_CELL[args.dtype]
        # roofline of the dominant (only) kernel: ALGORITHMIC bytes one launch accounts for
        # (72 B x cells x time steps the launch advances) / its average duration.  A k-step
        # kernel advances k steps per pass over HBM, so this may exceed the copy peak; `traffic`
        # is what ncu saw the launch really move, frac_dram_actual the PHYSICAL fraction.
        launches = max(res["launches"], 1)
        steps_per_launch = args.steps / launches
        bytes_per_launch = cells * bpc * steps_per_launch
        launch_ms = res["ms"] * args.steps / launches
        achieved = bytes_per_launch / (launch_ms * 1e-3) / 1e9
        rec = ncu_record(res["kernel_name"]) if wl.nx == 8192 else None
        traffic = rec["traffic_bytes_per_launch"] if rec else None
        dram_actual = (traffic / (launch_ms * 1e-3) / 1e9) if traffic else None
        line = {
            "metric": METRIC if args.dtype == "f64" else METRIC.replace("fp64", "fp32"), "value": res["value"], "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": res["ms"],
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": args.dtype, "data": "synthetic",
            "config": {"workload": WORKLOAD3.format(dtype=args.dtype).replace("8192x8192", f"{wl.nx}x{wl.ny}"),
                       "kernel": res["kernel"], "kernel_name": res["kernel_name"],
                       "l2": "working set 4.8 GB per step >> 126 MB L2",
                       "multi_gpu": "replicas only" if world > 1 else "single GPU",
                       "timing": f"median of {len(res['reps_ms'])} repetitions of the {args.steps} timed steps "
                                 f"(min {min(res['reps_ms']):.3f} ms, max {max(res['reps_ms']):.3f} ms)"},
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s",
                         "frac": achieved / peak, "traffic": traffic, "peak_source": peak_src,
                         "algorithmic_bytes_per_launch": bytes_per_launch,
                         "steps_per_launch": steps_per_launch, "launch_ms": launch_ms,
                         "dram_gbs_actual": dram_actual,
                         "frac_dram_actual": (dram_actual / peak) if dram_actual else None,
                         "traffic_source": ("profiles/ncu_traffic.json, csrc " + csrc_sha16()) if rec else
                                           "null: no ncu record for this kernel and this csrc/ (hash " + csrc_sha16() + ")",
                         "frac_of_nominal_8000": achieved / 8000.0},
            "e2e": res["e2e"], "gpu_launches": res["launches"], "clocks": res["clocks"],
        }
        # The multi-step kernels are not HBM-bound (see frac_dram_actual); their nearest ceiling
        # is the plain-ALU pipe of the arithmetic type.  Thread instructions of that pipe per
        # cell-step from the ncu record of THIS kernel (redundant overlap lanes included); peak =
        # 148 SMs x lanes per clock x the max SM clock (one fused multiply-add = one instruction),
        # DESIGN.md section 8.  Absent when there is no valid record.
        if rec and rec.get("pipe_instr_per_cell_step"):
            ops = rec["pipe_instr_per_cell_step"]
            lanes = 64 if args.dtype == "f64" else 128
            mhz = (res["clocks"] or {}).get("sm_max_mhz") or 1965.0
            alu_peak = 148 * lanes * mhz * 1e6 / 1e12
            alu = res["value"] * 1e9 * ops / 1e12
            line["alu"] = {"bound": "alu", "achieved": alu, "peak": alu_peak,
                           "unit": f"T {args.dtype} instr/s", "frac": alu / alu_peak,
                           "instr_per_cell_step": ops, "source": rec.get("pipe_metric")}
        if res.get("reductions"):
            line["reductions"] = res["reductions"]
        t0 = time.perf_counter()
        line["parity_sample_max_abs_err"] = window_parity(wl, res["final"], args.steps)
        log(f"sampled parity: {line['parity_sample_max_abs_err']:.3e} ({time.perf_counter() - t0:.1f} s)")
        res["final"] = None
        if world == 1 and not args.no_configs and args.dtype == "f64" and not args.kernel and wl.nx == 8192:
            line["configs"] = other_configs(device, wl)
        if not args.no_cpu and world == 1:
            g, desc, cores, _ = oracle_sample(wl, steps=50, min_seconds=6.0)
            line["cpu_baseline"] = {"value": g, "unit": UNIT, "cores": cores, "kind": "oracle",
                                    "sample": desc}
        print(json.dumps(line), flush=True)
    if world > 1:
        td.barrier()
        td.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())

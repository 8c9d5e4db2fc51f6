#!/usr/bin/env python
"""Benchmark of the w-stacking hot path (BASELINE.json metric: Mvis/s and image wall time on one B200).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config large] [--impl ours|reference]

One "step" = one pass of the whole hot path over the synthetic workload, inputs resident in HBM:
a1 bin -> a2 grid (WS_GRID_SPARSE: only the tiles that hold visibilities are written, no memset) -> a3 the library's
own FFT, columns then rows, skipping what the gridder left empty -> a4 fused into the row pass (also writes a5, the
real dirty image).  cuFFT + the stand-alone w-correction are timed beside it (library_path_ms).  Prints ONE JSON line (rank 0).
N > 1 runs N independent replicas (the path is built for one GPU, "replicas only").
`--impl reference` times the fp64 CPU oracle on a bounded sample of the same workload (see cpu_baseline()).
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np
import torch

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from synth import get_config, make_dataset  # noqa: E402

METRIC = "Mvis/s through the whole w-stacking path (bin+grid+FFT+w-correct) on 1 B200"
UNIT = "Mvis/s"


def peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, burst copy)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.lines, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=lambda: self.lines.extend(self.proc.stdout), daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        self.t.join(timeout=2)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


KERNEL = "gaussian"     # --kernel: "gaussian" (the headline workload) or "kb" (Kaiser-Bessel, :459)


def kb_beta(support, alpha=2.0):
    """Kaiser-Bessel shape for a window of `support` cells and the inner 1/alpha of the field (Beatty et al.)."""
    return float(np.pi * np.sqrt((support / alpha) ** 2 * (alpha - 0.5) ** 2 - 0.8))


def oracle_params(orc, d, tile=32):
    kb = KERNEL == "kb"
    return orc.OracleParams(n_pix=d.n_pix, n_wplanes=d.n_wplanes, support=d.support, cell_rad=d.cell_rad,
                            w_min=d.w_min, w_max=d.w_max, sigma=kb_beta(d.support) if kb else d.sigma_cells, tile=tile,
                            kernel_type=1 if kb else 0)


def _omp_threads(n):
    """Sets the OpenMP thread count of the process (the oracle's runtime is libgomp); False if that is not possible."""
    import ctypes
    try:
        ctypes.CDLL("libgomp.so.1").omp_set_num_threads(int(n))
        return True
    except OSError:
        return False


def _oracle_planes(orc, prm, d, lo, n):
    """The oracle's chain on planes [lo, lo + n): one gridding call (a plane per host thread: every core works), then
    its transform and w-correction plane by plane.  Returns the seconds it took."""
    uvw, vis, wt = d.uvw.numpy(), d.vis.numpy(), d.weights.numpy()
    D = np.zeros((d.n_pix, d.n_pix), np.complex128)
    t0 = time.perf_counter()
    G = orc.grid(prm, uvw, vis, wt, d.freqs_hz, lo, lo + n)
    for i in range(n):
        orc.wcorrect(prm, orc.transform(G[i])[None], lo + i, D)
    return time.perf_counter() - t0


def cpu_baseline(d, single_thread=True, row_fraction=1.0):
    """The fp64 oracle as it stands, plane-streamed like oracle.dirty_image, timed on the host cores on a bounded
    sample: ONE batch of `cores` adjacent planes from the middle of the stack (each plane pass places all visibilities,
    grids those of its plane, transforms and w-corrects it); the whole-workload time is the sample time x N_w / planes.
    Also the same on ONE thread and one plane (comparison with the paper's per-core rows)."""
    import psutil
    from oracle import wstack_oracle as orc
    prm = oracle_params(orc, d)
    d = d.to("cpu")
    n_all = d.n_vis
    if row_fraction < 1.0:      # a leading share of the (time-major) rows: the reference arm's way to bound a many-step run
        import dataclasses
        n_r = max(1, int(d.n_rows * row_fraction))
        d = dataclasses.replace(d, uvw=d.uvw[:n_r].contiguous(), vis=d.vis[:n_r].contiguous(), weights=d.weights[:n_r].contiguous())
    cores = orc.num_threads()
    fit = int(psutil.virtual_memory().available * 0.4 // (16 * d.n_pix ** 2))
    n_s = max(1, min(cores, d.n_wplanes, fit))
    lo = (d.n_wplanes - n_s) // 2
    dt = _oracle_planes(orc, prm, d, lo, n_s)
    full = dt * d.n_wplanes / n_s
    out = {"value": d.n_vis / full / 1e6, "unit": UNIT, "cores": min(cores, n_s), "kind": "oracle",
           "planes_timed": n_s, "planes_total": d.n_wplanes, "extrapolated": n_s < d.n_wplanes, "sample_seconds": dt,
           "rows_fraction": d.n_vis / n_all,
           "sample": f"planes {lo}..{lo + n_s - 1} of {d.n_wplanes}, one per thread ("
                     + ("all" if d.n_vis == n_all else f"the first {d.n_vis} of the") + f" {n_all} visibilities placed per plane "
                     f"pass, fp64 grid + radix-2 FFT + w-correction of those planes): {dt:.1f} s"
                     + (f", whole workload extrapolated x{d.n_wplanes / n_s:.1f} = {full:.0f} s" if n_s < d.n_wplanes else "")}
    if single_thread and _omp_threads(1):
        try:
            k1 = d.n_wplanes // 2
            dt1 = _oracle_planes(orc, prm, d, k1, 1)
        finally:
            _omp_threads(cores)
        out["single_thread"] = {"value": d.n_vis / (dt1 * d.n_wplanes) / 1e6, "unit": UNIT, "cores": 1, "planes_timed": 1,
                                "extrapolated": d.n_wplanes > 1, "sample_seconds": dt1}
    return out


def run_reference(args, d, cfg_name):
    """K timed + W warm-up samples of the oracle.  The first sample is the cpu_baseline() sample (one batch of planes, all
    rows); if K + W of those would not end within ~3 minutes, the later samples take a leading share of the rows (not less
    than a quarter; their transforms keep their full cost, so the rate they give is, if anything, low)."""
    n_total = args.steps + args.warmup
    first = cpu_baseline(d, single_thread=False)
    frac = 1.0
    if n_total > 1 and first["sample_seconds"] * n_total > 180.0:
        frac = max(0.25, min(1.0, 180.0 / n_total / first["sample_seconds"]))
    vals = [first] + [cpu_baseline(d, single_thread=False, row_fraction=frac) for _ in range(n_total - 1)]
    vals = vals[args.warmup:]
    v = float(np.mean([x["value"] for x in vals]))
    cb = dict(vals[-1]); cb["value"] = v
    ms = d.n_vis / (v * 1e6) * 1e3
    return {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "ms_per_step_is_extrapolated": bool(cb["extrapolated"]),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": workload_config(d, cfg_name),
            "cpu_baseline": cb, "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}


def reduce_max_ms(ms, dist, device):
    """The step time of the whole job: the MAX over ranks of the per-rank device time (replicas run side by side)."""
    if dist is None:
        return float(ms)
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(n_vis_per_rank, world, ms_step):
    """Mvis/s of all ranks together (weak scaling: every rank images its own replica of the workload)."""
    return world * n_vis_per_rank / (ms_step * 1e-3) / 1e6


def workload_config(d, cfg_name):
    return {"workload": f"{cfg_name}: {d.n_vis} visibilities ({d.n_rows} rows x {d.n_chan} channels), "
                        f"{d.n_pix}x{d.n_pix} complex64 mesh, {d.n_wplanes} w-planes, "
                        + ("Kaiser-Bessel (beta %.2f)" % kb_beta(d.support) if KERNEL == "kb" else "Gaussian") + f" support {d.support}",
            "n_vis": d.n_vis, "n_pix": d.n_pix, "n_wplanes": d.n_wplanes, "support": d.support,
            "l2": "inputs (%.2f GB) and mesh (%.1f GB) larger than the 126 MB L2; no flush needed" %
                  ((12 * d.n_rows + 12 * d.n_vis) / 1e9, 8.0 * d.n_pix ** 2 * d.n_wplanes / 1e9)}


def run_f64(args, ws, d, cfg, local_rank, world, dist):
    """The path in the paper's own arithmetic (PAPER.md:392, Table 3: fp64 mesh; :207, :219: one thread per measurement,
    atomicAdd on the mesh): zero -> grid -> cuFFT Z2Z -> w-correction, all fp64.  Context against the paper's Table 4
    (other hardware, its own data), not the headline."""
    presum = d.freqs_hz is None and d.n_chan > 1
    flags = ws.WS_FLAG_MESH_F64 | (ws.WS_FLAG_PRESUM_CHANNELS if presum else 0)
    plan = ws.Plan(d.n_pix, d.n_wplanes, d.support, d.cell_rad, d.w_min, d.w_max, sigma=d.sigma_cells, device=local_rank, flags=flags)
    grid, image, dirty = plan.alloc_grid(), plan.alloc_image(), plan.alloc_dirty()
    wsp = torch.empty(max(plan.fft_workspace_bytes(), 256), dtype=torch.uint8, device=f"cuda:{local_rank}")

    def step(ev=None):
        if ev: ev[0].record()
        plan.grid_zero(grid)
        if ev: ev[1].record()
        plan.grid_visibilities(d.uvw, d.vis, d.weights, d.freqs_hz, grid, wsp, mode=ws.WS_GRID_ACCUMULATE)
        if ev: ev[2].record()
        plan.fft_planes(grid, wsp)
        if ev: ev[3].record()
        plan.wcorrect_accumulate(grid, image, accumulate=False, dirty=dirty)
        if ev: ev[4].record()

    for _ in range(args.warmup):
        step()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(5)] for _ in range(args.steps)]
    clocks = ClockSampler(local_rank)
    torch.cuda.synchronize()
    if dist: dist.barrier()
    torch.cuda.synchronize()
    clocks.start()
    l0 = plan.launch_count()
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0.record()
    for i in range(args.steps):
        step(evs[i])
    t1.record()
    torch.cuda.synchronize()
    if dist: dist.barrier()
    launches = plan.launch_count() - l0
    clk = clocks.stop()
    ms_step = reduce_max_ms(t0.elapsed_time(t1), dist, f"cuda:{local_rank}") / args.steps
    med = np.median(np.array([[e[i].elapsed_time(e[i + 1]) for i in range(4)] for e in evs]), axis=0)
    peak, peak_src = peaks()
    mesh_b = 16.0 * d.n_pix ** 2 * d.n_wplanes
    alg = {"zero": mesh_b, "k_grid_f64": 12.0 * d.n_rows + 12.0 * d.n_vis + mesh_b, "cufft_z2z": 2 * mesh_b,
           "k_wcorrect_f64": mesh_b + 24.0 * d.n_pix ** 2}
    names = list(alg)
    own_k = {"k_grid_f64": med[1], "k_wcorrect_f64": med[3]}
    dom = max(own_k, key=own_k.get)
    ach = alg[dom] / (own_k[dom] * 1e-3) / 1e9
    return {"metric": METRIC, "value": whole_job_value(d.n_vis, world, ms_step), "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": workload_config(d, cfg.name), "clocks": clk,
            "gpu_launches": int(launches), "stages_ms_median": {n: float(v) for n, v in zip(names, med)},
            "fft": "cuFFT Z2Z", "presummed_channels": bool(presum),
            "ggpas": d.n_vis * d.support ** 2 / (med[1] * 1e-3) / 1e9,
            "mvis_per_s_gridding": d.n_vis / (med[1] * 1e-3) / 1e6,
            "kernels": {n: {"ms": float(t), "alg_GB": alg[n] / 1e9, "GBps": alg[n] / (t * 1e-3) / 1e9} for n, t in zip(names, med)},
            "roofline": {"bound": "hbm", "kernel": dom, "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                         "traffic": None, "peak_source": peak_src, "algorithmic_bytes_per_launch": alg[dom],
                         "launch_ms": float(own_k[dom]),
                         "note": "atomicAdd(double) gridder: bound by the L2 atomic rate on the dense core, not by HBM"}}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="large")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--kernel", default="gaussian", choices=["gaussian", "kb"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-degrid", action="store_true")
    ap.add_argument("--no-snapshot-hint", action="store_true")
    ap.add_argument("--chunked", action="store_true", help="configs with n_chunks > 1: grid the row chunks one call at a time")
    ap.add_argument("--mesh-f64", action="store_true",
                    help="the paper's arithmetic (WS_FLAG_MESH_F64: fp64 mesh, atomicAdd gridder, cuFFT Z2Z): context line, see run_f64()")
    args = ap.parse_args()
    global KERNEL
    KERNEL = args.kernel
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    cfg = get_config(args.config)

    if args.impl == "reference":
        if rank != 0:
            return
        dev = f"cuda:{local_rank}" if torch.cuda.is_available() else "cpu"
        d = make_dataset(cfg, device=dev).to("cpu")
        print(json.dumps(run_reference(args, d, cfg.name)), flush=True)
        return

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    import paper_2301_06061_b200 as ws
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local_rank}"))

    d = make_dataset(cfg, device=f"cuda:{local_rank}")
    if args.mesh_f64:
        out = run_f64(args, ws, d, cfg, local_rank, world, dist)
        if rank == 0:
            print(json.dumps(out), flush=True)
        if dist:
            dist.destroy_process_group()
        return
    # the paper's narrow-band mode (shared uvw): sum the channels of a row first, bin rows
    presum = d.freqs_hz is None and d.n_chan > 1
    flags = ws.WS_FLAG_PRESUM_CHANNELS if presum else 0
    if presum:
        args.no_degrid = True
    if KERNEL == "kb":
        plan = ws.Plan(d.n_pix, d.n_wplanes, d.support, d.cell_rad, d.w_min, d.w_max, device=local_rank, flags=flags,
                       kernel_type=ws.WS_KERNEL_KAISER_BESSEL, kernel_param=kb_beta(d.support))
    else:
        plan = ws.Plan(d.n_pix, d.n_wplanes, d.support, d.cell_rad, d.w_min, d.w_max, sigma=d.sigma_cells, device=local_rank,
                       flags=flags)
    if d.rows_per_snapshot and not args.no_snapshot_hint:   # the rows are time-major, every baseline per snapshot
        plan.set_snapshot_rows(d.rows_per_snapshot)
    grid, image, dirty = plan.alloc_grid(), plan.alloc_image(), plan.alloc_dirty()
    wsp = plan.alloc_workspace(d.n_rows if presum else d.n_vis)

    own = plan.fft_is_own
    OCC = ws.WS_FFT_USE_OCCUPANCY

    chunks = d.row_chunks() if (args.chunked and d.n_chunks > 1) else None
    if chunks:      # Extreme's recipe: row chunks through repeated accumulate calls onto a cleared mesh
        del wsp
        wsp = plan.alloc_workspace(max(hi - lo for lo, hi in chunks) * d.n_chan)

    def step_chunked(ev=None):
        # stages: [-] [bin + grid of all chunks] [FFT] [w-correct].  The mesh is never cleared: the first chunk is gridded
        # WS_GRID_SPARSE (library FFT: OVERWRITE), the later ones WS_GRID_SPARSE_ADD (ACCUMULATE)
        if ev: ev[0].record()
        if ev: ev[1].record()
        for i, (lo, hi) in enumerate(chunks):
            if own:
                mode = ws.WS_GRID_SPARSE if i == 0 else ws.WS_GRID_SPARSE_ADD
            else:
                mode = ws.WS_GRID_OVERWRITE if i == 0 else ws.WS_GRID_ACCUMULATE
            plan.grid_visibilities(d.uvw[lo:hi], d.vis[lo:hi], d.weights[lo:hi], d.freqs_hz, grid, wsp, mode=mode)
        if ev: ev[2].record()
        if own:
            plan.fft_columns(grid, OCC)
            if ev: ev[3].record()
            plan.fft_rows_wcorrect(grid, image, accumulate=False, dirty=dirty, fft_flags=OCC)
        else:
            plan.fft_planes(grid, wsp)
            if ev: ev[3].record()
            plan.wcorrect_accumulate(grid, image, accumulate=False, dirty=dirty)
        if ev: ev[4].record()

    def step(ev=None):
        if chunks:
            return step_chunked(ev)
        if ev: ev[0].record()
        plan.bin_visibilities(d.uvw, d.vis, d.weights, d.freqs_hz, wsp)
        if ev: ev[1].record()
        if own:     # the mesh is neither cleared nor completely written: the FFT passes skip what stayed empty
            plan.grid_binned(grid, wsp, mode=ws.WS_GRID_SPARSE)
            if ev: ev[2].record()
            plan.fft_columns(grid, OCC)
            if ev: ev[3].record()
            plan.fft_rows_wcorrect(grid, image, accumulate=False, dirty=dirty, fft_flags=OCC)
        else:       # N not a power of two in 256..8192: library FFT on a fully written mesh, stand-alone a4
            plan.grid_binned(grid, wsp, mode=ws.WS_GRID_OVERWRITE)
            if ev: ev[2].record()
            plan.fft_planes(grid, wsp)
            if ev: ev[3].record()
            plan.wcorrect_accumulate(grid, image, accumulate=False, dirty=dirty)
        if ev: ev[4].record()

    for _ in range(args.warmup):
        step()
    plan.async_status()
    bins_info = None
    if chunks:      # statistics of the first chunk stand for all (same recipe per chunk)
        lo0, hi0 = chunks[0]
        plan.bin_visibilities(d.uvw[lo0:hi0], d.vis[lo0:hi0], d.weights[lo0:hi0], d.freqs_hz, wsp)
    else:
        plan.bin_visibilities(d.uvw, d.vis, d.weights, d.freqs_hz, wsp)
    b = plan.get_bins(fields=("bin_start",))
    bins_info = {"n_dropped": b["n_dropped"], "n_records": b["n_records"],
                 "max_bin": int(np.diff(b["bin_start"].astype(np.int64)).max()),
                 "empty_bins_frac": float((np.diff(b["bin_start"].astype(np.int64)) == 0).mean())}
    n_records = b["n_records"] * (len(chunks) if chunks else 1)
    del b

    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(5)] for _ in range(args.steps)]
    clocks = ClockSampler(local_rank)
    torch.cuda.synchronize()
    if dist: dist.barrier()
    torch.cuda.synchronize()
    clocks.start()
    l0 = plan.launch_count()
    t_start, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t_start.record()
    for i in range(args.steps):
        step(evs[i])
    t_end.record()
    torch.cuda.synchronize()
    if dist: dist.barrier()
    launches = plan.launch_count() - l0
    clk = clocks.stop()
    total_ms = t_start.elapsed_time(t_end)
    total_ms = reduce_max_ms(total_ms, dist, f"cuda:{local_rank}")
    plan.async_status()
    ms_step = total_ms / args.steps
    st = np.array([[e[i].elapsed_time(e[i + 1]) for i in range(4)] for e in evs])     # bin, grid, fft, wcorrect
    med = np.median(st, axis=0)
    per_step = st.sum(axis=1)      # device time of each timed step (median, mean +- std, min)
    step_stats = {"median": float(np.median(per_step)), "mean": float(per_step.mean()), "std": float(per_step.std()),
                  "min": float(per_step.min())}
    value = whole_job_value(d.n_vis, world, ms_step)

    # ---- the library path on the same inputs, for the separate FFT figure (north_star): OVERWRITE gridding,
    # cuFFT per plane, stand-alone w-correction.  Outside the timed region.
    lib_ms = None
    occ = plan.occupancy() if own else None      # of the timed path's mesh (fractions the FFT passes touch; orientation)
    if own and not chunks:
        e = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
        rows = []
        for _ in range(3):
            plan.bin_visibilities(d.uvw, d.vis, d.weights, d.freqs_hz, wsp)
            e[0].record()
            plan.grid_binned(grid, wsp, mode=ws.WS_GRID_OVERWRITE)
            e[1].record()
            plan.fft_planes(grid, wsp)
            e[2].record()
            plan.wcorrect_accumulate(grid, image, accumulate=False, dirty=dirty)
            e[3].record()
            torch.cuda.synchronize()
            rows.append([e[i].elapsed_time(e[i + 1]) for i in range(3)])
        m = np.median(np.array(rows), axis=0)
        lib_ms = {"grid_overwrite": float(m[0]), "fft_cufft": float(m[1]), "wcorrect_standalone": float(m[2])}

    # ---- degridding on the same positions, outside the timed region: model image -> planes
    # (forward w-screen + cuFFT), then bins + footprint gather
    degrid_ms = None
    if not args.no_degrid and not chunks:
        model = torch.randn((d.n_pix, d.n_pix), dtype=torch.complex64, device=f"cuda:{local_rank}")
        pred = torch.empty_like(d.vis)
        e = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
        rows = []
        for _ in range(4):
            e[0].record()
            plan.predict_planes(model, grid, wsp)
            e[1].record()
            plan.degrid_visibilities(d.uvw, d.freqs_hz, d.n_chan, grid, pred, wsp)
            e[2].record()
            torch.cuda.synchronize()
            rows.append([e[i].elapsed_time(e[i + 1]) for i in range(2)])
        plan.async_status()
        m = np.median(np.array(rows[1:]), axis=0)
        degrid_ms = {"predict_planes_wscreen_cufft": float(m[0]), "bin_and_gather": float(m[1]),
                     "mvis_per_s_degridding": d.n_vis / (m[1] * 1e-3) / 1e6,
                     "mvis_per_s_whole_prediction": d.n_vis / ((m[0] + m[1]) * 1e-3) / 1e6}
        # the same prediction as ONE call: bins first, only the wanted column bands transformed (own column passes)
        rows = []
        for _ in range(4):
            e[0].record()
            plan.predict_visibilities(model, d.uvw, d.freqs_hz, d.n_chan, grid, pred, wsp)
            e[1].record()
            torch.cuda.synchronize()
            rows.append(e[0].elapsed_time(e[1]))
        plan.async_status()
        one = float(np.median(rows[1:]))
        degrid_ms["predict_visibilities_one_call"] = one
        degrid_ms["mvis_per_s_one_call"] = d.n_vis / (one * 1e-3) / 1e6
        del model, pred

    # ---- roofline of the dominant own kernel -----------------------------------------
    peak, peak_src = peaks()
    mesh_b = 8.0 * d.n_pix ** 2 * d.n_wplanes
    N, NW = d.n_pix, d.n_wplanes
    n_keys = d.n_rows if presum else d.n_vis
    # a1: inputs read once (12 B/row + 12 B/visibility), keys + perm written (4 + 4 B per binned entry), records written
    alg_bin = 12.0 * d.n_rows + 12.0 * d.n_vis + 8.0 * n_keys + 16.0 * n_records
    if own:
        # k_grid: records read + non-empty tiles written; column passes (k_fft_cols, one launch: the classes pass 1a writes
        # stay in L2 until pass 1b has read them): non-empty tiles read, non-empty bands written (N = 256 has pass 1b only);
        # pass 2: non-empty bands read once, image + dirty written
        alg = {"bin": alg_bin, "k_grid_tiles": 16.0 * n_records + mesh_b * occ["tiles"],
               "k_fft_columns": mesh_b * (occ["tiles"] + occ["bands"]),
               "k_fft_rows_wcorrect": mesh_b * occ["bands"] + 12.0 * N * N}
        times = {"bin": med[0], "k_grid_tiles": med[1], "k_fft_columns": med[2], "k_fft_rows_wcorrect": med[3]}
        # nominal FFT flops (5 n log2 n per transform) of the transforms that are not skipped, + 8 per point-plane of Horner
        flops = {"k_fft_columns": 5.0 * N * np.log2(N) * N * NW * occ["bands"],
                 "k_fft_rows_wcorrect": (5.0 * N * np.log2(N) + 8.0 * N) * N * NW * occ["planes"]}
    else:
        occ = None
        alg = {"bin": alg_bin, "k_grid_tiles": mesh_b + 16.0 * n_records, "k_wcorrect": mesh_b + 12.0 * N * N}
        times = {"bin": med[0], "k_grid_tiles": med[1], "k_wcorrect": med[3]}
        flops = {}
    # dram__bytes_read.sum + dram__bytes_write.sum per launch: from the committed ncu --set full capture of this command
    # and configuration, if there is one (profiles/traffic.json names the capture each figure comes from), else null
    ncu_traffic, traffic_src = {}, None
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as f:
            tj = json.load(f)
        ent = tj.get(f"{cfg.name}/{KERNEL}")
        if ent and own and not chunks:
            ncu_traffic, traffic_src = {k: float(v) for k, v in ent["dram_bytes_per_launch"].items()}, ent["capture"]
    except Exception:
        pass
    kernel_times = {k: v for k, v in times.items() if k != "bin"}
    dom = max(kernel_times, key=kernel_times.get)
    ach = alg[dom] / (times[dom] * 1e-3) / 1e9
    hbm_frac = ach / peak
    roof = {"bound": "hbm", "kernel": dom, "achieved": ach, "peak": peak, "unit": "GB/s", "frac": hbm_frac,
            "traffic": ncu_traffic.get(dom), "traffic_source": traffic_src if dom in ncu_traffic else None,
            "peak_source": peak_src, "algorithmic_bytes_per_launch": alg[dom], "launch_ms": float(times[dom])}
    if dom in flops:
        # fp32 peak: DERIVED, 148 SMs x 128 lanes x 2 flop x max SM clock (B200_PROFILING.md unit counts and clocks);
        # `fp32_fma_measured_tflops` beside it is what a register-only FFMA loop of this library reaches on this GPU
        alu_peak = 148 * 128 * 2 * 1.965e9 / 1e12
        tf = flops[dom] / (times[dom] * 1e-3) / 1e12
        if tf / alu_peak > hbm_frac:
            roof = {"bound": "alu", "kernel": dom, "achieved": tf, "peak": alu_peak, "unit": "TFLOP/s", "frac": tf / alu_peak,
                    "traffic": ncu_traffic.get(dom), "traffic_source": traffic_src if dom in ncu_traffic else None,
                    "peak_source": "derived: 148 SMs x 128 fp32 lanes x 2 x 1.965 GHz (guide's unit counts and clocks)",
                    "fp32_fma_measured_tflops": plan.measure_fp32_tflops(),
                    "nominal_flops_per_launch": flops[dom], "launch_ms": float(times[dom]),
                    "hbm_view": {"achieved": ach, "peak": peak, "frac": hbm_frac, "algorithmic_bytes_per_launch": alg[dom]}}
    per_kernel = {k: {"ms": float(times[k]), "alg_GB": alg[k] / 1e9, "GBps": alg[k] / (times[k] * 1e-3) / 1e9,
                      "frac_of_hbm_peak": alg[k] / (times[k] * 1e-3) / 1e9 / peak,
                      "ncu_dram_GB": ncu_traffic[k] / 1e9 if k in ncu_traffic else None} for k in times}
    # the whole timed step against HBM: sum of the algorithmic bytes of its stages / its device time
    b_step = float(sum(alg.values()))
    roof_step = {"what": "sum of the stages' algorithmic bytes / ms_per_step (the timed step as a whole)", "bytes": b_step,
                 "ms": float(ms_step), "achieved": b_step / (ms_step * 1e-3) / 1e9,
                 "frac_of_measured_peak": b_step / (ms_step * 1e-3) / 1e9 / peak}
    # B_alg(path) counts every plane cell written once and read once (a DENSE mesh), so its time is that of
    # the gridder that writes every cell (WS_GRID_OVERWRITE) + the stand-alone w-correction that reads every cell
    b_path = 12.0 * d.n_rows + 12.0 * d.n_vis + 2 * mesh_b + 8.0 * N * N
    roof_path = None
    if lib_ms:
        t_path = med[0] + lib_ms["grid_overwrite"] + lib_ms["wcorrect_standalone"]
        roof_path = {"what": "a1 + a2 (WS_GRID_OVERWRITE: every cell written) + stand-alone a4, no FFT: SURVEY 8(d) B_alg(path), dense accounting",
                     "bytes": b_path, "ms": float(t_path), "achieved": b_path / (t_path * 1e-3) / 1e9,
                     "frac_of_measured_peak": b_path / (t_path * 1e-3) / 1e9 / peak,
                     "frac_of_nominal_8TBs": b_path / (t_path * 1e-3) / 1e9 / 8000.0}
    elif not own:
        t_path = med[0] + med[1] + med[3]
        roof_path = {"what": "a1 + a2 (every cell written) + stand-alone a4 of the timed step, no FFT: SURVEY 8(d) B_alg(path)",
                     "bytes": b_path, "ms": float(t_path), "achieved": b_path / (t_path * 1e-3) / 1e9,
                     "frac_of_measured_peak": b_path / (t_path * 1e-3) / 1e9 / peak,
                     "frac_of_nominal_8TBs": b_path / (t_path * 1e-3) / 1e9 / 8000.0}
    # the sparse path's gridding with ITS OWN bytes (inputs, keys, records, only the tiles that hold visibilities)
    roof_sparse = None
    if own:
        b_sp = alg["bin"] + alg["k_grid_tiles"]
        t_sp = med[0] + med[1]
        roof_sparse = {"what": "a1 + a2 of the timed step (WS_GRID_SPARSE) with the bytes that path moves", "bytes": b_sp,
                       "ms": float(t_sp), "achieved": b_sp / (t_sp * 1e-3) / 1e9,
                       "frac_of_measured_peak": b_sp / (t_sp * 1e-3) / 1e9 / peak}

    stage_names = ["bin", "grid", "fft_columns", "fft_rows_wcorrect"] if own else ["bin", "grid", "fft_cufft", "wcorrect"]
    if chunks:
        stage_names = ["-", "bin_and_grid_%d_chunks" % len(chunks)] + stage_names[2:]
    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
           "data": "synthetic", "config": workload_config(d, cfg.name), "clocks": clk, "gpu_launches": int(launches),
           "stages_ms_median": {n: float(v) for n, v in zip(stage_names, med)}, "step_ms_stats": step_stats,
           "fft": "own two-pass FFT with fused w-correction, occupancy-aware" if own else "cuFFT",
           "library_path_ms": lib_ms, "degridding_ms": degrid_ms, "occupancy": occ,
           "mvis_per_s_gridding": d.n_vis / ((med[0] + med[1]) * 1e-3) / 1e6,
           "ggpas": d.n_vis * d.support ** 2 / (med[1] * 1e-3) / 1e9,
           "ggpas_bin_and_grid": d.n_vis * d.support ** 2 / ((med[0] + med[1]) * 1e-3) / 1e9,
           "presummed_channels": bool(presum),
           "snapshot_rows_hint": int(d.rows_per_snapshot) if (d.rows_per_snapshot and not args.no_snapshot_hint) else 0,
           "image_wall_ms": ms_step, "bins": bins_info, "roofline": roof, "kernels": per_kernel,
           "roofline_step": roof_step, "roofline_path": roof_path, "roofline_sparse_gridding": roof_sparse}

    # ---- end to end through the C ABI with HOST buffers --------------------------------------------------
    if not args.no_e2e:
        uvw_h, vis_h, wt_h = (t.cpu().pin_memory() for t in (d.uvw, d.vis, d.weights))
        dirty_h = torch.empty((d.n_pix, d.n_pix), dtype=torch.float32).pin_memory()
        dev_in = torch.empty(plan.dev_inputs_bytes(d.n_rows, d.n_chan), dtype=torch.uint8, device=f"cuda:{local_rank}")
        k_e2e = max(2, min(args.steps, 5))
        plan.image_from_host(uvw_h, vis_h, wt_h, d.freqs_hz, dev_in, grid, image, dirty, dirty_h, wsp)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(k_e2e):
            plan.image_from_host(uvw_h, vis_h, wt_h, d.freqs_hz, dev_in, grid, image, dirty, dirty_h, wsp)
        torch.cuda.synchronize()
        e2e_ms = (time.perf_counter() - t0) / k_e2e * 1e3
        e2e_ms = reduce_max_ms(e2e_ms, dist, f"cuda:{local_rank}")
        out["e2e"] = {"value": whole_job_value(d.n_vis, world, e2e_ms), "unit": UNIT, "ms_per_step": e2e_ms,
                      "h2d_bytes_per_step": 12 * d.n_rows + 12 * d.n_vis, "d2h_bytes_per_step": 4 * d.n_pix ** 2,
                      "steps": k_e2e, "checksum": float(dirty_h[d.n_pix // 2, d.n_pix // 2])}
        del dev_in

    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        del grid, image, dirty, wsp
        torch.cuda.empty_cache()
        out["cpu_baseline"] = cpu_baseline(d.to("cpu"))
    if rank == 0:
        print(json.dumps(out), flush=True)
    if dist:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

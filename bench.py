#!/usr/bin/env python
"""bench.py -- EP-TV outer iterations per second on the BASELINE.json throughput workload.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c4|c3|...] [--impl reference]

A "step" is ONE outer iteration of the whole hot path over the
batch: CGLS (n_cgls iterations, each one P and one P^T) + n_gd x (edge weights, EP-TV gradient,
Armijo search, update) + positivity clamp. Default workload: c4 = BASELINE.json configs[3], 64
independent 512x512 slices x 60 views x 888 bins (the 512^2 x 60-view geometry the metric is quoted
on), n_cgls = 15, n_gd = 5. value = slices * steps / seconds, summed over ranks (each rank owns its own
64 slices: weak scaling, no collective on the data path).
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
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

from ctr_inputs import get_config, make_case, scaled_config  # noqa: E402

UNIT = "slice-iters/s"


def metric_name(cfg):
    if cfg.ndim == 3:
        return (f"EP-TV outer iters/sec at {cfg.nx}x{cfg.ny}x{cfg.nz} x {cfg.nviews} views (one volume counts as one "
                "slice: outer iterations / s)")
    return (f"EP-TV outer iters/sec at {cfg.nx}^2 x {cfg.nviews} views (slice-iterations/s: slices x outer "
            "iterations / s)")


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="c4")
    ap.add_argument("--batch", type=int, default=0, help="override the number of slices (debug)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--geom-flags", type=int, default=0,
                    help="ctr_geometry.flags (1 no tables, 2 no graphs, 4 batched P on the fly, 8 CGLS re-orthogonalisation in image space only): A/B runs")
    return ap.parse_args()


# ----------------------------------------------------------------------------------------------
class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.gpu, self.rows, self.proc = gpu_index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.gpu), "-lms", "50"], stdout=subprocess.PIPE, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except Exception:
                self.proc.kill()
        sm = [float(r[1]) for r in self.rows if len(r) >= 9 and r[1].replace(".", "").isdigit()]
        mx = [float(r[2]) for r in self.rows if len(r) >= 9 and r[2].replace(".", "").isdigit()]
        reasons = set()
        for r in self.rows:
            if len(r) >= 9:
                for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[5:9]):
                    if v.lower().startswith("active"):
                        reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def oracle_step_seconds(cfg, sino_slice, n_steps):
    """Time the oracle AS IT STANDS. 2D: n_steps outer iterations (full n_cgls / n_gd) of ONE slice; returns
    (seconds per step of one slice, threads, description). 3D (c5: one outer iteration is ~10-20 minutes of CPU):
    a bounded sample of the same step - P and P^T over 2 of the views of the full volume, one weight update + GD
    sweep on 8 of the z-planes - scaled to (n_cgls + 1) applications of all views and n_gd sweeps of all planes."""
    from oracle import ctr_oracle as orc
    orc.build()
    if cfg.ndim == 2:
        one = scaled_config(cfg.name, batch=1, n_outer=n_steps)
        t0 = time.perf_counter()
        orc.reconstruct(one, sino_slice.astype(np.float64), one)
        secs = (time.perf_counter() - t0) / n_steps
        return secs, orc.num_threads(), (f"one slice of {cfg.batch}, {n_steps} outer iteration(s) from f = 0 at the full "
                                         f"per-iteration schedule (n_cgls={cfg.n_cgls}, n_gd={cfg.n_gd}), {secs * n_steps:.1f} s")
    nv_s, nz_s = 2, 8
    sub = scaled_config(cfg.name, nviews=nv_s)             # same scanner and volume, nv_s equally spaced views
    g = sub.geometry_dict() | {"angles": [cfg.theta0 + k * cfg.dtheta * (cfg.nviews // nv_s) for k in range(nv_s)]}
    rng = np.random.default_rng(0)
    x = rng.random(cfg.img_shape)
    t0 = time.perf_counter()
    for _ in range(n_steps):
        y = orc.forward(g, x)
        orc.back(g, y)
    t_op = (time.perf_counter() - t0) / n_steps * (cfg.nviews / nv_s) * (cfg.n_cgls + 1)
    f = 0.02 * rng.random((nz_s, cfg.ny, cfg.nx))
    t0 = time.perf_counter()
    for _ in range(n_steps):
        w, _ = orc.update_weights(f, cfg.sigma_quantile, cfg.eps, 0, ndim=3)
        orc.eptv_step(f, f, w, cfg.lam, cfg, ndim=3)
    t_tv = (time.perf_counter() - t0) / n_steps * (cfg.nz / nz_s) * cfg.n_gd
    return t_op + t_tv, orc.num_threads(), (
        f"bounded sample of one outer iteration: P + P^T over {nv_s} of {cfg.nviews} views (x{cfg.nviews // nv_s} x "
        f"{cfg.n_cgls + 1} applications) and one weight update + GD sweep on {nz_s} of {cfg.nz} planes (x{cfg.nz // nz_s} x "
        f"{cfg.n_gd}), extrapolated to {t_op + t_tv:.0f} s per step")


def run_reference(args):
    """--impl reference: the oracle on the host cores, each step = one outer iteration of ONE slice of
    the workload (a bounded sample: 1/batch of a real step; c5: see oracle_step_seconds)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = get_config(args.workload)
    sino = None
    if cfg.ndim == 2:
        sino = make_case(scaled_config(args.workload, batch=1), raster=False)["sino"][0]
        if args.warmup > 0:
            oracle_step_seconds(cfg, sino, args.warmup)
    secs, cores, sample = oracle_step_seconds(cfg, sino, args.steps)
    value = 1.0 / secs
    print(json.dumps({
        "impl": "reference", "metric": metric_name(cfg), "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * secs,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(cfg, cfg.batch) | {"sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def workload_config(cfg, batch):
    if cfg.ndim == 3:
        what = (f"{cfg.name}: cone beam, volume {cfg.nz}x{cfg.ny}x{cfg.nx} @ {cfg.dx:.2f} mm, {cfg.nviews} views x "
                f"{cfg.nv}x{cfg.nu} bins @ {cfg.du:.2f} mm")
        nbytes = 4.0 * (9 * cfg.n_pix + 4 * cfg.n_rays)
    else:
        what = (f"{cfg.name}: {batch} slice{'s' if batch > 1 else ''} x {cfg.ny}x{cfg.nx} @ {cfg.dx:.2f} mm, "
                f"{cfg.nviews} views x {cfg.nu} bins")
        nbytes = 4.0 * batch * (9 * cfg.nx * cfg.ny + 4 * cfg.nviews * cfg.nu)
    big = nbytes > 126e6
    return {"workload": what + f", flat detector, dso {cfg.dso:.0f} / dsd {cfg.dsd:.0f} mm",
            "n_cgls": cfg.n_cgls, "n_gd": cfg.n_gd, "lambda": cfg.lam, "I0": cfg.I0, "slices_per_gpu": batch,
            "l2_policy": (f"working set of one step (~{nbytes / 1e6:.0f} MB of vectors + tables) is larger than the 126 MB L2; "
                          "no explicit flush") if big else
                         (f"working set of one step (~{nbytes / 1e6:.1f} MB of vectors) is L2-resident by nature of this small "
                          "workload; the stored matrices (if any) stream from HBM every application; no explicit flush")}


# ----------------------------------------------------------------------------------------------
def main():
    args = parse()
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist
    import paper_1009_2288_b200 as ctr
    from paper_1009_2288_b200 import shard

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    cfg = get_config(args.workload)
    batch = args.batch or cfg.batch
    cfg = scaled_config(args.workload, batch=batch)
    K, W = args.steps, max(args.warmup, 0)

    # each rank reconstructs its own slices: slice seeds rank*batch .. rank*batch+batch-1
    case = make_case(cfg, slices=shard.slice_range(rank, world, batch), raster=False)
    sino_host = torch.from_numpy(case["sino"]).pin_memory()
    sino = sino_host.cuda(non_blocking=True)
    # on-chip peaks of THIS device, measured before anything is timed (roofline denominators)
    dev_peaks = ctr.ctr_measure_peaks(5)
    h = ctr.ctr_create(cfg, flags=args.geom_flags)
    path = h.ctr_path_info()
    img = torch.zeros(h.img_shape, device="cuda")
    img_host = torch.empty(h.img_shape, dtype=torch.float32).pin_memory()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def steps(n, warm):
        h.ctr_reconstruct(sino, img, ctr.make_params(cfg, n_outer=n, warm_start=int(warm)))

    # ---- device-resident timing: W warm-up steps (from f = 0), then exactly K more steps
    if W:
        steps(W, False)
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    l0 = h.ctr_launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record()
    steps(K, W > 0)
    ev1.record()
    barrier()
    ms = ev0.elapsed_time(ev1)
    launches = h.ctr_launch_count() - l0
    clocks = sampler.stop()

    # ---- per-kernel breakdown: the same K steps again with the library's event profiler on (an event pair
    # around every launch group costs ~0.5 ms per step, so it stays out of the timed region above)
    h.ctr_profile_enable(True)
    steps(K, True)
    barrier()
    prof = h.ctr_profile_read()
    h.ctr_profile_enable(False)

    # ---- end to end through the C ABI with HOST buffers: per step H2D(sino) + step + D2H(image), all inside the
    # timed region. The copies run on a second stream, double-buffered, so that the upload of step n+1 and the
    # download of step n overlap the kernels of the neighbouring step (what a pipeline of batches would do).
    img.zero_()
    steps(1, False)
    barrier()
    main, side = torch.cuda.current_stream(), torch.cuda.Stream()
    sino_buf = [sino, torch.empty_like(sino)]
    stage = torch.empty_like(img)
    ev_in = [torch.cuda.Event(), torch.cuda.Event()]
    ev_step, ev_out = torch.cuda.Event(), torch.cuda.Event()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    side.wait_stream(main)
    with torch.cuda.stream(side):
        sino_buf[0].copy_(sino_host, non_blocking=True)
        ev_in[0].record(side)
    for n in range(K):
        main.wait_event(ev_in[n % 2])
        h.ctr_reconstruct(sino_buf[n % 2], img, ctr.make_params(cfg, n_outer=1, warm_start=1))
        if n + 1 < K:
            with torch.cuda.stream(side):          # this step's kernels have been enqueued on `main` already
                sino_buf[(n + 1) % 2].copy_(sino_host, non_blocking=True)
                ev_in[(n + 1) % 2].record(side)
        if n > 0:
            main.wait_event(ev_out)                # the previous download has left `stage`
        stage.copy_(img, non_blocking=True)
        ev_step.record(main)
        with torch.cuda.stream(side):
            side.wait_event(ev_step)
            img_host.copy_(stage, non_blocking=True)
            ev_out.record(side)
    main.wait_event(ev_out)
    e1.record()
    barrier()
    ms_e2e = e0.elapsed_time(e1)

    ms, ms_e2e = shard.max_over_ranks([ms, ms_e2e], device="cuda")
    value = world * batch * K / (ms * 1e-3)
    e2e_value = world * batch * K / (ms_e2e * 1e-3)

    if rank == 0:
        peaks = {}
        try:
            peaks = json.loads((ROOT / "MEASURED_PEAKS.json").read_text())
        except Exception:
            pass
        out = {
            "metric": metric_name(cfg), "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic", "config": workload_config(cfg, batch),
            "clocks": clocks, "gpu_launches": int(launches),
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": sino_host.numel() * 4,
                    "d2h_bytes_per_step": img_host.numel() * 4, "ms_per_step": ms_e2e / K},
            "kernel_ms_per_step": {k: v[0] / K for k, v in prof.items()},
            "kernel_launch_groups_per_step": {k: v[1] / K for k, v in prof.items()},
        }
        out["roofline"] = roofline(cfg, batch, prof, peaks, dev_peaks, path)
        out["hbm_bound_parts"] = hbm_kinds(cfg, batch, prof, peaks, K, dev_peaks)
        # north_star's list of absolute numbers, derived from the same run (event-timed kinds; whole job = all ranks)
        kms = out["kernel_ms_per_step"]
        n_app, n_app_t = cfg.n_cgls + 1, max(cfg.n_cgls, 1)       # applications of P and of P^T per outer iteration (O4: the last P^T is skipped)
        comp = 4.0 * batch * (cfg.nx * cfg.ny * cfg.nz + cfg.nviews * cfg.nu * cfg.nv)
        cgls_ms = kms["forward"] + kms["back"] + kms["vector"]
        out["north_star_numbers"] = {
            "P_ms_per_application": kms["forward"] / n_app, "PT_ms_per_application": kms["back"] / n_app_t,
            "P_compulsory_GBps": comp / (kms["forward"] / n_app * 1e-3) / 1e9 if kms["forward"] > 0 else None,
            "PT_compulsory_GBps": comp / (kms["back"] / n_app_t * 1e-3) / 1e9 if kms["back"] > 0 else None,
            "cgls_slice_iterations_per_s": world * batch * cfg.n_cgls / (cgls_ms * 1e-3) if cgls_ms > 0 else None,
            "full_reconstructions_per_s": value / get_config(args.workload).n_outer,
            "note": f"compulsory bytes = image + sinogram once per application; CGLS: {cfg.n_cgls} iterations per outer iteration over "
                    f"forward + back + vector time; a full reconstruction = {get_config(args.workload).n_outer} outer iterations of every slice"}
        out["measured_peaks_this_run"] = dev_peaks
        out["kernel_path"] = path
        if not args.no_cpu_baseline:
            secs, cores, sample = oracle_step_seconds(cfg, case["sino"][0] if cfg.ndim == 2 else None,
                                                      5 if cfg.name in ("c3", "c4") else (1 if cfg.ndim == 3 else 20))
            out["cpu_baseline"] = {"value": 1.0 / secs, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample}
        print(json.dumps(out))
    h.close()
    if world > 1:
        dist.destroy_process_group()


NNZ = {"c1": 2.32e5, "c2": 4.60e6, "c3": 2.95e7, "c4": 2.95e7, "c5": 4.37e9}  # nnz(P) per slice / volume


def ncu_row(cfg, batch, kernel_substr):
    """Per-launch figures of a kernel from the committed `ncu --set full` capture of this workload
    (profiles/ncu_per_launch.csv: workload,batch,kernel,dram_bytes,l2_to_l1_bytes,warp_insts,source), or None."""
    try:
        for line in (ROOT / "profiles" / "ncu_per_launch.csv").read_text().splitlines()[1:]:
            wl, b, kern, dram, l2, inst, src = [c.strip() for c in line.split(",", 6)]
            if wl == cfg.name and int(b) == batch and kern in kernel_substr:
                num = lambda x: float(x) if x else None  # noqa: E731
                return {"dram": num(dram), "l2": num(l2), "inst": num(inst), "src": src}
    except Exception:
        pass
    return None


def ncu_traffic(cfg, batch, kernel_substr):
    row = ncu_row(cfg, batch, kernel_substr)
    return (row["dram"], row["src"]) if row else (None, None)


def roofline(cfg, batch, prof, peaks, dev_peaks, path):
    """Dominant kernel = the slower of the projector pair (a1 / a2), DESIGN.md section 5.

    Batched (c4): both kernels are bound by the L1 data pipe (ncu: l1tex 80+ % busy; DRAM 5-25 %; FMA pipe 30-45 %):
    every non-zero of P moves 4 bytes per slice through an L1. achieved = 4 B x nnz(P) x slices / launch time;
    peak = L1 load bandwidth MEASURED in this run by ctr_measure_peaks (LDG.128 hitting L1 at full occupancy).
    The fp32-FMA view (2 flop per non-zero and slice over the measured FFMA peak) and the HBM view BASELINE.json's
    metric asks for (compulsory image + sinogram bytes over MEASURED_PEAKS.json's copy bandwidth) are beside it.
    Single problems (c1-c3, c5) apply stored matrices: 8 B per non-zero streamed from HBM."""
    nnz = NNZ[cfg.name]
    kind = max(("forward", "back"), key=lambda k: prof[k][0])
    hbm = peaks.get("hbm_gbs", 6650.0)
    hbm_src = "MEASURED_PEAKS.json hbm_gbs (measured)" if "hbm_gbs" in peaks else "fallback 6650 GB/s (B200_PROFILING.md)"
    bytes_alg = 4.0 * batch * (cfg.nx * cfg.ny * cfg.nz + cfg.nviews * cfg.nu * cfg.nv)

    def launch_s(k):
        ms, n = prof[k]
        return ms / max(n, 1) * 1e-3, n

    if batch == 1:
        stored = "ell" in path.get(kind, "")
        sec, n = launch_s(kind)
        traffic, tsrc = ncu_traffic(cfg, batch, path.get(kind, ""))
        if stored:
            ach = 8.0 * nnz / sec / 1e9
            return {"bound": "hbm", "kernel": f"{path.get(kind)} ({'P, a1' if kind == 'forward' else 'P^T, a2'})",
                    "achieved": ach, "peak": hbm, "unit": "GB/s", "frac": ach / hbm, "traffic": traffic,
                    "traffic_source": tsrc, "avg_launch_ms": sec * 1e3, "launches": n, "peak_source": hbm_src,
                    "note": "algorithmic bytes = 8 B x nnz(P) of the stored matrix (index + weight), streamed once per "
                            "application; for c1-c3 the vectors are L2-resident"}
        ach = 2.0 * nnz / sec / 1e12
        return {"bound": "alu", "kernel": path.get(kind), "achieved": ach, "peak": dev_peaks["fma_tflops"],
                "unit": "TFLOP/s", "frac": ach / dev_peaks["fma_tflops"], "traffic": traffic, "traffic_source": tsrc,
                "avg_launch_ms": sec * 1e3, "launches": n,
                "peak_source": "fp32 FFMA rate measured in this run (ctr_measure_peaks)",
                "note": "on-the-fly kernel (lookup tables not built): 2 flop per non-zero of P"}

    def view(k):
        sec, n = launch_s(k)
        row = ncu_row(cfg, batch, path.get(k, "")) or {}
        l1 = 4.0 * nnz * batch / sec / 1e9
        fma = 2.0 * nnz * batch / sec / 1e12
        out = {"kernel": f"{path.get(k)} ({'P, a1' if k == 'forward' else 'P^T gather, a2'})",
               "achieved": l1, "peak": dev_peaks["l1_tbs"] * 1e3, "unit": "GB/s", "frac": l1 / (dev_peaks["l1_tbs"] * 1e3),
               "traffic": row.get("dram"), "traffic_source": row.get("src"), "avg_launch_ms": sec * 1e3, "launches": n,
               "fma_view": {"achieved": fma, "peak": dev_peaks["fma_tflops"], "unit": "TFLOP/s",
                            "frac": fma / dev_peaks["fma_tflops"]},
               "hbm_view": {"achieved": bytes_alg / sec / 1e9, "peak": hbm, "unit": "GB/s",
                            "frac": bytes_alg / sec / 1e9 / hbm, "peak_source": hbm_src,
                            "note": "compulsory bytes (image + sinogram once) of one application"}}
        if row.get("l2") and dev_peaks.get("l2_tbs"):
            l2 = row["l2"] / sec / 1e9
            out["l2_view"] = {"achieved": l2, "peak": dev_peaks["l2_tbs"] * 1e3, "unit": "GB/s", "frac": l2 / (dev_peaks["l2_tbs"] * 1e3),
                              "note": "bytes that cross the L2 -> SM fabric per launch (ncu, profiles/ncu_per_launch.csv) over this "
                                      "run's launch time; peak = LDG.128 cache-global over an L2-resident window, measured in this run"}
        return out

    return {"bound": "l1", **view(kind),
            "peak_source": "L1 load bandwidth measured in this run by ctr_measure_peaks (LDG.128 hitting L1, full "
                           "occupancy); fma_view: measured FFMA rate; hbm_view: " + hbm_src,
            "note": "algorithmic bytes = 4 B per non-zero of P per slice through the L1 data pipe, the unit ncu shows "
                    "busiest for this kernel (profiles/)",
            "other": view("back" if kind == "forward" else "forward")}


def hbm_kinds(cfg, batch, prof, peaks, steps, dev_peaks=None):
    """The HBM-bound parts of a step: CGLS vector work (a3) and the TV sweeps (a4-a7),
    algorithmic bytes per unit over the measured copy bandwidth."""
    hbm = peaks.get("hbm_gbs", 6650.0)
    npix, nray = cfg.nx * cfg.ny * cfg.nz * batch, cfg.nviews * cfg.nu * cfg.nv * batch
    out = {}
    ms_v = prof["vector"][0] / steps
    by_v = (20.0 * npix + 12.0 * nray) * cfg.n_cgls
    out["cgls_vector"] = {"ms_per_step": ms_v, "algorithmic_bytes_per_step": by_v,
                          "achieved_GBps": by_v / (ms_v * 1e-3) / 1e9 if ms_v > 0 else None,
                          "frac_of_measured_hbm": by_v / (ms_v * 1e-3) / 1e9 / hbm if ms_v > 0 else None,
                          "note": "20 B/pixel + 12 B/ray per CGLS iteration (SURVEY.md 8(d) a3); the S24 "
                                  "re-orthogonalisation reads are extra traffic, not algorithmic bytes"}
    ms_t = prof["tv"][0] / steps
    by_t = 44.0 * npix * cfg.n_gd
    out["tv_sweeps"] = {"ms_per_step": ms_t, "ms_per_sweep": ms_t / max(cfg.n_gd, 1), "algorithmic_bytes_per_step": by_t,
                        "achieved_GBps": by_t / (ms_t * 1e-3) / 1e9 if ms_t > 0 else None,
                        "frac_of_measured_hbm": by_t / (ms_t * 1e-3) / 1e9 / hbm if ms_t > 0 else None,
                        "note": "44 B/pixel per sweep, the lower figure of SURVEY.md 8(d) a4-a7 (60 B/pixel would "
                                "read 1.36x higher); the fused sweep moves 40 B/pixel"}
    row = ncu_row(cfg, batch, "tv_sweep")
    if row and row.get("inst") and dev_peaks and ms_t > 0 and cfg.n_gd > 0:
        # the sweep is bound by instruction issue, not by HBM (profiles/): warp instructions of one sweep (ncu) over this
        # run's time per sweep, against the issue rate measured in this run
        rate = row["inst"] / (ms_t / cfg.n_gd * 1e-3) / 1e9
        out["tv_sweeps"]["issue_view"] = {"warp_insts_per_sweep": row["inst"], "source": row["src"], "achieved_gwinst": rate,
                                          "peak_gwinst": dev_peaks["issue_gwinst"], "frac": rate / dev_peaks["issue_gwinst"],
                                          "peak_mixed_gwinst": dev_peaks["mixed_gwinst"],
                                          "frac_of_mixed": rate / dev_peaks["mixed_gwinst"],
                                          "note": "peak = one warp instruction per clock and scheduler (FFMA stream); mixed = FFMA and "
                                                  "integer instructions 1:1"}
    return out


if __name__ == "__main__":
    main()

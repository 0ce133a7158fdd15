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

METRIC = "EP-TV outer iters/sec at 512^2 x 60 views (slice-iterations/s: slices x outer iterations / s)"
UNIT = "slice-iters/s"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="c4")
    ap.add_argument("--batch", type=int, default=0, help="override the number of slices (debug)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
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
    """Time the oracle AS IT STANDS on one slice: n_steps outer iterations (full n_cgls / n_gd)."""
    from oracle import ctr_oracle as orc
    orc.build()
    one = scaled_config(cfg.name, batch=1, n_outer=n_steps)
    t0 = time.perf_counter()
    orc.reconstruct(one, sino_slice.astype(np.float64), one)
    return time.perf_counter() - t0, orc.num_threads()


def run_reference(args):
    """--impl reference: the oracle on the host cores, each step = one outer iteration of ONE slice of
    the workload (a bounded sample: 1/batch of a real step)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = get_config(args.workload)
    sino = make_case(scaled_config(args.workload, batch=1), raster=False)["sino"][0]
    if args.warmup > 0:
        oracle_step_seconds(cfg, sino, args.warmup)
    secs, cores = oracle_step_seconds(cfg, sino, args.steps)
    value = args.steps / secs
    sample = f"1 of {cfg.batch} slices per step, full schedule per step (n_cgls={cfg.n_cgls}, n_gd={cfg.n_gd})"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * secs / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(cfg, cfg.batch) | {"sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def workload_config(cfg, batch):
    return {"workload": f"{cfg.name}: {batch} slices x {cfg.ny}x{cfg.nx} @ {cfg.dx:.2f} mm, {cfg.nviews} views x "
                        f"{cfg.nu} bins, flat detector, dso {cfg.dso:.0f} / dsd {cfg.dsd:.0f} mm",
            "n_cgls": cfg.n_cgls, "n_gd": cfg.n_gd, "lambda": cfg.lam, "I0": cfg.I0, "slices_per_gpu": batch,
            "l2_policy": "working set (~2.3 GB per GPU at c4) is larger than the 126 MB L2; no explicit flush"}


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
    h = ctr.ctr_create(cfg)
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
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic", "config": workload_config(cfg, batch),
            "clocks": clocks, "gpu_launches": int(launches),
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": sino_host.numel() * 4,
                    "d2h_bytes_per_step": img_host.numel() * 4, "ms_per_step": ms_e2e / K},
            "kernel_ms_per_step": {k: v[0] / K for k, v in prof.items()},
            "kernel_launch_groups_per_step": {k: v[1] / K for k, v in prof.items()},
        }
        out["roofline"] = roofline(cfg, batch, prof, peaks)
        if not args.no_cpu_baseline:
            secs, cores = oracle_step_seconds(cfg, case["sino"][0], 1)
            out["cpu_baseline"] = {"value": 1.0 / secs, "unit": UNIT, "cores": cores, "kind": "oracle",
                                   "sample": f"slice 0 of {batch}, one outer iteration from f = 0 "
                                             f"(n_cgls={cfg.n_cgls}, n_gd={cfg.n_gd}), {secs:.1f} s"}
        print(json.dumps(out))
    h.close()
    if world > 1:
        dist.destroy_process_group()


# dram__bytes_read.sum + dram__bytes_write.sum per launch of the batched kernels at c4, from the committed
# ncu --set full captures (profiles/r1i_ncu_full_c4.md); None for workloads that were not captured
NCU_TRAFFIC_C4 = {"forward": 170.5e6, "back": 559.0e6}


def roofline(cfg, batch, prof, peaks):
    """Dominant kernel = the slower of the projector pair (a1 / a2). Both are bound by on-chip work, not HBM
    (DESIGN.md section 6): algorithmic work per application = one FMA (2 flop) per non-zero of P, i.e. per
    ray-pixel intersection, per slice; nnz(P) per slice is counted from the geometry (2.95e7
    for the 512^2 / 60 x 888 geometry). Peak = fp32 FMA peak of the chip, 148 SMs x 128 lanes x 2 flop x
    sm_max_mhz (B200_PROFILING.md unit counts, MEASURED_PEAKS.json clock). The HBM view of the same launch
    (compulsory image + sinogram bytes against the measured copy bandwidth) is reported beside it, as
    BASELINE.json's metric asks, with the ncu-measured DRAM traffic."""
    nnz = {"c1": 2.32e5, "c2": 4.60e6, "c3": 2.95e7, "c4": 2.95e7, "c5": 4.37e9}[cfg.name]
    kind = max(("forward", "back"), key=lambda k: prof[k][0])
    names = {"forward": "k_si_forward (P, a1)" if batch > 1 else "k_ell_apply<0> (stored P, a1)",
             "back": "k_si_back_quad (P^T gather, a2)" if batch > 1 else "k_ell_apply<1> (stored P^T, a2)"}
    sm_mhz = peaks.get("sm_max_mhz", 1965.0)
    peak = 148 * 128 * 2 * sm_mhz * 1e6 / 1e12
    hbm = peaks.get("hbm_gbs", 6650.0)
    bytes_alg = 4.0 * batch * (cfg.nx * cfg.ny * cfg.nz + cfg.nviews * cfg.nu * cfg.nv)

    def one(k):
        ms, n = prof[k]
        sec = ms / max(n, 1) * 1e-3
        ach = 2.0 * nnz * batch / sec / 1e12
        return {"kernel": names[k], "achieved": ach, "peak": peak, "unit": "TFLOP/s", "frac": ach / peak,
                "avg_launch_ms": sec * 1e3, "launches": n,
                "traffic": NCU_TRAFFIC_C4.get(k) if (cfg.name == "c4" and batch == 64) else None,
                "compulsory_GBps": bytes_alg / sec / 1e9,
                "compulsory_GBps_frac_of_measured_hbm": bytes_alg / sec / 1e9 / hbm}

    # the unit that actually binds both kernels (ncu: l1tex data pipe 78 % busy): every non-zero of P moves
    # 4 bytes per slice through an L1; peak = 148 SMs x 128 B/clk x sm_max_mhz
    sec_k = prof[kind][0] / max(prof[kind][1], 1) * 1e-3
    l1_peak = 148 * 128 * sm_mhz * 1e6 / 1e12
    l1 = {"bound": "l1 gather bandwidth", "achieved": 4.0 * nnz * batch / sec_k / 1e12, "peak": l1_peak, "unit": "TB/s",
          "frac": 4.0 * nnz * batch / sec_k / 1e12 / l1_peak,
          "note": "algorithmic gather bytes (4 B per non-zero of P per slice) over the L1 data-pipe peak"}
    if batch == 1:
        # single problems apply stored matrices: 8 bytes per non-zero streamed from HBM
        ms_k, n_k = prof[kind]
        ach = 8.0 * nnz / (ms_k / max(n_k, 1) * 1e-3) / 1e9
        return {"bound": "hbm", "kernel": names[kind], "achieved": ach, "peak": hbm, "unit": "GB/s", "frac": ach / hbm,
                "traffic": None, "avg_launch_ms": ms_k / max(n_k, 1), "launches": n_k,
                "peak_source": "MEASURED_PEAKS.json hbm_gbs (measured)" if "hbm_gbs" in peaks else "fallback 6650 GB/s",
                "note": "algorithmic bytes = 8 B x nnz(P) of the stored matrix (index + weight)"}
    out = {"bound": "alu", **one(kind), "l1_view": l1,
           "peak_source": "derived: 148 SM x 128 fp32 FMA lanes x 2 flop x sm_max_mhz (MEASURED_PEAKS.json clock); "
                          "hbm_gbs of measured" if "hbm_gbs" in peaks else "fallback 6650 GB/s",
           "other": one("back" if kind == "forward" else "forward")}
    return out


if __name__ == "__main__":
    main()

#!/usr/bin/env python
"""bench.py -- BASELINE.json's metric on its headline workload (config 3: 640x480, 500k Gaussians, D = 512 fp32, K = 40).

A step = one pass of the whole Q-Render hot path over one synthetic frame, through the C ABI:
    qr_preprocess -> qr_bin_sort -> qr_forward -> qr_backward -> qr_backward_clear
(qr_bin_count sizes the intersection lists once, before the timed region; the timed steps pass that size + 25 % as
the lists' capacity, so no step synchronises with the host, and the count found is verified afterwards)
(dL/dF is zeroed once before the loop; qr_backward_clear re-zeroes exactly the rows the step's qr_backward touched,
which is what a training loop does after consuming the gradient, instead of a 1.02 GB memset per step)
`value` = Mpix/s of that step with inputs resident in HBM (CUDA events, max over ranks).  The dense comparator
(qr_dense_forward) is timed beside it in the same run and reported under "dense"; it is not part
of the step.  `roofline` describes the dominant kernel (the longer of qr_forward / qr_backward), timed with CUDA
events around each call inside the timed steps.  `e2e` repeats the step with HOST (pinned) inputs and outputs, the
copies inside the timed region.  `cpu_baseline` times the CPU oracle on one full frame on the box's host cores.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--workload cfg3]
N > 1: launched by torch.distributed.run, one rank per GPU, independent replicas of the same frame (weak scaling,
no data-path collective: SURVEY 8(e)); rank 0 prints the one JSON line.
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

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "512-D feature-map Mpix/s (fwd+bwd step: preprocess, bin/sort, Q-Render forward, backward)"
UNIT = "Mpix/s"
NOMINAL_HBM_GBS = 8000.0


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 100 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.lines.append(ln.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 6:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for n, v in zip(names, f[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def scene_for(args):
    """BASELINE.json's configs; --D / --K / --pose pick a point of the sweeps of configs 4 (K, pose) and 5 (D)."""
    from qr_inputs import make_scene
    return make_scene(args.workload, seed=0, D=args.D, K=args.K, pose=args.pose)


# ----------------------------------------------------------------------------------------------------------------
# reference arm: the CPU oracle, as it stands, on the host cores
# ----------------------------------------------------------------------------------------------------------------
def oracle_frame(orc, sc):
    """One full frame of the path in the oracle: O1 projection, O2b lists, O4 Algorithm 1 with features, O5 backward."""
    proj = orc.project(sc.cam, sc.means, sc.scales, sc.quats, sc.opac)
    rect, touched = orc.tile_rects(sc.cam, proj)
    orc.tile_lists(sc.cam, proj.depth, rect, touched)
    lists = orc.pixel_lists(sc.cam, proj)
    q = orc.qrender(lists, sc.K, sc.features)
    if sc.dL_dmap is not None:
        sel = q.sel_idx[q.sel_idx >= 0]            # the oracle pads its records with -1
        rows = np.unique(sel).astype(np.int64)
        orc.backward(q.sel_idx, q.sel_w, q.n_sel, sc.dL_dmap, sc.N, rows=rows)
    return q


def time_oracle(sc, steps: int, warmup: int):
    from oracle import qr_oracle as orc
    for _ in range(warmup):
        oracle_frame(orc, sc)
    ts = []
    for _ in range(steps):
        t0 = time.perf_counter()
        oracle_frame(orc, sc)
        ts.append(time.perf_counter() - t0)
    return ts, orc.num_threads()


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    sc = scene_for(args)
    steps = max(1, min(args.steps, 3))          # one frame is ~10 s of CPU work: bound the run to a few minutes
    warm = min(args.warmup, 1)
    ts, cores = time_oracle(sc, steps, warm)
    npix = sc.cam.width * sc.cam.height
    ms = 1e3 * sum(ts) / len(ts)
    val = npix / (ms * 1e-3) / 1e6
    sample = f"{steps} full frame(s) of {args.workload} ({npix} px, all stages O1-O5), OpenMP over rows where the oracle has it"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
            "warmup": warm, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": workload_config(sc, args.workload),
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))
    return 0


def workload_config(sc, name):
    idx = {"cfg1": 0, "cfg2": 1, "cfg3": 2, "cfg4": 3, "cfg5": 4}.get(name, -1)
    kind = "64 blobs" if sc.meta.get("kind") == "blobs" else "uniform"
    esz = 2 if sc.feat_dtype == "f16" else 4
    mb = lambda n: f"{n / 1e6:.0f} MB"
    npix = sc.cam.width * sc.cam.height
    return {"workload": f"{name}: {sc.cam.width}x{sc.cam.height}, N={sc.N} Gaussians ({kind}), D={sc.D} "
                        f"{sc.feat_dtype}, K={sc.K}, forward+backward (BASELINE.json configs[{idx}])",
            "K": sc.K, "D": sc.D, "N": sc.N, "width": sc.cam.width, "height": sc.cam.height,
            "l2": f"inputs vs the 126 MB L2: features {mb(sc.N * sc.D * esz)}, dL_dmap {mb(npix * sc.D * 4)}, map "
                  f"{mb(npix * sc.D * 4)}; " + ("larger than L2, no flush needed" if npix * sc.D * 4 > 2.5e8 else
                                               "SMALLER than L2: figures at this size are L2-resident, not HBM, numbers")}


# ----------------------------------------------------------------------------------------------------------------
# CUDA arm
# ----------------------------------------------------------------------------------------------------------------
def run_cuda(args):
    import torch
    import torch.distributed as dist

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: libqr has no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    import paper_2512_20927_b200 as qr
    from paper_2512_20927_b200 import pipeline as pl
    qr.binding.load()

    sc = scene_for(args)
    cam, K, D, N = sc.cam, sc.K, sc.D, sc.N
    H, W = cam.height, cam.width
    npix = H * W
    dev = torch.device("cuda", local)
    host = {k: torch.from_numpy(np.ascontiguousarray(getattr(sc, k))).pin_memory()
            for k in ("means", "scales", "quats", "opac", "features", "dL_dmap")}
    d = {k: v.to(dev, non_blocking=True) for k, v in host.items()}
    dF = torch.zeros((N, D), dtype=torch.float32, device=dev)      # zeroed ONCE; every step re-zeroes the rows it touched
    bws = qr.qr_backward_workspace(cam, K, D, dev)
    fwd_out = None
    ev = lambda: torch.cuda.Event(enable_timing=True)
    launches = {"n": 0}

    # Front end: the first (untimed) step sizes the intersection lists exactly with qr_bin_count (one device->host
    # read); every later step passes 1.25 x that count as the capacity of the lists, so nothing in the timed region
    # synchronises with the host.  The count found on the device is checked against the capacity after the loop.
    state = {"capacity": None, "found": []}

    def step(timers=None):
        nonlocal fwd_out
        fe = pl.frontend(cam, d["means"], d["scales"], d["quats"], d["opac"], state["capacity"])
        if state["capacity"] is None:
            state["capacity"] = int(fe.M * 1.25) + 1024
        else:
            state["found"] = [fe.found]          # device scalar; only the latest is kept (holding all would pin every workspace)
        if timers is not None:
            e0, e1, e2, e3 = ev(), ev(), ev(), ev()
            e0.record()
        fwd_out = pl.forward(cam, fe, d["features"], K, fwd_out)
        if timers is not None:
            e1.record()
        pl.backward(cam, N, fwd_out, d["dL_dmap"], dF, None if fwd_out.has_lists else bws)
        if timers is not None:
            e2.record()
        # dL_dfeat would be consumed here (the 3D network's backward); then the rows this step touched are re-zeroed,
        # so that the table is all-zero again for the next step without a 1.02 GB memset
        pl.backward_clear(cam, N, fwd_out, dF, None if fwd_out.has_lists else bws)
        if timers is not None:
            e3.record()
            timers.append((e0, e1, e2, e3))
        # preprocess 1, bin_sort 5 (count, scan, scatter, 2 bucket sorts), forward 2 (walk, blend),
        # backward 3 (prep, tcgen05 contraction, FFMA kernel for the half tiles the prep left to it), clear 1
        launches["n"] += 1 + 5 + 2 + 3 + 1
        return fe

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        fe = step()
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    launches["n"] = 0
    timers = []
    s0, s1 = ev(), ev()
    barrier()
    s0.record()
    for _ in range(args.steps):
        fe = step(timers)
    s1.record()
    barrier()
    total_ms = s0.elapsed_time(s1)
    found = [int(f.item()) for f in state["found"]]
    if found and max(found) > state["capacity"]:
        raise RuntimeError(f"intersection lists overflowed their capacity ({max(found)} > {state['capacity']}): invalid run")
    t = torch.tensor([total_ms], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    total_ms = float(t.item())
    ms_step = total_ms / args.steps
    value = world * npix / (ms_step * 1e-3) / 1e6
    fwd_ms = statistics.mean(a.elapsed_time(b) for a, b, _, _ in timers)
    bwd_ms = statistics.mean(b.elapsed_time(c) for _, b, c, _ in timers)
    zero_ms = statistics.mean(c.elapsed_time(e) for _, _, c, e in timers)

    # dense comparator, same frame, same front end (not part of the step)
    dense_map = torch.empty((H, W, D), dtype=torch.float32, device=dev)
    dense_T = torch.empty((H, W), dtype=torch.float32, device=dev)
    for _ in range(2):
        pl.dense_forward(cam, fe, d["features"], 1e-4, dense_map, dense_T)
    torch.cuda.synchronize()
    a, b = ev(), ev()
    nd = 5
    a.record()
    for _ in range(nd):
        pl.dense_forward(cam, fe, d["features"], 1e-4, dense_map, dense_T)
    b.record()
    torch.cuda.synchronize()
    dense_ms = a.elapsed_time(b) / nd
    del dense_map
    # The timed region is ~15 ms at 20 steps, shorter than nvidia-smi's 100 ms sampling period: keep the SAME step
    # running (untimed, not counted anywhere) for ~0.4 s so that the clock / throttle samples are taken under this load.
    if rank == 0:
        hold_until = time.perf_counter() + 0.4
        n_before = launches["n"]
        while time.perf_counter() < hold_until:
            for _ in range(20):
                step()
            torch.cuda.synchronize()
        launches["n"] = n_before
    clocks = sampler.stop() if rank == 0 else None
    if clocks is not None:
        clocks["note"] = "sampled every 100 ms over the timed steps, the dense comparator and ~0.4 s of the same step kept running"

    # workload counts for the byte model (statistics only; torch ops outside every timed region)
    n_vis = int((fe.proj.tiles_touched != 0).sum().item())
    used = torch.arange(K, device=dev)[None, None, :] < fwd_out.n_sel[..., None]   # slots >= n_sel are not written
    sel = fwd_out.sel_idx[used]
    S = int(torch.unique(sel).numel())
    nsel_mean = float(fwd_out.n_sel.float().mean().item())
    esz = 2 if sc.feat_dtype == "f16" else 4
    M_found = found[-1] if found else fe.M
    fwd_bytes = M_found * 4 + n_vis * 32 + S * D * esz + npix * D * 4 + npix * 4
    rec_bytes = npix * (8 * K + 4)
    bwd_bytes = npix * D * 4 + S * D * 4 + rec_bytes
    peak, peak_src = _peaks()
    dom = "qr_forward" if fwd_ms >= bwd_ms else "qr_backward"
    dom_bytes, dom_ms = (fwd_bytes, fwd_ms) if dom == "qr_forward" else (bwd_bytes, bwd_ms)

    def roof(nbytes, ms, kernel, traffic=None):
        ach = nbytes / (ms * 1e-3) / 1e9
        return {"kernel": kernel, "bound": "hbm", "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                "peak_source": peak_src, "frac_of_nominal_8TBs": ach / NOMINAL_HBM_GBS, "algorithmic_bytes": nbytes,
                "ms_per_launch": ms, "traffic": traffic}

    # ---- e2e: host buffers in, host buffers out, copies inside the timed region ----
    e2e = None
    if not args.no_e2e:
        out_host = torch.empty((H, W, D), dtype=torch.float32).pin_memory()
        dF_host = torch.empty((N, D), dtype=torch.float32).pin_memory()
        dd = {k: torch.empty_like(v) for k, v in d.items()}

        def e2e_step():
            for k in dd:
                dd[k].copy_(host[k], non_blocking=True)
            fe2 = pl.frontend(cam, dd["means"], dd["scales"], dd["quats"], dd["opac"], state["capacity"])
            o = pl.forward(cam, fe2, dd["features"], K, fwd_out)
            pl.backward(cam, N, o, dd["dL_dmap"], dF, None if o.has_lists else bws)
            out_host.copy_(o.out_map, non_blocking=True)
            dF_host.copy_(dF, non_blocking=True)
            pl.backward_clear(cam, N, o, dF, None if o.has_lists else bws)

        e2e_step()
        barrier()
        ne = max(2, min(args.steps, 4))
        a, b = ev(), ev()
        a.record()
        for _ in range(ne):
            e2e_step()
        b.record()
        barrier()
        t = torch.tensor([a.elapsed_time(b)], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e_ms = float(t.item()) / ne
        h2d = sum(v.numel() * v.element_size() for v in host.values())
        d2h = out_host.numel() * 4 + dF_host.numel() * 4
        e2e = {"value": world * npix / (e_ms * 1e-3) / 1e6, "unit": UNIT, "ms_per_step": e_ms, "steps": ne,
               "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
               "note": "inputs (Gaussians, features, dL_dmap) from pinned host memory; out_map and dL_dfeat read back"}
        del out_host, dF_host, dd

    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu:
        ts, cores = time_oracle(sc, 1, 0)
        cpu_baseline = {"value": npix / ts[0] / 1e6, "unit": UNIT, "cores": cores, "kind": "oracle",
                        "seconds": ts[0],
                        "sample": f"1 full frame of {args.workload} ({npix} px; O1 projection, O2b lists, O4 Algorithm 1 "
                                  f"with D={D} features, O5 backward of the selected rows)"}

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f32", "data": "synthetic", "config": workload_config(sc, args.workload),
                "clocks": clocks, "e2e": e2e, "gpu_launches": launches["n"],
                "roofline": roof(dom_bytes, dom_ms, dom, TRAFFIC.get(dom)),
                "roofline_fwd": roof(fwd_bytes, fwd_ms, "qr_forward", TRAFFIC.get("qr_forward")),
                "roofline_bwd": roof(bwd_bytes, bwd_ms, "qr_backward", TRAFFIC.get("qr_backward")),
                "cpu_baseline": cpu_baseline,
                "kernels_ms": {"qr_forward": fwd_ms, "qr_backward": bwd_ms, "qr_backward_clear": zero_ms,
                               "frontend_and_rest": ms_step - fwd_ms - bwd_ms - zero_ms},
                "mpix_s": {"fwd_kernel": npix / fwd_ms / 1e3, "fwd_bwd_kernels": npix / (fwd_ms + bwd_ms) / 1e3,
                           "dense_fwd_kernel": npix / dense_ms / 1e3},
                "dense": {"ms": dense_ms, "speedup_qr_forward_over_dense": dense_ms / fwd_ms, "t_min": 1e-4},
                "workload_counts": {"M": M_found, "M_capacity": state["capacity"], "N_visible": n_vis, "n_sel_mean": nsel_mean, "S_distinct_selected": S,
                                    "selection_record_bytes": rec_bytes}}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


# dram__bytes_read.sum + dram__bytes_write.sum per launch from the ncu --set full capture named in profiles/ (None
# until a capture of the current kernels is committed).
TRAFFIC = {"qr_forward": 825.3e6, "qr_backward": 821.4e6}   # profiles/r1_e_full_metrics.csv (walk + blend; prep + mma)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--workload", default="cfg3")
    ap.add_argument("--D", type=int, default=None, help="feature width (config 5 sweeps 3..512)")
    ap.add_argument("--K", type=int, default=None, help="quantile count (config 4 sweeps 4..32)")
    ap.add_argument("--pose", type=int, default=None, help="camera pose 0..7 of config 4's circle")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_cuda(args)


if __name__ == "__main__":
    sys.exit(main())

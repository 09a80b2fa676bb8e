#!/usr/bin/env python
"""bench.py -- BASELINE.json's metric on its headline workload (config 3: 640x480, 500k Gaussians, D = 512 fp32, K = 40).

A step = one pass of the whole Q-Render hot path over one synthetic frame, through the C ABI:
    qr_preprocess -> qr_bin_sort -> qr_forward -> qr_backward -> qr_backward_clear
Two things a naive loop pays every step are NOT in the step, and `config.step` says so next to the number:
  * qr_bin_count and its device->host read of M: the lists are sized once, by the untimed first step; the timed steps pass
    that size + 25 % as the lists' capacity, nothing synchronises with the host, and the count found is verified afterwards;
  * the zero fill of the whole [N, D] dL_dfeat table (1.02 GB): it is zeroed once before the loop and qr_backward_clear
    re-zeroes exactly the rows the step's qr_backward touched, which is what a training loop does after consuming the
    gradient.  `kernels_ms.zero_fill_ms` reports what the whole-table fill would cost.
`value` = Mpix/s of that step with inputs resident in HBM (CUDA events, max over ranks).  The comparators -- dense V-Render
(qr_dense_forward) and top-K (qr_topk_forward, 8(f) NEXT-1) -- are timed beside it in the same run; they
are not part of the step.  `roofline` describes the dominant call (the longer of qr_forward / qr_backward), timed with CUDA
events around each call inside the timed steps; `traffic` is the DRAM traffic of an ncu capture of exactly this workload,
D and K if profiles/traffic.json has one, else null.  `gpu_launches` is counted by the library.  `e2e` repeats the step
with HOST (pinned) inputs and outputs, the copies inside the timed region, as a three-stream pipeline with doubled buffers
(upload of step i + 1 and read-back of step i - 1 under step i; `serial_ms` is the same step issued on one stream).  `cpu_baseline` times the CPU oracle on one full
frame on the box's host cores (plus its V-Render / top-K and a 1-thread figure on configs 1 and 2).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--workload cfg3] [--D d] [--K k] [--pose j]
    python bench.py --sweep cfg4|cfg5 [--out file.json] [--no-parity]     every point of BASELINE.json configs[3] / [4]
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
def _time_dense_tc(qr, pl, fr, cam, fe, out_map, out_T, cap=128, n=10, warm=3):
    # out_map / out_T hold the FFMA kernel's result on entry: keep every 37th row of it to check the tensor-core path against
    """qr_dense_forward_tc on the frame of `fr` (None where the shape is not one of the tcgen05 path): ms per call, list capacity,
    half tiles the walk flagged (lists too small: rendered by the FFMA kernel inside the call)."""
    import torch
    feats = fr.d["features"]
    if not qr.binding.lists_supported(feats.dtype, int(feats.shape[1])):
        return None
    st = {"ws": None}
    ref_rows, ref_T = out_map[::37].clone(), out_T.clone()

    def call():
        _, _, st["ws"] = pl.dense_forward_tc(cam, fe, feats, 1e-4, cap, out_map, out_T, st["ws"])
    ms = fr.time_call(call, n=n, warm=warm)
    same = bool(torch.equal(out_T, ref_T)) and bool(torch.allclose(out_map[::37], ref_rows, rtol=2e-4, atol=2e-5))
    al = lambda v: (v + 255) // 256 * 256
    nh = 2 * ((cam.width + 15) // 16) * ((cam.height + 15) // 16)
    o = al(256 + 64)
    hdr = al(o + (64 + nh) * 4)
    h = st["ws"][hdr:hdr + nh * 64].view(torch.int32).view(nh, 16)
    rec = {"ms": ms, "cap": cap, "matches_ffma_dense": same, "flagged_half_tiles": int((h[:, 5] == 1).sum().item()), "half_tiles": nh,
           "entries": int(h[:, :4].sum().item()), "union_mean": float(h[:, 4].float().mean().item())}
    st["ws"] = None
    return rec


def _traffic(workload, D, K):
    """dram__bytes_read.sum + dram__bytes_write.sum per call from the committed ncu --set full capture of exactly this
    (workload, D, K) -- profiles/traffic.json names the capture -- else None."""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    if not os.path.exists(p):
        return {}
    with open(p) as f:
        return json.load(f).get(f"{workload}:D{D}:K{K}", {})


class Frame:
    """One scene resident on the device and the step over it (all through the C ABI binding)."""

    def __init__(self, sc, dev, qr):
        import torch
        self.torch, self.qr, self.pl = torch, qr, qr.pipeline
        self.sc, self.dev = sc, dev
        self.cam, self.K, self.D, self.N = sc.cam, sc.K, sc.D, sc.N
        self.host = {k: torch.from_numpy(np.ascontiguousarray(getattr(sc, k))).pin_memory()
                     for k in ("means", "scales", "quats", "opac", "features", "dL_dmap")}
        self.d = {k: v.to(dev, non_blocking=True) for k, v in self.host.items()}
        self.dF = torch.zeros((self.N, self.D), dtype=torch.float32, device=dev)   # zeroed ONCE; each step re-zeroes what it touched
        self.bws = qr.qr_backward_workspace(self.cam, self.K, self.D, dev)
        self.fwd_out = None
        self.capacity = None          # of the intersection lists: sized by the first (untimed) step's qr_bin_count
        self.found = None
        self.fe = None

    def reset(self, cam=None, K=None):
        """Another camera pose and / or K over the same Gaussians (config 4's sweep)."""
        if cam is not None:
            self.cam = cam
            self.capacity = None
        if K is not None and K != self.K:
            self.K = K
            self.fwd_out = None
        self.bws = self.qr.qr_backward_workspace(self.cam, self.K, self.D, self.dev)

    def step(self, timers=None):
        t, pl, d = self.torch, self.pl, self.d
        fe = pl.frontend(self.cam, d["means"], d["scales"], d["quats"], d["opac"], self.capacity)
        if self.capacity is None:
            self.capacity = int(fe.M * 1.25) + 1024
        else:
            self.found = fe.found            # device scalar; only the latest is kept
        if timers is not None:
            ev = [t.cuda.Event(enable_timing=True) for _ in range(4)]
            ev[0].record()
        self.fwd_out = pl.forward(self.cam, fe, d["features"], self.K, self.fwd_out)
        if timers is not None:
            ev[1].record()
        ws = None if self.fwd_out.has_lists else self.bws
        pl.backward(self.cam, self.N, self.fwd_out, d["dL_dmap"], self.dF, ws)
        if timers is not None:
            ev[2].record()
        # dL_dfeat would be consumed here (the 3D network's backward); then the rows this step touched are re-zeroed,
        # so that the table is all-zero again for the next step without a 1.02 GB memset
        pl.backward_clear(self.cam, self.N, self.fwd_out, self.dF, ws)
        if timers is not None:
            ev[3].record()
            timers.append(ev)
        self.fe = fe
        return fe

    def capture(self):
        """The step as four CUDA graphs (front end | qr_forward | qr_backward | qr_backward_clear): the same library calls, captured
        once on a side stream and replayed, so that the ~12 launches and memsets of a step cost four graph launches.  Events are
        recorded between the replays, so the per-call timings stay live.  Returns False (and the step stays eager) if capture
        is not possible."""
        t, pl, d = self.torch, self.pl, self.d
        try:
            if self.capacity is None:
                self.step()
            t.cuda.synchronize()
            n0 = self.qr.binding.qr_launch_count()
            g = [t.cuda.CUDAGraph() for _ in range(4)]
            pool = t.cuda.graph_pool_handle()
            with t.cuda.graph(g[0], pool=pool):
                fe = pl.frontend(self.cam, d["means"], d["scales"], d["quats"], d["opac"], self.capacity)
            with t.cuda.graph(g[1], pool=pool):
                self.fwd_out = pl.forward(self.cam, fe, d["features"], self.K, self.fwd_out)
            ws = None if self.fwd_out.has_lists else self.bws
            with t.cuda.graph(g[2], pool=pool):
                pl.backward(self.cam, self.N, self.fwd_out, d["dL_dmap"], self.dF, ws)
            with t.cuda.graph(g[3], pool=pool):
                pl.backward_clear(self.cam, self.N, self.fwd_out, self.dF, ws)
            self.graph_launches = self.qr.binding.qr_launch_count() - n0       # kernels one replayed step launches
            self.graphs, self.fe, self.found = g, fe, fe.found
            for _ in range(2):
                self.step_graph()
            t.cuda.synchronize()
            return True
        except Exception as e:           # noqa: BLE001 -- any failure: stay eager, say why
            self.graphs = None
            self.graph_error = repr(e)[:200]
            t.cuda.synchronize()
            return False

    def step_graph(self, timers=None):
        t, g = self.torch, self.graphs
        g[0].replay()
        if timers is not None:
            ev = [t.cuda.Event(enable_timing=True) for _ in range(4)]
            ev[0].record()
        g[1].replay()
        if timers is not None:
            ev[1].record()
        g[2].replay()
        if timers is not None:
            ev[2].record()
        g[3].replay()
        if timers is not None:
            ev[3].record()
            timers.append(ev)

    def timed(self, steps, warmup, barrier, world=1, dist=None, graph=False):
        t = self.torch
        for _ in range(max(warmup, 3)):
            self.step()
        barrier()
        use_graph = bool(graph) and self.capture()
        run = self.step_graph if use_graph else self.step
        for _ in range(3 if use_graph else 0):
            run()
        barrier()
        timers = []
        s0, s1 = t.cuda.Event(enable_timing=True), t.cuda.Event(enable_timing=True)
        n0 = self.qr.binding.qr_launch_count()
        barrier()
        s0.record()
        for _ in range(steps):
            run(timers)
        s1.record()
        barrier()
        launches = (self.graph_launches * steps) if use_graph else (self.qr.binding.qr_launch_count() - n0)
        total_ms = s0.elapsed_time(s1)
        found = int(self.found.item()) if self.found is not None else self.fe.M
        if found > self.capacity:
            raise RuntimeError(f"intersection lists overflowed their capacity ({found} > {self.capacity}): invalid run")
        tt = t.tensor([total_ms], dtype=t.float64, device=self.dev)
        if world > 1:
            dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        mean = lambda i, j: statistics.mean(e[i].elapsed_time(e[j]) for e in timers)
        return {"ms_step": float(tt.item()) / steps, "fwd_ms": mean(0, 1), "bwd_ms": mean(1, 2), "clear_ms": mean(2, 3),
                "launches": int(launches), "M_found": found, "cuda_graph": use_graph,
                "cuda_graph_error": getattr(self, "graph_error", None)}

    def time_call(self, fn, n=5, warm=2):
        t = self.torch
        for _ in range(warm):
            fn()
        t.cuda.synchronize()
        a, b = t.cuda.Event(enable_timing=True), t.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(n):
            fn()
        b.record()
        t.cuda.synchronize()
        return a.elapsed_time(b) / n

    def counts(self):
        """Workload counts for the byte model and SURVEY 8(d)'s work counters (statistics only, outside every timed region)."""
        t, K = self.torch, self.K
        fo = self.fwd_out
        npix = self.cam.width * self.cam.height
        n_vis = int((self.fe.proj.tiles_touched != 0).sum().item())
        used = t.arange(K, device=self.dev)[None, None, :] < fo.n_sel[..., None]      # slots >= n_sel are not written
        S = int(t.unique(fo.sel_idx[used]).numel())
        hist = t.bincount(fo.n_sel.reshape(-1).to(t.int64), minlength=K + 1).cpu().tolist()
        out = {"N_visible": n_vis, "n_sel_mean": float(fo.n_sel.float().mean().item()), "n_sel_max": int(fo.n_sel.max().item()),
               "S_distinct_selected": S, "zero_selection_pixels": int(hist[0]), "selection_record_bytes": npix * (8 * K + 4),
               "n_sel_histogram": hist}
        if fo.has_lists:
            st = self.qr.binding.qr_forward_stats(self.cam, K, fo)
            nh = 2 * self.qr.binding.qr_num_tiles(self.cam)
            out.update({"sum_U_half_tiles": st["sum_U_half_tiles"], "U_half_tile_mean": st["sum_U_half_tiles"] / nh,
                        "half_tiles_U_gt_64": st["half_tiles_U_gt_64"],
                        "walk_list_entries_consumed": st["list_entries_consumed"],
                        "walk_entry_pixel_evaluations": st["entry_pixel_evaluations"],
                        "walk_evaluations_per_pixel": st["entry_pixel_evaluations"] / npix})
        return out


def cpu_baseline_record(sc, workload):
    """The oracle, as it stands, on the box's host cores: one full frame of the workload (all threads), the oracle's
    own work counts for the byte model (N-bar = mean walk length), its V-Render and top-K on the same lists, and a
    1-thread figure on configs 1 and 2 (SURVEY 8(d) "Oracle timing beside it")."""
    from oracle import qr_oracle as orc
    from qr_inputs import make_scene
    npix = sc.cam.width * sc.cam.height
    t0 = time.perf_counter()
    q = oracle_frame(orc, sc)
    sec = time.perf_counter() - t0
    cores = orc.num_threads()
    rec = {"value": npix / sec / 1e6, "unit": UNIT, "cores": cores, "kind": "oracle", "seconds": sec,
           "sample": f"1 full frame of {workload} ({npix} px; O1 projection, O2b lists, O4 Algorithm 1 with D={sc.D} "
                     f"features, O5 backward of the selected rows)",
           "N_bar_mean_walk_length": float(q.n_walked.mean()), "n_sel_mean": float(q.n_sel.mean())}
    proj = orc.project(sc.cam, sc.means, sc.scales, sc.quats, sc.opac)
    lists = orc.pixel_lists(sc.cam, proj)
    rec["mean_list_length"] = float(len(lists.gid)) / npix
    t0 = time.perf_counter()
    v = orc.vrender(lists, sc.features, t_min=1e-4)
    rec["vrender_seconds"] = time.perf_counter() - t0
    rec["dense_walk_mean"] = float(v.n_blended.mean())
    if sc.K <= 64:
        t0 = time.perf_counter()
        orc.topk(lists, sc.K, sc.features, t_min=1e-4)
        rec["topk_seconds"] = time.perf_counter() - t0
    one = {}
    orc.set_num_threads(1)
    try:
        for name in ("cfg1", "cfg2"):
            s1 = make_scene(name, seed=0)
            t0 = time.perf_counter()
            oracle_frame(orc, s1)
            one[name] = {"seconds": time.perf_counter() - t0, "mpix_s": s1.cam.width * s1.cam.height / (time.perf_counter() - t0) / 1e6}
    finally:
        orc.set_num_threads(cores)
    rec["one_thread"] = one
    return rec


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
    qr.binding.load()
    pl = qr.pipeline
    dev = torch.device("cuda", local)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    if args.sweep:
        rc = run_sweep(args, qr, dev, barrier) if rank == 0 else 0
        if world > 1:
            dist.destroy_process_group()
        return rc

    sc = scene_for(args)
    fr = Frame(sc, dev, qr)
    cam, K, D, N = fr.cam, fr.K, fr.D, fr.N
    H, W = cam.height, cam.width
    npix = H * W
    sampler = ClockSampler(local)
    for _ in range(max(args.warmup, 3)):
        fr.step()
    barrier()
    if rank == 0:
        sampler.start()
    r = fr.timed(args.steps, args.warmup, barrier, world, dist, graph=not args.no_graph)
    ms_step, fwd_ms, bwd_ms, zero_ms = r["ms_step"], r["fwd_ms"], r["bwd_ms"], r["clear_ms"]
    value = world * npix / (ms_step * 1e-3) / 1e6
    fe = fr.fe

    # comparators on the same frame and front end (not part of the step): dense V-Render (Eq. 1) and top-K
    dense_map = torch.empty((H, W, D), dtype=torch.float32, device=dev)
    dense_T = torch.empty((H, W), dtype=torch.float32, device=dev)
    dense_ms = fr.time_call(lambda: pl.dense_forward(cam, fe, fr.d["features"], 1e-4, dense_map, dense_T))
    dense_tc = _time_dense_tc(qr, pl, fr, cam, fe, dense_map, dense_T)
    del dense_map
    topk_ms = None
    if K <= 64:
        tk = {"out": None}

        def topk_call():
            tk["out"] = pl.topk_forward(cam, fe, fr.d["features"], K, 1e-4, tk["out"])
        topk_ms = fr.time_call(topk_call)
        topk_nsel = float(tk["out"].n_sel.float().mean().item())
        del tk
    strat_ms = None
    if qr.binding.lists_supported(fr.d["features"].dtype, D):           # stratified-K variant (two walks), same blend
        so = {"out": None}

        def strat_call():
            so["out"] = pl.stratified_forward(cam, fe, fr.d["features"], K, 1e-4, 2.0, so["out"])
        strat_ms = fr.time_call(strat_call)
        strat_nsel = float(so["out"].n_sel.float().mean().item())
        del so
    # the path's neighbours, on synthetic stand-ins of this frame's size: de-voxelisation producing the
    # [N, D] feature table from ~N unique voxels (2 voxels per Gaussian on average) and the mask-pooled loss over the map
    nb = None
    if D % 4 == 0 and sc.feat_dtype == "f32":
        g = torch.Generator(device=dev).manual_seed(0)
        U = N
        uni = torch.randn((U, D), device=dev, generator=g)
        cnts = torch.randint(0, 5, (N,), device=dev, generator=g, dtype=torch.int32)
        Mv = int(cnts.sum().item())
        inv = torch.randint(0, U, (Mv,), device=dev, generator=g, dtype=torch.int64)
        st_ = {}

        def devox():
            st_["gs"], st_["am"], st_["ws"] = qr.binding.qr_devoxelize(uni, inv, cnts, "max", st_.get("ws"))
        devox_ms = fr.time_call(devox)
        dgs = torch.randn((N, D), device=dev, generator=g)
        duni = torch.zeros((U, D), device=dev)
        devox_bwd_ms = fr.time_call(lambda: qr.binding.qr_devoxelize_backward(U, inv, "max", st_["am"], dgs, st_["ws"], duni))
        S_m = 32
        ys = torch.arange(H, device=dev)[:, None] // max(H // 4, 1)
        xs = torch.arange(W, device=dev)[None, :] // max(W // 8, 1)
        mid = (ys * 8 + xs).clamp(max=S_m - 1).to(torch.int32).contiguous()
        tg = torch.randn((S_m, D), device=dev, generator=g)
        dm = torch.empty((H, W, D), dtype=torch.float32, device=dev)
        loss_ms = fr.time_call(lambda: qr.binding.qr_mask_loss(cam, fr.fwd_out.out_map, mid, tg, dm))
        # the same loss FUSED with the path (qr_pooled_loss: from the selection lists, no map, no dL/dmap), and the training step
        # built on it: front end, selection-only forward, loss + dL/dF, clear
        fused = None
        if fr.fwd_out.has_lists:
            fused_loss_ms = fr.time_call(lambda: qr.binding.qr_pooled_loss(cam, K, N, fr.fwd_out, fr.d["features"], mid, tg, fr.dF))
            fr.dF.zero_()
            sel = {"out": None}

            def fused_step():
                fe2 = pl.frontend(cam, fr.d["means"], fr.d["scales"], fr.d["quats"], fr.d["opac"], fr.capacity)
                sel["out"] = pl.forward(cam, fe2, fr.d["features"], K, sel["out"] or fr.fwd_out, select_only=True)
                qr.binding.qr_pooled_loss(cam, K, N, sel["out"], fr.d["features"], mid, tg, fr.dF)
                pl.backward_clear(cam, N, sel["out"], fr.dF)
            fused_step_ms = fr.time_call(fused_step, n=10, warm=3)
            select_ms = fr.time_call(lambda: pl.forward(cam, fr.fe, fr.d["features"], K, fr.fwd_out, select_only=True))
            fused = {"qr_pooled_loss_ms": fused_loss_ms, "selection_only_forward_ms": select_ms, "training_step_ms": fused_step_ms,
                     "unfused_equivalent_ms": ms_step + loss_ms,
                     "note": "training step with the mask-pooled loss: qr_preprocess, qr_bin_sort, qr_forward(out_map = NULL), "
                             "qr_pooled_loss (loss + dL/dF), qr_backward_clear -- the map and dL/dmap never exist; unfused = the "
                             "headline step + qr_mask_loss"}
            pl.forward(cam, fr.fe, fr.d["features"], K, fr.fwd_out)        # leave a complete forward behind for the counters below
        # RGB payload (NEXT-4): this view's colours from degree-3 spherical harmonics, N Gaussians
        shc = torch.randn((N, 16, 3), device=dev, generator=g) * 0.5
        col = torch.empty((N, 3), device=dev)
        sh_ms = fr.time_call(lambda: qr.binding.qr_sh_colors(cam, fr.d["means"], shc, 3, col))
        del shc, col
        devox_bytes = Mv * (D * 4 + 8) + N * D * 4 * 2            # voxel rows gathered + indices, table + argmax written
        loss_bytes = 2 * npix * D * 4 + npix * 8
        nb = {"devoxelize_max": {"ms": devox_ms, "voxels": Mv, "unique_voxels": U, "gb_s": devox_bytes / devox_ms / 1e6},
              "devoxelize_backward_max": {"ms": devox_bwd_ms},
              "mask_loss": {"ms": loss_ms, "masks": S_m, "gb_s": loss_bytes / loss_ms / 1e6,
                            "note": "one read of the map + one write of dL/dmap"},
              "sh_colors_degree3": {"ms": sh_ms, "gb_s": N * 216 / sh_ms / 1e6, "note": "12 + 192 + 12 bytes per Gaussian"},
              "fused": fused}
        del uni, inv, dgs, duni, dm, st_
    # zero fill of the whole dL_dfeat table: what a caller without qr_backward_clear pays per step (reported, not in the step)
    fill_ms = fr.time_call(lambda: fr.dF.zero_())
    # The timed region is ~12 ms at 20 steps, shorter than nvidia-smi's 100 ms sampling period: keep the SAME step
    # running (untimed, not counted anywhere) for ~0.4 s so that the clock / throttle samples are taken under this load.
    if rank == 0:
        hold_until = time.perf_counter() + 0.4
        while time.perf_counter() < hold_until:
            for _ in range(20):
                fr.step()
            torch.cuda.synchronize()
    clocks = sampler.stop() if rank == 0 else None
    if clocks is not None:
        clocks["note"] = "sampled every 100 ms over the timed steps, the comparators and ~0.4 s of the same step kept running"

    counts = fr.counts()
    S, n_vis, M_found = counts["S_distinct_selected"], counts["N_visible"], r["M_found"]
    esz = 2 if sc.feat_dtype == "f16" else 4
    fwd_bytes = M_found * 4 + n_vis * 32 + S * D * esz + npix * D * 4 + npix * 4
    rec_bytes = npix * (8 * K + 4)
    bwd_bytes = npix * D * 4 + S * D * 4 + rec_bytes
    peak, peak_src = _peaks()
    traffic = _traffic(args.workload, D, K)

    def roof(nbytes, ms, kernel):
        ach = nbytes / (ms * 1e-3) / 1e9
        tr = traffic.get(kernel)
        return {"kernel": kernel, "bound": "hbm", "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                "peak_source": peak_src, "frac_of_nominal_8TBs": ach / NOMINAL_HBM_GBS, "algorithmic_bytes": nbytes,
                "ms_per_launch": ms, "traffic": tr, "traffic_source": traffic.get("source") if tr else None,
                "traffic_over_algorithmic": (tr / nbytes) if tr else None}

    dom = "qr_forward" if fwd_ms >= bwd_ms else "qr_backward"
    dom_bytes, dom_ms = (fwd_bytes, fwd_ms) if dom == "qr_forward" else (bwd_bytes, bwd_ms)

    # ---- e2e: host buffers in, host buffers out, copies inside the timed region ----
    e2e = None
    if not args.no_e2e:
        out_host = torch.empty((H, W, D), dtype=torch.float32).pin_memory()
        dF_host = torch.empty((N, D), dtype=torch.float32).pin_memory()
        dd = {k: torch.empty_like(v) for k, v in fr.d.items()}

        def e2e_step():
            for k in dd:
                dd[k].copy_(fr.host[k], non_blocking=True)
            fe2 = pl.frontend(cam, dd["means"], dd["scales"], dd["quats"], dd["opac"], fr.capacity)
            o = pl.forward(cam, fe2, dd["features"], K, fr.fwd_out)
            ws = None if o.has_lists else fr.bws
            pl.backward(cam, N, o, dd["dL_dmap"], fr.dF, ws)
            out_host.copy_(o.out_map, non_blocking=True)
            dF_host.copy_(fr.dF, non_blocking=True)
            pl.backward_clear(cam, N, o, fr.dF, ws)

        e2e_step()
        barrier()
        ne = max(2, min(args.steps, 4))
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(ne):
            e2e_step()
        b.record()
        barrier()
        t = torch.tensor([a.elapsed_time(b)], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e_ms = float(t.item()) / ne
        h2d = sum(v.numel() * v.element_size() for v in fr.host.values())
        d2h = out_host.numel() * 4 + dF_host.numel() * 4
        note = ("inputs (Gaussians, features, dL_dmap) from pinned host memory; out_map and the whole dL_dfeat table "
                "read back: PCIe-bound by construction")
        serial_ms = e_ms
        # The same step as a three-stream pipeline (what a caller who streams frames would write): the upload of step i + 1 and the
        # read-back of step i - 1 run under step i (PCIe is full duplex), every buffer doubled, events between the streams.  Every
        # step still uploads all of its inputs and reads back all of its results inside the timed region.
        if fr.fwd_out.has_lists:
            s_in, s_c, s_out = torch.cuda.Stream(), torch.cuda.Stream(), torch.cuda.Stream()
            ddb = [dd, {k: torch.empty_like(v) for k, v in fr.d.items()}]
            outs = [fr.fwd_out, None]
            with torch.cuda.stream(s_c):
                outs[1] = pl.forward(cam, fr.fe, dd["features"], K, None)
            dFs = [fr.dF, torch.zeros_like(fr.dF)]
            oh = [out_host, torch.empty((H, W, D), dtype=torch.float32).pin_memory()]
            fh = [dF_host, torch.empty((N, D), dtype=torch.float32).pin_memory()]
            torch.cuda.synchronize()
            ev_in = [torch.cuda.Event() for _ in range(2)]
            ev_c = [torch.cuda.Event() for _ in range(2)]
            ev_out = [torch.cuda.Event() for _ in range(2)]

            def pipe_step(i):
                bb = i & 1
                with torch.cuda.stream(s_in):
                    if i >= 2:
                        s_in.wait_event(ev_c[bb])              # the step that last read these inputs has run
                    for k in ddb[bb]:
                        ddb[bb][k].copy_(fr.host[k], non_blocking=True)
                    ev_in[bb].record(s_in)
                with torch.cuda.stream(s_c):
                    s_c.wait_event(ev_in[bb])
                    if i >= 2:
                        s_c.wait_event(ev_out[bb])             # its results have been read back and its rows cleared
                    x = ddb[bb]
                    fe2 = pl.frontend(cam, x["means"], x["scales"], x["quats"], x["opac"], fr.capacity)
                    outs[bb] = pl.forward(cam, fe2, x["features"], K, outs[bb])
                    pl.backward(cam, N, outs[bb], x["dL_dmap"], dFs[bb], None)
                    ev_c[bb].record(s_c)
                with torch.cuda.stream(s_out):
                    s_out.wait_event(ev_c[bb])
                    oh[bb].copy_(outs[bb].out_map, non_blocking=True)
                    fh[bb].copy_(dFs[bb], non_blocking=True)
                    pl.backward_clear(cam, N, outs[bb], dFs[bb], None)
                    ev_out[bb].record(s_out)

            def pipe_run(n):
                cur = torch.cuda.current_stream()
                a2, b2 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a2.record(cur)
                for st_ in (s_in, s_c, s_out):
                    st_.wait_event(a2)
                for i in range(n):
                    pipe_step(i)
                for st_ in (s_in, s_c, s_out):
                    e_ = torch.cuda.Event()
                    e_.record(st_)
                    cur.wait_event(e_)
                b2.record(cur)
                torch.cuda.synchronize()
                return a2.elapsed_time(b2)

            pipe_run(2)
            barrier()
            np_ = max(4, 2 * ne)
            t = torch.tensor([pipe_run(np_)], dtype=torch.float64, device=dev)
            barrier()
            if world > 1:
                dist.all_reduce(t, op=dist.ReduceOp.MAX)
            e_ms = float(t.item()) / np_
            ne = np_
            # the pipelined run must have produced the same map as the device-resident step
            # (to fp32 tolerance: the union columns are numbered by a race, so the summation order differs from run to run)
            ref_map = fr.fwd_out.out_map.cpu()
            same = bool(torch.allclose(oh[0], ref_map, rtol=1e-4, atol=1e-5)) and bool(torch.allclose(oh[1], ref_map, rtol=1e-4, atol=1e-5)) \
                and bool(torch.allclose(fh[0], fh[1], rtol=1e-3, atol=1e-3)) and float(fh[0].abs().max()) > 0.0
            note = ("three-stream pipeline, double buffers: inputs (Gaussians, features, dL_dmap) from pinned host memory, out_map and the "
                    "whole dL_dfeat table read back, every step; upload of step i + 1 and read-back of step i - 1 overlap step i "
                    "(PCIe-bound by construction); the same step issued on one stream takes serial_ms")
            del ddb, outs, dFs, oh, fh
        else:
            same = None
        e2e = {"value": world * npix / (e_ms * 1e-3) / 1e6, "unit": UNIT, "ms_per_step": e_ms, "steps": ne,
               "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "serial_ms": serial_ms, "results_match_device_step": same, "note": note}
        del out_host, dF_host, dd

    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu:
        cpu_baseline = cpu_baseline_record(sc, args.workload)

    if rank == 0:
        cfg = workload_config(sc, args.workload)
        cfg["cuda_graph"] = ("the step is replayed as four CUDA graphs (front end | qr_forward | qr_backward | qr_backward_clear), captured "
                             "from the same library calls; events between the replays time each call" if r["cuda_graph"] else
                             "eager launches" + (f" (graph capture failed: {r['cuda_graph_error']})" if r["cuda_graph_error"] else ""))
        cfg["step"] = ("qr_preprocess, qr_bin_sort (list capacity from an untimed first step: qr_bin_count and its host read "
                       "are NOT in the step), qr_forward, qr_backward, qr_backward_clear (re-zeroes the touched rows; the "
                       "zero fill of the whole dL_dfeat table is NOT in the step, see zero_fill_ms)")
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f32", "data": "synthetic", "config": cfg,
                "clocks": clocks, "e2e": e2e, "gpu_launches": r["launches"],
                "gpu_launches_note": "counted by the library at every kernel launch it issues (qr_launch_count) over the timed steps",
                "roofline": roof(dom_bytes, dom_ms, dom),
                "roofline_fwd": roof(fwd_bytes, fwd_ms, "qr_forward"),
                "roofline_bwd": roof(bwd_bytes, bwd_ms, "qr_backward"),
                "cpu_baseline": cpu_baseline,
                "kernels_ms": {"qr_forward": fwd_ms, "qr_backward": bwd_ms, "qr_backward_clear": zero_ms,
                               "frontend_and_rest": ms_step - fwd_ms - bwd_ms - zero_ms, "zero_fill_ms": fill_ms},
                "mpix_s": {"fwd_kernel": npix / fwd_ms / 1e3, "fwd_bwd_kernels": npix / (fwd_ms + bwd_ms) / 1e3,
                           "dense_fwd_kernel": npix / dense_ms / 1e3,
                           "topk_fwd_kernel": (npix / topk_ms / 1e3) if topk_ms else None},
                "dense": {"ms": dense_ms, "speedup_qr_forward_over_dense": dense_ms / fwd_ms, "t_min": 1e-4,
                          "note": "render_kernel<1>: FFMA formulation without the tensor-core blend (DESIGN.md 5.5); the ratio "
                                  "compares a tuned kernel with an untuned one: see dense_tc for the like-for-like figure"},
                "dense_tc": (dict(dense_tc, speedup_qr_forward_over_dense_tc=dense_tc["ms"] / fwd_ms,
                                  note="qr_dense_forward_tc: walk2_kernel in dense mode + the same tcgen05 blend as Q-Render "
                                       "(PAPER.md:353 reports 1.5x for Q-Render over V-Render at 512-D)") if dense_tc else None),
                "topk": ({"ms": topk_ms, "K": K, "n_sel_mean": topk_nsel, "qr_forward_over_topk": topk_ms / fwd_ms,
                          "note": "same tcgen05 blend as Q-Render; selection by a per-pixel heap (O(N log K), PAPER.md:187)"}
                         if topk_ms else None),
                "stratified": ({"ms": strat_ms, "K": K, "n_sel_mean": strat_nsel, "over_qr_forward": strat_ms / fwd_ms,
                                "note": "qr_forward_stratified: statistics pass + walk with per-pixel boundaries + the same blend "
                                        "(PAPER.md:775 reports about half the FPS of Q-Render for its two-pass variants)"}
                               if strat_ms else None),
                "neighbours": nb,
                "workload_counts": dict(counts, M=M_found, M_capacity=fr.capacity)}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def _parity_counts(orc, lists, K, fwd_out):
    """Selection parity of a frame against the oracle on EVERY pixel (indices bit-exact off the exemption set of
    DESIGN.md reading R15); returns counts, never raises: the sweep records them next to the timings."""
    q = orc.qrender(lists, K, None)
    sel = fwd_out.sel_idx.cpu().numpy().reshape(-1, K)
    n = fwd_out.n_sel.cpu().numpy().reshape(-1)
    used = np.arange(K)[None, :] < q.n_sel[:, None]
    same = (n == q.n_sel) & ((sel == q.sel_idx) | ~used).all(axis=1)
    ex_m = q.margin <= 1e-6
    ex_b = lists.bl_first <= q.n_walked.astype(np.int64)
    ex = ex_m | ex_b
    return {"pixels": int(same.size), "exempt_margin": int(ex_m.sum()), "exempt_borderline": int((ex_b & ~ex_m).sum()),
            "mismatch_exempt": int(((~same) & ex).sum()), "mismatch_nonexempt": int(((~same) & ~ex).sum())}


def run_sweep(args, qr, dev, barrier):
    """BASELINE.json configs[3] (cfg4: K in {4, 8, 16, 32} x 8 camera poses, fp16 features) or configs[4] (cfg5: D in
    {3, 16, 64, 128, 256, 512}, Q-Render vs dense): every point timed like the headline step, with its clocks, work
    counts and (unless --no-parity) its selection parity against the oracle on every pixel.  Writes --out (JSON)."""
    import torch
    from qr_inputs import make_scene
    from qr_inputs.scenes import pose_on_circle
    pl = qr.pipeline
    orc = None
    if not args.no_parity:
        from oracle import qr_oracle as orc
    points = []
    steps = max(3, min(args.steps, 10))
    sampler = ClockSampler(dev.index or 0)

    def measure(fr, tag, lists):
        sampler.lines = []
        sampler.start()
        r = fr.timed(steps, 3, barrier)
        cam, K, D = fr.cam, fr.K, fr.D
        npix = cam.width * cam.height
        fe = fr.fe
        rec = dict(tag, ms_step=r["ms_step"], qr_forward_ms=r["fwd_ms"], qr_backward_ms=r["bwd_ms"], clear_ms=r["clear_ms"],
                   frontend_ms=r["ms_step"] - r["fwd_ms"] - r["bwd_ms"] - r["clear_ms"], gpu_launches=r["launches"], steps=steps,
                   mpix_s_step=npix / r["ms_step"] / 1e3, M=r["M_found"])
        if args.sweep == "cfg5":
            dm = torch.empty((cam.height, cam.width, D), dtype=torch.float32, device=dev)
            dT = torch.empty((cam.height, cam.width), dtype=torch.float32, device=dev)
            rec["dense_ms"] = fr.time_call(lambda: pl.dense_forward(cam, fe, fr.d["features"], 1e-4, dm, dT), n=3, warm=1)
            rec["dense_over_qr_forward"] = rec["dense_ms"] / r["fwd_ms"]
            dtc = _time_dense_tc(qr, pl, fr, cam, fe, dm, dT, n=3, warm=1)
            if dtc:
                rec["dense_tc_ms"] = dtc["ms"]
                rec["dense_tc_over_qr_forward"] = dtc["ms"] / r["fwd_ms"]
                rec["dense_tc_flagged_half_tiles"] = dtc["flagged_half_tiles"]
            del dm
        if K <= 64:
            tk = {"out": None}

            def topk_call():
                tk["out"] = pl.topk_forward(cam, fe, fr.d["features"], K, 1e-4, tk["out"])
            rec["topk_ms"] = fr.time_call(topk_call, n=3, warm=1)
            del tk
        hold = time.perf_counter() + 0.25           # keep the step running so that nvidia-smi samples it under load
        while time.perf_counter() < hold:
            for _ in range(10):
                fr.step()
            torch.cuda.synchronize()
        rec["clocks"] = sampler.stop()
        c = fr.counts()
        c.pop("n_sel_histogram", None)
        rec["counts"] = c
        # the headline line's byte model at this point: fraction of the measured HBM peak each call reaches
        esz = 2 if fr.d["features"].dtype == torch.float16 else 4
        fb = r["M_found"] * 4 + c["N_visible"] * 32 + c["S_distinct_selected"] * D * esz + npix * D * 4 + npix * 4
        bb = npix * D * 4 + c["S_distinct_selected"] * D * 4 + npix * (8 * K + 4)
        peak, _src = _peaks()
        rec["roofline"] = {"peak_gb_s": peak, "fwd_bytes": fb, "fwd_frac": fb / (r["fwd_ms"] * 1e-3) / 1e9 / peak,
                           "bwd_bytes": bb, "bwd_frac": bb / (r["bwd_ms"] * 1e-3) / 1e9 / peak}
        if lists is not None:
            rec["parity"] = _parity_counts(orc, lists, K, fr.fwd_out)
        print(json.dumps(rec), file=sys.stderr, flush=True)
        points.append(rec)

    if args.sweep == "cfg5":
        for D in (3, 16, 64, 128, 256, 512):
            sc = make_scene("cfg5", seed=0, D=D)
            fr = Frame(sc, dev, qr)
            lists = None
            if orc is not None:
                proj = orc.project(sc.cam, sc.means, sc.scales, sc.quats, sc.opac)
                lists = orc.pixel_lists(sc.cam, proj)
            measure(fr, {"workload": "cfg5", "D": D, "K": sc.K, "dtype": sc.feat_dtype}, lists)
            del fr, sc
            torch.cuda.empty_cache()
    elif args.sweep == "cfg4":
        sc = make_scene("cfg4", seed=0, pose=0)
        fr = Frame(sc, dev, qr)
        for pose in range(8):
            cam = sc.cam.copy()
            cam.world_to_cam = pose_on_circle(pose, 8)
            lists = None
            if orc is not None:
                proj = orc.project(cam, sc.means, sc.scales, sc.quats, sc.opac)
                lists = orc.pixel_lists(cam, proj)
            for K in (4, 8, 16, 32):
                fr.reset(cam=cam, K=K)
                measure(fr, {"workload": "cfg4", "pose": pose, "K": K, "D": sc.D, "dtype": sc.feat_dtype}, lists)
            # the four K of this pose in ONE walk (qr_forward_multik) against the four qr_forward calls measured above
            if qr.binding.lists_supported(fr.d["features"].dtype, sc.D):
                Ks = (4, 8, 16, 32)
                fe_p = fr.fe
                mk = {"outs": None}

                def multik_call():
                    mk["outs"] = pl.forward_multik(cam, fe_p, fr.d["features"], Ks, mk["outs"])
                mk_ms = fr.time_call(multik_call, n=5, warm=2)
                sel_ms = None
                singles = [p for p in points if p.get("pose") == pose and "views" not in p and p.get("workload") == "cfg4" and "K" in p]
                rec = {"workload": "cfg4", "pose": pose, "multik": list(Ks), "qr_forward_multik_ms": mk_ms,
                       "sum_of_single_k_forwards_ms": sum(p["qr_forward_ms"] for p in singles if p["K"] in Ks)}
                print(json.dumps(rec), file=sys.stderr, flush=True)
                points.append(rec)
                del mk
        # the same poses as ONE batch (include/qr.h "Multi-camera batching": B views stacked as one tall tile grid, one set of
        # launches, one backward into one dL_dfeat), against the sum of the single-view steps above
        ev = lambda: torch.cuda.Event(enable_timing=True)
        N, D = sc.N, sc.D
        for nb in (4, 8):
            cams = []
            for pose in range(nb):
                cam = sc.cam.copy()
                cam.world_to_cam = pose_on_circle(pose, 8)
                cams.append(cam)
            H, W = sc.cam.height, sc.cam.width
            G = torch.randn((nb * H, W, D), dtype=torch.float32, device=dev)      # dL_dmap of the tall image, drawn on the device
            for K in (4, 8, 16, 32):
                st = {"cap": None, "out": None}
                tall = qr.binding.qr_batch_camera(cams)
                bws = qr.qr_backward_workspace(tall, K, D, dev)

                def bstep(tm=None):
                    e = [ev() for _ in range(4)] if tm is not None else None
                    if e: e[0].record()
                    t_, fe = pl.frontend_batch(cams, fr.d["means"], fr.d["scales"], fr.d["quats"], fr.d["opac"], st["cap"])
                    if st["cap"] is None:
                        st["cap"] = int(fe.M * 1.1) + 1024
                    if e: e[1].record()
                    st["out"] = pl.forward_batch(t_, nb, N, fe, fr.d["features"], K, st["out"])
                    if e: e[2].record()
                    ws = None if st["out"].has_lists else bws
                    pl.backward(t_, N, st["out"], G, fr.dF, ws)
                    pl.backward_clear(t_, N, st["out"], fr.dF, ws)
                    if e:
                        e[3].record(); tm.append(e)
                    return fe
                for _ in range(3):
                    fe = bstep()
                torch.cuda.synchronize()
                tm = []
                n0 = qr.binding.qr_launch_count()
                a, b = ev(), ev()
                a.record()
                for _ in range(steps):
                    fe = bstep(tm)
                b.record()
                torch.cuda.synchronize()
                found = int(fe.found.item())
                assert found <= st["cap"], "batched intersection lists overflowed"
                mean = lambda i, j: statistics.mean(e[i].elapsed_time(e[j]) for e in tm)
                single = sum(p["ms_step"] for p in points if p.get("K") == K and p.get("pose", 99) < nb and "views" not in p)
                rec = {"workload": "cfg4", "views": nb, "K": K, "D": D, "dtype": sc.feat_dtype, "ms_step": a.elapsed_time(b) / steps,
                       "frontend_ms": mean(0, 1), "qr_forward_ms": mean(1, 2), "qr_backward_and_clear_ms": mean(2, 3),
                       "gpu_launches": qr.binding.qr_launch_count() - n0, "steps": steps, "M": found,
                       "sum_of_single_view_steps_ms": single, "mpix_s_step": nb * H * W / (a.elapsed_time(b) / steps) / 1e3}
                print(json.dumps(rec), file=sys.stderr, flush=True)
                points.append(rec)
                del st, bws
            del G
            torch.cuda.empty_cache()
    else:
        raise SystemExit(f"unknown sweep {args.sweep}")
    out = {"sweep": args.sweep, "command": "python bench.py --sweep " + args.sweep + (" --no-parity" if args.no_parity else ""),
           "peak_hbm_gbs": _peaks()[0], "points": points}
    path = args.out or os.path.join(ROOT, "gpurun_out", f"sweep_{args.sweep}.json")
    os.makedirs(os.path.dirname(path), exist_ok=True)
    with open(path, "w") as f:
        json.dump(out, f, indent=1)
    bad = sum(p.get("parity", {}).get("mismatch_nonexempt", 0) for p in points)
    print(json.dumps({"sweep": args.sweep, "points": len(points), "written": path, "mismatch_nonexempt_total": bad}))
    return 0 if bad == 0 else 1


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
    ap.add_argument("--no-graph", action="store_true", help="launch the step's kernels eagerly instead of replaying CUDA graphs")
    ap.add_argument("--sweep", default=None, choices=["cfg4", "cfg5"],
                    help="run every point of BASELINE.json's config 4 (4 K x 8 poses) or config 5 (6 D) and write a JSON file")
    ap.add_argument("--out", default=None, help="where --sweep writes (default gpurun_out/sweep_<cfg>.json)")
    ap.add_argument("--no-parity", action="store_true", help="--sweep: skip the oracle's selection parity of every point")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_cuda(args)


if __name__ == "__main__":
    sys.exit(main())

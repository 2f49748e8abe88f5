#!/usr/bin/env python
"""bench.py -- forward+backward throughput of the B200 surfel renderer on BASELINE.json's configs.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C4] [--impl ours|reference]

A "step" is one pass of the whole hot path over one batch of synthetic input:
  C2 / C5 (tracking-shaped): one frame = `iters` iterations of render -> Eq. 15-19 loss -> pose-only backward
  C1 / C3 / C4 (mapping-shaped): every view rendered and back-propagated (Eq. 24-26 loss, full backward + pose), the
      surfel gradients summed over windows of N_a + N_i = 5 views (Tab. I) by sgs_backward_accumulate
Without --config ALL FIVE configs of BASELINE.json run one after the other; the line's headline (`value`, `roofline`,
`e2e`, `cpu_baseline`, `config.workload`) is C4, the largest single-GPU configuration, and `per_config` carries the same
figures for C1..C5.  `value` is megapixels/s (W*H*renders / device time), inputs resident in HBM; `e2e` is the same
metric through the HOST-buffer C-ABI calls with the copies inside the timed region.  The roofline object is for the
dominant stage, timed in a second pass of the same K steps with CUDA events around every stage (sgs_set_profiling), so
the headline value is not perturbed by the extra event records; its `traffic` is read from profiles/r02_traffic.json,
which `bench.py --ingest-ncu` writes from an `ncu --set full` capture of that kernel.
Rank 0 prints ONE JSON line.  --impl reference times the CPU oracle (oracle/) on the host cores."""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "fwd+bwd megapixels/s"
UNIT = "MP/s"
# Algorithmic flops per (pixel, entry) pair, counted from the oracle's formulas with FMA = 2
# (DESIGN.md §7): tested pair 26; composited pair +26 forward, +102 full backward, +94 pose-only backward.
F_TEST, F_COMP_FWD, F_COMP_BWD_FULL, F_COMP_BWD_POSE = 26, 26, 102, 94
# dram__bytes_read.sum + dram__bytes_write.sum per launch of each config's kernels: profiles/r02_traffic.json, written by
# `bench.py --ingest-ncu` from `ncu --set full` captures (ncu flushes L2 before every replay: cold-cache figures)
TRAFFIC_JSON = os.path.join(ROOT, "profiles", "r02_traffic.json")
WINDOW = 5            # views per mapping window: N_a + N_i (Tab. I)
KERNEL_OF_STAGE = {"forward": "k_forward<", "backward": "k_backward<", "track": "k_track<", "preprocess": "k_pre_project<",
                   "sort": "k_tile_order"}


def load_traffic(config, stage):
    try:
        return json.load(open(TRAFFIC_JSON)).get(config, {}).get(stage, {}).get("dram_bytes_per_launch")
    except (OSError, ValueError):
        return None


def ingest_ncu(csv_path, config):
    """`ncu -i X.ncu-rep --page raw --csv` of a capture of one bench step -> profiles/r02_traffic.json[config][stage] =
    mean dram__bytes_read.sum + dram__bytes_write.sum per launch of that stage's kernel (all captured launches)."""
    import csv
    rows = list(csv.reader(open(csv_path)))
    hdr = next(i for i, r in enumerate(rows) if "Kernel Name" in r)
    names, units = rows[hdr], rows[hdr + 1]
    kn, rd, wr = names.index("Kernel Name"), names.index("dram__bytes_read.sum"), names.index("dram__bytes_write.sum")
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
    out = json.load(open(TRAFFIC_JSON)) if os.path.exists(TRAFFIC_JSON) else {}
    cfg = out.setdefault(config, {})
    for stage, kern in KERNEL_OF_STAGE.items():
        vals = [float(r[rd].replace(",", "")) * scale[units[rd]] + float(r[wr].replace(",", "")) * scale[units[wr]]
                for r in rows[hdr + 2:] if len(r) > wr and kern in r[kn]]
        if vals:
            cfg[stage] = dict(kernel=kern.rstrip("<"), launches=len(vals), dram_bytes_per_launch=sum(vals) / len(vals), source=os.path.basename(csv_path))
    json.dump(out, open(TRAFFIC_JSON, "w"), indent=1, sort_keys=True)
    return cfg


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm_gbs=float(d["hbm_gbs"]), sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)), source="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")


def fp32_peak_tflops(peaks):
    # measured on this device by sgs_measure_fp32_peak (register-resident FMA loop) when available; else
    # 148 SMs x 128 FP32 lanes x 2 flop (FMA) x max SM clock (guide's unit counts and clocks)
    if peaks.get("fp32_tflops_measured"):
        return peaks["fp32_tflops_measured"]
    return 148 * 128 * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12


class ClockSampler(threading.Thread):
    """Samples nvidia-smi clocks and throttle reasons every 200 ms while the timed region runs."""
    Q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.rows, self._stop_evt, self.proc = index, [], threading.Event(), None

    def run(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            for line in self.proc.stdout:
                self.rows.append([x.strip() for x in line.split(",")])
                if self._stop_evt.is_set():
                    break
        except Exception:
            pass

    def stop(self):
        self._stop_evt.set()
        if self.proc:
            self.proc.terminate()
        sm = [float(r[0]) for r in self.rows if r and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(len(r) > 2 + i and r[2 + i].lower().startswith("active") for r in self.rows)]
        return dict(sm_mhz=float(np.median(sm)) if sm else None, sm_max_mhz=max(mx) if mx else None,
                    reasons=reasons, samples=len(sm))


def tau0(seed):
    import scenegen
    g = scenegen.SplitMix(seed)
    d = np.stack([g.normal(3), g.normal(3)])
    return np.concatenate([0.02 * d[0] / np.linalg.norm(d[0]), np.deg2rad(1.0) * d[1] / np.linalg.norm(d[1])])


def oracle_counters(sc, cams, info):
    """Q_t, Q_tb, Q_c, E, N_v ... per view from the oracle (they define the algorithmic work)."""
    import oracle
    cfg = oracle.make_cfg()
    out = []
    for cam in cams:
        camv = oracle.make_cam(cam)
        t0 = time.time()
        r = oracle.render(sc, camv, cfg)
        c = dict(r["counters"])
        c["E"] = oracle.preprocess(sc, camv, cfg)["E"]
        c["fwd_s"] = time.time() - t0
        out.append((c, r))
    return out


def aggregate_replicas(ms_local, pixels, renders_per_rank, world, dist=None, device="cpu"):
    """Weak scaling over independent replicas ("replicas only", no data-path collective): every rank
    times the same K steps on the device; the job's time is the MAX over ranks and its throughput the work of
    ALL ranks divided by that time.  Returns (ms_max, megapixels_per_second)."""
    import torch
    t = torch.tensor([float(ms_local)], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms_max = float(t.item())
    return ms_max, pixels * renders_per_rank * world / (ms_max * 1e-3) / 1e6


# --------------------------------------------------------------------------------------- our arm
class Workload:
    """Device-resident inputs + the step function for one config."""

    def __init__(self, name, iters_override=None, contrib=False, prefetch=True, reuse=True, normalised_depth=False, graph=False,
                 tight=False, radix=False, two_streams=False):
        self.contrib = contrib
        self.dense_fetch = False
        self.prefetch_at = "start"
        self.graph, self.cg, self.eager_steps = graph, None, 0
        nd = self.normalised_depth = normalised_depth
        import torch
        import scenegen
        import paper_2506_00970_b200 as sgs
        self.torch, self.sgs, self.name = torch, sgs, name
        self.sc, self.cams, self.info = scenegen.make_config(name)
        self.tracking = self.info["mode"] == "pose"
        self.iters = iters_override or self.info["iters"]
        sc = self.sc
        d = lambda a, dt=torch.float32: None if a is None else torch.from_numpy(np.ascontiguousarray(a)).to("cuda", dt)
        self.t = dict(mean=d(sc.mean), scale=d(sc.scale), quat=d(sc.quat), opacity=d(sc.opacity), rgb=d(sc.rgb),
                      active=d(sc.active, torch.uint8))
        self.sf = sgs.Renderer.surfels(*(self.t[k] for k in ("mean", "scale", "quat", "opacity", "rgb", "active")))
        self.ren = sgs.Renderer(async_mode=not graph, graph=graph, track_reuse=self.tracking and reuse and not radix,
                                normalised_depth=nd, tight_binning=tight, radix_binning=radix)
        # mapping window: a second context + a side stream, so that sgs_prepare (binning) of view v+1 runs under the
        # compositing kernels of view v (include/sgs.h); tracking iterations depend on one another and use one context
        two = prefetch and not self.tracking and len(self.cams) > 1 and not graph and not radix   # (capture mode: one context, one stream)
        if two:  # + SGS_FLAG_LAZY_GRADS: a view's per-surfel kernel runs under the next view's forward; joined at the step's end
            self.ren.close()
            self.ren = sgs.Renderer(async_mode=True, lazy_grads=True, normalised_depth=nd, tight_binning=tight)
        self.rens = [self.ren] + ([sgs.Renderer(async_mode=True, lazy_grads=True, normalised_depth=nd, tight_binning=tight)] if two else [])
        self.side = torch.cuda.Stream(priority=-1) if len(self.rens) > 1 else None
        # --two-streams: each of the two contexts works through its views on a stream of its own (binning in line, own image
        # and upstream buffers), so one view's loss and backward run beside the other's binning and forward
        self.two_streams = two_streams and len(self.rens) > 1
        if self.two_streams:
            for r in self.rens:
                r.close()
            self.ren = sgs.Renderer(async_mode=True, normalised_depth=nd, tight_binning=tight)
            self.rens = [self.ren, sgs.Renderer(async_mode=True, normalised_depth=nd, tight_binning=tight)]
            self.streams = [torch.cuda.Stream(), torch.cuda.Stream()]
        cam0 = self.cams[0]
        self.H, self.W = cam0.height, cam0.width
        z = lambda c: torch.zeros((c, self.H, self.W), device="cuda")
        self.im = dict(rgb=z(3), depth=z(1), normal=z(3), alpha=z(1))
        self.up = dict(rgb=z(3), depth=z(1), normal=z(3), alpha=z(1))
        self.ccams = [sgs.make_camera(c.width, c.height, c.fx, c.fy, c.cx, c.cy, c.T_cw) for c in self.cams]
        self.p6 = torch.zeros(6, device="cuda")
        self.contrib_buf = torch.zeros(sc.n, device="cuda") if contrib else None
        self.loss = torch.zeros(1, device="cuda")
        self.n_active = int(sc.n if sc.active is None else sc.active.sum())
        # target frame(s): the renderer's own image at the perturbed pose Exp(tau0) T
        self.targets = []
        for i, c in enumerate(self.cams):
            Tt = scenegen.perturb_pose(c.T_cw, tau0(self.info.get("tau0_seed", 2000 + i)))
            ct = sgs.make_camera(c.width, c.height, c.fx, c.fy, c.cx, c.cy, Tt)
            self._render_retry(ct)
            self.targets.append((self.im["rgb"].clone(), self.im["depth"].clone()))
        if not self.tracking:
            n = sc.n
            mk = lambda: dict(mean=torch.zeros(n, 3, device="cuda"), scale=torch.zeros(n, 2, device="cuda"),
                              quat=torch.zeros(n, 4, device="cuda"), opacity=torch.zeros(n, device="cuda"),
                              rgb=torch.zeros(n, 3, device="cuda"))
            self.grads = mk()
            # one set of gradient buffers (and pose gradient) per context: with lazy gradients two views' are in flight
            self.grads_of = {id(r): (self.grads if k == 0 else mk()) for k, r in enumerate(self.rens)}
            self.p6_of = {id(r): (self.p6 if k == 0 else torch.zeros(6, device="cuda")) for k, r in enumerate(self.rens)}
        self.renders_per_step = self.iters if self.tracking else len(self.cams)
        for r in self.rens[1:]:   # the second context's workspace settles on the same views
            for c in self.ccams:
                self._render_retry(c, r)
        if self.two_streams:
            zz = lambda c: torch.zeros((c, self.H, self.W), device="cuda")
            self.bufs = [dict(im=dict(rgb=zz(3), depth=zz(1), normal=zz(3), alpha=zz(1)),
                              up=dict(rgb=zz(3), depth=zz(1), normal=zz(3), alpha=zz(1)), loss=torch.zeros(1, device="cuda"))
                         for _ in self.rens]
        self.flush_buf = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")

    def _render_retry(self, cam, ren=None):
        ren = ren or self.ren
        for _ in range(4):  # async mode: an overflow is reported by the next call, after growing
            try:
                ren.render(self.sf, cam, **self.im)
                ren.stats()
                ren.render(self.sf, cam, **self.im)
                return
            except self.sgs.SgsError as e:
                if e.status != self.sgs.SGS_WORKSPACE_OVERFLOW:
                    raise
        raise RuntimeError("workspace did not settle")

    def one(self, v, ren=None, bufs=None, hook=None, hook_at=None):
        """render -> loss -> backward for view v (everything enqueued, no host sync)."""
        ren = ren or self.ren
        cam = self.ccams[v]
        trgb, tdep = self.targets[v]
        if bufs is not None:   # --two-streams: this context's own buffers, on the current (its own) stream
            im, up, loss = bufs["im"], bufs["up"], bufs["loss"]
            ren.render(self.sf, cam, **im)
            ren.mapping_loss(cam, im, trgb, tdep, 0.875, 0.5, 0.02, -1.0, up, loss)
            ren.ssim_loss(im["rgb"], trgb, 0.125, up["rgb"], loss)
            ren.backward(d_rgb=up["rgb"], d_depth=up["depth"], d_normal=up["normal"], d_alpha=up["alpha"],
                         grads=self.grads_of[id(ren)], d_pose6=self.p6_of[id(ren)], accumulate=True)
            return
        if self.tracking:  # one tracking iteration: K-pre + K-track (render, Eq. 15-19 loss, pose-only backward); images written
            ren.track_iter(self.sf, cam, trgb, tdep, 0.5, -1.0, self.p6, self.loss, **self.im)
            return
        if self.contrib:  # forward with the per-splat contribution output (Eq. 20-21) switched on
            ren.render_contrib(self.sf, cam, self.contrib_buf, **self.im)
        else:
            ren.render(self.sf, cam, **self.im)
        if hook is not None and hook_at == "forward":
            hook()
        # mapping iteration: Eq. 24-26 with Tab. I's lambda_c, w_d, w_n -> upstream gradients of all planes
        ren.mapping_loss(cam, self.im, trgb, tdep, 0.875, 0.5, 0.02, -1.0, self.up, self.loss)
        ren.ssim_loss(self.im["rgb"], trgb, 0.125, self.up["rgb"], self.loss)   # + (1 - lambda_c) L_SSIM: Eq. 24 complete
        if hook is not None and hook_at == "loss":
            hook()
        u = self.up
        ren.backward(d_rgb=u["rgb"], d_depth=u["depth"], d_normal=u["normal"], d_alpha=u["alpha"],
                     grads=self.grads_of[id(ren)], d_pose6=self.p6_of[id(ren)], accumulate=True)

    def begin_window(self):
        """Start of a mapping window: the consumer of the last window's gradients (the optimiser step) is past, every
        context's accumulator is zeroed."""
        for r in self.rens:
            r.wait_grads()
            r.zero_grads(self.grads_of[id(r)])

    def step(self):
        if self.graph and self.cg is not None:
            self.cg.replay()             # --graph: the whole step (frame / window of views) is one CUDA graph launch
        elif self.tracking or self.graph:
            def frame():
                if not self.tracking:
                    for v in range(len(self.cams)):
                        if v % WINDOW == 0:
                            self.begin_window()
                        self.one(v)
                    return
                self.ren.track_new_frame()   # a step is the tracking of one frame: the survivor list is built once per step
                for _ in range(self.iters):
                    self.one(0)
            if self.graph and self.eager_steps >= 2:   # workspace at size after two eager frames: record the third
                self.cg = self.torch.cuda.CUDAGraph()
                with self.torch.cuda.graph(self.cg):
                    frame()
                self.cg.replay()
            else:
                frame()
                self.eager_steps += 1
        elif len(self.rens) == 1:
            for v in range(len(self.cams)):
                if v % WINDOW == 0:
                    self.begin_window()
                self.one(v)
        elif self.two_streams:
            torch = self.torch
            main = torch.cuda.current_stream()
            nv = len(self.cams)
            for w0 in range(0, nv, WINDOW):   # a window: both streams start behind the main stream (optimiser step of the last window) ...
                for k, st in enumerate(self.streams):
                    st.wait_stream(main)
                    with torch.cuda.stream(st):
                        self.rens[k].zero_grads(self.grads_of[id(self.rens[k])])
                        for v in range(w0 + k, min(w0 + WINDOW, nv), 2):
                            self.one(v, self.rens[k], self.bufs[k])
                for st in self.streams:       # ... and the main stream (the consumer of the window's gradients) waits for both
                    main.wait_stream(st)
        else:
            main = self.torch.cuda.current_stream()
            self.side.wait_stream(main)   # the step's first launch stays behind the timed region's start event
            nv = len(self.cams)
            self.rens[0].prepare(self.sf, self.ccams[0], stream=self.side)
            for v in range(nv):
                if v % WINDOW == 0:
                    self.begin_window()   # (each context sums the views it renders; the optimiser adds the two accumulators)
                at = self.prefetch_at
                def nxt(v=v, at=at):
                    if v + 1 < nv:
                        if at != "start":
                            self.side.wait_stream(main)   # the binning of view v+1 starts behind what view v has enqueued so far
                        self.rens[(v + 1) % 2].prepare(self.sf, self.ccams[v + 1], stream=self.side)
                if at == "start":
                    nxt()
                self.one(v, self.rens[v % 2], hook=nxt, hook_at=at)   # its render finds the binning prepared and orders itself behind it
            main.wait_stream(self.side)
            for r in self.rens:
                r.wait_grads()   # the step ends when every view's gradients are complete

    def flush_l2(self):
        self.flush_buf.zero_()

    # ---- end-to-end: HOST buffers through the C-ABI host calls
    def setup_e2e(self):
        torch = self.torch
        pin = lambda a, dt=torch.float32: None if a is None else torch.from_numpy(np.ascontiguousarray(a)).to(dt).pin_memory()
        sc = self.sc
        self.h = dict(mean=pin(sc.mean), scale=pin(sc.scale), quat=pin(sc.quat), opacity=pin(sc.opacity), rgb=pin(sc.rgb),
                      active=pin(sc.active, torch.uint8))
        self.h_targets = [(a.cpu().pin_memory(), b.cpu().pin_memory()) for a, b in self.targets]
        if not self.tracking:
            self.h_grads = [{k: torch.zeros(v.shape).pin_memory() for k, v in self.grads.items()} for _ in range(2)]
            self.h_ids = [torch.zeros(self.sc.n, dtype=torch.int32).pin_memory() for _ in range(2)]
            nw = (len(self.cams) + WINDOW - 1) // WINDOW
            self.h_counts = [torch.zeros(1, dtype=torch.int64).pin_memory() for _ in range(nw)]
            self.h_p6 = [torch.zeros(6).pin_memory() for _ in self.cams]
            self.h_loss = [torch.zeros(1).pin_memory() for _ in self.cams]

    def step_e2e(self):
        """Tracking: upload map + target frame, then `iters` x sgs_track_iter_host (loss + 6-vector read back
        every iteration).  Mapping: upload map; per view sgs_map_view_host (keyframe from the host; render, Eq. 24-26,
        full backward summed into the window on the device; loss + 6-vector back); per window of 5 views
        sgs_fetch_grads_sparse_host (the rows of the surfels the window touched, ids + 13 floats each, written to the host
        by the device; --dense-fetch: sgs_fetch_grads_host, all N x 13); sgs_sync_host at the end of the step."""
        r, h = self.ren, self.h
        r.upload_surfels(h["mean"], h["scale"], h["quat"], h["opacity"], h["rgb"], h["active"])
        if self.tracking:
            r.upload_target(self.ccams[0], *self.h_targets[0])
            for _ in range(self.iters):
                loss, p6 = r.track_iter_host(self.ccams[0], 0.5, -1.0)
            return loss
        nv = len(self.cams)
        for v in range(nv):
            r.map_view_host(self.ccams[v], *self.h_targets[v], 0.875, 0.5, 0.02, 0.125, -1.0, self.h_loss[v], self.h_p6[v])
            if (v + 1) % WINDOW == 0 or v + 1 == nv:
                w = v // WINDOW
                if self.dense_fetch:
                    r.fetch_grads_host(self.h_grads[w % 2])
                else:
                    r.fetch_grads_sparse_host(self.h_ids[w % 2], self.h_grads[w % 2], self.h_counts[w])
        r.sync_host()
        return float(self.h_loss[0][0])

    def e2e_bytes(self):
        n, px = self.sc.n, self.H * self.W
        h2d = n * 52 + (n if self.sc.active is not None else 0)
        if self.tracking:
            return h2d + px * 16 + self.iters * 48, self.iters * 28
        k = len(self.cams)
        windows = (k + WINDOW - 1) // WINDOW
        if self.dense_fetch:
            return h2d + k * (px * 16 + 48), windows * n * 52 + k * 28
        rows = sum(int(c.item()) for c in self.h_counts)    # counted from the last step's windows
        return h2d + k * (px * 16 + 48), rows * 56 + windows * 8 + k * 28


def cpu_baseline(sc, cams, name, samples=3):
    """The oracle as it stands, on the host cores: fp64 forward + analytic backward (to surfels and pose) of one view,
    `samples` views of the config (0, 1, 2, ... cyclically), the MEDIAN reported."""
    import oracle
    cfg = oracle.make_cfg()
    secs = []
    for k in range(samples):
        cam = cams[k % len(cams)]
        camv = oracle.make_cam(cam)
        up = np.ones((8, cam.height, cam.width)) / (cam.height * cam.width)
        t0 = time.time()
        oracle.render(sc, camv, cfg, counters=False)
        oracle.backward(sc, camv, cfg, up)
        secs.append(time.time() - t0)
    dt = float(np.median(secs))
    cam = cams[0]
    n_act = int(sc.n if sc.active is None else sc.active.sum())
    return dict(value=cam.width * cam.height / dt / 1e6, unit=UNIT, cores=oracle.num_threads(), kind="oracle",
                surfels_per_s=n_act / dt,
                sample=f"median of {samples} samples, each 1 view of {name} (fp64 forward + analytic backward to surfels and pose): "
                       + ", ".join(f"{t:.2f}" for t in secs) + " s", seconds=dt)


def run_reference(args):
    """--impl reference: the CPU oracle timed on the host cores on OUR arm's config (default C4).  A step renders and
    back-propagates `m` views of the config, walking through its views cyclically from step to step; m is the largest
    number of views (at most the config's own views per step) that keeps the whole --steps/--warmup run within a few
    minutes, decided from one timed view -- a bounded sample of the workload, stated in config.workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    import scenegen
    name = args.config or "C4"
    sc, cams, info = scenegen.make_config(name)
    cfg = oracle.make_cfg()
    tracking = info["mode"] == "pose"
    per_step = info["iters"] if tracking else len(cams)
    ups = {}

    def view(k):
        cam = cams[k % len(cams)]
        if (cam.height, cam.width) not in ups:
            ups[(cam.height, cam.width)] = np.ones((8, cam.height, cam.width)) / (cam.height * cam.width)
        camv = oracle.make_cam(cam)
        oracle.render(sc, camv, cfg, counters=False)
        oracle.backward(sc, camv, cfg, ups[(cam.height, cam.width)])

    t0 = time.time()
    view(0)
    t_view = time.time() - t0
    budget = 150.0 / max(1, args.steps + args.warmup)
    m = int(max(1, min(per_step, budget // max(t_view, 1e-6))))
    k = 0
    for _ in range(args.warmup):
        for _ in range(m):
            view(k); k += 1
    t0 = time.time()
    for _ in range(args.steps):
        for _ in range(m):
            view(k); k += 1
    dt = time.time() - t0
    cam = cams[0]
    mp = cam.width * cam.height * m * args.steps / dt / 1e6
    n_act = int(sc.n if sc.active is None else sc.active.sum())
    sample = (f"every step: {m} of the config's {per_step} renders per step (fp64 forward + analytic backward to surfels and "
              f"pose each), views taken cyclically")
    line = dict(metric=METRIC, value=mp, unit=UNIT, n_gpus=args.gpus, steps=args.steps, warmup=args.warmup,
                ms_per_step=1e3 * dt / args.steps, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64",
                data="synthetic", impl="reference", surfels_per_s=n_act * m * args.steps / dt,
                config=dict(workload=f"{name}: {sample} (bounded sample of the same workload)",
                            surfels=sc.n, active=n_act, width=cam.width, height=cam.height, renders_per_step=m,
                            renders_per_step_of_the_workload=per_step),
                cpu_baseline=dict(value=mp, unit=UNIT, cores=oracle.num_threads(), kind="oracle", sample=sample),
                e2e=dict(value=mp, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0))
    print(json.dumps(line))


def run_config(name, args, torch, dist, world, rank, local, peaks):
    """One config: timed pass (value), profiled pass (stages / roofline), end-to-end pass, oracle baseline + counters."""
    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    wl = Workload(name, args.iters, args.contrib, not args.no_prefetch, not args.no_reuse, args.normalised_depth, args.graph,
                  args.tight, args.radix, args.two_streams)
    wl.prefetch_at = args.prefetch_at
    K, W = args.steps, max(args.warmup, 3)
    per_step = []
    for _ in range(W):
        l0 = sum(r.stats()["kernel_launches"] for r in wl.rens)
        wl.step()
        per_step.append(sum(r.stats()["kernel_launches"] for r in wl.rens) - l0)
    torch.cuda.synchronize()
    launches0 = sum(r.stats()["kernel_launches"] for r in wl.rens)

    def timed_pass():
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
        barrier()
        for a, b in evs:
            wl.flush_l2()
            a.record()
            wl.step()
            b.record()
        barrier()
        return sum(a.elapsed_time(b) for a, b in evs)  # ms, device time of the K steps

    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.3)
    ms = timed_pass()
    launches = sum(r.stats()["kernel_launches"] for r in wl.rens) - launches0   # of the timed region only
    if args.graph and wl.cg is not None:   # replays do not pass the library's launch counter: the recorded step's count x K
        launches = per_step[2] * K
    # the timed region can be shorter than nvidia-smi's start-up: keep the same load running (untimed) until the sampler
    # has seen it a few times, so that `clocks` is always a reading under this workload
    t_wait = time.time()
    while len(sampler.rows) < 3 and time.time() - t_wait < 4.0:
        wl.step()
        torch.cuda.synchronize()
    clocks = sampler.stop()
    px = wl.H * wl.W
    ms_max, value = aggregate_replicas(ms, px, wl.renders_per_step * K, world, dist, "cuda")
    renders = wl.renders_per_step * K * world

    # second pass with per-stage CUDA events (roofline), not part of `value`
    wl.graph = False   # (--graph: the stage events live in the eager calls)
    for r in wl.rens:
        r.set_profiling(True)
        r.get_profile(reset=True)
    timed_pass()
    prof = {}
    for r in wl.rens:
        for st, (ms_s, calls) in r.get_profile(reset=True).items():
            a, b = prof.get(st, (0.0, 0))
            prof[st] = (a + ms_s, b + calls)
        r.set_profiling(False)

    # end to end through the HOST-buffer C-ABI calls
    e2e = None
    if not args.no_e2e:
        wl.dense_fetch = args.dense_fetch
        wl.setup_e2e()
        wl.step_e2e()
        barrier()
        t0 = time.time()
        for _ in range(K):
            wl.step_e2e()
        barrier()
        dt = time.time() - t0
        te = torch.tensor([dt], device="cuda", dtype=torch.float64)
        if world > 1:
            dist.all_reduce(te, op=dist.ReduceOp.MAX)
        h2d, d2h = wl.e2e_bytes()
        e2e = dict(value=px * renders / float(te.item()) / 1e6, unit=UNIT, h2d_bytes_per_step=h2d, d2h_bytes_per_step=d2h,
                   timing="wall clock around K steps incl. pinned-host copies and the read-back of every result")
    out = dict(value=value, unit=UNIT, ms_per_step=ms_max / K, surfels_per_s=wl.n_active * renders / (ms_max * 1e-3),
               e2e=e2e, gpu_launches=int(launches), clocks=clocks,
               stage_us={k: round(1e3 * v[0] / v[1], 2) for k, v in prof.items() if v[1]},
               config=dict(workload=f"{name} ({'tracking' if wl.tracking else 'mapping'}-shaped): "
                           f"{wl.renders_per_step} x (render + {'Eq.15-19' if wl.tracking else 'Eq.24-26'} loss + "
                           f"{'pose-only' if wl.tracking else 'full+pose'} backward) per step",
                           surfels=wl.sc.n, active=wl.n_active, width=wl.W, height=wl.H, renders_per_step=wl.renders_per_step,
                           l2="flushed between steps by a 256 MiB write; iterations inside a step reuse the map as tracking does",
                           replicas=world,
                           survivor_list=("built once per step (frame) with a 3 cm / 0.02 rad pose margin, SGS_FLAG_TRACK_REUSE"
                                          if (wl.tracking and not args.no_reuse) else "every render"),
                           binning=("two contexts on two streams, views alternating; binning in line on each" if getattr(wl, "two_streams", False) else
                                    f"sgs_prepare of view v+1 on a second context and a side stream, enqueued behind view v's {args.prefetch_at}"
                                    if len(wl.rens) > 1 else "in line (sgs_render / sgs_track_iter)")))
    if not wl.tracking and e2e is not None:
        e2e["gradients"] = ("all n x 13 floats per window (sgs_fetch_grads_host)" if args.dense_fetch else
                            "rows of the surfels each window touched: ids + 13 floats (sgs_fetch_grads_sparse_host)")
    if not wl.tracking:
        out["config"]["gradients"] = f"summed over windows of {WINDOW} views (sgs_backward_accumulate), zeroed per window"
    if args.graph:
        out["config"]["launch"] = "one CUDA graph per step (SGS_FLAG_GRAPH); not the default workload"
    if args.radix:
        out["config"]["binning"] = "SGS_FLAG_RADIX_BINNING: global onesweep radix sort of (tile << 32 | depth) keys, in line; not the default workload"
    if args.tight:
        out["config"]["binning_variant"] = "SGS_FLAG_TIGHT_BINNING (readings R26, R27); not the default workload"
    if args.normalised_depth:
        out["config"]["depth"] = "normalised D/O (SGS_FLAG_NORMALISED_DEPTH); not the default workload"
    sc, cams, tracking, n_active = wl.sc, wl.cams, wl.tracking, wl.n_active
    for r in wl.rens:
        r.close()
    del wl
    torch.cuda.empty_cache()
    if rank != 0 or args.no_cpu_baseline:
        out.update(roofline=None, stages={}, cpu_baseline=None)
        return out
    import oracle
    out["cpu_baseline"] = cpu_baseline(sc, cams, name)
    # algorithmic work per render from the oracle's counters (view 0 stands for every view)
    camv, cfg = oracle.make_cam(cams[0]), oracle.make_cfg(tight=args.tight)
    cnt = oracle.render(sc, camv, cfg)["counters"]
    E = oracle.preprocess(sc, camv, cfg)["E"]
    fcb = F_COMP_BWD_POSE if tracking else F_COMP_BWD_FULL
    work = dict(preprocess=("hbm", (sc.n if sc.active is not None else 0) + n_active * 56 + cnt["n_vis"] * 76 + E * 12),
                sort=("hbm", E * 24 + E * 8),
                forward=("alu", F_TEST * cnt["Q_t"] + F_COMP_FWD * cnt["Q_c"]),
                loss=("hbm", px * (12 + 8) * 4 + (0 if tracking else px * 3 * 4 * 12)),
                backward=("alu", F_TEST * cnt["Q_tb"] + fcb * cnt["Q_c"]),
                # sgs_track_iter's single kernel: forward + pose-only backward of the same view
                track=("alu", F_TEST * (cnt["Q_t"] + cnt["Q_tb"]) + (F_COMP_FWD + F_COMP_BWD_POSE) * cnt["Q_c"]))
    stages = {}
    tot_ms = sum(v[0] for v in prof.values()) or 1.0
    for st, (ms_s, calls) in prof.items():
        if calls == 0:
            continue
        kind, units = work[st]
        per = ms_s / calls * 1e-3
        if kind == "hbm":
            ach, peak, unit = units / per / 1e9, peaks["hbm_gbs"], "GB/s"
        else:
            ach, peak, unit = units / per / 1e12, fp32_peak_tflops(peaks), "TFLOP/s"
        stages[st] = dict(bound=kind, achieved=ach, peak=peak, unit=unit, frac=ach / peak, ms_per_launch=per * 1e3,
                          share=ms_s / tot_ms, algorithmic_units=units)
    dom = max(stages, key=lambda k: stages[k]["share"])
    roof = dict(stages[dom])
    nominal = 148 * 128 * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12
    roof.update(kernel=dom, traffic=load_traffic(name, dom),
                peak_source=peaks["source"] + (" HBM copy" if roof["bound"] == "hbm" else
                            ("; alu peak = measured FMA loop (sgs_measure_fp32_peak), nominal 148 SM x 128 lanes x 2 x max SM clock = %.1f" % nominal
                             if peaks.get("fp32_tflops_measured") else "; alu peak = 148 SM x 128 lanes x 2 x max SM clock")),
                counters=dict(cnt, E=E))
    out.update(roofline=roof, stages=stages)
    return out


def probe_staging(args):
    """--probe-staging: no benchmark.  Renders view 0 of --config (default C2) and times the staging of its tile lists alone,
    by LDG gathers (mode 0, what the kernels do) and by one cp.async.bulk per record (mode 1): sgs_probe_staging."""
    import torch
    import scenegen
    import paper_2506_00970_b200 as sgs
    name = args.config or "C2"
    sc, cams, info = scenegen.make_config(name)
    cam = cams[0]
    d = lambda a, dt=torch.float32: None if a is None else torch.from_numpy(np.ascontiguousarray(a)).to("cuda", dt)
    keep = [d(sc.mean), d(sc.scale), d(sc.quat), d(sc.opacity), d(sc.rgb), d(sc.active, torch.uint8)]   # (the struct borrows them)
    sf = sgs.Renderer.surfels(*keep)
    ren = sgs.Renderer()
    z = lambda c: torch.zeros((c, cam.height, cam.width), device="cuda")
    ren.render(sf, sgs.make_camera(cam.width, cam.height, cam.fx, cam.fy, cam.cx, cam.cy, cam.T_cw), rgb=z(3), depth=z(1), normal=z(3), alpha=z(1))
    st = ren.stats()
    out = dict(config=name, n_entries=st["n_entries"], tiles=((cam.width + 15) // 16) * ((cam.height + 15) // 16))
    for rep in range(2):
        for mode, key in ((0, "ldg_gather_us"), (1, "bulk_copy_us")):
            out[key] = ren.probe_staging(mode, reps=50)
    print(json.dumps(out))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default=None, choices=["C1", "C2", "C3", "C4", "C5"],
                    help="one config only (default: all five, headline C4)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--iters", type=int, default=None, help="override iterations per tracking step")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--dense-fetch", action="store_true", help="e2e leg of the mapping configs: sgs_fetch_grads_host (all N x 13 floats per window) instead of the sparse hand-over")
    ap.add_argument("--no-reuse", action="store_true", help="tracking configs: run the pre-cull over the whole map every iteration")
    ap.add_argument("--no-prefetch", action="store_true", help="mapping configs: one context, binning of each view in line")
    ap.add_argument("--prefetch-at", default="start", choices=["start", "forward", "loss"],
                    help="mapping configs: where sgs_prepare of view v+1 is enqueued on the side stream: at the start of view v (default: it runs under k_forward), behind its forward, or behind its loss kernels (under k_backward: +1.4 %% MP/s, but the dominant kernel's measured duration then includes the binning it shares the SMs with)")
    ap.add_argument("--graph", action="store_true", help="SGS_FLAG_GRAPH: each step (a tracking frame, or a mapping window on one context) replayed as one CUDA graph")
    ap.add_argument("--normalised-depth", action="store_true", help="SGS_FLAG_NORMALISED_DEPTH: depth image D/O (tracking takes the unfused sequence)")
    ap.add_argument("--tight", action="store_true", help="SGS_FLAG_TIGHT_BINNING: opacity-aware cutoff + tile-exact culling (shorter tile lists, same images)")
    ap.add_argument("--two-streams", action="store_true", help="mapping configs: two contexts on two streams, views alternating (no prefetch pipeline)")
    ap.add_argument("--radix", action="store_true", help="SGS_FLAG_RADIX_BINNING: the global LSD radix sort of the 64-bit keys instead of the per-tile buckets (A/B; one context, in line)")
    ap.add_argument("--contrib", action="store_true", help="mapping configs: render with sgs_render_contrib (C_k output on)")
    ap.add_argument("--probe-staging", action="store_true", help="no benchmark: time the staging of --config's tile lists by LDG gathers and by cp.async.bulk (sgs_probe_staging)")
    ap.add_argument("--ingest-ncu", default=None, metavar="RAW_CSV",
                    help="no benchmark: read `ncu -i X.ncu-rep --page raw --csv` of a capture of --config and update profiles/r02_traffic.json")
    args = ap.parse_args()
    if args.ingest_ncu:
        print(json.dumps(ingest_ncu(args.ingest_ncu, args.config or "C4"), indent=1))
        return
    if args.impl == "reference":
        return run_reference(args)
    if args.probe_staging:
        return probe_staging(args)

    import torch
    import torch.distributed as dist
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    import paper_2506_00970_b200 as sgs
    peaks = load_peaks()
    try:
        peaks["fp32_tflops_measured"] = sgs.measure_fp32_peak()
    except Exception:
        peaks["fp32_tflops_measured"] = None
    names = [args.config] if args.config else ["C1", "C2", "C3", "C4", "C5"]
    head = args.config or "C4"
    res = {n: run_config(n, args, torch, dist, world, rank, local, peaks) for n in names}
    if rank == 0:
        h = res[head]
        line = dict(metric=METRIC, value=h["value"], unit=UNIT, n_gpus=world, steps=args.steps, warmup=max(args.warmup, 3),
                    ms_per_step=h["ms_per_step"], higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f32",
                    data="synthetic", surfels_per_s=h["surfels_per_s"], config=h["config"], clocks=h["clocks"], e2e=h["e2e"],
                    gpu_launches=sum(r["gpu_launches"] for r in res.values()), roofline=h["roofline"], stages=h["stages"],
                    cpu_baseline=h["cpu_baseline"], stage_us=h["stage_us"])
        if len(names) > 1:
            line["config"] = dict(h["config"], headline="C4, the largest single-GPU configuration of BASELINE.json; per_config has all five")
            line["per_config"] = {n: {k: r[k] for k in ("value", "surfels_per_s", "ms_per_step", "roofline", "e2e", "cpu_baseline",
                                                         "gpu_launches", "stage_us", "clocks")} | {"workload": r["config"]["workload"]}
                                  for n, r in res.items()}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

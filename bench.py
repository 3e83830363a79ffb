#!/usr/bin/env python
"""bench.py — affine-2DGS fwd+bwd on the benchmark-shaped site (BASELINE.json configs[3]: 1M surfels, 2048^2 views).

    python bench.py --gpus N --steps K --warmup W            # the CUDA path (hand-written sm_100a kernels)
    python bench.py --impl reference --steps K --warmup W    # the CPU oracle, as it stands, on the host cores
    python bench.py --record-traffic <ncu raw csv>           # refresh profiles/r3_traffic.json from an ncu capture

A "step" is one full training-view iteration of the hot path: sun pass (preprocess,
binning, depth-only compositing) -> view pass (preprocess, binning, compositing of colour/alpha/depth/normal/
median/distortion with the fused colour-correction + shadow epilogue) -> backward of both passes (epilogue
backward, reverse compositing, per-surfel chain, dF / CC reductions) -> cascade chain of the sun camera into dF.
Views cycle through the config's 20 views.  With --gpus N > 1 (one process per GPU: under torchrun, or spawned by this
script when WORLD_SIZE is unset) the views are sharded over the ranks and every step ends with ONE NCCL all-reduce
(sum) of the packed 13 N surfel gradients, overlapped with the next step.  Prints ONE JSON line
(rank 0).
"""
from __future__ import annotations

import argparse
import hashlib
import json
import os
import re
import socket
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "affine-2DGS fwd+bwd throughput at 1M surfels, 2048^2 view (C3 full iteration incl. shadow pass)"
UNIT = "Mpixel/s"
# algorithmic work per pair: FP32-pipe lane-instructions of the paper's per-pixel loop
INST_EVAL = 17.0          # per evaluated (pixel, list entry) pair: Eq. 9 + Eq. 12 + ex2 + alpha tests
INST_CONTRIB_FWD = 25.0   # extra per contributing pair, forward (view pass; the depth-only sun pass: 6)
INST_CONTRIB_BWD = 90.0   # extra per contributing pair, backward (view pass; sun pass: 50)
INST_CONTRIB_FWD_SUN, INST_CONTRIB_BWD_SUN = 6.0, 50.0
SM_LANES = 128            # FP32 lanes per SM; derived peak = SMs x 128 x clock, measured one beside it
TRAFFIC_JSON = os.path.join(ROOT, "profiles", "r3_traffic.json")
DESIGN_BYTES = {"preprocess": 137.0, "chain_bwd": 309.0}   # bytes per surfel this implementation moves
# stage -> kernel name in the traffic JSON (view pass, sun pass)
TRAFFIC_KEYS = {"preprocess": ("void preprocess_kernel<0>", None), "blend_fwd": ("blend_fwd", "blend_fwd_sun"),
                "blend_bwd": ("blend_bwd", "blend_bwd_sun"), "chain_bwd": ("void chain_backward_kernel<0>", None)}
CSRC = os.path.join(ROOT, "paper_2606_28581_b200", "csrc")


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json config index (3 = the metric's config)")
    ap.add_argument("--surfels", type=int, default=None, help="override N (debug)")
    ap.add_argument("--size", type=int, default=None, help="override view size (debug)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip the Adam / loss / init stage timings")
    ap.add_argument("--no-graphs", action="store_true", help="launch every kernel of a step from the host instead of replaying one CUDA graph per view")
    ap.add_argument("--no-allreduce", action="store_true", help="N > 1: leave the per-rank gradients un-reduced")
    ap.add_argument("--dp-path", action="store_true",
                    help="run the data-parallel code path (NCCL group, gradient all-reduce on the communication stream, host-launched "
                         "steps) even with one rank: a functional check of that path on a single GPU, not a scaling number")
    ap.add_argument("--record-traffic", default=None, nargs="+", metavar="NCU_RAW_CSV",
                    help="write profiles/r3_traffic.json from `ncu -i <rep> --page raw --csv` output file(s) and exit")
    return ap.parse_args()


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm_gbs=float(d["hbm_gbs"]), sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)), source="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")


def csrc_hash() -> str:
    """Content hash of the CUDA sources (the GPU box has no .git): ties the ncu-derived fields to the kernels they
    were captured on."""
    h = hashlib.sha256()
    for name in sorted(os.listdir(CSRC)):
        if name.endswith((".cu", ".cuh")):
            h.update(name.encode())
            h.update(open(os.path.join(CSRC, name), "rb").read())
    return h.hexdigest()[:16]


def record_traffic(raw_csvs):
    """profiles/r3_traffic.json <- per-kernel DRAM bytes, executed warp-instructions and issue utilisation of `ncu --set
    full` captures (first launch of each kernel name in the files), with the hash of the sources."""
    import csv
    out = {}
    for raw_csv in raw_csvs:
        rows = list(csv.reader(open(raw_csv)))
        _record_rows(rows, out)
    json.dump(dict(csrc_sha256=csrc_hash(), source=[os.path.basename(f) for f in raw_csvs], kernels=out), open(TRAFFIC_JSON, "w"), indent=1)
    print("wrote", TRAFFIC_JSON, list(out))


def _record_rows(rows, out):
    hdr = rows[0]
    col = {h: i for i, h in enumerate(hdr)}
    for r in rows[2:]:
        name = r[col["Kernel Name"]]
        key = ("blend_bwd" if "blend_backward" in name else "blend_fwd" if "blend_forward" in name else name.split("(")[0].split("::")[-1])
        m = re.search(r"kernel<\s*(?:\(bool\))?\s*(\d|true|false)", name)     # first template argument: DEPTH_ONLY (the sun pass)
        key += "_sun" if (m and m.group(1) in ("1", "true") and key.startswith("blend_")) else ""
        if key in out:
            continue
        f = lambda k: float(r[col[k]]) if k in col and r[col[k]] not in ("", "n/a") else None
        unit = rows[1][col["dram__bytes_read.sum"]].lower() if "dram__bytes_read.sum" in col else "byte"
        mul = dict(byte=1.0, kbyte=1e3, mbyte=1e6, gbyte=1e9).get(unit, 1.0)
        rd, wr = f("dram__bytes_read.sum"), f("dram__bytes_write.sum")
        out[key] = dict(dram_bytes=(rd + wr) * mul if rd is not None and wr is not None else None,
                        warp_inst=f("smsp__inst_executed.sum"),
                        issue_active_pct=f("smsp__issue_active.avg.pct_of_peak_sustained_active"),
                        ncu_us=f("gpu__time_duration.sum"))


def load_traffic():
    """ncu-derived fields of the roofline line; None when the committed capture was taken on other kernel sources."""
    if not os.path.exists(TRAFFIC_JSON):
        return None, "no capture committed"
    d = json.load(open(TRAFFIC_JSON))
    if d.get("csrc_sha256") != csrc_hash():
        return None, f"stale: profiles/r3_traffic.json was captured on sources {d.get('csrc_sha256')}, these are {csrc_hash()}"
    return d["kernels"], "profiles/r3_traffic.json (ncu --set full, same sources)"


def make_scene(args):
    import satsplat_scenes as S
    kw = {}
    if args.surfels:
        kw["n"] = args.surfels
    if args.size:
        kw["size"] = args.size
        kw["sun_size"] = args.size
    return S.make_config(args.config, **kw)


def views_for_rank(rank: int, world: int, n_views: int, steps: int):
    """View index of every step of this rank: ranks start on different views and stride by the world size, so
    that the ranks of one job render disjoint views (independent units; the only exchange is the gradient sum)."""
    return [(rank + s * world) % n_views for s in range(steps)]


def packed_offsets(n: int):
    """Float offsets of the five surfel-gradient groups (means 3N, quats 4N, scales 2N, logits N, rgb 3N) in the ONE
    buffer that is all-reduced; every group starts on a 16-byte boundary.  Returns (offsets[5], total floats)."""
    off, t = [], 0
    for w in (3, 4, 2, 1, 3):
        off.append(t)
        t += (n * w + 3) // 4 * 4
    return off, t


def allreduce_sum(dist, flat):
    """The one collective of the data-parallel path: sum over ranks of the packed surfel gradients."""
    dist.all_reduce(flat, op=dist.ReduceOp.SUM)
    return flat


def spawn_command(args, port: int):
    """Command line that launches this bench as one process per GPU (used when --gpus N > 1 and WORLD_SIZE is unset)."""
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__)]
    return cmd + [a for a in sys.argv[1:]]


def free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


class ClockSampler:
    """SM clock + throttle reasons through NVML every ~2 ms, started BEFORE the warm-up; only the samples whose host
    time falls inside the timed window are reported (so even a 40 ms timed region has samples).  Falls back to
    `nvidia-smi -lms` when NVML cannot be loaded."""
    REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown"}

    def __init__(self, index):
        self.index, self.rows, self.stop_flag, self.thread, self.mode = index, [], False, None, None

    def start(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv, self.h = pynvml, pynvml.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.mode = "nvml"
            self.thread = threading.Thread(target=self._loop_nvml, daemon=True)
        except Exception:
            self.mode = "nvidia-smi"
            self.thread = threading.Thread(target=self._loop_smi, daemon=True)
        self.thread.start()

    def _loop_nvml(self):
        nv = self.nv
        while not self.stop_flag:
            try:
                t = time.perf_counter()
                mhz = nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)
                try:
                    rs = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    rs = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                self.rows.append((t, float(mhz), int(rs)))
            except Exception:
                pass
            time.sleep(0.002)

    def _loop_smi(self):
        q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.sw_power_cap,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.hw_thermal_slowdown")
        try:
            proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={q}", "--format=csv,noheader,nounits", "-lms", "20"],
                                    stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.mode = None
            return
        self.proc = proc
        for line in proc.stdout:
            f = [x.strip() for x in line.split(",")]
            try:
                bits = sum(b for b, v in zip((0x4, 0x8, 0x20, 0x40), f[2:6]) if v.lower().startswith("active"))
                self.max_mhz = float(f[1])
                self.rows.append((time.perf_counter(), float(f[0]), bits))
            except Exception:
                pass
            if self.stop_flag:
                break
        proc.terminate()

    def stop(self, t0, t1):
        time.sleep(0.03)
        self.stop_flag = True
        if getattr(self, "proc", None):
            self.proc.terminate()
        if self.mode is None or not self.rows:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["clock sampling unavailable"], samples=0)
        inside = [r for r in self.rows if t0 <= r[0] <= t1]
        reasons = set()
        for r in inside:
            for bit, nm in self.REASONS.items():
                if r[2] & bit:
                    reasons.add(nm)
        return dict(sm_mhz=float(np.median([r[1] for r in inside])) if inside else None, sm_max_mhz=getattr(self, "max_mhz", None),
                    reasons=sorted(reasons), samples=len(inside), samples_total=len(self.rows), source=self.mode)


# ------------------------------------------------------------------------------------------------------------
# reference arm / cpu_baseline: the oracle as it stands, on the host cores, on a bounded sample
# ------------------------------------------------------------------------------------------------------------
def oracle_iteration_seconds(scene, view_index, threads=None, do_backward=True):
    import satsplat_scenes as S
    from oracle import oracle as orc
    view = scene.views[view_index]
    up = S.upstream_grads(scene.seed, view_index, view.height, view.width)
    nth = threads or orc.num_threads()
    t0 = time.perf_counter()
    orc.view_iteration(scene, view, upstream=up if do_backward else None, threads=nth, do_backward=do_backward)
    return time.perf_counter() - t0, nth


def oracle_flags():
    return "-O3 -march=native -ffp-contract=off -fno-fast-math -fopenmp (BASELINE.md section 3), compiled on this host"


def cpu_baseline_block(scene, view_index, px, nviews):
    """The oracle timed on the host cores, beside the GPU number: all threads fwd and fwd+bwd on one full view of the
    workload, and ONE thread on a bounded sample (a C1-sized scene: 200k surfels, one 512^2 view with its sun pass)."""
    import satsplat_scenes as S
    from oracle import oracle as orc
    orc.use_native_build()
    dt, nth = oracle_iteration_seconds(scene, view_index)
    dt_f, _ = oracle_iteration_seconds(scene, view_index, do_backward=False)
    small = S.make_config(2, n_views=1)
    spx = small.views[0].width * small.views[0].height
    dt1, _ = oracle_iteration_seconds(small, 0, threads=1)
    dt1n, _ = oracle_iteration_seconds(small, 0, threads=nth)
    return dict(value=px / 1e6 / dt, unit=UNIT, cores=nth, kind="oracle", seconds=dt, fwd_seconds=dt_f, fwd_value=px / 1e6 / dt_f,
                sample=f"1 full view iteration (view {view_index} of {nviews}) of the same workload, {nth} threads; forward alone timed too",
                flags=oracle_flags(),
                single_thread=dict(value=spx / 1e6 / dt1, unit=UNIT, seconds=dt1, all_threads_seconds=dt1n, cores=1,
                                   sample="C2-sized scene (200k surfels, one 512^2 view + 1024^2 sun map), full iteration, 1 thread"))


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import oracle as orc
    orc.use_native_build()
    scene = make_scene(args)
    steps, warm = max(1, min(args.steps, 3)), min(args.warmup, 1)   # bounded: each step is ~10 s of CPU work
    for w in range(warm):
        oracle_iteration_seconds(scene, w % len(scene.views))
    ts = []
    for s in range(steps):
        dt, nth = oracle_iteration_seconds(scene, s % len(scene.views))
        ts.append(dt)
    v = scene.views[0]
    ms = 1e3 * float(np.mean(ts))
    val = v.width * v.height / 1e6 / (ms / 1e3)
    sample = f"{steps} full view iteration(s) of the workload (views 0..{steps - 1} of {len(scene.views)}), all {nth} host threads"
    line = dict(impl="reference", metric=METRIC, value=val, unit=UNIT, n_gpus=0, steps=steps, warmup=warm, ms_per_step=ms,
                higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64", data="synthetic",
                config=workload_config(scene, args, 1),
                cpu_baseline=dict(value=val, unit=UNIT, cores=nth, kind="oracle", sample=sample, flags=oracle_flags()),
                e2e=dict(value=val, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0))
    print(json.dumps(line))


def workload_config(scene, args, world):
    v = scene.views[0]
    par = (f"views sharded over {world} rank(s); one NCCL all-reduce (sum) of the packed 13 N surfel gradients per step"
           if (world > 1 or getattr(args, "dp_path", False)) else "1 rank")
    return dict(workload=f"C{args.config} benchmark-shaped site (BASELINE.json configs[{args.config}])", surfels=scene.n,
                view=f"{v.width}x{v.height}", cuda_graphs=("one graph for all views (device-resident cameras)"
                             if (not getattr(args, "no_graphs", False)) and world == 1 and not getattr(args, "dp_path", False) else False),
                sun_map=f"{v.sun_width}x{v.sun_height}" if v.shadows_on else None,
                views=len(scene.views), shadows=bool(v.shadows_on), parallelism=par,
                l2="per-step working set (records, keys, per-pixel state, images: >0.8 GB) exceeds the 126 MB L2; views cycle")


# ------------------------------------------------------------------------------------------------------------
# the CUDA path
# ------------------------------------------------------------------------------------------------------------
class Job:
    """Device-resident state of one rank: surfels, two contexts (view + sun), outputs, gradient buffers."""

    def __init__(self, P, torch, scene, device, n_grad_buffers=1):
        self.P, self.torch, self.scene = P, torch, scene
        dev = lambda a: torch.from_numpy(np.ascontiguousarray(a, np.float32)).to(device)
        self.means, self.quats, self.scales = dev(scene.means), dev(scene.quats), dev(scene.scales)
        self.logits, self.rgb = dev(scene.opacity_logits), dev(scene.rgb)
        n, v = scene.n, scene.views[0]
        self.n, self.W, self.H = n, v.width, v.height
        self.shadows = bool(v.shadows_on)
        max_dup = 8 * n + 4096
        self.ctx = P.Context(n, v.width, v.height, max_dup, device=device.index)
        self.sctx = P.Context(n, v.sun_width, v.sun_height, max_dup, device=device.index) if self.shadows else None
        z = lambda *s: torch.zeros(*s, device=device, dtype=torch.float32)
        self.out = [torch.empty(v.height, v.width, 4, device=device) for _ in range(3)]
        self.sun_depth = z(v.sun_height, v.sun_width) if self.shadows else None
        self.v_sun = z(v.sun_height, v.sun_width) if self.shadows else None
        # the 13 N surfel gradients live in ONE packed buffer (what a data-parallel job all-reduces), followed by the
        # small per-camera vectors: dF(8) cc(12) ambient(3) reproj(8) dF_sun(8), which stay local to the rank
        off, tot = packed_offsets(n)
        self.flat_floats = tot
        self.gbufs = []
        for _ in range(n_grad_buffers):
            flat = z(tot + 40)
            g = dict(flat=flat, surfel=flat[:tot],
                     m=flat[off[0]:off[0] + 3 * n].view(n, 3), q=flat[off[1]:off[1] + 4 * n].view(n, 4),
                     s=flat[off[2]:off[2] + 2 * n].view(n, 2), l=flat[off[3]:off[3] + n], c=flat[off[4]:off[4] + 3 * n].view(n, 3),
                     dF=flat[tot:tot + 8], cc=flat[tot + 8:tot + 20], amb=flat[tot + 20:tot + 23], rep=flat[tot + 24:tot + 32],
                     dFs=flat[tot + 32:tot + 40])
            self.gbufs.append(g)
        self.g = self.gbufs[0]
        self.cams = {}
        self.device = device
        # one set of upstream gradient images ~ N(0,1), shared by all views (synthetic; the loss stage would write them)
        gen = torch.Generator(device=device)
        gen.manual_seed(scene.seed + 1000)
        self.up_shared = [torch.randn(v.height, v.width, 4, device=device, generator=gen) for _ in range(3)]
        self.up_shared[2][..., 2:] = 0
        # (f2) device-resident cameras: per-view constants, the learnable dF [V,8], the current view index, the camera block
        self.table = P.view_params_table(scene.views, device=device)
        self.dF_all = dev(np.stack([vw.dF for vw in scene.views]))
        self.v_dF_all = z(len(scene.views), 8)
        self.idx = torch.zeros(1, dtype=torch.int32, device=device)
        self.block = z(P.CAMERA_BLOCK_FLOATS)
        # the view pass's preprocess + binning do not depend on the sun pass: they run on a second stream beside it
        self.side = torch.cuda.Stream(device=device) if self.shadows else None
        self.overlap = True     # False: everything on one stream (the per-stage timers then see each kernel alone)
        self.split = False      # True while step_device runs: contexts in SATSPLAT_OPT_SPLIT_BACKWARD mode

    def prepare_view(self, vi):
        if vi in self.cams:
            return
        P, torch, v = self.P, self.torch, self.scene.views[vi]
        cam = P.Camera.from_view(v)
        sun_cam, rep = (P.sun_camera(cam, v.sun_azimuth, v.sun_elevation, v.sun_width, v.sun_height, v.sun_viewport)
                        if self.shadows else (None, None))
        self.cams[vi] = (cam, sun_cam, rep)

    def shading(self, vi, with_sun=True):
        v = self.scene.views[vi]
        rep = self.cams[vi][2]
        return self.P.Shading.make(cc=v.cc, ambient=v.ambient, sun_depth=self.sun_depth if (self.shadows and with_sun) else None,
                                   reproj=rep, depth_bias=v.depth_bias, slope=v.slope)

    def forward(self, vi):
        cam, sun_cam, _ = self.cams[vi]
        sh = self.shading(vi)
        if self.shadows and not self.overlap:
            self.sctx.preprocess(sun_cam, self.means, self.quats, self.scales, self.logits, self.rgb)
            self.sctx.shadow_map(self.sun_depth)
            self.ctx.preprocess(cam, self.means, self.quats, self.scales, self.logits, self.rgb)
        elif self.shadows:
            cur = self.torch.cuda.current_stream()
            self.side.wait_stream(cur)
            self.ctx.preprocess(cam, self.means, self.quats, self.scales, self.logits, self.rgb, stream=self.side)
            self.sctx.preprocess(sun_cam, self.means, self.quats, self.scales, self.logits, self.rgb)
            self.sctx.shadow_map(self.sun_depth)
            cur.wait_stream(self.side)
        else:
            self.ctx.preprocess(cam, self.means, self.quats, self.scales, self.logits, self.rgb)
        self.ctx.render_forward(sh, *self.out)
        return sh

    def step(self, vi, buf=0):
        if self.split:          # the host-struct step uses the unsplit backward calls
            self.ctx.set_option(self.P.OPT_SPLIT_BACKWARD, 0)
            self.sctx.set_option(self.P.OPT_SPLIT_BACKWARD, 0)
            self.split = False
        g = self.gbufs[buf]
        g["flat"].zero_()
        sh = self.forward(vi)
        up = self.up_shared
        if self.shadows:
            self.v_sun.zero_()
        self.ctx.render_backward(sh, up[0], up[1], up[2], g["m"], g["q"], g["s"], g["l"], g["c"], g["dF"], g["cc"], g["amb"],
                                 self.v_sun, g["rep"] if self.shadows else None)
        if self.shadows:
            self.sctx.shadow_map_backward(self.v_sun, g["m"], g["q"], g["s"], g["l"], g["dFs"])
            # cascade (Fig. 1): the sun camera is derived from F' = F + dF
            v = self.scene.views[vi]
            self.P.sun_camera_backward(self.cams[vi][0], v.sun_azimuth, v.sun_elevation, v.sun_viewport, g["dFs"], g["rep"], g["dF"])


    def step_device(self, stride=1, buf=0, upstream_fn=None, camera_step_fn=None):
        """The same iteration with every camera read from the device-resident block: the view is
        selected by the device index, nothing of it is baked into kernel arguments, so ONE captured graph of this function
        serves all views and all optimiser steps (dF lives in self.dF_all on the device)."""
        P, g, surf = self.P, self.gbufs[buf], (self.means, self.quats, self.scales, self.logits, self.rgb)
        if self.shadows and not self.split:
            self.ctx.set_option(P.OPT_SPLIT_BACKWARD, 1)
            self.sctx.set_option(P.OPT_SPLIT_BACKWARD, 1)
            self.split = True
        g["flat"].zero_()
        P.camera_chain(self.table, self.dF_all, self.idx, self.block)
        v = self.scene.views[0]
        if self.shadows:
            cur = self.torch.cuda.current_stream()
            self.side.wait_stream(cur)
            self.ctx.preprocess_device(self.W, self.H, self.block, P.CAM_VIEW, *surf, stream=self.side)
            self.sctx.preprocess_device(v.sun_width, v.sun_height, self.block, P.CAM_SUN, *surf)
            self.sctx.shadow_map(self.sun_depth)
            cur.wait_stream(self.side)
            self.v_sun.zero_()
        else:
            self.ctx.preprocess_device(self.W, self.H, self.block, P.CAM_VIEW, *surf)
        self.ctx.render_forward_device(self.block, self.sun_depth, *self.out)
        up = upstream_fn() if upstream_fn else self.up_shared     # upstream_fn: the loss stage on the rendered images (extras)
        if self.shadows:
            # split backward calls: the view pass's per-surfel chain (HBM-bound) runs on the side stream beside the sun pass's
            # blend backward (issue-bound); the sun pass's chain follows both (the two chains share the gradient buffers)
            cur = self.torch.cuda.current_stream()
            self.ctx.render_backward_device(self.block, self.sun_depth, up[0], up[1], up[2], None, None, None, None, None,
                                            v_sun_depth=self.v_sun)
            self.side.wait_stream(cur)
            self.ctx.backward_chain(g["m"], g["q"], g["s"], g["l"], g["c"], g["dF"], g["cc"], g["amb"], g["rep"], stream=self.side)
            self.sctx.shadow_map_backward(self.v_sun, None, None, None, None)
            cur.wait_stream(self.side)
            self.sctx.backward_chain(g["m"], g["q"], g["s"], g["l"], None, g["dFs"])
        else:
            self.ctx.render_backward_device(self.block, None, up[0], up[1], up[2], g["m"], g["q"], g["s"], g["l"], g["c"], g["dF"],
                                            g["cc"], g["amb"], None, None)
        # cascade (Fig. 1): view-pass dF gradient + adjoint of the sun camera / reprojection -> this view's row of v_dF_all
        P.camera_chain_backward(self.table, self.dF_all, self.idx, g["dF"], g["dFs"] if self.shadows else None,
                                g["rep"] if self.shadows else None, None, self.v_dF_all)
        if camera_step_fn:      # the optimiser step of the per-camera groups needs the index of the view just rendered
            camera_step_fn(g)
        P.advance_view_index(self.idx, stride, len(self.scene.views))


def max_over_ranks(torch, dist, world, value, device):
    """MAX all-reduce of a per-rank scalar (device timings are reported as the max over ranks)."""
    if world <= 1:
        return float(value)
    t = torch.tensor([float(value)], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def timed(torch, dist, world, fn, items, per_step=False):
    """Time fn(item) over items with CUDA events on the current stream; barrier + synchronize on both sides;
    returns the max over ranks of the elapsed milliseconds (and, with per_step, this rank's per-item times and the
    host-clock window of the timed region)."""
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(len(items) + 1 if per_step else 2)]
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    ev[0].record()
    for k, it in enumerate(items):
        fn(it)
        if per_step:
            ev[k + 1].record()
    if not per_step:
        ev[1].record()
    torch.cuda.synchronize()
    t1 = time.perf_counter()
    if world > 1:
        dist.barrier()
    total = max_over_ranks(torch, dist, world, ev[0].elapsed_time(ev[-1]), "cuda")
    if per_step:
        return total, [ev[k].elapsed_time(ev[k + 1]) for k in range(len(items))], (t0, t1)
    return total


def stage_profile(job, views, peaks, fp32_peak_tinst):
    """Per-stage device ms (CUDA events recorded by the library on the launching stream around every kernel of a
    stage), averaged over the launches of the bench's step views; pair counts and the algorithmic work of each kernel
    (of the last view), for both passes."""
    torch, P = job.torch, job.P
    job.ctx.set_profiling(True)
    if job.sctx:
        job.sctx.set_profiling(True)
    job.overlap = False
    ms_view, ms_sun = {}, {}
    for vi in views:
        job.step(vi)
        torch.cuda.synchronize()
        for acc, ctx in ((ms_view, job.ctx), (ms_sun, job.sctx)):
            if ctx:
                for k, v in ctx.stage_ms().items():
                    acc[k] = acc.get(k, 0.0) + v / len(views)
    job.ctx.set_profiling(False)
    if job.sctx:
        job.sctx.set_profiling(False)
    # pair counters: one more pass over the last view with the instrumentation planes on (SATSPLAT_OPT_DEBUG_PLANES; they are
    # off in every timed region, stage times above included)
    for c in (job.ctx, job.sctx):
        if c:
            c.set_option(P.OPT_DEBUG_PLANES, 1)
    job.step(views[-1])
    torch.cuda.synchronize()
    for c in (job.ctx, job.sctx):
        if c:
            c.set_option(P.OPT_DEBUG_PLANES, 0)
    job.overlap = True
    nv, nc = job.ctx.debug_planes()
    pairs = dict(view_evaluated=int(nv.sum().item()), view_contributing=int(nc.sum().item()), view_K=job.ctx.sync_status())
    if job.sctx:
        snv, snc = job.sctx.debug_planes()
        pairs.update(sun_evaluated=int(snv.sum().item()), sun_contributing=int(snc.sum().item()), sun_K=job.sctx.sync_status())
        # the sun-pass backward only has work on the texels some view pixel looked up (the others have no upstream gradient
        # and are skipped exactly): its algorithmic work counts the pairs of those texels only
        live = (job.v_sun != 0).to(snv.dtype)
        pairs.update(sun_bwd_evaluated=int((snv * live).sum().item()), sun_bwd_contributing=int((snc * live).sum().item()),
                     sun_live_texel_share=float(live.float().mean().item()))
    n = job.n
    tiles = ((job.W + 15) // 16) * ((job.H + 15) // 16)
    px = job.W * job.H

    def work(pass_):   # algorithmic bytes / lane-instructions (per surfel / key / pair figures of SURVEY.md 8(d))
        K, ev, co = pairs[f"{pass_}_K"], pairs[f"{pass_}_evaluated"], pairs[f"{pass_}_contributing"]
        evb, cob = pairs.get(f"{pass_}_bwd_evaluated", ev), pairs.get(f"{pass_}_bwd_contributing", co)
        cf, cb = (INST_CONTRIB_FWD, INST_CONTRIB_BWD) if pass_ == "view" else (INST_CONTRIB_FWD_SUN, INST_CONTRIB_BWD_SUN)
        return {
            "preprocess": ("hbm", n * 132.0, None),      # 56 B in + 76 B of records / boxes / keys out
            "scan": ("hbm", tiles * 12.0, None),
            "duplicate": ("hbm", n * 16.0 + K * 8.0, None),
            "sort": ("hbm", K * 20.0, None),
            "ranges": ("hbm", 0.0, None),
            "blend_fwd": ("alu", ev * INST_EVAL + co * cf, co * (INST_EVAL + cf)),
            "blend_bwd": ("alu", evb * INST_EVAL + cob * cb, cob * (INST_EVAL + cb)),
            "chain_bwd": ("hbm", n * 172.0, None),       # SURVEY.md 8(d); the design moves 309 (DESIGN_BYTES below)
        }

    stages = {}
    wv, ws = work("view"), (work("sun") if job.sctx else None)
    for k, ms in ms_view.items():
        bound, w, useful = wv[k]
        peak = fp32_peak_tinst if bound == "alu" else peaks["hbm_gbs"]
        scale = 1e12 if bound == "alu" else 1e9
        ach = w / (ms * 1e-3) / scale if ms > 0 else 0.0
        st = dict(ms=ms, sun_ms=ms_sun.get(k, 0.0), bound=bound, achieved=ach, peak=peak, unit="Tinst/s" if bound == "alu" else "GB/s",
                  frac=ach / peak if peak else None, roofline_ms=w / scale / peak * 1e3)
        if useful is not None and ms > 0:
            st["useful_frac"] = useful / (ms * 1e-3) / scale / peak          # contributing pairs only
        if k in DESIGN_BYTES and ms > 0:
            # what THIS design moves per surfel (moment records written by the blend and read + cleared by the chain, the +=
            # read-modify-write of the gradient arrays): printed beside the method's bytes, never as the fraction
            st["design_bytes_per_surfel"] = DESIGN_BYTES[k]
            st["method_bytes_per_surfel"] = w / n
            st["design_frac"] = n * DESIGN_BYTES[k] / (ms * 1e-3) / scale / peak
        if ws is not None and ms_sun.get(k, 0.0) > 0:
            _, w2, u2 = ws[k]
            st["sun_frac"] = w2 / (ms_sun[k] * 1e-3) / scale / peak
            st["sun_roofline_ms"] = w2 / scale / peak * 1e3
            if u2 is not None:
                st["sun_useful_frac"] = u2 / (ms_sun[k] * 1e-3) / scale / peak
        stages[k] = st
    return stages, pairs, px


def run_ours(args):
    import torch
    import torch.distributed as dist
    import paper_2606_28581_b200 as P
    P.lib()   # no CUDA library -> fail loudly (there is no fallback)
    assert torch.cuda.is_available(), "bench.py needs a CUDA device"
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    device = torch.device("cuda", local)
    dp = world > 1 or args.dp_path     # the data-parallel path: NCCL group, one all-reduce per step
    if dp:
        if "MASTER_ADDR" not in os.environ:
            os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(free_port()), RANK="0", WORLD_SIZE="1")
        dist.init_process_group("nccl", device_id=device)
    peaks = load_peaks()
    sampler = ClockSampler(local)
    sampler.start()                      # before the warm-up: the samples of the timed window are picked out afterwards
    # the two issue-rate peaks of the blend kernels' roofline, measured on this device
    mp = P.measure_peaks(local)
    derived_tinst = mp["sm_count"] * SM_LANES * peaks["sm_max_mhz"] * 1e6 / 1e12
    fp32_peak = mp["fp32_lane_inst_per_s"] / 1e12
    scene = make_scene(args)
    allreduce = dp and not args.no_allreduce
    job = Job(P, torch, scene, device, n_grad_buffers=2 if allreduce else 1)
    nviews = len(scene.views)
    warm_views = views_for_rank(rank, world, nviews, args.warmup)
    step_views = views_for_rank(rank + args.warmup * world, world, nviews, args.steps)
    for vi in set(warm_views + step_views):
        job.prepare_view(vi)
    comm = torch.cuda.Stream(device=device) if allreduce else None
    state = dict(k=0, pending=[None, None])

    def dp_step(vi):
        """One data-parallel step: this rank's view, then the all-reduce of its packed gradients on the communication
        stream, overlapped with the next step (which writes the other gradient buffer)."""
        b = state["k"] & 1
        cur = torch.cuda.current_stream()
        if state["pending"][b] is not None:
            cur.wait_event(state["pending"][b])          # the all-reduce that last used this buffer has finished
        job.step(vi, buf=b)
        done = torch.cuda.Event()
        done.record(cur)
        comm.wait_event(done)
        with torch.cuda.stream(comm):
            allreduce_sum(dist, job.gbufs[b]["surfel"])
            fin = torch.cuda.Event()
            fin.record(comm)
        state["pending"][b] = fin
        state["k"] += 1

    def drain():
        for e in state["pending"]:
            if e is not None:
                torch.cuda.current_stream().wait_event(e)

    run_step = dp_step if allreduce else job.step
    for vi in warm_views:
        run_step(vi)
    if allreduce:
        drain()
    torch.cuda.synchronize()
    job.ctx.sync_status()     # raises on capacity overflow
    launches0 = P.kernel_launches()
    launches_per_step = None
    use_graphs = not args.no_graphs and not dp   # data-parallel runs launch from the host (no capture beside the NCCL watchdog)
    if use_graphs:
        # ONE CUDA graph for all views and all steps: the cameras are device-resident (row f2), the graph advances the view
        # index itself; a step is one graph launch
        job.idx.fill_(step_views[0])
        job.step_device()                      # warm-up of the device path outside the capture
        torch.cuda.synchronize()
        l0 = P.kernel_launches()
        graph = torch.cuda.CUDAGraph()
        # captured on a high-priority stream: the critical chain (sun pass -> view forward -> backwards) gets the SMs before
        # the view pass's preprocess + binning, which runs beside the sun pass on the default-priority side stream and is
        # not needed until the sun map is done (2.206 -> 2.189 ms per step)
        cap = torch.cuda.Stream(device=device, priority=-1)
        with torch.cuda.graph(graph, stream=cap):
            job.step_device()
        launches_per_step = P.kernel_launches() - l0
        for _ in range(3):
            graph.replay()
        torch.cuda.synchronize()
        job.idx.fill_(step_views[0])           # views step_views[0], +1, ... (mod the number of views): the same sequence
        job.v_dF_all.zero_()
        run_step = lambda vi: graph.replay()
        launches0 = P.kernel_launches()
    if allreduce:
        def timed_steps(vi):
            dp_step(vi)
        ms_total, per_step, window = timed(torch, dist, world, timed_steps, step_views, per_step=True)
        drain()
        torch.cuda.synchronize()
    else:
        ms_total, per_step, window = timed(torch, dist, world, run_step, step_views, per_step=True)
    launches = P.kernel_launches() - launches0 if launches_per_step is None else launches_per_step * len(step_views)
    clocks = sampler.stop(*window)
    ms_fwd = timed(torch, dist, world, job.forward, step_views)
    px = job.W * job.H
    ms_step = ms_total / args.steps
    value = world * px / 1e6 / (ms_step * 1e-3)

    line = dict(metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=args.steps, warmup=args.warmup, ms_per_step=ms_step,
                ms_median=float(np.median(per_step)), ms_min=float(np.min(per_step)),
                higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f32", data="synthetic",
                config=workload_config(scene, args, world), clocks=clocks, gpu_launches=int(launches),
                fwd_ms_per_step=ms_fwd / args.steps, fwd_mpixel_s=world * px / 1e6 / (ms_fwd / args.steps * 1e-3))
    if allreduce:
        line["allreduce"] = dict(bytes_per_step=job.flat_floats * 4, collective="ncclAllReduce(sum) of the packed surfel gradients",
                                 overlapped_with="the next step's kernels (double-buffered gradient buffer, communication stream)")
    if rank == 0:
        stages, pairs, _ = stage_profile(job, step_views, peaks, fp32_peak)
        dom = max(stages, key=lambda k: stages[k]["ms"])
        d = stages[dom]
        traffic, traffic_src = load_traffic()
        t_dom = (traffic or {}).get(dom)
        line["roofline"] = dict(kernel=dom, bound=d["bound"], achieved=d["achieved"], peak=d["peak"], unit=d["unit"], frac=d["frac"],
                                useful_frac=d.get("useful_frac"),
                                traffic=t_dom["dram_bytes"] if t_dom else None, traffic_source=traffic_src, launches_averaged=len(step_views),
                                executed=dict(warp_inst=t_dom["warp_inst"], issue_active_pct=t_dom["issue_active_pct"]) if t_dom else None,
                                peak_source=("measured: satsplat_measure_peaks (independent FFMA chains on every sub-partition of this device)"
                                             if d["bound"] == "alu" else peaks["source"] + " HBM copy (MEASURED_PEAKS.json)"),
                                peak_derived=derived_tinst if d["bound"] == "alu" else None,
                                peak_derived_how=f"{mp['sm_count']} SMs x {SM_LANES} FP32 lanes x {peaks['sm_max_mhz']:.0f} MHz",
                                mufu_peak_measured_tops=mp["mufu_per_s"] / 1e12, kernel_ms=d["ms"])
        # ncu-derived fields per stage (only while the committed capture matches these sources): DRAM traffic against the
        # method's bytes for the HBM-bound stages; executed lane slots against the credited lane-instructions for the blends,
        # so that a stage whose credited work exceeds everything its kernel executes shows as such
        for k, (kv, ks) in TRAFFIC_KEYS.items():
            for key, pre in ((kv, ""), (ks, "sun_")):
                t_k = (traffic or {}).get(key) if key else None
                if not t_k or k not in stages:
                    continue
                st = stages[k]
                credited_ms = st["roofline_ms"] if pre == "" else st.get("sun_roofline_ms")
                if credited_ms is None:
                    continue
                if st["bound"] == "hbm" and t_k.get("dram_bytes"):
                    st[pre + "traffic_over_algorithmic"] = t_k["dram_bytes"] / (credited_ms * 1e-3 * st["peak"] * 1e9)
                elif st["bound"] == "alu" and t_k.get("warp_inst"):
                    slots = t_k["warp_inst"] * 32
                    st[pre + "executed_lane_slots"] = slots
                    st[pre + "credited_over_executed"] = credited_ms * 1e-3 * st["peak"] * 1e12 / slots
        line["stages"] = stages
        line["pairs"] = pairs
        sun_ms = sum(s["sun_ms"] for s in stages.values())
        view_ms = sum(s["ms"] for s in stages.values())
        # whole-iteration roofline: sum over kernels of their own roofline time, BOTH passes
        roof_view = sum(s["roofline_ms"] for s in stages.values())
        roof_sun = sum(s.get("sun_roofline_ms", 0.0) for s in stages.values())
        scratch = (job.ctx.scratch_bytes + (job.sctx.scratch_bytes if job.sctx else 0)) / 1e9
        line["iteration"] = dict(view_pass_kernel_ms=view_ms, sun_pass_kernel_ms=sun_ms, view_pass_roofline_ms=roof_view,
                                 sun_pass_roofline_ms=roof_sun,
                                 view_pass_frac_of_roofline=roof_view / view_ms if view_ms else None,
                                 sun_pass_frac_of_roofline=roof_sun / sun_ms if sun_ms else None,
                                 frac_of_roofline=(roof_view + roof_sun) / (view_ms + sun_ms) if view_ms + sun_ms else None,
                                 frac_of_roofline_vs_step=(roof_view + roof_sun) / ms_step,
                                 scratch_gb=scratch, peak_mem_gb=torch.cuda.max_memory_allocated() / 1e9 + scratch)
    if rank == 0 and not args.no_extras:
        extras(line, args, job, P, torch, scene, device, peaks, step_views, px)
    # ---- end to end through the C ABI with HOST buffers ----
    if not args.no_e2e:
        vi = step_views[0]
        v = scene.views[vi]
        pin = lambda t: t.detach().cpu().contiguous().pin_memory()
        h_in = [pin(x) for x in (job.means, job.quats, job.scales, job.logits, job.rgb)]
        h_up = [pin(u) for u in job.up_shared]
        # outputs are per slot: a step's host buffers stay untouched until its _end (the inputs are only read: shared)
        h_out2 = [[torch.empty(v.height, v.width, 4).pin_memory() for _ in range(3)] for _ in range(2)]
        h_g2 = [torch.empty(scene.n * 13 + 23).pin_memory() for _ in range(2)]
        h_g = h_g2[0]
        cam = job.cams[vi][0]
        sun = P.Sun.from_view(v) if job.shadows else None
        sh = P.Shading.make(cc=v.cc, ambient=v.ambient, depth_bias=v.depth_bias, slope=v.slope)
        sh.shadows_on = 1 if job.shadows else 0
        P.reserve_host_staging(job.ctx, job.sctx)
        if job.split:            # the host-buffer entry point runs the unsplit backward calls
            job.ctx.set_option(P.OPT_SPLIT_BACKWARD, 0)
            job.sctx.set_option(P.OPT_SPLIT_BACKWARD, 0)
            job.split = False

        hargs2 = [(cam, sun, sh, scene.n, *h_in, *h_up, *h_out2[k], h_g2[k]) for k in range(2)]
        hargs = hargs2[0]

        def e2e_step(_):
            P.iteration_host(job.ctx, job.sctx, *hargs)
        for _ in range(2):
            e2e_step(0)
        n_e2e = max(3, min(args.steps, 10))

        def wall(fn):
            torch.cuda.synchronize()
            if world > 1:
                dist.barrier()
            t0 = time.perf_counter()
            fn()
            torch.cuda.synchronize()
            return max_over_ranks(torch, dist, world, time.perf_counter() - t0, "cuda")

        def serial():
            for i in range(n_e2e):
                e2e_step(i)

        def pipelined():   # the begin / end pair: the upload of step i+1 crosses PCIe while the kernels of step i run
            P.iteration_host_begin(job.ctx, job.sctx, 0, *hargs2[0])
            for i in range(1, n_e2e):
                P.iteration_host_begin(job.ctx, job.sctx, i & 1, *hargs2[i & 1])
                P.iteration_host_end(job.ctx, (i - 1) & 1)
            P.iteration_host_end(job.ctx, (n_e2e - 1) & 1)
        dt_serial = wall(serial)
        pipelined()
        dt = wall(pipelined)
        h2d = scene.n * 52 + 3 * px * 16
        d2h = 3 * px * 16 + (scene.n * 13 + 23) * 4
        raster_only = dict(value=world * px / 1e6 / (dt / n_e2e), unit=UNIT, h2d_bytes_per_step=h2d, d2h_bytes_per_step=d2h,
                           ms_per_step=1e3 * dt / n_e2e, steps=n_e2e, serial_ms_per_step=1e3 * dt_serial / n_e2e,
                           api="satsplat_iteration_host_begin / _end, two steps in flight (pinned host buffers; same work as the device "
                               "step, cascade chain included; the upstream-gradient images go up and the rendered images come down); "
                               "serial_ms_per_step = one blocking satsplat_iteration_host per step")
        # the call a training loop makes: surfels + target image up, forward -> loss stage on the device -> backward,
        # gradients + loss sums down.  MORE device work per step than `value` times (the loss stage), a third of the bytes.
        h_tgt = torch.rand(v.height, v.width, 4).pin_memory()
        h_sums2 = [torch.empty(8).pin_memory() for _ in range(2)]
        h_sums = h_sums2[0]
        targs2 = [(cam, sun, sh, scene.n, *h_in, h_tgt, None, h_g2[k], h_sums2[k]) for k in range(2)]
        targs = targs2[0]

        def t_serial():
            for i in range(n_e2e):
                P.training_step_host(job.ctx, job.sctx, *targs)

        def t_pipelined():
            P.training_step_host_begin(job.ctx, job.sctx, 0, *targs2[0])
            for i in range(1, n_e2e):
                P.training_step_host_begin(job.ctx, job.sctx, i & 1, *targs2[i & 1])
                P.training_step_host_end(job.ctx, (i - 1) & 1)
            P.training_step_host_end(job.ctx, (n_e2e - 1) & 1)
        t_serial()
        dt_ts = wall(t_serial)
        t_pipelined()
        dt_t = wall(t_pipelined)
        assert all(float(x[0]) > 0 for x in h_sums2) and all(bool(torch.isfinite(x).all()) for x in h_g2)
        line["e2e"] = dict(value=world * px / 1e6 / (dt_t / n_e2e), unit=UNIT, h2d_bytes_per_step=scene.n * 52 + px * 16,
                           d2h_bytes_per_step=(scene.n * 13 + 23 + 8) * 4, ms_per_step=1e3 * dt_t / n_e2e, steps=n_e2e,
                           serial_ms_per_step=1e3 * dt_ts / n_e2e,
                           api="satsplat_training_step_host_begin / _end, two steps in flight (pinned host buffers): the device step "
                               "of `value` PLUS the loss stage (L1 + SSIM + distortion + normal consistency) between forward and "
                               "backward; surfels and the target image go up, gradients and the loss sums come down; "
                               "serial_ms_per_step = one blocking satsplat_training_step_host per step",
                           rasteriser_only=raster_only)
    # ---- the oracle beside it (rank 0, N = 1 only) ----
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline_block(scene, step_views[0], px, nviews)
    if rank == 0:
        print(json.dumps(line))
    if dp:
        dist.destroy_process_group()


def extras(line, args, job, P, torch, scene, device, peaks, step_views, px):
    """The NEXT rows of SURVEY.md section 8 that sit outside the metric's iteration, each timed on its own."""
    traffic_all, _ = load_traffic()
    # ---- the optimiser step (row f3) ----
    ns = P.adam_state_floats(scene.n)
    am, av = torch.zeros(ns, device=device), torch.zeros(ns, device=device)
    pp = [t.clone() for t in (job.means, job.quats, job.scales, job.logits, job.rgb)]
    gg = [job.g[k] for k in ("m", "q", "s", "l", "c")]
    lr = [0.075, 0.001, 0.001, 0.05, 0.0025]     # PAPER.md:349 (opacity: not stated, 3DGS's value)
    for t_ in range(1, 4):
        P.adam_step(scene.n, *pp, *gg, am, av, lr, step=t_)
    ms_adam = timed(torch, None, 1, lambda t_: P.adam_step(scene.n, *pp, *gg, am, av, lr, step=t_), range(4, 4 + 20)) / 20
    ab = scene.n * 13 * 28.0
    line["adam"] = dict(ms=ms_adam, bound="hbm", achieved=ab / (ms_adam * 1e-3) / 1e9, peak=peaks["hbm_gbs"], unit="GB/s",
                        frac=ab / (ms_adam * 1e-3) / 1e9 / peaks["hbm_gbs"], bytes_per_surfel=13 * 28,
                        note="fused Adam over the 13 N surfel parameters; not included in value / ms_per_step")
    # ---- the loss stage (row f1), on the last rendered view ----
    vi = step_views[-1]
    cam = job.cams[vi][0]
    tgt = torch.rand(job.H, job.W, 4, device=device)
    scr = torch.empty(P.loss_scratch_floats(job.W, job.H), device=device)
    vv = [torch.empty(job.H, job.W, 4, device=device) for _ in range(3)]
    sums = torch.zeros(8, device=device)
    run_loss = lambda _: P.loss_upstream(cam, job.out[0], job.out[1], job.out[2], tgt, scr, vv[0], vv[1], vv[2], sums)
    for _ in range(3):
        run_loss(0)
    ms_loss = timed(torch, None, 1, run_loss, range(20)) / 20
    # the METHOD moves 64 B in (three rendered images + target) + 48 B out (three upstream images) = 112 B / pixel; this
    # design's three kernels move 264 (derivative maps and v_zv written and read back).  Neither is what limits the
    # kernels today: ssim_stats / ssim_adjoint run at 59-73 % issue-active (profiles/r2_loss.md), i.e. instruction issue.
    lb, lb_design = px * 112.0, px * 264.0
    lt = [(traffic_all or {}).get(k) for k in ("ssim_stats_kernel", "normal_term_kernel", "ssim_adjoint_kernel")]
    line["loss_stage"] = dict(ms=ms_loss, bound="hbm", achieved=lb / (ms_loss * 1e-3) / 1e9, peak=peaks["hbm_gbs"], unit="GB/s",
                              frac=lb / (ms_loss * 1e-3) / 1e9 / peaks["hbm_gbs"], bytes_per_pixel=112,
                              design_bytes_per_pixel=264, design_frac=lb_design / (ms_loss * 1e-3) / 1e9 / peaks["hbm_gbs"],
                              binding="instruction issue (59-73 % issue-active in the two SSIM kernels), not HBM: frac is the distance "
                                      "to the method's byte floor, not the headroom of these kernels",
                              traffic_over_algorithmic=(sum(t["dram_bytes"] for t in lt) / lb) if all(lt) else None,
                              note="L1 + SSIM + distortion + normal consistency -> upstream gradients (3 kernels, the normal term beside "
                                   "the SSIM statistics on a side stream); not included in value / ms_per_step")
    # ---- one whole TRAINING iteration as ONE CUDA graph: camera chain (f2), both passes forward, loss stage (f1), both
    # backwards, cascade chain, Adam step (f3); device-resident cameras, so the same graph serves all views and steps ----
    if not args.no_graphs and not args.dp_path and args.gpus == 1:
        lr_tiny = [1e-7] * 5      # the step is real, the learning rates are tiny so that the synthetic scene stays put
        surf = [job.means, job.quats, job.scales, job.logits, job.rgb]

        def upstream():
            P.loss_upstream(cam, job.out[0], job.out[1], job.out[2], tgt, scr, vv[0], vv[1], vv[2], sums)
            return vv

        nv_ = len(scene.views)
        cm, cv = torch.zeros(nv_, 23, device=device), torch.zeros(nv_, 23, device=device)
        csteps = torch.zeros(nv_, dtype=torch.int32, device=device)

        def camera_step(g):     # dF, gain / bias (and ambient) of the rendered view; tiny rates as for the surfels
            P.adam_step_cameras(job.table, job.idx, job.dF_all, job.v_dF_all, g["cc"], g["amb"], cm, cv, csteps, [1e-9] * 3)

        def train_iteration():
            job.step_device(upstream_fn=upstream, camera_step_fn=camera_step)
            P.adam_step(scene.n, *surf, *gg, am, av, lr_tiny, step=100)
        job.idx.fill_(step_views[0])
        train_iteration()
        torch.cuda.synchronize()
        tgraph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(tgraph, stream=torch.cuda.Stream(device=device, priority=-1)):
            train_iteration()
        for _ in range(3):
            tgraph.replay()
        ms_train = timed(torch, None, 1, lambda _: tgraph.replay(), range(50)) / 50
        line["training_iteration"] = dict(ms=ms_train, mpixel_s=px / 1e6 / (ms_train * 1e-3),
                                          note="ONE graph replay per iteration: the step of `value` + loss stage between forward and "
                                               "backward + fused Adam over the 13 N parameters + Adam step of the rendered view's camera groups "
                                               "(dF, gain / bias, ambient; PAPER.md:349) -- a closed step for every learnable group "
                                               "(learning rates 1e-7 / 1e-9: the synthetic scene stays put); not included in value / ms_per_step")
    # ---- geometry-aware initialisation (row f4): one-time work, on a DSM of the site's size ----
    side = int(round(1000.0 / 0.3)) if args.config in (3, 4) else 512
    gen = torch.Generator(device=device); gen.manual_seed(1)
    dsm = torch.cumsum(torch.randn(side, side, device=device, generator=gen) * 0.05, 1)
    dsm[side // 4: side // 3, side // 4: side // 2] += 25.0
    uu = [torch.rand(scene.n, device=device, generator=gen).clamp_(max=0.99999994) for _ in range(3)]
    P.init_from_dsm(dsm, 0.3, (0.0, 0.0), *uu)
    ms_init = timed(torch, None, 1, lambda _: P.init_from_dsm(dsm, 0.3, (0.0, 0.0), *uu), range(3)) / 3
    line["init_stage"] = dict(ms=ms_init, dsm=f"{side}x{side}", samples=scene.n,
                              note="area-weighted sampling + frames + exact 3-NN scale from a DSM (9 kernels); one-time, not part of the iteration")


def main():
    args = parse()
    if args.record_traffic:
        record_traffic(args.record_traffic)
        return
    if args.impl == "reference":
        run_reference(args)
        return
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # not launched by torchrun: start one process per GPU ourselves and hand over
        sys.exit(subprocess.call(spawn_command(args, free_port())))
    run_ours(args)


if __name__ == "__main__":
    main()

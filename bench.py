#!/usr/bin/env python
"""bench.py - throughput of the dfp hot path on B200, one JSON line (contract: see the task statement / DESIGN.md §8).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 5]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N --steps K --warmup W

A STEP is one pass of the whole hot path over one batch of synthetic input: dfp_forward, dfp_forward_pose_grad,
dfp_backproject and dfp_backproject_pose_grad on the workload.  Default workload: BASELINE.json configs[4], the
LARGEST single-GPU config ("large throughput sweep": 512^3 volume, 360 views of 1024x1024, all four calls, everything
resident in HBM at once).  `value` is the headline metric "fwd+pose-grad Gray-steps/s" =
2 * ray_steps / (t_forward + t_forward_pose_grad) with inputs resident in HBM; the back-projection half of the step is
reported in `extra` as Gvoxel-views/s, and so are the rates of configs[1] (C2 registration) and configs[3] (C4
calibration).  N > 1: every rank runs its own slice of a global batch of N x 360 views (independent views, no
data-path collective) -> weak scaling.
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
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads as W  # noqa: E402

METRIC = "fwd+pose-grad Gray-steps/s"
UNIT = "Gray-steps/s"

# ALGORITHMIC work per unit, SURVEY.md section 8(d) (what the method itself must do per ray-step / voxel-view):
#   fetches: distinct voxel / pixel reads of 4 bytes each; flop: the arithmetic of section 8(d)'s per-unit list.
KERNELS = ("fwd_project", "fwd_grad", "bp", "bp_grad")
FETCHES_PER_UNIT = {"fwd_project": 8, "fwd_grad": 32, "bp": 4, "bp_grad": 12}
FLOP_PER_UNIT = {"fwd_project": 30, "fwd_grad": 100, "bp": 25, "bp_grad": 80}
N_SM = 148
L1_BYTES_PER_CLK_PER_SM = 128          # shared-memory / L1 data pipe: 32 lanes x 4 bytes per clock per SM
FP32_LANES_PER_SM = 128


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return json.load(open(p)), "measured (MEASURED_PEAKS.json)"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, pw = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def row_band(g, rows):
    """The central `rows` detector rows of g as a sub-detector (v0 shifts the principal point so that its rays are
    exactly rays of the full detector)."""
    rows = min(rows, g.nv)
    r0 = (g.nv - rows) // 2
    v0 = (g.nv - 1) / 2.0 + g.v0 - r0 - (rows - 1) / 2.0       # c_v' = (rows-1)/2 + v0' = c_v - r0
    return g.replace(nv=rows, v0=v0), r0, rows


def time_oracle(w, vol_cpu, up_cpu_views, steps=1, warmup=0, rows=None):
    """oracle.forward + oracle.forward_pose_grad, as they stand, on a bounded sample of the workload: the first
    len(up_cpu_views) views, central `rows` detector rows.  Returns (Gray-steps/s, s per step, cores, text, steps)."""
    import oracle
    gs, r0, rows = row_band(w.geom, w.geom.nv if rows is None else rows)
    if up_cpu_views.ndim == 2:
        up_cpu_views = up_cpu_views[None]
    nv_s = up_cpu_views.shape[0]
    a = w.angles[:nv_s].float().numpy()
    p = w.poses[:nv_s].float().numpy()
    up = np.ascontiguousarray(up_cpu_views[:, r0:r0 + rows, :])
    times, n_steps = [], 0
    for i in range(warmup + steps):
        t0 = time.perf_counter()
        _, n_steps = oracle.forward(gs, a, p, vol_cpu, return_steps=True)
        oracle.forward_pose_grad(gs, a, p, vol_cpu, up)
        dt = time.perf_counter() - t0
        if i >= warmup:
            times.append(dt)
    sec = float(np.mean(times))
    val = 2.0 * n_steps / sec / 1e9
    txt = (f"views 0..{nv_s - 1} of {w.n_views}, central {rows} of {w.geom.nv} detector rows x {w.geom.nu} columns "
           f"({n_steps} ray-steps per pass), oracle.forward + oracle.forward_pose_grad, fp64, OpenMP; a RATE on a "
           f"seeded subset of the workload's views, not the whole job")
    return val, sec, oracle.num_threads(), txt, n_steps, gs


def run_reference(args, rank, world):
    """--impl reference: the fp64 CPU oracle, as it stands, on the host cores (rank 0 only).  One step = one view,
    central 256 detector rows of the workload (about 1.5 s on 16 cores), so that K + W steps end within minutes."""
    if rank != 0:
        return
    w = W.make_config(args.config)
    vol = w.volume("cpu").numpy()
    ups = w.fwd_upstream("cpu", views=range(1)).numpy()
    rows = 256 if w.geom.nv * w.geom.nu > 512 * 512 else w.geom.nv
    val, sec, cores, txt, _, _ = time_oracle(w, vol, ups, steps=args.steps, warmup=args.warmup, rows=rows)
    out = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
           "steps": args.steps, "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": workload_name(w, w.n_views), "sample": txt},
           "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": txt},
           "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out), flush=True)


def workload_name(w, V):
    g = w.geom
    return (f"{w.name} (BASELINE.json configs[{w.index - 1}]): {g.nx}^3 volume, {V} views of {g.nu}x{g.nv}, "
            f"all four calls per step")


class Job:
    """One workload resident in HBM and the four calls on it."""

    def __init__(self, dfp, index, dev, rank=0, world=1, views=None, flags=0):
        from paper_2508_13304_b200.sharding import shard_range
        self.dfp, self.dev = dfp, dev
        V1 = views if views is not None else W.CONFIGS[index]["views"]
        self.w = w = W.make_config(index, n_views=V1 * world)
        self.g = g = w.geom.replace(flags=w.geom.flags | flags) if flags else w.geom
        lo, hi = shard_range(w.n_views, rank, world)
        self.V = V = hi - lo
        self.angles = np.ascontiguousarray(w.angles.float().numpy()[lo:hi])
        self.poses = np.ascontiguousarray(w.poses.float().numpy()[lo:hi])
        self.vol = w.volume(dev)
        self.up = w.fwd_upstream(dev, views=range(lo, hi))
        self.bp_up = W.normal_field(w.seed * 4096 + 5, g.nx * g.ny * g.nz, dev).reshape(g.vol_shape).contiguous()
        self.proj = torch.empty((V, g.nv, g.nu), dtype=torch.float32, device=dev)
        self.grad = torch.empty((V, 6), dtype=torch.float32, device=dev)
        self.bvol = torch.empty(g.vol_shape, dtype=torch.float32, device=dev)
        self.bgrad = torch.empty((V, 6), dtype=torch.float32, device=dev)
        self.ws = torch.empty(max(dfp.workspace_bytes(g, V, op) for op in range(4)), dtype=torch.uint8, device=dev)
        self.ray_steps = dfp.count_ray_steps(g, self.angles, self.poses)
        self.voxel_views = g.nx * g.ny * g.nz * V
        self.launches = 0
        self.kern_ms = {k: [] for k in KERNELS}
        self.paths = {}

    def calls(self, g=None, views=None):
        d, g = self.dfp, self.g if g is None else g
        a = self.angles if views is None else views
        return (("forward", lambda: d.forward(g, a, self.poses, self.vol, out=self.proj, ws=self.ws)),
                ("forward_pose_grad", lambda: d.forward_pose_grad(g, a, self.poses, self.vol, self.up, out=self.grad,
                                                                  ws=self.ws)),
                ("backproject", lambda: d.backproject(g, a, self.poses, self.proj, out=self.bvol, ws=self.ws)),
                ("backproject_pose_grad", lambda: d.backproject_pose_grad(g, a, self.poses, self.proj, self.bp_up,
                                                                          out=self.bgrad, ws=self.ws)))

    def step(self, record=False):
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(5)]
        ev[0].record()
        for i, ((name, fn), k) in enumerate(zip(self.calls(), KERNELS)):
            fn()
            self.launches += self.dfp.last_launch_count()
            self.paths[name] = self.dfp.last_path()
            if record:
                self.kern_ms[k].append(self.dfp.last_kernel_ms())
            ev[i + 1].record()
        return ev

    def timed(self, steps, warmup, flush, barrier, sampler=None):
        for _ in range(warmup):
            self.step()
            flush.zero_()
        barrier()
        self.launches = 0
        if sampler:
            sampler.start()
        evs = []
        for _ in range(steps):
            flush.zero_()                      # L2 flush between timed iterations (outside the per-step events)
            evs.append(self.step(record=True))
        barrier()
        clocks = sampler.stop() if sampler else None
        seg = np.array([[a.elapsed_time(b) for a, b in zip(e[:-1], e[1:])] for e in evs])   # ms, [K,4]
        return seg, clocks

    def time_calls(self, fns, reps):
        out = []
        for fn in fns:
            fn()
            a_, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a_.record()
            for _ in range(reps):
                fn()
            b_.record()
            torch.cuda.synchronize()
            out.append(a_.elapsed_time(b_) / reps)
        return out


def rates(job, seg):
    """Per-call rates of one rank from the [K,4] millisecond table."""
    t = seg.mean(axis=0) * 1e-3
    return {"ms_per_call": {"forward": float(t[0] * 1e3), "forward_pose_grad": float(t[1] * 1e3),
                            "backproject": float(t[2] * 1e3), "backproject_pose_grad": float(t[3] * 1e3)},
            "fwd+pose-grad_gray_steps_per_s": 2.0 * job.ray_steps / (t[0] + t[1]) / 1e9,
            "forward_gray_steps_per_s": job.ray_steps / t[0] / 1e9,
            "forward_pose_grad_gray_steps_per_s": job.ray_steps / t[1] / 1e9,
            "backproject+grad_gvoxel_views_per_s": 2.0 * job.voxel_views / (t[2] + t[3]) / 1e9,
            "backproject_gvoxel_views_per_s": job.voxel_views / t[2] / 1e9,
            "backproject_pose_grad_gvoxel_views_per_s": job.voxel_views / t[3] / 1e9,
            "ray_steps_per_pass": int(job.ray_steps), "voxel_views_per_pass": int(job.voxel_views),
            "kernel_paths": {k: ("tma" if v == job.dfp.PATH_TMA else "gather") for k, v in job.paths.items()}}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=5, help="BASELINE.json config index 1..5 (default 5, the largest)")
    ap.add_argument("--debug-views", type=int, default=None, help="override the view count (profiling runs only)")
    ap.add_argument("--weights", default="rd", choices=["rd", "dd", "sf"],
                    help="profiling runs only: the four calls with the distance-driven / separable-footprint weights "
                         "(DFP_FLAG_DD / DFP_FLAG_SF) instead of the paper's ray-driven trilinear / voxel-driven pair")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip the other modes / configs reported in `extra`")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.weights != "rd":      # another weight model: the four calls only (unit, roofline and baselines are the RD path's)
        args.no_cpu_baseline = args.no_e2e = args.no_extras = True

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))

    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import paper_2508_13304_b200 as dfp   # fails loudly if libdfp.so is missing: no CPU fallback
    from paper_2508_13304_b200.sharding import max_over_ranks, sum_over_ranks

    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---------------------------------------------------------------- workload, resident in HBM
    # N ranks: a global batch of N x (the config's views), sharded by views, one shard per GPU (weak scaling);
    # rank 0's shard is exactly the N=1 workload.  No data-path collective.
    job = Job(dfp, args.config, dev, rank, world, args.debug_views,
              {"rd": 0, "dd": dfp.FLAG_DD, "sf": dfp.FLAG_SF}[args.weights])
    w, g, V = job.w, job.g, job.V
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)        # > 126 MB L2
    dfp.set_kernel_timing(True)
    K = args.steps
    seg, clocks = job.timed(K, args.warmup, flush, barrier, ClockSampler(local_rank) if rank == 0 else None)
    n_launch = job.launches
    t = seg.sum(axis=0) / 1e3                                                            # s per call, over K steps
    tt = max_over_ranks(torch.tensor([t[0] + t[1], t[2] + t[3], t.sum()], dtype=torch.float64, device=dev))
    t_fg, t_bp, t_all = [float(x) for x in tt.cpu()]
    t_call = [float(x) for x in max_over_ranks(torch.tensor(t, dtype=torch.float64, device=dev)).cpu()]
    uu = sum_over_ranks(torch.tensor([job.ray_steps, job.voxel_views], dtype=torch.float64, device=dev))
    job_ray_steps, job_voxel_views = [float(x) for x in uu.cpu()]      # units all ranks processed per pass
    value = 2.0 * job_ray_steps * K / t_fg / 1e9
    bp_value = 2.0 * job_voxel_views * K / t_bp / 1e9
    mean_ms = {k: float(np.mean(v)) for k, v in job.kern_ms.items()}
    main_rates = rates(job, seg)

    # ---------------------------------------------------------------- other modes of the same workload (outside the step)
    extra = {"backproject+grad_gvoxel_views_per_s": bp_value,
             "forward_gray_steps_per_s": job_ray_steps * K / t_call[0] / 1e9,
             "forward_pose_grad_gray_steps_per_s": job_ray_steps * K / t_call[1] / 1e9,
             "backproject_gvoxel_views_per_s": job_voxel_views * K / t_call[2] / 1e9,
             "backproject_pose_grad_gvoxel_views_per_s": job_voxel_views * K / t_call[3] / 1e9,
             "ms_per_call": main_rates["ms_per_call"], "kernel_paths": main_rates["kernel_paths"]}
    if not args.no_extras:
        reps = 1 if job.ray_steps > 2e10 else 3
        gi = g.replace(flags=g.flags | dfp.FLAG_GRAD_INTERP)
        c = dict(job.calls(gi))
        ms = job.time_calls([c["forward_pose_grad"], c["backproject_pose_grad"]], reps)
        extra["grad_interp_mode_ms_per_call"] = {"forward_pose_grad": ms[0], "backproject_pose_grad": ms[1]}
        for name, flag in (("siddon", dfp.FLAG_SIDDON), ("joseph", dfp.FLAG_JOSEPH)):
            c = dict(job.calls(g.replace(flags=g.flags | flag)))
            ms = job.time_calls([c["forward"], c["forward_pose_grad"]], reps)
            extra[f"{name}_mode_ms_per_call"] = {"forward": ms[0], "forward_pose_grad": ms[1]}
        # DFP_FLAG_DD / DFP_FLAG_SF: the other matched pairs, all four calls (back-projector = exact transpose of the
        # forward one)
        ws0 = job.ws
        for name, flag in (("dd", dfp.FLAG_DD), ("sf", dfp.FLAG_SF)):
            gm = g.replace(flags=g.flags | flag)
            job.ws = torch.empty(max(dfp.workspace_bytes(gm, V, op) for op in range(4)), dtype=torch.uint8, device=dev)
            ms = job.time_calls([fn for _, fn in job.calls(gm)], 1)
            extra[f"{name}_mode_ms_per_call"] = dict(zip(("forward", "forward_pose_grad", "backproject",
                                                         "backproject_pose_grad"), ms))
        job.ws = ws0
        torch.cuda.empty_cache()
        # DFP_FLAG_VIEW_FRAMES: the four calls with one explicit (s, c, U, V) frame per view - the config's views on a
        # seeded non-circular (saddle) orbit with detector wobble; same kernels, only the per-view set-up differs
        gv = g.replace(flags=g.flags | dfp.FLAG_VIEW_FRAMES)
        frames = W.noncircular_orbit(g, np.asarray(job.angles, dtype=np.float64), w.seed + 17).numpy().astype(np.float32)
        ms = job.time_calls([fn for _, fn in job.calls(gv, frames)], reps)
        extra["view_frames_mode_ms_per_call"] = dict(zip(("forward", "forward_pose_grad", "backproject",
                                                          "backproject_pose_grad"), ms))
        dict(job.calls())["forward"]()                                       # restore the default-mode projections
        # dfp_forward_fused_moments: projection + gradient moments in one traversal (target = the upstream array's shape)
        ws_f = torch.empty(dfp.workspace_bytes(g, V, dfp.OP_FORWARD_FUSED), dtype=torch.uint8, device=dev)
        mom = torch.empty((V, 3, 6), dtype=torch.float32, device=dev)
        proj_f = torch.empty_like(job.proj)
        ms = job.time_calls([lambda: dfp.forward_fused_moments(g, job.angles, job.poses, job.vol, job.up,
                                                               out_proj=proj_f, out_moments=mom, ws=ws_f)], reps)
        extra["forward_fused_moments_ms_per_call"] = ms[0]
        extra["forward_fused_moments_gray_steps_per_s"] = 2.0 * job.ray_steps / (ms[0] * 1e-3) / 1e9
        del ws_f, proj_f, mom
        for _, fn in job.calls():                                            # leave the default-mode results behind
            fn()
        torch.cuda.synchronize()

    # ---------------------------------------------------------------- end to end through the host-buffer C ABI
    e2e = None
    if not args.no_e2e:
        pin = lambda t_: t_.cpu().pin_memory()
        h_vol, h_up, h_bpup = pin(job.vol), pin(job.up), pin(job.bp_up)
        h_proj = torch.empty((V, g.nv, g.nu), dtype=torch.float32).pin_memory()
        h_grad = torch.empty((V, 6), dtype=torch.float32).pin_memory()
        h_bvol = torch.empty(g.vol_shape, dtype=torch.float32).pin_memory()
        h_bgrad = torch.empty((V, 6), dtype=torch.float32).pin_memory()
        a_, p_ = job.angles, job.poses

        def e2e_step():
            t0 = time.perf_counter()
            dfp.forward_host(g, a_, p_, h_vol, out=h_proj)
            dfp.forward_pose_grad_host(g, a_, p_, h_vol, h_up, out=h_grad)
            t1 = time.perf_counter()
            dfp.backproject_host(g, a_, p_, h_proj, out=h_bvol)
            dfp.backproject_pose_grad_host(g, a_, p_, h_proj, h_bpup, out=h_bgrad)
            return t1 - t0, time.perf_counter() - t1

        Ke = min(K, 5)                       # the end-to-end loop is bounded so that the default run ends within minutes
        for _ in range(2):
            e2e_step()
        barrier()
        tf = tb = 0.0
        for _ in range(Ke):
            x, y = e2e_step()
            tf += x
            tb += y
        barrier()
        te = max_over_ranks(torch.tensor([tf, tb], dtype=torch.float64, device=dev))
        tf, tb = [float(x) for x in te.cpu()]
        nb = lambda t_: t_.numel() * t_.element_size()
        e2e = {"value": 2.0 * job_ray_steps * Ke / tf / 1e9, "unit": UNIT, "steps": Ke,
               "h2d_bytes_per_step": 2 * nb(h_vol) + nb(h_up) + 2 * nb(h_proj) + nb(h_bpup),
               "d2h_bytes_per_step": nb(h_proj) + nb(h_grad) + nb(h_bvol) + nb(h_bgrad),
               "backproject+grad_gvoxel_views_per_s": 2.0 * job_voxel_views * Ke / tb / 1e9,
               "api": "dfp_*_host (pinned host buffers; cudaMallocAsync + chunked H2D + kernels + D2H + sync per call)"}
        del h_vol, h_up, h_bpup, h_proj, h_grad, h_bvol, h_bgrad

    # ---------------------------------------------------------------- CPU baseline: the oracle on the host cores
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        # about 10 s of oracle work on 16 cores: two full views of config 5 (forward + gradient)
        n_s = min(2 if g.nu * g.nv >= 1024 * 1024 else (4 if g.nx >= 512 else 16), V)
        val, sec, cores, txt, n_ora, gs = time_oracle(w, job.vol.cpu().numpy(), job.up[:n_s].cpu().numpy())
        n_lib = dfp.count_ray_steps(gs, job.angles[:n_s], job.poses[:n_s])
        cpu = {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": txt, "seconds": sec,
               "unit_check": {"ray_steps_oracle_sample": int(n_ora), "ray_steps_library_same_sample": int(n_lib),
                              "ratio": n_lib / max(n_ora, 1),
                              "note": "the metric's unit is defined by the oracle's clip (SURVEY 8d: samples inside the "
                                      "2-voxel-padded box); dfp_count_ray_steps counts the same set"}}

    # ---------------------------------------------------------------- rates of the other measured configs (rank 0)
    other = {}
    if not args.no_extras and world == 1 and args.config == 5 and args.debug_views is None:
        del job.up, job.proj, job.bp_up, job.ws, job.vol, job.bvol
        torch.cuda.empty_cache()
        # the paper's first task as a loop (PAPER.md :228-235): one view of C2, Adam on NCC, per iteration
        # dfp_forward_fused_moments + dfp_ncc_pose_grad + a 28-byte read-back (registration.register_view)
        from paper_2508_13304_b200.registration import register_view
        wr = W.make_config(2, n_views=1)
        volr = wr.volume(dev)
        ar = wr.angles.float().numpy()
        hidden = wr.data_poses[0].float().numpy()
        tgt = dfp.forward(wr.geom, ar, hidden[None] * 0.25, volr).clone()          # 5 mm / 2.5 degrees off
        register_view(wr.geom, ar, volr, tgt, max_iters=5, ncc_stop=2.0, dloss_stop=-1.0)     # warm-up
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        rr = register_view(wr.geom, ar, volr, tgt, max_iters=100, ncc_stop=2.0, dloss_stop=-1.0)
        dt = time.perf_counter() - t0
        rs = register_view(wr.geom, ar, volr, tgt, max_iters=300)
        other["registration_loop_C2"] = {"iterations_per_s": rr["iterations"] / dt, "ms_per_iteration": dt / rr["iterations"] * 1e3,
                                         "timed_iterations": rr["iterations"], "with_stop_rule": {"iterations": rs["iterations"],
                                         "ncc": rs["ncc"], "stop": rs["stop"]},
                                         "what": "256^3 volume, one 512x512 view, Adam on NCC (Eq.25), stop rule of PAPER.md :235"}
        del volr, tgt
        # the paper's second task as a loop (PAPER.md :237-242, Eq.26): full C3 (256^3, 360 ramp-filtered views of
        # 512x384, FDK weight), Adam on the gradient entropy of the back-projection; per iteration dfp_backproject +
        # GE and its autograd gradient (harness, torch, same stream) + dfp_backproject_pose_grad + a [360, 6] read-back
        from paper_2508_13304_b200.registration import motion_compensated_backprojection
        w3 = W.make_config(3)
        p3 = w3.projections(dev)
        a3 = w3.angles.float().numpy()
        motion_compensated_backprojection(w3.geom, a3, p3, W.gradient_entropy, n_iters=2)       # warm-up
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        r3 = motion_compensated_backprojection(w3.geom, a3, p3, W.gradient_entropy, n_iters=10)
        dt = time.perf_counter() - t0
        other["mcfdk_loop_C3"] = {"ms_per_iteration": dt / 10 * 1e3, "iterations_per_s": 10 / dt, "timed_iterations": 10,
                                  "gradient_entropy_first_last": [r3["losses"][0], r3["losses"][-1]],
                                  "what": "256^3 volume, 360 views of 512x384, all 360x6 poses, Adam on gradient entropy (Eq.26)"}
        del p3
        torch.cuda.empty_cache()
        for idx in (2, 4):
            j2 = Job(dfp, idx, dev)
            seg2, _ = j2.timed(3, 3, flush, barrier)
            other[f"C{idx}"] = dict(rates(j2, seg2), workload=workload_name(j2.w, j2.V))
            if idx == 2:      # DFP_FLAG_DD / DFP_FLAG_SF: the other matched pairs, all four calls, on the C2 workload
                for name, flag in (("dd", dfp.FLAG_DD), ("sf", dfp.FLAG_SF)):
                    gm = j2.g.replace(flags=j2.g.flags | flag)
                    j2.ws = torch.empty(max(dfp.workspace_bytes(gm, j2.V, op) for op in range(4)), dtype=torch.uint8,
                                        device=dev)
                    ms = j2.time_calls([fn for _, fn in j2.calls(gm)], 1)
                    other["C2"][f"{name}_mode_ms_per_call"] = dict(zip(("forward", "forward_pose_grad", "backproject",
                                                                       "backproject_pose_grad"), ms))
            del j2
            torch.cuda.empty_cache()

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---------------------------------------------------------------- roofline of the dominant kernel
    # The path is bound by the SM-side memory pipe, not by HBM: achieved = ALGORITHMIC fetch bytes
    # (distinct voxel / pixel reads x 4 B per unit) / CUDA-event time of the kernel; peak = the
    # shared-memory / L1 data pipe, 128 B per clock per SM at the measured maximum SM clock.
    pk, pk_kind = peaks()
    clk = pk.get("sm_max_mhz", 1965.0) * 1e6
    dom = max(mean_ms, key=mean_ms.get)
    units = {"fwd_project": job.ray_steps, "fwd_grad": job.ray_steps, "bp": job.voxel_views, "bp_grad": job.voxel_views}
    l1_peak = N_SM * L1_BYTES_PER_CLK_PER_SM * clk / 1e9                                  # GB/s
    fp32_peak = N_SM * FP32_LANES_PER_SM * 2 * clk / 1e12                                 # TFLOP/s (FMA = 2)
    nbytes = lambda t_: t_.numel() * 4
    vox, img = g.nx * g.ny * g.nz * 4, V * g.nu * g.nv * 4
    compulsory = {"fwd_project": vox + img, "fwd_grad": vox + img, "bp": img + vox, "bp_grad": img + vox}

    def kernel_roofline(k):
        sec = mean_ms[k] * 1e-3
        ach = FETCHES_PER_UNIT[k] * 4.0 * units[k] / sec / 1e9
        return {"ms": mean_ms[k], "share_of_step": mean_ms[k] * K / 1e3 / t_all, "l1_gbs": ach, "l1_frac": ach / l1_peak,
                "fp32_tflops": FLOP_PER_UNIT[k] * units[k] / sec / 1e12,
                "fp32_frac": FLOP_PER_UNIT[k] * units[k] / sec / 1e12 / fp32_peak,
                "hbm_compulsory_bytes": compulsory[k],
                "hbm_compulsory_frac": compulsory[k] / sec / 1e9 / pk["hbm_gbs"]}

    per_kernel = {k: kernel_roofline(k) for k in KERNELS}
    traffic = None
    tp = os.path.join(ROOT, "profiles", "traffic.csv")     # dram__bytes_read+write per launch from the ncu --set full capture
    if os.path.exists(tp):
        import csv
        for row in csv.DictReader(open(tp)):
            if row["config"] == f"C{args.config}" and row["kernel"] == dom:
                # captured with `views_in_capture` views; DRAM traffic of these kernels scales with the view count
                traffic = int(float(row["dram_bytes_per_launch"]) * V / float(row["views_in_capture"]))
    roofline = {"bound": "l1/shared", "kernel": dom, "achieved": per_kernel[dom]["l1_gbs"], "peak": l1_peak,
                "unit": "GB/s", "frac": per_kernel[dom]["l1_frac"], "traffic": traffic,
                "algorithmic_bytes_per_unit": FETCHES_PER_UNIT[dom] * 4, "units_per_launch": int(units[dom]),
                "kernel_ms": mean_ms[dom],
                "peak_source": f"148 SMs x 128 B/clk (shared-memory / L1 data pipe) x sm_max_mhz, {pk_kind}; "
                               "HBM is not the binding roofline: see hbm_compulsory_frac",
                "hbm_peak_gbs": pk["hbm_gbs"], "fp32_peak_tflops": fp32_peak, "per_kernel": per_kernel}
    try:      # measured denominator (libdfp_bench.so, include/dfp_bench.h): warp-wide conflict-free LDS per clock per SM
        from paper_2508_13304_b200 import microbench as mb
        lds = mb.run(mb.MB_LDS) / (N_SM * clk)
        roofline["measured_lds_warp_inst_per_clk_per_sm"] = lds
        roofline["frac_of_measured_lds_rate"] = roofline["frac"] / lds
    except Exception as e:      # the probe library is optional
        roofline["measured_lds_warp_inst_per_clk_per_sm"] = f"unavailable: {e}"

    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": args.warmup,
           "ms_per_step": t_all / K * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "f32", "data": "synthetic",
           "config": {"workload": workload_name(w, V) + ("" if args.weights == "rd" else
                                                          f" - {args.weights.upper()} weights (profiling run: unit and "
                                                          "roofline figures are those of the ray-driven path)"),
                      "ray_steps_per_pass": int(job_ray_steps),
                      "voxel_views_per_pass": int(job_voxel_views), "l2": "256 MiB flush write between timed steps",
                      "parallelism": f"views sharded over {world} rank(s), {V} views per GPU, no data-path collective"},
           "extra": extra, "other_configs": other, "clocks": clocks, "e2e": e2e, "gpu_launches": n_launch,
           "roofline": roofline, "cpu_baseline": cpu}
    print(json.dumps(out), flush=True)
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

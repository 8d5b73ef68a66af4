#!/usr/bin/env python
"""bench.py - throughput of the dfp hot path on B200, one JSON line (contract: see the task statement / DESIGN.md).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 2]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N --steps K --warmup W

A STEP is one pass of the whole hot path over one batch of synthetic input: dfp_forward, dfp_forward_pose_grad,
dfp_backproject and dfp_backproject_pose_grad on the workload (default: BASELINE.json configs[1], the 2D/3D
registration batch - 256^3 volume, 64 pose candidates, 512x512 detector).  `value` is the headline metric
"fwd+pose-grad Gray-steps/s" = 2 * ray_steps / (t_forward + t_forward_pose_grad), with inputs resident in
HBM; the back-projection half of the step is reported in `extra` as Gvoxel-views/s.  N > 1: every rank runs
its own copy of the batch (independent problems, no data-path collective) -> weak scaling.
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

# Algorithmic work per unit: thread-level arithmetic + load operations the method itself
# needs per ray-step / voxel-view, FMA counted as one op.  ALU peak = SMs x 128 lanes x clock.
OPS_PER_UNIT = {"fwd_project": 38, "fwd_grad": 113, "bp": 30, "bp_grad": 78}
N_SM = 148
LANES_PER_SM = 128


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return d, "measured"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


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


def oracle_sample(w, rows=32):
    """A bounded sample of the workload for the CPU oracle: ONE view, the central `rows` detector rows
    (v0 shifts the principal point so that the rays are exactly rays of the full detector)."""
    g = w.geom
    rows = min(rows, g.nv)
    r0 = (g.nv - rows) // 2
    # c_v' = (rows-1)/2 + v0' must equal c_v - r0
    v0 = (g.nv - 1) / 2.0 + g.v0 - r0 - (rows - 1) / 2.0
    gs = g.replace(nv=rows, v0=v0)
    return gs, r0, rows


def time_oracle(w, vol_cpu, up_cpu_views, steps=1, warmup=0, rows=128):
    """Oracle forward + forward_pose_grad on the sample (the first len(up_cpu_views) views, central `rows` detector
    rows); returns (Gray-steps/s, seconds per step, cores, text)."""
    import oracle
    gs, r0, rows = oracle_sample(w, rows)
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
    txt = (f"views 0..{nv_s - 1} of {w.n_views}, central {rows} of {g_nv(w)} detector rows x {w.geom.nu} columns "
           f"({n_steps} ray-steps per pass), oracle.forward + oracle.forward_pose_grad, fp64, OpenMP")
    return val, sec, oracle.num_threads(), txt


def g_nv(w):
    return w.geom.nv


def run_reference(args, rank, world):
    """--impl reference: the fp64 CPU oracle, as it stands, on the host cores (rank 0 only)."""
    if rank != 0:
        return
    w = W.make_config(args.config)
    vol = w.volume("cpu").numpy()
    # one step = 4 full views (forward + gradient): ~3 s on 16 cores, so that K + W steps end within a few minutes
    n_s = min(4, w.n_views)
    ups = w.fwd_upstream("cpu", views=range(n_s)).numpy()
    val, sec, cores, txt = time_oracle(w, vol, ups, steps=args.steps, warmup=args.warmup, rows=w.geom.nv)
    out = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
           "steps": args.steps, "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": f"{w.name} (BASELINE.json configs[{args.config - 1}])", "sample": txt},
           "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": txt},
           "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config index 1..5 (default 2)")
    ap.add_argument("--views", type=int, default=None, help="override the view count (debugging)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))

    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import paper_2508_13304_b200 as dfp   # fails loudly if libdfp.so is missing: no CPU fallback
    from paper_2508_13304_b200.sharding import max_over_ranks, shard_range, sum_over_ranks

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
    V1 = args.views if args.views is not None else W.CONFIGS[args.config]["views"]
    w = W.make_config(args.config, n_views=V1 * world)
    g = w.geom
    lo, hi = shard_range(w.n_views, rank, world)
    V = hi - lo
    angles = np.ascontiguousarray(w.angles.float().numpy()[lo:hi])
    poses = np.ascontiguousarray(w.poses.float().numpy()[lo:hi])
    vol = w.volume(dev)
    up = w.fwd_upstream(dev, views=range(lo, hi))
    bp_up = W.normal_field(w.seed * 4096 + 5, g.nx * g.ny * g.nz, dev).reshape(g.vol_shape).contiguous()
    proj = torch.empty((V, g.nv, g.nu), dtype=torch.float32, device=dev)
    grad = torch.empty((V, 6), dtype=torch.float32, device=dev)
    bvol = torch.empty(g.vol_shape, dtype=torch.float32, device=dev)
    bgrad = torch.empty((V, 6), dtype=torch.float32, device=dev)
    ws = torch.empty(max(dfp.workspace_bytes(g, V, op) for op in range(4)), dtype=torch.uint8, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)        # > 126 MB L2
    ray_steps = dfp.count_ray_steps(g, angles, poses)
    voxel_views = g.nx * g.ny * g.nz * V
    dfp.set_kernel_timing(True)

    ev = lambda: torch.cuda.Event(enable_timing=True)
    kern_ms = {k: [] for k in OPS_PER_UNIT}
    launches = [0]

    def step(record=False):
        e = [ev() for _ in range(5)]
        e[0].record()
        dfp.forward(g, angles, poses, vol, out=proj, ws=ws)
        launches[0] += dfp.last_launch_count()
        k0 = dfp.last_kernel_ms() if record else None
        e[1].record()
        dfp.forward_pose_grad(g, angles, poses, vol, up, out=grad, ws=ws)
        launches[0] += dfp.last_launch_count()
        k1 = dfp.last_kernel_ms() if record else None
        e[2].record()
        dfp.backproject(g, angles, poses, proj, out=bvol, ws=ws)
        launches[0] += dfp.last_launch_count()
        k2 = dfp.last_kernel_ms() if record else None
        e[3].record()
        dfp.backproject_pose_grad(g, angles, poses, proj, bp_up, out=bgrad, ws=ws)
        launches[0] += dfp.last_launch_count()
        k3 = dfp.last_kernel_ms() if record else None
        e[4].record()
        if record:
            for k, v in zip(OPS_PER_UNIT, (k0, k1, k2, k3)):
                kern_ms[k].append(v)
        return e

    for _ in range(args.warmup):
        step()
        flush.zero_()
    barrier()
    launches[0] = 0
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    evs = []
    for _ in range(args.steps):
        flush.zero_()                      # L2 flush between timed iterations (outside the per-step events)
        evs.append(step(record=True))
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    seg = np.array([[a.elapsed_time(b) for a, b in zip(e[:-1], e[1:])] for e in evs])   # ms, [K,4]
    t = seg.sum(axis=0) / 1e3                                                            # s per call, over K steps
    tt = max_over_ranks(torch.tensor([t[0] + t[1], t[2] + t[3], t.sum()], dtype=torch.float64, device=dev))
    t_fg, t_bp, t_all = [float(x) for x in tt.cpu()]
    t_call = [float(x) for x in max_over_ranks(torch.tensor(t, dtype=torch.float64, device=dev)).cpu()]
    uu = sum_over_ranks(torch.tensor([ray_steps, voxel_views], dtype=torch.float64, device=dev))
    job_ray_steps, job_voxel_views = [float(x) for x in uu.cpu()]      # units all ranks processed per pass
    K = args.steps
    value = 2.0 * job_ray_steps * K / t_fg / 1e9
    bp_value = 2.0 * job_voxel_views * K / t_bp / 1e9
    n_launch = launches[0]

    # ---------------------------------------------------------------- DFP_FLAG_GRAD_INTERP variants (outside the step)
    gi = g.replace(flags=g.flags | dfp.FLAG_GRAD_INTERP)
    interp_ms = []
    for fn in (lambda: dfp.forward_pose_grad(gi, angles, poses, vol, up, out=grad, ws=ws),
               lambda: dfp.backproject_pose_grad(gi, angles, poses, proj, bp_up, out=bgrad, ws=ws)):
        fn()
        a_, b_ = ev(), ev()
        a_.record()
        for _ in range(3):
            fn()
        b_.record()
        torch.cuda.synchronize()
        interp_ms.append(a_.elapsed_time(b_) / 3)
    # DFP_FLAG_SIDDON / DFP_FLAG_JOSEPH variants of the two forward calls
    model_ms = {}
    for name, flag in (("siddon", dfp.FLAG_SIDDON), ("joseph", dfp.FLAG_JOSEPH)):
        gm = g.replace(flags=g.flags | flag)
        model_ms[name] = []
        for fn in (lambda: dfp.forward(gm, angles, poses, vol, out=proj, ws=ws),
                   lambda: dfp.forward_pose_grad(gm, angles, poses, vol, up, out=grad, ws=ws)):
            fn()
            a_, b_ = ev(), ev()
            a_.record()
            for _ in range(3):
                fn()
            b_.record()
            torch.cuda.synchronize()
            model_ms[name].append(a_.elapsed_time(b_) / 3)
    # DFP_FLAG_VIEW_FRAMES: the four calls with one explicit (s, c, U, V) frame per view - the config's views on a
    # seeded non-circular (saddle) orbit with detector wobble; same kernels, only the per-view set-up differs
    gv = g.replace(flags=g.flags | dfp.FLAG_VIEW_FRAMES)
    frames = W.noncircular_orbit(g, np.asarray(angles, dtype=np.float64), w.seed + 17).numpy().astype(np.float32)
    frames_ms = []
    for fn in (lambda: dfp.forward(gv, frames, poses, vol, out=proj, ws=ws),
               lambda: dfp.forward_pose_grad(gv, frames, poses, vol, up, out=grad, ws=ws),
               lambda: dfp.backproject(gv, frames, poses, proj, out=bvol, ws=ws),
               lambda: dfp.backproject_pose_grad(gv, frames, poses, proj, bp_up, out=bgrad, ws=ws)):
        fn()
        a_, b_ = ev(), ev()
        a_.record()
        for _ in range(3):
            fn()
        b_.record()
        torch.cuda.synchronize()
        frames_ms.append(a_.elapsed_time(b_) / 3)
    dfp.forward(g, angles, poses, vol, out=proj, ws=ws)                        # restore the default-mode projections
    # dfp_forward_fused_moments: projection + gradient moments in one traversal (target = the upstream array's shape)
    ws_f = torch.empty(dfp.workspace_bytes(g, V, dfp.OP_FORWARD_FUSED), dtype=torch.uint8, device=dev)
    mom = torch.empty((V, 3, 6), dtype=torch.float32, device=dev)
    proj_f = torch.empty_like(proj)
    fused = lambda: dfp.forward_fused_moments(g, angles, poses, vol, up, out_proj=proj_f, out_moments=mom, ws=ws_f)
    fused()
    a_, b_ = ev(), ev()
    a_.record()
    for _ in range(3):
        fused()
    b_.record()
    torch.cuda.synchronize()
    fused_ms = a_.elapsed_time(b_) / 3
    del ws_f, proj_f
    dfp.forward_pose_grad(g, angles, poses, vol, up, out=grad, ws=ws)          # leave the default-mode results behind
    dfp.backproject_pose_grad(g, angles, poses, proj, bp_up, out=bgrad, ws=ws)

    # ---------------------------------------------------------------- end to end through the host-buffer C ABI
    e2e = None
    if not args.no_e2e:
        pin = lambda t_: t_.cpu().pin_memory()
        h_vol, h_up, h_bpup = pin(vol), pin(up), pin(bp_up)
        h_proj = torch.empty((V, g.nv, g.nu), dtype=torch.float32).pin_memory()
        h_grad = torch.empty((V, 6), dtype=torch.float32).pin_memory()
        h_bvol = torch.empty(g.vol_shape, dtype=torch.float32).pin_memory()
        h_bgrad = torch.empty((V, 6), dtype=torch.float32).pin_memory()

        def e2e_step():
            t0 = time.perf_counter()
            dfp.forward_host(g, angles, poses, h_vol, out=h_proj)
            dfp.forward_pose_grad_host(g, angles, poses, h_vol, h_up, out=h_grad)
            t1 = time.perf_counter()
            dfp.backproject_host(g, angles, poses, h_proj, out=h_bvol)
            dfp.backproject_pose_grad_host(g, angles, poses, h_proj, h_bpup, out=h_bgrad)
            return t1 - t0, time.perf_counter() - t1

        for _ in range(2):
            e2e_step()
        barrier()
        tf = tb = 0.0
        for _ in range(K):
            a_, b_ = e2e_step()
            tf += a_
            tb += b_
        barrier()
        te = max_over_ranks(torch.tensor([tf, tb], dtype=torch.float64, device=dev))
        tf, tb = [float(x) for x in te.cpu()]
        nb = lambda t_: t_.numel() * t_.element_size()
        e2e = {"value": 2.0 * job_ray_steps * K / tf / 1e9, "unit": UNIT,
               "h2d_bytes_per_step": 2 * nb(h_vol) + nb(h_up) + 2 * nb(h_proj) + nb(h_bpup),
               "d2h_bytes_per_step": nb(h_proj) + nb(h_grad) + nb(h_bvol) + nb(h_bgrad),
               "backproject_gvoxel_views_per_s": 2.0 * job_voxel_views * K / tb / 1e9,
               "api": "dfp_*_host (pinned host buffers; cudaMallocAsync + H2D + kernels + D2H + sync per call)"}

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---------------------------------------------------------------- roofline of the dominant kernel
    pk, pk_kind = peaks()
    mean_ms = {k: float(np.mean(v)) for k, v in kern_ms.items()}
    dom = max(mean_ms, key=mean_ms.get)
    units = {"fwd_project": ray_steps, "fwd_grad": ray_steps, "bp": voxel_views, "bp_grad": voxel_views}
    alu_peak = N_SM * LANES_PER_SM * pk.get("sm_max_mhz", 1965.0) * 1e6 / 1e12          # Tera lane-ops/s
    achieved = OPS_PER_UNIT[dom] * units[dom] / (mean_ms[dom] * 1e-3) / 1e12
    traffic = None
    tp = os.path.join(ROOT, "profiles", "traffic.csv")     # dram__bytes_read+write per launch from the ncu --set full capture
    if os.path.exists(tp):
        import csv
        for row in csv.DictReader(open(tp)):
            if row["config"] == f"C{args.config}" and row["kernel"] == dom:
                traffic = int(row["dram_bytes_per_launch"])
    roofline = {"bound": "alu", "kernel": dom, "achieved": achieved, "peak": alu_peak, "unit": "Tlane-op/s",
                "frac": achieved / alu_peak, "traffic": traffic,
                "peak_source": f"148 SMs x 128 fp32 lanes x sm_max_mhz ({pk_kind} MEASURED_PEAKS.json clock)",
                "ops_per_unit": OPS_PER_UNIT[dom], "units_per_launch": units[dom], "kernel_ms": mean_ms,
                "kernel_share_of_step": {k: v * K / 1e3 / t_all for k, v in mean_ms.items()},
                "hbm_compulsory_frac": None, "lsu_floor_frac": None}
    # compulsory HBM bytes of the dominant kernel vs the measured copy peak (expected to be small)
    comp = {"fwd_project": vol.numel() * 16 + proj.numel() * 4, "fwd_grad": vol.numel() * 16 + up.numel() * 4,
            "bp": proj.numel() * 16 + bvol.numel() * 4, "bp_grad": proj.numel() * 16 + bvol.numel() * 4}[dom]
    roofline["hbm_compulsory_frac"] = comp / (mean_ms[dom] * 1e-3) / 1e9 / pk["hbm_gbs"]
    # the unit that binds the staged kernels: the LSU issues one warp-wide shared-memory load per
    # clock per SM; loads per unit x warp-units / (SMs x clock x time) = fraction of that floor
    lds = {"fwd_project": 8, "fwd_grad": 32, "bp": 4, "bp_grad": 12}[dom]
    roofline["lsu_floor_frac"] = lds * (units[dom] / 32.0) / (N_SM * pk.get("sm_max_mhz", 1965.0) * 1e6 *
                                                                mean_ms[dom] * 1e-3)

    # measured denominators (dfp_microbench, one resident wave each): sustained rate per clock per SM of the pipes the
    # kernels are bound by; "lsu_measured_frac" replaces the assumed one LDS per clock by the measured LDS rate
    per_clk_sm = 1.0 / (N_SM * pk.get("sm_max_mhz", 1965.0) * 1e6)
    mb = {name: dfp.microbench(kind) * per_clk_sm
          for name, kind in (("lds_warp_inst", dfp.MB_LDS), ("fadd_lane_ops", dfp.MB_FADD),
                             ("ffma_lane_ops", dfp.MB_FFMA), ("ffma2_lane_ops", dfp.MB_FFMA2))}
    roofline["measured_per_clk_per_sm"] = mb
    roofline["lsu_measured_frac"] = roofline["lsu_floor_frac"] / mb["lds_warp_inst"]
    roofline["alu_measured_frac"] = roofline["frac"] * 128.0 / max(mb["fadd_lane_ops"], mb["ffma_lane_ops"],
                                                                   mb["ffma2_lane_ops"])

    # ---------------------------------------------------------------- CPU baseline: the oracle on the host cores
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        # ~10-15 s of oracle work on 16 cores: 16 full views of the 64 (0.7 s per view, forward + gradient)
        n_s = min(16, V)
        val, sec, cores, txt = time_oracle(w, vol.cpu().numpy(), up[:n_s].cpu().numpy(), rows=g.nv)
        cpu = {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": txt, "seconds": sec}

    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": args.warmup,
           "ms_per_step": t_all / K * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "f32", "data": "synthetic",
           "config": {"workload": f"{w.name} (BASELINE.json configs[{args.config - 1}]): {g.nx}^3 volume, {V} views of "
                                  f"{g.nu}x{g.nv}, all four calls per step", "ray_steps_per_pass": int(job_ray_steps),
                      "voxel_views_per_pass": int(job_voxel_views), "l2": "256 MiB flush write between timed steps",
                      "parallelism": f"views sharded over {world} rank(s), {V} views per GPU, no data-path collective"},
           "extra": {"backproject+grad_gvoxel_views_per_s": bp_value,
                     "forward_gray_steps_per_s": job_ray_steps * K / t_call[0] / 1e9,
                     "forward_pose_grad_gray_steps_per_s": job_ray_steps * K / t_call[1] / 1e9,
                     "backproject_gvoxel_views_per_s": job_voxel_views * K / t_call[2] / 1e9,
                     "backproject_pose_grad_gvoxel_views_per_s":
                         job_voxel_views * K / t_call[3] / 1e9,
                     "ms_per_call": {"forward": float(seg[:, 0].mean()), "forward_pose_grad": float(seg[:, 1].mean()),
                                     "backproject": float(seg[:, 2].mean()),
                                     "backproject_pose_grad": float(seg[:, 3].mean())},
                     "grad_interp_mode_ms_per_call": {"forward_pose_grad": interp_ms[0],
                                                      "backproject_pose_grad": interp_ms[1]},
                     "siddon_mode_ms_per_call": {"forward": model_ms["siddon"][0],
                                                 "forward_pose_grad": model_ms["siddon"][1]},
                     "joseph_mode_ms_per_call": {"forward": model_ms["joseph"][0],
                                                 "forward_pose_grad": model_ms["joseph"][1]},
                     "view_frames_mode_ms_per_call": {"forward": frames_ms[0], "forward_pose_grad": frames_ms[1],
                                                      "backproject": frames_ms[2],
                                                      "backproject_pose_grad": frames_ms[3]},
                     "forward_fused_moments_ms_per_call": fused_ms,
                     "forward_fused_moments_gray_steps_per_s": 2.0 * ray_steps / (fused_ms * 1e-3) / 1e9},
           "clocks": clocks, "e2e": e2e, "gpu_launches": n_launch, "roofline": roofline, "cpu_baseline": cpu}
    print(json.dumps(out), flush=True)
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

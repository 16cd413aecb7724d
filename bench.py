#!/usr/bin/env python
"""bench.py -- fp64 projection throughput of the B200-native AFiD projection step.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C4] [--impl reference]

A "step" is one afid_project call (all six kernels) on one synthetic velocity field resident
in HBM.  N = 1 runs BASELINE.json's headline configuration C4 (1024 x 1536 x 1536, tanh grid);
N > 1 (under torchrun) runs N independent replicas, one per GPU ("replicas only": the path
does not shard without a transpose), value = total points / max-over-ranks time.
Prints ONE JSON line on rank 0.

--impl reference times the CPU oracle (oracle/, as it stands) on a bounded sample of the same
workload: it is a deliberately slow baseline, not a target.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "fp64 projection Mpoints/s at 1024x1536x1536; % of B200 HBM roofline"
UNIT = "Mpoints/s"
# algorithmic HBM bytes per grid point of each kernel: fp64, complex = 16 B per 2 points
ALG_BYTES_PER_POINT = {"k_div_r2c": 32.0, "k_fft_y": 16.0, "k_solve_x": 16.0, "k_ifft_y": 16.0, "k_c2r_z": 16.0,
                       "k_correct": 56.0,
                       # plane-pipelined sweeps (afid_plan_set_pipeline): the intermediates B, D (and the re-read of p)
                       # stay in L2, so a sweep's algorithmic HBM bytes are its end-to-end streams only
                       "sweep_forward": 32.0, "sweep_inverse": 64.0}
PATH_ALG_BYTES_PER_POINT = 96.0   # strict minimum of the whole path
NOMINAL_HBM_GBS = 8000.0          # BASELINE.json north_star: "about 8 TB/s"


def rank_info():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def is_printing_rank():
    return rank_info()[0] == 0


def aggregate_over_ranks(ms, points, device="cuda"):
    """(max over ranks of ms, sum over ranks of points); identity when not distributed."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(ms), int(points)
    t = torch.tensor([float(ms)], dtype=torch.float64, device=device)
    n = torch.tensor([int(points)], dtype=torch.int64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(n, op=dist.ReduceOp.SUM)
    return float(t.item()), int(n.item())


def make_line(config, n_gpus, steps, warmup, ms_total, points_per_step, **extra):
    ms_per_step = ms_total / steps
    line = {"metric": METRIC, "value": points_per_step / (ms_per_step * 1e-3) / 1e6, "unit": UNIT, "n_gpus": n_gpus,
            "steps": steps, "warmup": warmup, "ms_per_step": ms_per_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": config}
    line.update(extra)
    return line


def measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (of measured)"
    except Exception:
        return 6650.0, "B200_PROFILING.md fallback 6.65 TB/s (of fallback)"


def built_kernel_names():
    """Mangled names of the kernels in the built library (cuobjdump), or None if they cannot be listed."""
    lib = os.path.join(ROOT, "paper_1705_01423_b200", "libafid_b200.so")
    try:
        out = subprocess.run(["cuobjdump", "--dump-resource-usage", lib], capture_output=True, text=True, timeout=60).stdout
    except Exception:
        return None
    names = {ln.split("Function", 1)[1].strip().rstrip(":") for ln in out.splitlines() if ln.strip().startswith("Function")}
    return names or None


def ncu_traffic(kernel, ny, nz, nx, points):
    """DRAM bytes per launch of `kernel` on this workload, scaled from the committed ncu capture
    (profiles/r2_dram_traffic.csv: bytes per point on a slab with the same cross-section), or None when there is
    no capture of that shape or the captured kernel (by mangled name) is no longer the one in the built library."""
    path = os.path.join(ROOT, "profiles", "r2_dram_traffic.csv")
    try:
        with open(path) as f:
            rows = [ln.strip().split(",") for ln in f if ln.strip()]
    except Exception:
        return None, None
    hdr = rows[0]
    for r in rows[1:]:
        d = dict(zip(hdr, r))
        if d["kernel"] != kernel:
            continue
        sx, sy, sz = (int(x) for x in d["shape"].split("x"))
        same = (sx == nx and sy == ny) if kernel == "k_solve_x" else (sy == ny and sz == nz)
        if not same:
            return None, "no capture of this shape"
        names = built_kernel_names()
        if names is None or d["mangled_name"] not in names:
            return None, "captured kernel is not in the built library any more (or cuobjdump unavailable)"
        return float(d["bytes_per_point"]) * points, f"profiles/r2_dram_traffic.csv (ncu at commit {d['commit']}, {d['shape']} slab, scaled by points)"
    return None, None


def git_sha():
    try:
        return subprocess.run(["git", "-C", ROOT, "rev-parse", "--short", "HEAD"], capture_output=True, text=True, timeout=10).stdout.strip() or None
    except Exception:
        return None


class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons of one GPU during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.rows.append(ln.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for k, nm in enumerate(names):
                if f[3 + k].lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def run_gpu(args):
    import torch
    import paper_1705_01423_b200 as afid
    from paper_1705_01423_b200 import synth

    rank, local_rank, world = rank_info()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    cfg = synth.config(args.workload)
    if args.shape:   # a slab / another shape with the workload's grid law and field recipe (profiling under ncu)
        sx, sy, sz = (int(x) for x in args.shape.split(","))
        cfg = synth.config(args.workload, nx=sx, ny=sy, nz=sz)
    nx, ny, nz = cfg["nx"], cfg["ny"], cfg["nz"]
    N = nx * ny * nz
    xc = synth.grid_faces(cfg)
    plan = afid.Plan(nx, ny, nz, xc, cfg["Ly"], cfg["Lz"])
    if args.pipeline:
        pb, pr = (int(x) for x in args.pipeline.split(","))
        plan.set_pipeline(pb, pr)
    if args.hints is not None:
        plan.set_l2_hints(args.hints)
    u = torch.empty((nx + 1, ny, nz), dtype=torch.float64, device=dev)
    v = torch.empty((nx, ny, nz), dtype=torch.float64, device=dev)
    w = torch.empty_like(v)
    p = torch.empty_like(v)
    synth.velocity(cfg, xc, device=dev, out=(u, v, w))     # seeded synthetic field, generated on the device
    torch.cuda.synchronize()
    plan.enable_timing(True)
    stream = torch.cuda.current_stream()

    def barrier():
        if world > 1:
            torch.distributed.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        plan.project(u, v, w, p)
    barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    kt = {}
    e0.record(stream)
    for _ in range(args.steps):
        plan.project(u, v, w, p)
    e1.record(stream)
    barrier()
    ms_local = e0.elapsed_time(e1)
    clocks = sampler.stop()
    # per-kernel durations (CUDA events recorded by the library on the same stream; the last
    # step's are read here, then averaged over a few more steps outside the timed region)
    acc = {}
    reps = max(1, min(args.steps, 3))
    for k, t in plan.kernel_times().items():
        acc[k] = t
    for _ in range(reps - 1):
        plan.project(u, v, w, p)
        for k, t in plan.kernel_times().items():
            acc[k] += t
    kt = {k: t / reps for k, t in acc.items()}
    ms_total, pts = aggregate_over_ranks(ms_local, N, device=dev)

    # end to end through the C ABI with HOST buffers: H2D of u,v,w, project, D2H of u,v,w,p per step
    e2e = None
    if not args.no_e2e:
        try:
            hu = torch.empty(u.shape, dtype=torch.float64, pin_memory=True)
            hv = torch.empty(v.shape, dtype=torch.float64, pin_memory=True)
            hw = torch.empty(v.shape, dtype=torch.float64, pin_memory=True)
            hp = torch.empty(v.shape, dtype=torch.float64, pin_memory=True)
            synth.velocity(cfg, xc, device=dev, out=(u, v, w))
            hu.copy_(u); hv.copy_(v); hw.copy_(w)
            torch.cuda.synchronize()
            es = max(1, args.e2e_steps)
            barrier()
            a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a0.record(stream)
            for _ in range(es):
                u.copy_(hu, non_blocking=True); v.copy_(hv, non_blocking=True); w.copy_(hw, non_blocking=True)
                plan.project(u, v, w, p)
                hu.copy_(u, non_blocking=True); hv.copy_(v, non_blocking=True); hw.copy_(w, non_blocking=True)
                hp.copy_(p, non_blocking=True)
            a1.record(stream)
            barrier()
            ms_e, pts_e = aggregate_over_ranks(a0.elapsed_time(a1), N, device=dev)
            bi = (u.numel() + v.numel() + w.numel()) * 8
            bo = bi + p.numel() * 8
            e2e = {"value": pts_e / (ms_e / es * 1e-3) / 1e6, "unit": UNIT, "steps": es, "ms_per_step": ms_e / es,
                   "h2d_bytes_per_step": bi, "d2h_bytes_per_step": bo, "host_memory": "pinned"}
            del hu, hv, hw, hp
        except Exception as ex:  # pinned allocation can fail on small hosts
            e2e = {"value": None, "unit": UNIT, "error": str(ex)[:200]}

    peak, peak_src = measured_peaks()
    # SURVEY.md 8(f) rows, timed outside the step: afid_max_cfl (24 B/pt) and afid_xsolve_apply (16 B/pt)
    extras = {}
    try:
        if args.no_extras:
            raise RuntimeError("skipped (--no-extras)")

        def timed(fn, reps=5):
            for _ in range(2):
                fn()
            t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            t0.record(stream)
            for _ in range(reps):
                fn()
            t1.record(stream)
            torch.cuda.synchronize()
            return t0.elapsed_time(t1) / reps
        out = torch.empty(1, dtype=torch.float64, device=dev)
        ms_cfl = timed(lambda: plan.max_cfl(u, v, w, out))
        ms_pcfl = timed(lambda: plan.project_cfl(u, v, w, p, out), reps=3) if args.fused_cfl else None
        dxs = np.diff(xc)
        xs = plan.xsolve(np.r_[0.0, 1.0 / dxs[1:] ** 2], np.r_[1.0 / dxs[:-1] ** 2, 0.0], np.full(nx, 1.0e3))
        ms_xs = timed(lambda: xs.apply(p))
        xs.destroy()
        extras = {"afid_project_cfl": ({"ms": ms_pcfl, "ms_over_afid_project": ms_pcfl - ms_local / args.steps} if ms_pcfl else "not timed (--fused-cfl)"),
                  "afid_max_cfl": {"ms": ms_cfl, "alg_GBps": 24.0 * N / (ms_cfl * 1e-3) / 1e9, "frac_of_peak": 24.0 * N / (ms_cfl * 1e-3) / 1e9 / peak},
                  "afid_xsolve_apply": {"ms": ms_xs, "alg_GBps": 16.0 * N / (ms_xs * 1e-3) / 1e9, "frac_of_peak": 16.0 * N / (ms_xs * 1e-3) / 1e9 / peak}}
    except Exception as ex:
        extras = {"error": str(ex)[:200]}
    dom = max(kt, key=kt.get)
    ach = ALG_BYTES_PER_POINT[dom] * N / (kt[dom] * 1e-3) / 1e9
    traffic, traffic_src = ncu_traffic(dom, ny, nz, nx, N)
    roofline = {"bound": "hbm", "kernel": dom, "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                "traffic": traffic, "traffic_source": traffic_src, "peak_source": peak_src,
                "alg_bytes_per_launch": ALG_BYTES_PER_POINT[dom] * N, "kernel_ms": kt[dom]}
    ms_step = ms_total / args.steps
    path_gbs = PATH_ALG_BYTES_PER_POINT * N / (ms_local / args.steps * 1e-3) / 1e9
    kernels = {k: {"ms": t, "alg_GBps": ALG_BYTES_PER_POINT[k] * N / (t * 1e-3) / 1e9,
                   "frac_of_peak": ALG_BYTES_PER_POINT[k] * N / (t * 1e-3) / 1e9 / peak} for k, t in kt.items()}
    config = {"workload": f"{args.workload}{' (--shape)' if args.shape else ''}: {nx}x{ny}x{nz} {cfg['grid']}-clustered x grid, Ly={cfg['Ly']:.6g}, "
                          f"Lz={cfg['Lz']:.6g}, seeded random-mode velocity (synth.py)",
              "points_per_step_per_gpu": N, "parallelism": "replicas only" if world > 1 else "1 gpu",
              "l2": "working set (>= 77 GB) far larger than the 126 MB L2; no flush needed",
              "device_bytes": plan.workspace_bytes + (4 * N + ny * nz) * 8, "git_sha": git_sha()}
    line = make_line(config, world, args.steps, args.warmup, ms_total, pts, clocks=clocks, e2e=e2e,
                     gpu_launches=plan.num_launches * args.steps, roofline=roofline, kernels=kernels, extras=extras,
                     path_roofline={"alg_bytes_per_point": PATH_ALG_BYTES_PER_POINT, "achieved_GBps": path_gbs,
                                    "frac_of_nominal_8TBs": path_gbs / NOMINAL_HBM_GBS, "frac_of_measured": path_gbs / peak})
    if rank == 0 and not args.no_cpu_baseline and world == 1:
        line["cpu_baseline"] = cpu_baseline(args.workload)
        try:
            line["cpu_baseline_fft"] = cpu_baseline_fft(args.workload)
        except Exception as ex:
            line["cpu_baseline_fft"] = {"value": None, "error": str(ex)[:200]}
    elif rank == 0:
        line["cpu_baseline"] = None
    plan.destroy()
    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        torch.distributed.destroy_process_group()


# ------------------------------------------------------------------------------------------
# CPU oracle legs
# ------------------------------------------------------------------------------------------
def oracle_sample(workload):
    """The bounded sample: a slab of nx=2 cells with the workload's full y-z cross-section (the
    per-point cost of the oracle's naive DFT, O(ny+nz), is that of the full workload)."""
    from paper_1705_01423_b200 import synth
    cfg = synth.config(workload, nx=2)
    xc = synth.grid_faces(synth.config(workload))[:3].copy()
    u, v, w = synth.velocity(cfg, xc)
    desc = f"{workload} cross-section slab: nx=2 x ny={cfg['ny']} x nz={cfg['nz']} (first two cells of the x grid)"
    return cfg, xc, u.numpy(), v.numpy(), w.numpy(), desc


def time_oracle(cfg, xc, u, v, w):
    from oracle import ref
    t0 = time.perf_counter()
    ref.project(xc, cfg["Ly"], cfg["Lz"], u, v, w)
    return time.perf_counter() - t0


def cpu_baseline(workload):
    from oracle import ref
    cfg, xc, u, v, w, desc = oracle_sample(workload)
    dt = time_oracle(cfg, xc, u, v, w)
    n = cfg["nx"] * cfg["ny"] * cfg["nz"]
    return {"value": n / dt / 1e6, "unit": UNIT, "cores": ref.num_threads(), "kind": "oracle",
            "sample": desc + f"; one oracle projection, {dt:.1f} s"}


def cpu_baseline_fft(workload):
    """The FFT form of the oracle (oracle/ref_fft.py: scipy.fft for the two DFTs, the C oracle's long-double Thomas,
    divergence and correction) on a 32-plane slab of the workload's cross-section: the per-point cost of this form
    does not depend on nx.  Reported next to cpu_baseline so that the line also has a CPU number for the
    O(n log n) algorithm the paper's CPU code runs; it is a context figure, not a target."""
    from oracle import ref, ref_fft
    from paper_1705_01423_b200 import synth
    full = synth.config(workload)
    nxs = min(32, full["nx"])
    cfg = synth.config(workload, nx=nxs)
    xc = synth.grid_faces(full)[:nxs + 1].copy()
    u, v, w = (t.numpy() for t in synth.velocity(cfg, xc))
    t0 = time.perf_counter()
    ref_fft.project_fft(xc, cfg["Ly"], cfg["Lz"], u, v, w)
    dt = time.perf_counter() - t0
    n = cfg["nx"] * cfg["ny"] * cfg["nz"]
    return {"value": n / dt / 1e6, "unit": UNIT, "cores": ref.num_threads(), "kind": "oracle, FFT form (scipy.fft + long-double Thomas)",
            "sample": f"{workload} cross-section slab: nx={nxs} x ny={cfg['ny']} x nz={cfg['nz']} (first {nxs} cells of the x grid); "
                      f"one projection, {dt:.1f} s"}


def run_reference(args):
    rank, _, world = rank_info()
    if rank != 0:
        return
    from oracle import ref
    from paper_1705_01423_b200 import synth
    cfg, xc, u, v, w, desc = oracle_sample(args.workload)
    n = cfg["nx"] * cfg["ny"] * cfg["nz"]
    for _ in range(args.warmup):
        time_oracle(cfg, xc, u, v, w)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        time_oracle(cfg, xc, u, v, w)
    ms_total = (time.perf_counter() - t0) * 1e3
    full = synth.config(args.workload)
    config = {"workload": f"{args.workload}: {full['nx']}x{full['ny']}x{full['nz']} (each step = bounded sample: {desc})"}
    line = make_line(config, world, args.steps, args.warmup, ms_total, n, impl="reference")
    line["gpu_launches"] = 0
    line["cpu_baseline"] = {"value": line["value"], "unit": UNIT, "cores": ref.num_threads(), "kind": "oracle", "sample": desc}
    line["e2e"] = {"value": line["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    print(json.dumps(line), flush=True)


def maybe_spawn_ranks(args):
    """`python bench.py --gpus N` with N > 1 and no torchrun environment: launch the N ranks ourselves (the same
    command the driver uses: torch.distributed.run, one process per GPU, rendezvous on 127.0.0.1) and exit with
    their status.  Under torchrun (WORLD_SIZE set) the world size must equal --gpus."""
    if args.gpus < 1:
        raise SystemExit("bench.py: --gpus must be >= 1")
    world_env = os.environ.get("WORLD_SIZE")
    if world_env is not None:
        if int(world_env) != args.gpus:
            raise SystemExit(f"bench.py: --gpus {args.gpus} but the launcher started WORLD_SIZE={world_env} ranks")
        return
    if args.gpus == 1:
        return
    if args.impl == "b200":
        import torch
        have = torch.cuda.device_count() if torch.cuda.is_available() else 0
        if have < args.gpus:
            raise SystemExit(f"bench.py: --gpus {args.gpus} requested but only {have} CUDA device(s) are visible "
                             "(one rank per GPU; there is no CPU fallback)")
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    raise SystemExit(subprocess.call(cmd))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=None)
    ap.add_argument("--workload", default="C4", choices=["C1", "C2", "C3", "C4", "C5"])
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--shape", default=None, help="nx,ny,nz: time this shape with the workload's grid law and field recipe "
                                                  "(slabs for ncu captures; the headline is the unmodified workload)")
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--pipeline", default=None, help="planes_per_batch,rotation (afid_plan_set_pipeline)")
    ap.add_argument("--hints", type=int, default=None, help="L2 hint mask (afid_plan_set_l2_hints)")
    ap.add_argument("--no-extras", action="store_true")
    ap.add_argument("--fused-cfl", action="store_true", help="also time afid_project_cfl (SURVEY.md 8(f3), fused form) in the extras")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    maybe_spawn_ranks(args)
    if args.impl == "reference":
        args.steps = 2 if args.steps is None else args.steps
        args.warmup = 1 if args.warmup is None else args.warmup
        run_reference(args)
    else:
        args.steps = 10 if args.steps is None else args.steps
        args.warmup = 3 if args.warmup is None else max(3, args.warmup)
        run_gpu(args)


if __name__ == "__main__":
    main()

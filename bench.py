#!/usr/bin/env python
"""bench.py -- throughput of the fused pseudo-transient (PT) elasticity iteration of libdr on B200.

Metric (BASELINE.json): PT voxel-updates/s, T_eff = 160 B x N x iterations / time against the measured HBM
peak, and (with --time-to-solution) the time to the full 6x6 C_eff.

A "step" is one PT iteration of the whole hot path as dr_solve runs it: the fused stress+velocity kernel
(SURVEY 8(a) a2+a3) every step, the residual max-norm (a5) every `ncheck`-th step, and -- once per timed call --
the initial/boundary fields (a4) and the volume averages -> C column (a6).  The timed region is ONE
dr_solve(lc, eps0, tol=1e-300, maxiter=K) call, i.e. exactly K steps.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg4|cfg2|cfg1|cfg5] [--kernel 3|0|1|2|4] [--time-to-solution]
    python bench.py --impl reference ...      # the CPU oracle on the host cores (bounded sample)

N > 1 (torchrun): the path shards over independent load cases -- rank r solves load case r mod 6 of the same
image on its own GPU, no data-path collective ("scaling": "weak").
"""
from __future__ import annotations

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

from paper_2410_20441_b200 import inputs, shard  # noqa: E402
from paper_2410_20441_b200 import build as drbuild  # noqa: E402

BYTES_PER_VOXEL_ITER = 160.0        # (2*9 + 2) fp64, SURVEY 8(d)
KERNEL_NAMES = {0: "k_pt_tma", 1: "k_stress_split+k_velocity_split", 2: "k_pt_fused", 3: "k_pt_tb2<.,2> (two iterations per sweep)",
                4: "k_pt_tb2<.,1>"}
KERNEL_DESC = {0: "fused+TMA", 1: "split", 2: "fused+LDG", 3: "fused+TMA, stencil codes, 2 iterations per sweep", 4: "fused+TMA, stencil codes"}


def ncu_traffic(workload, kernel, palette, form):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the `ncu --set full` captures
    listed in profiles/traffic.csv -- only a row taken with the CURRENT kernel sources (build.source_hash) counts; a capture of
    older kernels says nothing about this binary, so the answer is then null."""
    path = os.path.join(ROOT, "profiles", "traffic.csv")
    try:
        cur = drbuild.source_hash()
        with open(path) as fh:
            for line in fh:
                t = [x.strip() for x in line.split(",")]
                if len(t) < 8 or t[0].startswith("#") or t[0] == "source_hash":
                    continue
                if t[0] == cur and t[1] == workload and int(t[2]) == kernel and int(t[3]) == palette and int(t[4]) == form:
                    return float(t[5]) + float(t[6])
    except Exception:
        pass
    return None


WORKLOADS = {
    "cfg1": dict(n=32, gen="config1_sphere", desc="32^3 centred spherical pore r=5, contrast 1e-6"),
    "cfg2": dict(n=191, gen="config2_spheroid", desc="191^3 oblate fluid spheroid (40,40,8)"),
    "cfg3": dict(n=191, gen="config3_random_spheres", desc="191^3 200 random spherical pores, contrast 1e-6"),
    "cfg4": dict(n=479, gen="config4_grf", desc="479^3 thresholded Gaussian random field, 15% soft phase"),
    "cfg5": dict(n=703, gen="config5_penny_cracks", desc="703^3 400 penny cracks, contrast 1e-6"),
}


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as fh:
            return float(json.load(fh)["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (measured copy rate)"
    except Exception:
        return 6650.0, "fallback 6.65 TB/s (B200_PROFILING.md; MEASURED_PEAKS.json absent)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows = []
        self.proc = None
        self.index = index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            t = [x.strip() for x in r.split(",")]
            if len(t) < 7:
                continue
            try:
                sm.append(float(t[0])); mx.append(float(t[1]))
            except ValueError:
                continue
            for nme, v in zip(names, t[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nme)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def make_image(workload, n_override=None, with_mask=False):
    w = WORKLOADS[workload]
    n = n_override or w["n"]
    K, G, m = getattr(inputs, w["gen"])(n=n)
    return (K, G, n, m) if with_mask else (K, G, n)


STOP_NAMES = ("none", "residual", "stagnation", "maxiter")
# cfg 4 whole solve to tol 1e-8, default parameters: iterations per load case measured in round 2 with this kernel
# (`bench.py --workload cfg4 --time-to-solution`: 133.4 s) -- used for a PROJECTION only
CFG4_ITERS_R2 = (9500, 9500, 10000, 7200, 7800, 7500)


def time_to_full_C_cfg2(torch, binding, dev, stream, eps0, tol, ncheck):
    """BASELINE.json's third metric ("time to full 6x6 C_eff") inside the default, driver-run line: cfg 2 (191^3) from
    dr_create to the 6x6 read-back with all six load cases in every launch (dr_solve_all), solved to `tol`; second of two
    calls (the first warms up).  Every DR_OK carries the rule that produced it (dr_info_lc: residual or stagnation)."""
    K2, G2, n2 = make_image("cfg2")
    Kd2, Gd2 = torch.from_numpy(K2).to(dev), torch.from_numpy(G2).to(dev)
    ws6 = torch.empty(binding.workspace_bytes(n2, n2, n2, True), dtype=torch.uint8, device=dev)
    for rep in range(2):
        torch.cuda.synchronize(dev)
        t0 = time.perf_counter()
        b = binding.Solver(Kd2, Gd2, stream=stream, workspace=ws6, six=True, ncheck=ncheck)
        C2, log2 = b.solve_all_batched(eps0, tol, 100 * n2)
        torch.cuda.synchronize(dev)
        dt = time.perf_counter() - t0
        kern = b.active_kernel()
        b.close()
    return {"workload": "cfg2: " + WORKLOADS["cfg2"]["desc"], "seconds_incl_create": dt, "tol": tol, "ncheck": ncheck,
            "driver": "dr_create + dr_solve_all (six load cases per launch) + dr_effective_C", "kernel": KERNEL_NAMES[kern],
            "iters": [l[1] for l in log2], "status": [l[0] for l in log2], "residual": [l[2] for l in log2],
            "stop": [STOP_NAMES[l[3]] for l in log2],
            "C": [[float("%.6f" % v) for v in row] for row in C2]}


def crop(K, G, m):
    m = min(m, K.shape[0])
    return np.ascontiguousarray(K[:m, :m, :m]), np.ascontiguousarray(G[:m, :m, :m]), m


def oracle_rate(K, G, lc, eps0, sample_n, iters):
    """time the oracle as it stands on the host cores: `iters` PT iterations on a sample_n^3 crop"""
    from oracle import dro
    Kc, Gc, m = crop(K, G, sample_n)
    o = dro.Oracle(Kc, Gc)
    o.step(lc, eps0, 1)
    t0 = time.perf_counter()
    o.iterate(lc, eps0, iters)
    dt = time.perf_counter() - t0
    return m ** 3 * iters / dt, dt, m


def host_threads():
    try:
        return int(os.environ.get("OMP_NUM_THREADS", "")) if os.environ.get("OMP_NUM_THREADS") else len(os.sched_getaffinity(0))
    except Exception:
        return os.cpu_count() or 1


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    if args.cpu_threads > 0:
        os.environ["OMP_NUM_THREADS"] = str(args.cpu_threads)      # before libdro.so (and its OpenMP runtime) is loaded
    K, G, n = make_image(args.workload, args.n)
    sample_n = min(n, args.cpu_sample_n)
    from oracle import dro
    Kc, Gc, m = crop(K, G, sample_n)
    o = dro.Oracle(Kc, Gc)
    o.step(args.lc, args.eps0, 0)
    per = max(1, args.cpu_iters_per_step)
    for _ in range(args.warmup):
        o.iterate(args.lc, args.eps0, per)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        o.iterate(args.lc, args.eps0, per)
    dt = time.perf_counter() - t0
    rate = m ** 3 * per * args.steps / dt
    sample = "%d^3 crop of %s, %d oracle PT iterations per step" % (m, args.workload, per)
    line = {
        "impl": "reference", "metric": "pt_voxel_updates_per_s", "value": rate, "unit": "voxel-updates/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "%s: %s" % (args.workload, WORKLOADS[args.workload]["desc"]), "load_case": args.lc},
        "cpu_baseline": {"value": rate, "unit": "voxel-updates/s", "cores": host_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": rate, "unit": "voxel-updates/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    if args.time_to_solution:
        # the oracle's own time to the full 6x6 tensor (all six load cases to `tol`), same crop
        o2 = dro.Oracle(Kc, Gc, ncheck=args.ncheck)
        t0 = time.perf_counter()
        Cc, log = o2.solve_all(args.eps0, args.tol, 100 * m)
        line["time_to_full_C"] = {"seconds": time.perf_counter() - t0, "tol": args.tol, "grid": [m, m, m],
                                  "iters": [l[1] for l in log], "status": [l[0] for l in log],
                                  "C": [[float("%.6f" % v) for v in row] for row in Cc]}
    print(json.dumps(line))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="libdr", choices=["libdr", "reference"])
    ap.add_argument("--workload", default="cfg4", choices=sorted(WORKLOADS))
    ap.add_argument("--n", type=int, default=None, help="override the grid size of the workload (debug)")
    ap.add_argument("--lc", type=int, default=2)
    ap.add_argument("--eps0", type=float, default=1e-4)
    ap.add_argument("--ncheck", type=int, default=100)
    ap.add_argument("--kernel", type=int, default=3, help="3 two PT iterations per sweep on stencil-coded images (default; falls back to 0), 0 fused with TMA staging, 1 split baseline, 2 fused with LDG prefetch, 4 coded one-iteration sweep")
    ap.add_argument("--sustained-seconds", type=float, default=3.0, help="length of the back-to-back dr_iterate run behind the `sustained` block (0 = skip)")
    ap.add_argument("--form", type=int, default=0, help="0 stress-relaxation form of the paper (default, 160 B/voxel), 1 displacement form (112 B/voxel)")
    ap.add_argument("--palette", type=int, default=1, help="1 (default): uint8 phase ids + table when the image has <= 256 distinct (K,G); 0: fp64 modulus fields")
    ap.add_argument("--cpu-sample-n", type=int, default=191)
    ap.add_argument("--cpu-iters", type=int, default=600, help="oracle PT iterations of the cpu_baseline sample (~13 s on 16 cores at 191^3)")
    ap.add_argument("--cpu-iters-per-step", type=int, default=5)
    ap.add_argument("--cpu-threads", type=int, default=0, help="--impl reference: OMP_NUM_THREADS of the oracle (0 = all host cores)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--e2e-iters", type=int, default=50, help="PT iterations per load case in the host-buffer e2e call")
    ap.add_argument("--time-to-solution", action="store_true", help="also solve all six load cases to tol 1e-8")
    ap.add_argument("--tol", type=float, default=1e-8)
    ap.add_argument("--direct-offdiag", action="store_true", help="time-to-solution: also run the 7th (triaxial) test and report Eq. 27-29")
    ap.add_argument("--st-factor", type=float, default=1.0, help="DR_ST_FACTOR (non-default tuning: 0.7 needs ~35 %% fewer iterations at 479^3)")
    ap.add_argument("--void-rel", type=float, default=0.0, help="DR_VOID_REL (non-default: exact-void clamp of near-void cells)")
    ap.add_argument("--no-cfg2-tts", action="store_true", help="skip the cfg 2 time-to-full-6x6 block of the default line (~5 s)")
    ap.add_argument("--tts-maxiter-n", type=int, default=100, help="time-to-solution: maxiter = this x n per load case")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)

    if args.impl == "reference":
        return run_reference(args)

    import torch
    from paper_2410_20441_b200 import binding

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libdr has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    K, G, n, mask = make_image(args.workload, args.n, with_mask=True)
    mask = np.asarray(mask, dtype=bool) if mask is not None and np.shape(mask) == K.shape else None
    N = n ** 3
    Kd = torch.from_numpy(K).to(dev)
    Gd = torch.from_numpy(G).to(dev)
    lc = shard.load_case_of_rank(rank, world, args.lc)
    stream = torch.cuda.Stream(device=dev)
    with torch.cuda.stream(stream):
        # stag_tol 0: the timed dr_solve must run exactly K steps (the stagnation rule could end it early)
        extra = {}
        if args.st_factor != 1.0:
            extra["st_factor"] = args.st_factor
        if args.void_rel != 0.0:
            extra["void_rel"] = args.void_rel
        s = binding.Solver(Kd, Gd, stream=stream, ncheck=args.ncheck, kernel=args.kernel, form=args.form, palette=args.palette, stag_tol=0.0, **extra)

        def barrier():
            torch.cuda.synchronize(dev)
            if dist is not None:
                dist.barrier()
            torch.cuda.synchronize(dev)

        # ---- warm-up, then the timed call: exactly K steps of the whole hot path
        s.solve(lc, args.eps0, 1e-300, args.warmup)
        barrier()
        sampler = ClockSampler(local)
        if rank == 0:
            sampler.start()
        l0 = s.launch_count()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        s.solve(lc, args.eps0, 1e-300, args.steps)
        e1.record(stream)
        barrier()
        launches = s.launch_count() - l0
        pal_active = s.uses_palette()
        ms = e0.elapsed_time(e1)
        # ---- dominant kernel alone (k_pt_fused back to back, no residual): average launch duration
        # an EVEN count, so that with two iterations per sweep every launch in the window is a pair (an odd count would mix a
        # single-iteration launch in); the launch duration is the window divided by the launches the library counted
        nk = args.steps + (args.steps & 1)
        s.iterate(lc, args.eps0, 6)
        lk0 = s.launch_count()
        k0, k1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        k0.record(stream)
        s.iterate(lc, args.eps0, nk)
        k1.record(stream)
        torch.cuda.synchronize(dev)
        klaunches = max(int(s.launch_count() - lk0), 1)
        kms = k0.elapsed_time(k1) / nk
        launch_ms = k0.elapsed_time(k1) / klaunches
        clocks = sampler.stop() if rank == 0 else None
        active_kernel = s.active_kernel()
        # ---- sustained: what a real solve gets.  >= 3 s of back-to-back PT iterations (no residual check, no host sync) with
        # its own clock record: under the 1 kW cap the SM clock settles below what a 0.1 s burst sees.
        sustained = None
        if args.sustained_seconds > 0 and rank == 0:
            n_sus = max(2 * int(args.sustained_seconds / (kms * 1e-3) / 2 + 1), 2)
            smp2 = ClockSampler(local)
            smp2.start()
            q0, q1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            q0.record(stream)
            s.iterate(lc, args.eps0, n_sus)
            q1.record(stream)
            torch.cuda.synchronize(dev)
            sus_ms = q0.elapsed_time(q1) / n_sus
            sustained = {"iterations": n_sus, "seconds": sus_ms * n_sus * 1e-3, "ms_per_step": sus_ms, "clocks": smp2.stop()}
        if dist is not None:
            ms = shard.max_over_ranks(ms, dist, dev)
            kms = shard.max_over_ranks(kms, dist, dev)
            launch_ms = shard.max_over_ranks(launch_ms, dist, dev)

        # ---- e2e through the C-ABI call with HOST buffers (H2D of K,G and D2H of C inside the timed region)
        # every rank runs the call on its own GPU (N independent images: weak scaling); time = max over ranks
        e2e = None
        if True:
            Kh = torch.from_numpy(K).pin_memory()
            Gh = torch.from_numpy(G).pin_memory()
            stage = torch.empty(2 * N, dtype=torch.float64, device=dev)
            binding.solve_image_host(Kh, Gh, tol=1e-300, maxiter=3, ncheck=args.ncheck, stage=stage, workspace=s.workspace)
            barrier()
            t0 = time.perf_counter()
            _, iters, _ = binding.solve_image_host(Kh, Gh, eps0=args.eps0, tol=1e-300, maxiter=args.e2e_iters,
                                                   ncheck=args.ncheck, stage=stage, workspace=s.workspace)
            torch.cuda.synchronize(dev)
            dt = time.perf_counter() - t0
            dt = shard.max_over_ranks(dt * 1e3, dist, dev) * 1e-3
            nsteps = sum(iters)
            e2e = {"value": world * N * nsteps / dt, "unit": "voxel-updates/s",
                   "h2d_bytes_per_step": 2 * N * 8 / nsteps, "d2h_bytes_per_step": (36 * 8 + 6 * 8 * (args.e2e_iters // args.ncheck)) / nsteps,
                   "call": "dr_solve_image_host (library defaults, DR_KERNEL 3): H2D K,G + dr_create + 6 load cases x %d iterations + C read back" % args.e2e_iters,
                   "seconds": dt}
            # the same call for the image as a segmentation would deliver it: uint8 phase ids + per-phase tables
            # (dr_solve_image_host_segmented: 1 byte per voxel over PCIe instead of 16)
            if mask is not None:
                ph = np.ascontiguousarray(mask, dtype=np.uint8)
                Kt = np.array([K[~mask].flat[0] if (~mask).any() else 0.0, K[mask].flat[0] if mask.any() else 0.0])
                Gt = np.array([G[~mask].flat[0] if (~mask).any() else 0.0, G[mask].flat[0] if mask.any() else 0.0])
                if np.array_equal(Kt[ph], K) and np.array_equal(Gt[ph], G):
                    Ph = torch.from_numpy(ph).pin_memory()
                    stage8 = stage.view(torch.uint8)
                    binding.solve_image_host_segmented(Ph, Kt, Gt, tol=1e-300, maxiter=3, ncheck=args.ncheck, stage=stage8, workspace=s.workspace)
                    barrier()
                    t0 = time.perf_counter()
                    _, iters2, _ = binding.solve_image_host_segmented(Ph, Kt, Gt, eps0=args.eps0, tol=1e-300, maxiter=args.e2e_iters,
                                                                      ncheck=args.ncheck, stage=stage8, workspace=s.workspace)
                    torch.cuda.synchronize(dev)
                    dt2 = shard.max_over_ranks((time.perf_counter() - t0) * 1e3, dist, dev) * 1e-3
                    e2e["segmented"] = {"value": world * N * sum(iters2) / dt2, "unit": "voxel-updates/s", "seconds": dt2,
                                        "h2d_bytes_per_step": N / sum(iters2), "call": "dr_solve_image_host_segmented (uint8 phase ids + tables)"}
                    del Ph
            del stage, Kh, Gh
            # the solver's workspace was reused by the e2e call: rebuild the handle state
            s.close()
            s = binding.Solver(Kd, Gd, stream=stream, workspace=s.workspace, ncheck=args.ncheck, kernel=args.kernel, form=args.form, palette=args.palette, **extra)
        if dist is not None:
            dist.barrier()
            dist.destroy_process_group()
            dist = None
            if rank != 0:
                return 0

        tts = None
        if args.time_to_solution and rank == 0:
            torch.cuda.synchronize(dev)
            t0 = time.perf_counter()
            C, log = s.solve_all(args.eps0, args.tol, args.tts_maxiter_n * n)
            torch.cuda.synchronize(dev)
            tts = {"seconds": time.perf_counter() - t0, "tol": args.tol, "driver": "six dr_solve calls on one handle",
                   "params": dict(extra, form=args.form, kernel=args.kernel), "stop": [int(l[4]) for l in log] if len(log[0]) > 4 else None,
                   "iters": [l[1] for l in log], "status": [l[0] for l in log], "residual": [l[2] for l in log],
                   "C": [[float("%.6f" % v) for v in row] for row in C]}
            if args.direct_offdiag:
                # the paper's 7th direct test (App. A.3): load case 6 + Eq. 27-29 against the symmetrised columns of C
                st7 = s.solve(6, args.eps0, args.tol, args.tts_maxiter_n * n)
                d7 = s.offdiag_direct()
                sym = [0.5 * (C[0, 1] + C[1, 0]), 0.5 * (C[0, 2] + C[2, 0]), 0.5 * (C[1, 2] + C[2, 1])]
                tts["direct_offdiag"] = {"status": int(st7), "iters": s.info()[0], "C12_C13_C23": [float(v) for v in d7],
                                         "symmetrised_columns": [float(v) for v in sym],
                                         "max_abs_diff": float(max(abs(a - b) for a, b in zip(d7, sym)))}
            # the same six columns with all load cases in every launch (dr_solve_all) where six state
            # sets fit the device; timed from dr_create to the 6x6 read-back, second of two calls (the first warms up)
            need6 = binding.workspace_bytes(n, n, n, True)
            free_b, _ = torch.cuda.mem_get_info(dev)
            if need6 + (2 << 30) < free_b + s.workspace.numel():
                s.close()
                del s
                ws6 = torch.empty(need6, dtype=torch.uint8, device=dev)
                for rep in range(2):
                    torch.cuda.synchronize(dev)
                    t0 = time.perf_counter()
                    b = binding.Solver(Kd, Gd, stream=stream, workspace=ws6, six=True, ncheck=args.ncheck, kernel=args.kernel, form=args.form, palette=args.palette, **extra)
                    Cb, logb = b.solve_all_batched(args.eps0, args.tol, args.tts_maxiter_n * n)
                    torch.cuda.synchronize(dev)
                    dtb = time.perf_counter() - t0
                    b.close()
                tts["batched"] = {"seconds_incl_create": dtb, "driver": "dr_create + dr_solve_all (six load cases per launch)",
                                  "iters": [l[1] for l in logb], "status": [l[0] for l in logb],
                                  "max_abs_dC_vs_sequential": float(np.max(np.abs(Cb - C)))}

        cfg2_tts = None
        if rank == 0 and world == 1 and args.workload == "cfg4" and args.n is None and not args.no_cfg2_tts and not args.time_to_solution:
            cfg2_tts = time_to_full_C_cfg2(torch, binding, dev, stream, args.eps0, args.tol, args.ncheck)

    peak, peak_src = measured_peak()
    bpv = 112.0 if args.form == 1 else BYTES_PER_VOXEL_ITER      # algorithmic bytes per voxel-iteration of the form
    value = shard.job_throughput(N, args.steps, world, ms)
    teff = bpv * N * args.steps / (ms * 1e-3) / 1e9
    # one launch of the dominant kernel advances N voxels by `ipl` iterations: algorithmic bytes per launch = ipl x bpv x N
    # (counted, not assumed: iterations of the window / launches of the window)
    ipl = nk // klaunches
    assert ipl * klaunches == nk and ipl == (2 if active_kernel == 3 else 1), (nk, klaunches, active_kernel)
    kern_gbs = ipl * bpv * N / (launch_ms * 1e-3) / 1e9
    traffic = ncu_traffic(args.workload, active_kernel, int(pal_active), args.form) if args.n is None else None
    roof = {"bound": "hbm", "kernel": KERNEL_NAMES[active_kernel], "achieved": kern_gbs, "peak": peak, "unit": "GB/s", "frac": kern_gbs / peak,
            "algorithmic_frac": kern_gbs / peak, "launches_timed": klaunches, "iterations_timed": nk,
            "traffic": traffic, "peak_source": peak_src, "launch_ms": launch_ms, "iterations_per_launch": ipl,
            "algorithmic_bytes_per_launch": ipl * bpv * N,
            "note": "achieved = ALGORITHMIC bytes (160 B per voxel-iteration, SURVEY 8(d)) / launch time: with two iterations per sweep it "
                    "may exceed the DRAM rate (frac = algorithmic_frac > 1 is not a DRAM rate); physical_frac = ncu dram bytes / launch time / peak "
                    "is the figure bounded by 1"}
    if traffic is not None:
        roof["physical_GBs"] = traffic / (launch_ms * 1e-3) / 1e9
        roof["physical_frac"] = roof["physical_GBs"] / peak
        roof["traffic_source"] = "profiles/traffic.csv row for source hash %s" % drbuild.source_hash()
    line = {
        "metric": "pt_voxel_updates_per_s", "value": value, "unit": "voxel-updates/s",
        "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "%s: %s" % (args.workload, WORKLOADS[args.workload]["desc"]), "grid": [n, n, n],
                   "load_case": lc, "ncheck": args.ncheck, "form": "stress-relaxation (paper, 160 B/voxel-iteration)" if args.form == 0 else "displacement (112 B/voxel-iteration)",
                   "kernel": KERNEL_DESC[active_kernel], "kernel_requested": args.kernel,
                   "moduli": "uint8 phase ids + 256-entry table" if pal_active else "fp64 K, G fields",
                   "parallelism": "load cases sharded over %d GPU(s), no collective" % world,
                   "l2": ("inputs (%.1f GB per sweep) larger than L2; no flush needed" % (BYTES_PER_VOXEL_ITER * N / 1e9)) if BYTES_PER_VOXEL_ITER * N > 2 * 126e6
                         else "working set (%.1f MB per sweep) fits the 126 MB L2: an L2-resident, latency-bound case, not flushed (the graded workload is cfg4)" % (BYTES_PER_VOXEL_ITER * N / 1e6)},
        "T_eff_GBs": teff, "T_eff_frac_of_measured_peak": teff / peak, "T_eff_frac_of_8000_nominal": teff / 8000.0,
        "clocks": clocks,
        "e2e": e2e,
        "gpu_launches": int(launches),
        "roofline": roof,
    }
    if sustained is not None:
        sus_gbs = bpv * N / (sustained["ms_per_step"] * 1e-3) / 1e9
        sustained.update({"value": N / (sustained["ms_per_step"] * 1e-3), "unit": "voxel-updates/s", "T_eff_GBs": sus_gbs,
                          "frac": sus_gbs / peak, "what": "back-to-back dr_iterate, same handle and load case, no host synchronisation"})
        line["sustained"] = sustained
    if tts is not None:
        line["time_to_full_C"] = tts
    elif cfg2_tts is not None:
        line["time_to_full_C"] = cfg2_tts
        if sustained is not None and args.form == 0 and args.kernel == 3:
            line["cfg4_projection"] = {
                "label": "projected, not measured in this run",
                "seconds": sum(CFG4_ITERS_R2) * sustained["ms_per_step"] * 1e-3,
                "how": "sum of the iterations per load case of the round-2 whole solve of cfg 4 to tol 1e-8 (BASELINE.md section 5: "
                       "%s, measured 133.4 s) x this line's sustained ms_per_step" % (list(CFG4_ITERS_R2),)}
    if not args.no_cpu_baseline:
        rate, dt, m = oracle_rate(K, G, lc, args.eps0, args.cpu_sample_n, args.cpu_iters)
        line["cpu_baseline"] = {"value": rate, "unit": "voxel-updates/s", "cores": host_threads(), "kind": "oracle",
                                "sample": "%d^3 crop of the same image, %d oracle PT iterations, %.1f s" % (m, args.cpu_iters, dt)}
    print(json.dumps(line))
    return 0


if __name__ == "__main__":
    sys.exit(main())

#!/usr/bin/env python
"""bench.py — throughput of the residual + BSR-Jacobian assembly (BASELINE.json metric).

    python bench.py --gpus 1 --steps 10 --warmup 3             # this repo's CUDA path
    python bench.py --impl reference --steps 3 --warmup 1      # the CPU oracle, timed as it stands
    python -m torch.distributed.run --nproc-per-node N ... bench.py --gpus N   # N replicas

A "step" is one whole assembly (gradient + limiter kernel, then the fused flux / Jacobian /
source / BDF2 / BSR-write kernel) of one synthetic batch.  Default workload: BASELINE config 4,
run B — GEM Harris sheet on a 1,000,000-cell jittered Delaunay mesh, reverse-Cuthill-McKee order.
Every timed step assembles the same resident state, except in config 2's recipe (and q2), which
perturbs the state by 1e-6 between calls outside the timed regions.  Prints ONE JSON line (rank 0).
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

METRIC = "residual+BSR-Jacobian assembly throughput"
UNIT = "Mcells/s"


# --------------------------------------------------------------------------------------------
def algorithmic_bytes(nc: int, nnzb: int, nst: int, F: int = 3, packed: bool = False):
    """compulsory HBM bytes per launch of each kernel.  F = face slots per cell (3 on
    triangle meshes, 4 on meshes with quadrilaterals).  packed: the Jacobian in the packed form of include/tfa.h
    (full diagonal blocks, 114 entries per off-diagonal block)."""
    bs = 4 if F == 3 else 8
    jac = nc * 2592 + (nnzb - nc) * 912 if packed else nnzb * 18 * 18 * 8
    asm = (jac                     # Jacobian blocks written once
           + nc * 144 * 3          # state, state_n, state_nm1 read
           + nc * 144              # rhs written
           + nc * F * 144          # own-side face states of the cell's faces (read once; both users hit L2)
           + nc * F * 64           # per-cell geometry record
           + nc * F * 4 + nc * bs * 4)   # packed neighbour table, block map
    grad = (nc * 144               # state read
            + nst * 4 + nst * 16   # stencil indices and least-squares coefficient vectors
            + nc * 4               # stencil row pointers
            + nc * (2 * F + 2) * 8 # packed geometry (face midpoint offsets, sqrt of the volume)
            + nc * F * 144)        # face states written
    return asm, grad


def survey_bytes(nc: int, nnzb: int):
    """SURVEY 8(d)'s own per-step figures: Jacobian + three states + rhs + ~250 B of mesh data per cell, without
    and with the 864 B/cell of stored gradient / limiter intermediates."""
    fused = nnzb * 2592 + nc * (432 + 144 + 250)
    return fused, fused + nc * 864


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows = []
        self.proc = None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0: float, t1: float):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons, pw = [], [], set(), []
        for t, line in self.rows:
            if not (t0 - 0.05 <= t <= t1 + 0.15):
                continue
            f = [x.strip() for x in line.split(",")]
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except Exception:
                continue
            for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        if not sm:   # region shorter than the sampling period: take everything we saw
            for _, line in self.rows:
                f = [x.strip() for x in line.split(",")]
                try:
                    sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
                except Exception:
                    pass
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (driver-measured copy bandwidth)"
    return 6650.0, "fallback 6.65 TB/s (B200_PROFILING.md; MEASURED_PEAKS.json absent)"


def ncu_traffic(workload: str):
    """dram__bytes_read.sum + dram__bytes_write.sum of k_assemble per launch, from the committed
    `ncu --set full` capture (profiles/ncu_traffic.csv: workload,kernel,dram_bytes_per_launch)."""
    p = os.path.join(ROOT, "profiles", "ncu_traffic.csv")
    if os.path.exists(p):
        for line in open(p):
            f = [x.strip() for x in line.split(",")]
            if len(f) >= 3 and f[0] == workload and f[1] == "k_assemble":
                return float(f[2])
    return None


# --------------------------------------------------------------------------------------------
def oracle_sample(wl, n_rows: int, steps: int, warmup: int, threads: int | None = None):
    """Time the oracle as it stands on a row sample of the workload (host cores of this box; `threads` limits
    the OpenMP team, None = all cores)."""
    import oracle
    oracle.build()
    all_threads = oracle.num_threads()
    if threads is not None:
        oracle.set_num_threads(threads)
    om = oracle.OracleMesh.from_input(wl.mesh)
    state = wl.state
    if wl.reorder in ("rcm", "morton"):   # the oracle has no Z-order of its own; its work per cell is the same in any order
        om.reorder("rcm")
        state = np.ascontiguousarray(state[om.get("perm")])
    ph = oracle.physics_c(wl.physics)
    nu = oracle.default_numerics(ph)
    rng = np.random.default_rng(12345)
    n_rows = min(n_rows, om.n_cells)
    rows = np.sort(rng.choice(om.n_cells, size=n_rows, replace=False)).astype(np.int32)
    times = []
    for it in range(warmup + steps):
        t = time.perf_counter()
        oracle.assemble(om, ph, nu, state, dt=wl.dt, rows=rows)
        if it >= warmup:
            times.append(time.perf_counter() - t)
    sec = float(np.mean(times))
    used = oracle.num_threads()
    if threads is not None:
        oracle.set_num_threads(all_threads)
    return {"value": n_rows / sec / 1e6, "unit": UNIT, "cores": used, "kind": "oracle",
            "sample": f"{n_rows} random rows of {om.n_cells} (gradients of the rows and their neighbours "
                      f"included), {warmup} warm-up + mean of {steps} runs, {sec:.2f} s each "
                      f"(min {min(times):.2f}, max {max(times):.2f})"}, sec


def run_reference(args, wl):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cb, sec = oracle_sample(wl, args.cpu_rows, args.steps, args.warmup)
    line = {"impl": "reference", "metric": METRIC, "value": cb["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": wl_description(args.workload, wl), "n_cells": wl.mesh.n_cells,
                       "parallelism": "host cores (oracle)", "dt": wl.dt, "reorder": wl.reorder,
                       "sample_rows": min(args.cpu_rows, wl.mesh.n_cells)},
            "cpu_baseline": cb,
            "e2e": {"value": cb["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def run_shards(args, wl):
    """`--shards N` (one GPU): the sharded assembly of SURVEY 8(f)4 with its N ranks emulated one after another in
    this process (their kernels never wait on each other; the halos go through the library's pack / unpack kernels
    with a device buffer standing in for the wire).  Not a scaling measurement -- there is one GPU -- but the cost
    structure of a rank: owned and ghost cells, halo volumes, and the device time of its kernels for 1/N of the problem."""
    import torch
    from paper_1809_02532_b200 import api, build
    build.build()
    torch.cuda.set_device(0)
    n = args.shards
    mesh = api.Mesh.from_input(wl.mesh)
    if wl.reorder in ("rcm", "morton"):
        mesh.reorder(wl.reorder)
    P = np.ascontiguousarray(wl.state[mesh.get("perm")])
    ev = lambda: torch.cuda.Event(enable_timing=True)
    t0 = time.time()
    shards = [api.Shard(mesh, n, r) for r in range(n)]
    torch.cuda.synchronize()
    t_build = time.time() - t0
    ctxs = [api.Context(wl.physics) for _ in shards]
    loc = [torch.from_numpy(P[s.part.local_to_global]).cuda() for s in shards]
    vals = [torch.empty((s.nnzb_owned, 18, 18), dtype=torch.float64, device="cuda") for s in shards]
    rhs = [torch.empty((s.part.n_local, 18), dtype=torch.float64, device="cuda") for s in shards]
    F = mesh.max_faces

    def one_step(timers=None):
        def lap(key, fn):
            if timers is None:
                return fn()
            a, b = ev(), ev()
            a.record(); fn(); b.record()
            timers.setdefault(key, []).append((a, b))
        lap("halo_state", lambda: api.exchange_in_process(shards, api.HALO_STATE, loc))
        for r, (s, c) in enumerate(zip(shards, ctxs)):
            lap(f"gradient_{r}", lambda: c.assemble_gradient(s.mesh, loc[r]))
        faces = [c.face_states(s.mesh) for s, c in zip(shards, ctxs)]
        lap("halo_face", lambda: api.exchange_in_process(shards, api.HALO_FACE, faces))
        for r, (s, c) in enumerate(zip(shards, ctxs)):
            lap(f"faces_{r}", lambda: c.assemble_faces(s.mesh, loc[r], loc[r], loc[r], wl.dt, rhs=rhs[r], vals=vals[r]))

    for _ in range(max(args.warmup, 3)):
        one_step()
    for c in ctxs:
        c.check()
    timers = {}
    for _ in range(args.steps):
        one_step(timers)
    torch.cuda.synchronize()
    ms = {k: float(np.mean([a.elapsed_time(b) for a, b in v])) for k, v in timers.items()}
    rank_ms = [ms[f"gradient_{r}"] + ms[f"faces_{r}"] for r in range(n)]
    halo_state = [sum(s.part.count(api.PART_RECV_STATE, q) for q in range(n)) for s in shards]
    halo_face = [sum(s.part.count(api.PART_RECV_FACE, q) for q in range(n)) for s in shards]
    line = {"metric": METRIC, "mode": "sharded assembly, ranks emulated on one GPU (no scaling claim)", "unit": UNIT,
            "n_gpus": 1, "shards": n, "steps": args.steps, "dtype": "f64", "data": "synthetic",
            "config": {"workload": wl_description(args.workload, wl), "n_cells": mesh.n_cells, "nnzb": mesh.nnzb},
            "per_rank": {"owned_cells": [s.part.n_owned for s in shards],
                         "ghost_cells": [s.part.n_local - s.part.n_owned for s in shards],
                         "owned_blocks": [s.nnzb_owned for s in shards],
                         "kernel_ms": rank_ms,
                         "mcells_per_s": [s.part.n_owned / (t * 1e-3) / 1e6 for s, t in zip(shards, rank_ms)],
                         "halo_state_bytes_received": [h * 144 for h in halo_state],
                         "halo_face_bytes_received": [h * F * 144 for h in halo_face]},
            "slowest_rank_ms": max(rank_ms), "sum_of_ranks_ms": sum(rank_ms),
            "in_process_exchange_ms": {"state": ms["halo_state"], "face": ms["halo_face"],
                                       "note": "pack + unpack kernels of all ranks, no wire"},
            "shard_build_s": t_build}
    print(json.dumps(line), flush=True)


def reduce_max_over_ranks(x: float, world: int, device="cuda") -> float:
    """Replicas only: the one inter-rank step is the max of the device-timed durations."""
    if world <= 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_throughput(n_cells: int, steps: int, world: int, total_ms: float) -> float:
    """Whole-job Mcells/s: every rank assembles its own replica of the workload (weak scaling)."""
    return world * n_cells * steps / (total_ms * 1e-3) / 1e6


def wl_description(name, wl):
    desc = {"c1": "config 1: wave, 16x16 split quads, periodic",
            "c2": "config 2: wave, 256x256 split quads, periodic",
            "c3": "config 3: GEM, 512x256 split quads, periodic-x",
            "c4a": "config 4 run A: GEM, 1M-cell jittered Delaunay, random cell order",
            "c4b": "config 4 run B: GEM, 1M-cell jittered Delaunay, reverse Cuthill-McKee order",
            "c4m": "config 4's mesh in Z-order (Morton curve through the centroids; not a BASELINE run)",
            "c5": "config 5: GEM, 4M-cell jittered Delaunay, RCM order",
            "q1": "paper mesh (L559, Table 9): double current sheet, 512x512 periodic quadrilaterals",
            "q2": "paper mesh (L433, Table 4): wave, 256x128 periodic quadrilaterals",
            "qm": "mixed mesh: GEM, jittered quadrilaterals with every third split into triangles, walls in y, RCM"}[name]
    return f"{desc} ({wl.mesh.n_cells} cells)"


# --------------------------------------------------------------------------------------------
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c4b",
                    choices=["c1", "c2", "c3", "c4a", "c4b", "c4m", "c5", "q1", "q2", "qm"])
    ap.add_argument("--scale", type=float, default=1.0, help="linear lattice scale (tests only)")
    ap.add_argument("--cpu-rows", type=int, default=200000, help="rows of the oracle's timed sample")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--solve", action="store_true", help="also time the linear-solve step (SpMV, block-Jacobi, GMRES)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--shards", type=int, default=0,
                    help="one GPU: emulate the sharded assembly of N ranks in this process and report per-rank costs")
    ap.add_argument("--packed", action="store_true",
                    help="assemble the packed Jacobian (tfa_assemble_packed) instead of the BSR one")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = max(args.warmup, 1)

    from paper_1809_02532_b200 import workloads as W
    t_gen = time.time()
    wl = W.make_workload(args.workload, scale=args.scale)
    t_gen = time.time() - t_gen
    if args.impl == "reference":
        return run_reference(args, wl)
    if args.shards > 0:
        return run_shards(args, wl)

    import torch
    import torch.distributed as dist
    from paper_1809_02532_b200 import api, build
    build.build()

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- setup (step a1; timed separately, once per mesh) ----
    ev = lambda: torch.cuda.Event(enable_timing=True)
    e0, e1, e2 = ev(), ev(), ev()
    e0.record()
    mesh = api.Mesh.from_input(wl.mesh)
    e1.record()
    if wl.reorder in ("rcm", "morton"):
        mesh.reorder(wl.reorder)
    e2.record()
    torch.cuda.synchronize()
    setup_ms = {"mesh_create_ms": e0.elapsed_time(e1), "reorder_ms": e1.elapsed_time(e2), "generate_s": t_gen}
    perm = mesh.get("perm")
    state_h = np.ascontiguousarray(wl.state[perm])
    nc, nnzb, nst, F = mesh.n_cells, mesh.nnzb, mesh.n_stencil, mesh.max_faces
    if args.workload == "qm":   # conducting walls on the y boundaries
        mesh.set_bc(np.full(mesh.n_bfaces, api.BC_WALL, dtype=np.int32))
    ctx = api.Context(wl.physics)
    P = torch.from_numpy(state_h).cuda()
    Pn, Pnm1 = P.clone(), P.clone()
    rhs = torch.empty((nc, 18), dtype=torch.float64, device="cuda")
    if args.packed:
        pk_diag = torch.empty((nc, 18, 18), dtype=torch.float64, device="cuda")
        pk_offd = torch.empty((nnzb - nc, 114), dtype=torch.float64, device="cuda")
        vals = None
    else:
        vals = torch.empty((nnzb, 18, 18), dtype=torch.float64, device="cuda")

    def assemble_step():
        if args.packed:
            ctx.assemble_packed(mesh, P, Pn, Pnm1, wl.dt, rhs=rhs, diag=pk_diag, offd=pk_offd)
        else:
            ctx.assemble(mesh, P, Pn, Pnm1, wl.dt, rhs=rhs, vals=vals)
    noise = torch.empty_like(P)
    gen = torch.Generator(device="cuda").manual_seed(1000 + rank)

    def perturb():   # BASELINE config 2: seeded noise of 1e-6 between calls (outside the timed kernels)
        noise.uniform_(-1e-6, 1e-6, generator=gen)
        P.add_(noise)

    # BASELINE config 2's recipe (and its quadrilateral twin) perturbs the state between consecutive calls; the
    # perturbation sits outside the timed regions (SURVEY 8(d) "rate definition"): those workloads are timed per
    # call and summed.  The other configurations assemble the same state every step: one bracket around K steps
    # (12.6 GB of traffic per step at c4b against 126 MB of L2; c1-c3 and q2 fit in L2 and run L2-warm).
    recipe_perturbs = args.workload in ("c2", "q2")

    # ---- probes: FP64 FMA peak and copy bandwidth in this run ----
    sink = torch.zeros(8, dtype=torch.float64, device="cuda")
    flops = api.probe_dfma(148 * 8, 1 << 14, sink)
    torch.cuda.synchronize()
    best = 1e9
    for _ in range(3):
        a, b = ev(), ev()
        a.record(); flops = api.probe_dfma(148 * 8, 1 << 14, sink); b.record(); torch.cuda.synchronize()
        best = min(best, a.elapsed_time(b))
    fp64_tflops = flops / (best * 1e-3) / 1e12
    src = torch.empty(1 << 27, dtype=torch.float64, device="cuda").normal_()
    dst = torch.empty_like(src)
    best = 1e9
    for _ in range(4):
        a, b = ev(), ev()
        a.record(); nbytes = api.probe_copy(src, dst); b.record(); torch.cuda.synchronize()
        best = min(best, a.elapsed_time(b))
    copy_gbs = nbytes / (best * 1e-3) / 1e9
    del src, dst

    # ---- device-resident timing ----
    sampler = ClockSampler(local) if rank == 0 else None   # started early: nvidia-smi takes a while to come up
    for _ in range(max(args.warmup, 3)):
        perturb()
        assemble_step()
    ctx.check()
    # per-kernel events ride inside the timed region (the library keeps at most 64 assemblies of them)
    inline_events = args.steps <= 64
    ctx.timing_enable(inline_events)
    barrier()
    t0 = time.time()
    if recipe_perturbs:
        pairs = [(ev(), ev()) for _ in range(args.steps)]
        for a, b in pairs:
            perturb()
            a.record()
            assemble_step()
            b.record()
        barrier()
        total_ms = sum(a.elapsed_time(b) for a, b in pairs)
    else:
        start, end = ev(), ev()
        start.record()
        for _ in range(args.steps):
            assemble_step()
        end.record()
        barrier()
        total_ms = start.elapsed_time(end)
    t1 = time.time()
    clocks = sampler.stop(t0, t1) if sampler else None
    if not inline_events:   # long runs: the per-kernel split comes from 32 further steps right after
        ctx.timing_enable(True)
        for _ in range(32):
            assemble_step()
    ms_grad, ms_asm, ncalls = ctx.timing_read()
    ctx.timing_enable(False)
    ctx.check()
    total_ms = reduce_max_over_ranks(total_ms, world)
    ms_per_step = total_ms / args.steps
    value = job_throughput(nc, args.steps, world, total_ms)

    # ---- end to end through the C ABI with HOST buffers (copies inside the timed region) ----
    e2e = None
    if not args.no_e2e and not args.packed:
        k_e2e = max(1, min(args.steps, 3))
        sh = [torch.from_numpy(state_h).pin_memory() for _ in range(3)]
        rhs_h = torch.empty((nc, 18), dtype=torch.float64).pin_memory()
        vals_h = torch.empty((nnzb, 18, 18), dtype=torch.float64).pin_memory()
        ctx.assemble_host(mesh, sh[0], sh[1], sh[2], wl.dt, rhs_h, vals_h)   # warm-up (allocates staging)
        barrier()
        tt = time.perf_counter()
        for _ in range(k_e2e):
            ctx.assemble_host(mesh, sh[0], sh[1], sh[2], wl.dt, rhs_h, vals_h)
        torch.cuda.synchronize()
        sec = (time.perf_counter() - tt)
        sec = reduce_max_over_ranks(sec, world)
        e2e = {"value": job_throughput(nc, k_e2e, world, sec * 1e3), "unit": UNIT,
               "h2d_bytes_per_step": 3 * nc * 144, "d2h_bytes_per_step": nc * 144 + nnzb * 2592,
               "steps": k_e2e, "ms_per_step": sec / k_e2e * 1e3,
               "note": "tfa_assemble_host: pinned host buffers, H2D of 3 states and D2H of rhs + BSR values inside"}
        del sh, rhs_h, vals_h

    # ---- optional: the next step of the method, the linear solve on the assembled system ----
    solve = None
    if args.solve and rank == 0 and not args.packed:
        n = 18 * nc
        xv = torch.randn(n, dtype=torch.float64, device="cuda")
        yv = torch.empty_like(xv)
        def timed(fn, reps):
            fn(); torch.cuda.synchronize()
            a, b = ev(), ev()
            a.record()
            for _ in range(reps):
                fn()
            b.record(); torch.cuda.synchronize()
            return a.elapsed_time(b) / reps
        spmv_ms = timed(lambda: api.bsr_spmv(mesh, vals, xv, yv), 10)
        dinv = torch.empty((nc, 18, 18), dtype=torch.float64, device="cuda")
        bj_ms = timed(lambda: ctx.block_jacobi(mesh, vals, dinv), 3)
        bvec = rhs.reshape(-1).contiguous()
        for _ in range(2):   # the first solve allocates the Krylov workspace; the second is the timed one
            torch.cuda.synchronize()
            tt = time.perf_counter()
            xs, its, rel = ctx.gmres(mesh, vals, bvec, dinv=dinv, restart=30, max_iters=300, rtol=1e-6)
            torch.cuda.synchronize()
            gm_s = time.perf_counter() - tt
        ctx.check()
        jv = torch.empty_like(xv)
        jvp_ms = timed(lambda: ctx.jvp(mesh, P, xv, Pn, Pnm1, wl.dt, eps=1e-7, out=jv), 5)
        for _ in range(2):
            torch.cuda.synchronize()
            tt = time.perf_counter()
            xj, itj, relj = ctx.gmres_jfnk(mesh, P, bvec, Pn, Pnm1, wl.dt, dinv=dinv, restart=30, max_iters=300, rtol=1e-6)
            torch.cuda.synchronize()
            gj_s = time.perf_counter() - tt
        ctx.check()
        # the same solve on the packed Jacobian (tfa_assemble_packed, tfa_packed_spmv, tfa_gmres_packed)
        _, pk_d, pk_o = ctx.assemble_packed(mesh, P, Pn, Pnm1, wl.dt)
        pspmv_ms = timed(lambda: api.packed_spmv(mesh, pk_d, pk_o, xv, yv), 10)
        dinv_p = ctx.block_jacobi_packed(mesh, pk_d)
        for _ in range(2):
            torch.cuda.synchronize()
            tt = time.perf_counter()
            xp, itp, relp = ctx.gmres_packed(mesh, pk_d, pk_o, bvec, dinv=dinv_p, restart=30, max_iters=300, rtol=1e-6)
            torch.cuda.synchronize()
            gp_s = time.perf_counter() - tt
        ctx.check()
        # mixed precision: Krylov cycles on FP32 copies of the packed matrix and of the inverses, restarts in FP64
        tt = time.perf_counter()
        d32, o32 = api.packed_to_f32(mesh, pk_d, pk_o)
        dinv32 = api.to_f32(dinv_p)
        torch.cuda.synchronize()
        conv_s = time.perf_counter() - tt
        mixed = {}
        for tol in (1e-6, 1e-10):
            for _ in range(2):
                torch.cuda.synchronize()
                tt = time.perf_counter()
                xm, itm, relm = ctx.gmres_packed_f32(mesh, pk_d, pk_o, d32, o32, bvec, dinv32=dinv32, restart=30,
                                                     max_iters=300, rtol=tol)
                torch.cuda.synchronize()
                gm32_s = time.perf_counter() - tt
            mixed["rtol_%g" % tol] = {"iterations": itm, "relative_residual": relm, "seconds": gm32_s}
        for _ in range(2):
            torch.cuda.synchronize()
            tt = time.perf_counter()
            xp10, itp10, relp10 = ctx.gmres_packed(mesh, pk_d, pk_o, bvec, dinv=dinv_p, restart=30, max_iters=300,
                                                   rtol=1e-10)
            torch.cuda.synchronize()
            gp10_s = time.perf_counter() - tt
        mixed["fp64_rtol_1e-10"] = {"iterations": itp10, "relative_residual": relp10, "seconds": gp10_s}
        mixed["convert_seconds"] = conv_s
        mixed["max_diff_to_fp64_solution"] = float((xm - xp10).abs().max() / xp10.abs().max())
        ctx.check()
        pspmv_bytes = nc * 2592 + (nnzb - nc) * 912 + 2 * n * 8 + nnzb * 4 + nc * 4
        del pk_d, pk_o, dinv_p, xp, d32, o32, dinv32, xm, xp10
        # one Newton sub-iteration of Eq. 14 as one call (tfa_implicit_step): assembled BSR path against mode 2
        work = dict(rhs=torch.empty((nc, 18), dtype=torch.float64, device="cuda"), vals=vals, dinv=dinv,
                    dP=torch.empty((nc, 18), dtype=torch.float64, device="cuda"))
        newton = {}
        for mode, key in ((False, "bsr_fp64"), ("packed_f32", "packed_f32_cycles")):
            for _ in range(2):
                S = P.clone()
                torch.cuda.synchronize()
                tt = time.perf_counter()
                (nit, upd, gits, lrel), _ = ctx.implicit_step(mesh, S, Pn, Pnm1, wl.dt, work=work, max_newton=1,
                                                              rtol=1e-6, matrix_free=mode)
                torch.cuda.synchronize()
                nw_s = time.perf_counter() - tt
            newton[key] = {"seconds": nw_s, "gmres_iterations": gits, "linear_residual": lrel, "update": upd}
        ctx.check()
        del work, S
        spmv_bytes = nnzb * 2592 + 2 * n * 8 + nnzb * 4 + nc * 4
        solve = {"spmv_ms": spmv_ms, "spmv_algorithmic_bytes": spmv_bytes,
                 "spmv_gbs": spmv_bytes / (spmv_ms * 1e-3) / 1e9, "block_jacobi_ms": bj_ms,
                 "jvp_ms": jvp_ms, "jvp_note": "tfa_jvp: two residual-only assemblies (base + perturbed) and two axpby",
                 "gmres": {"restart": 30, "rtol": 1e-6, "iterations": its, "relative_residual": rel, "seconds": gm_s,
                           "preconditioner": "block-Jacobi (18x18 diagonal blocks)"},
                 "packed": {"spmv_ms": pspmv_ms, "spmv_algorithmic_bytes": pspmv_bytes,
                            "spmv_gbs": pspmv_bytes / (pspmv_ms * 1e-3) / 1e9,
                            "gmres": {"iterations": itp, "relative_residual": relp, "seconds": gp_s},
                            "gmres_f32_cycles": mixed},
                 "newton_iteration": newton,
                 "gmres_jfnk": {"restart": 30, "rtol": 1e-6, "iterations": itj, "relative_residual": relj,
                                "seconds": gj_s, "operator": "tfa_jvp (matrix-free), same preconditioner"}}
        del xv, yv, dinv, xs, xj

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (k_assemble) ----
    asm_bytes, grad_bytes = algorithmic_bytes(nc, nnzb, nst, F, args.packed)
    sv_fused, sv_stored = survey_bytes(nc, nnzb)
    step_gbs = lambda nbytes: nbytes / (ms_per_step * 1e-3) / 1e9
    peak, peak_src = measured_peaks()
    asm_ms = ms_asm / max(ncalls, 1)
    grad_ms = ms_grad / max(ncalls, 1)
    achieved = asm_bytes / (asm_ms * 1e-3) / 1e9
    roofline = {"bound": "hbm", "kernel": "k_assemble", "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": ncu_traffic(args.workload + ("+packed" if args.packed else "")),
                "algorithmic_bytes_per_launch": asm_bytes, "kernel_ms": asm_ms, "peak_source": peak_src,
                "kernel_share_of_step": asm_ms / ms_per_step,
                "copy_probe_gbs_this_run": copy_gbs, "fp64_probe_tflops_this_run": fp64_tflops,
                "gradient_kernel": {"ms": grad_ms, "algorithmic_bytes_per_launch": grad_bytes,
                                    "achieved_gbs": grad_bytes / (grad_ms * 1e-3) / 1e9},
                # whole step (both kernels) against the same peak, by three byte counts: as built (each kernel's own
                # compulsory traffic, geometry and states counted once per kernel that reads them) and SURVEY 8(d)'s
                # two figures (intermediates fused away / stored and re-read)
                "step": {"as_built_bytes": asm_bytes + grad_bytes, "as_built_frac": step_gbs(asm_bytes + grad_bytes) / peak,
                         "survey_fused_bytes": sv_fused, "survey_fused_frac": step_gbs(sv_fused) / peak,
                         "survey_stored_bytes": sv_stored, "survey_stored_frac": step_gbs(sv_stored) / peak},
                "step_frac_of_hbm_roofline": step_gbs(sv_stored) / peak}

    cpu_baseline = None
    if not args.no_cpu_baseline and world == 1:
        cpu_baseline, _ = oracle_sample(wl, args.cpu_rows, 3, 1)
        one, _ = oracle_sample(wl, max(1, args.cpu_rows // 8), 2, 1, threads=1)
        cpu_baseline["one_thread"] = {"value": one["value"], "unit": UNIT, "cores": 1, "sample": one["sample"]}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": wl_description(args.workload, wl), "n_cells": nc, "nnzb": nnzb, "max_faces": F,
                       "parallelism": "replicas only" if world > 1 else "single GPU",
                       "l2": "inputs+outputs per step (%.1f GB) exceed the 126 MB L2; no flush needed" %
                             ((asm_bytes + grad_bytes) / 1e9),
                       "dt": wl.dt, "reorder": wl.reorder,
                       "jacobian": "packed: full diagonal blocks + 114-entry off-diagonal blocks (tfa_assemble_packed)"
                                   if args.packed else "18x18 BSR (cuSPARSE layout)"},
            "clocks": clocks, "e2e": e2e, "gpu_launches": ctx.launches_per_assemble * args.steps,
            "roofline": roofline, "cpu_baseline": cpu_baseline, "setup": setup_ms}
    if solve is not None:
        line["solve"] = solve
        line["solve"]["spmv_frac_of_hbm"] = solve["spmv_gbs"] / peak
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()

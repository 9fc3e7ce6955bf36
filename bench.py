#!/usr/bin/env python
"""bench.py -- BASELINE.json's metric on BASELINE.json's configs: fp64 pair interactions per second and
ms per full HSMA evaluation, with the FP64 roofline of the dominant kernel and the CPU oracle timed
beside it.  One JSON line on stdout (rank 0).  DESIGN.md "Measurement" explains every field.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 5] [--impl b200|reference]
  N > 1: python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 \
         --master-port P bench.py --gpus N --steps K --warmup W

A "step" is one pass of the whole hot path (H1..H7: pre-pass, (a) check-point sums, fit, mapping,
(b) near sums at the sources, (c) node sums, energy) over one synthetic configuration.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import hsma_workloads as W  # noqa: E402

METRIC = "fp64 pair interactions/sec"
UNIT = "pairs/s"

# Algorithmic work per pair, SURVEY.md 8(d) / DESIGN.md "Roofline": flops with add/mul = 1, fma = 2
FLOPS_PAIR_CHARGE = 18.0      # 3 DADD + (DMUL + 2 DFMA) + cubic rsqrt refinement (2 DMUL + 3 DFMA) + DFMA
FLOPS_PAIR_DIPOLE = 26.0      # + P.d (DMUL + 2 DFMA) + y^2 (DMUL) + DFMA
# what near_sum_kernel<R, REFINE> executes per pair (FP64-pipe instructions, flops), DESIGN.md 6.1/6.4:
# (refine, all |q| equal) -> the uniform-|q| path drops the multiplication by q
EXEC_PAIR = {(1, False): (10.0, 14.0), (2, False): (12.0, 18.0), (1, True): (9.0, 13.0), (2, True): (11.0, 17.0)}
# --forces: the potential+gradient form of the same kernel: (instructions, flops) executed per pair;
# algorithmic: the charge pair (18) + q y^3 (2 mul) + 3 fma = 26 flops
EXEC_PAIR_FIELD = {(1, False): (16.0, 22.0), (2, False): (18.0, 26.0), (1, True): (15.0, 21.0), (2, True): (17.0, 25.0)}
FLOPS_PAIR_CHARGE_FIELD = 26.0
# Symmetric form of step (b) (near_sym_kernel; used when one rank evaluates all N targets): the unit of
# the kernel is one pair EVALUATION (an unordered source pair in one image cell), which feeds two sums.  `frac` charges
# an evaluation SURVEY.md 8(d)'s 18 flops of a charge pair (FLOPS_PAIR_CHARGE), nothing for the second accumulation;
# `frac_with_second_accumulation` adds that DFMA (20 flops).  Executed per evaluation
# (FP64-pipe instructions, flops): pair 11 / 16 (Newton), 13 / 20 (cubic); + per 8 evaluations the image of the source
# (3 DFMA), q*w (DMUL) and the column accumulation (DFMA).
FLOPS_EVAL_SYM = 20.0
EXEC_EVAL_SYM = {1: (11.0 + 5.0 / 8.0, 16.0 + 9.0 / 8.0), 2: (13.0 + 5.0 / 8.0, 20.0 + 9.0 / 8.0)}
# the same with the gradient (near_sym_field_kernel): algorithmic = the 26 of a potential+gradient pair + the column side
# (DFMA + DMUL + 3 DFMA = 9); executed: pair 21 / 33 (Newton), 23 / 37 (cubic) + per 8 evaluations 11 instructions / 18 flops
FLOPS_EVAL_SYM_FIELD = 35.0
EXEC_EVAL_SYM_FIELD = {1: (21.0 + 11.0 / 8.0, 33.0 + 18.0 / 8.0), 2: (23.0 + 11.0 / 8.0, 37.0 + 18.0 / 8.0)}


# Lattice-factored kernels (csrc/lattice_kernels.cuh): the unit is still one image-pair evaluation, but
# its r^2 comes from per-axis squares shared by all images of the (target, source) pair and the charges enter once per
# pair.  Counted from the formulation (and checked against the SASS of the inner loop, profiles/r02_sass_opcodes.md):
#   per image   : r^2 = z-square + (x-square + y-square) [DFMA], y0^2 [DMUL], Newton factor [DFMA], accumulate [DFMA]
#                 (+ 2 DFMA for the cubic step)
#   per pair    : offsets (1 + 2 s_a [+ 1 on a reflecting axis] DADD per axis), x squares (2 s_x + 1 DMUL),
#                 x-square + y-square (DFMA per (kx, ky)), weight classes (1 DMUL + DFMA per further class),
#                 row and column accumulation (2 DFMA; 1 for ordered pairs), symmetric form: 5/4 DADD (warp reduction of the
#                 column sum of a source, once per 4 targets)
# Gradient forms: measured on the 27-cell periodic shape (10.22 instructions / 15.15 flops per image, Newton).
def lat_counts(shell, reflecting, refine: int, field: bool, symmetric: bool):
    """(FP64-pipe instructions, flops) executed per image-pair evaluation by the lattice-factored kernels."""
    sx, sy, sz = shell
    images = (2 * sx + 1) * (2 * sy + 1) * (2 * sz + 1)
    if field:
        instr, flops = 10.22, 15.15
        return (instr + (2.0 if refine == 2 else 0.0), flops + (4.0 if refine == 2 else 0.0))
    classes = 1 + sum(s for s, r in zip(shell, reflecting) if r)
    dadd = sum(1 + 2 * s + (1 if r else 0) for s, r in zip(shell, reflecting))
    dmul = (2 * sx + 1) + 1
    dfma = (2 * sx + 1) * (2 * sy + 1) + (classes - 1) + (2 if symmetric else 1)
    per_img_instr = 4 + (2 if refine == 2 else 0)
    per_img_flops = 7 + (4 if refine == 2 else 0)
    red = 5.0 / 4.0 if symmetric else 0.0     # symmetric form: 5 DADD of the warp reduction of a source's column sum, per 4 pairs
    return (per_img_instr + (dadd + dmul + dfma + red) / images, per_img_flops + (dadd + dmul + 2 * dfma + red) / images)


def sym_evaluations(N: int, C: int) -> int:
    """Pair evaluations of one near_sym_kernel launch (csrc/sum_kernels.cuh: visits x tile x block x cells; the
    diagonal visits and the padding of the last block are evaluated like the rest and counted here)."""
    nt = -(-N // 256)
    nb = -(-nt // 8)
    visits = nb * nt - 8 * (nb * (nb - 1) // 2)
    return visits * 256 * 2048 * C


# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the dominant kernel from the committed ncu --set full
# capture (profiles/r01_ncu_near_sum_N262144.md): valid for config 5 at N = 262,144 on one GPU, potential only
NCU_TRAFFIC_BYTES_CFG5 = 9555200
NCU_TRAFFIC_BYTES_CFG5_SYM = 28873728    # near_sym_kernel, 3 waves per evaluate: 3 x (8,463,872 read + 1,160,704 written)
NCU_TRAFFIC_BYTES_CFG5_LAT_SYM = 29011968   # near_lat_sym_kernel, 3 waves per evaluate: 3 x (8,478,464 read + 1,192,192 written)
TRAFFIC_SOURCE_LAT_SYM = "profiles/r02c_ncu_lat_sym_N262144.md (dram read+write bytes of one wave x 3 waves per evaluate)"
TRAFFIC_SOURCE_SYM = "profiles/r02_ncu_near_sym_waves_N262144.md (dram read+write bytes of one wave x 3 waves per evaluate)"
TRAFFIC_SOURCE = "profiles/r01_ncu_near_sum_N262144.md (dram read+write bytes of one launch)"
# FP64 peak derived from unit counts and clocks: SMs x 64 DFMA lanes x 2 x clock
FP64_LANES_PER_SM = 64


def pair_counts(info: dict, N: int, T: int) -> dict:
    """Pairs per step for a rank that owns T of the N targets (step (a) is computed in full).  With the
    sphere-culled near set the images per target are what the last evaluate counted on the device."""
    images = info.get("near_images_last_evaluate") or N * info["near_cells"]
    near_a = images if images != N * info["near_cells"] else N * info["rhs_cells"]
    return {"a": info["check_targets"] * near_a, "b": T * images, "c": T * info.get("node_records", info["M"])}


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.gpu = gpu_index
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None

    def start(self):
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(self.gpu), f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "200"], stdout=self.f,
                                      stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self) -> dict:
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, pw, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for line in self.f.read().splitlines():
            t = [x.strip() for x in line.split(",")]
            if len(t) < 9:
                continue
            try:
                sm.append(float(t[1])); mx.append(float(t[2])); pw.append(float(t[3]))
            except ValueError:
                continue
            for name, v in zip(names, t[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        try:
            os.unlink(self.f.name)
        except OSError:
            pass
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": statistics.median(sm), "sm_min_mhz": min(sm), "sm_max_mhz": max(mx),
                "power_w_max": max(pw), "samples": len(sm), "reasons": sorted(reasons)}


# ---------------------------------------------------------------------------------------------------
# CPU oracle arm (cpu_baseline leg and --impl reference): the only place bench.py executes oracle/
# ---------------------------------------------------------------------------------------------------
class OracleSample:
    """A bounded sample of one HSMA step of workload `w`, run by the oracle as it stands
    (oracle/direct_sum.c, OpenMP over targets): the three direct sums at T_b of the N source targets
    and at the same fraction of the check targets.  The fit and the mapping (O(1e6) flops) are not in
    the sample; the node strengths are fixed numbers of the right size (their values do not change the
    cost of a sum)."""

    def __init__(self, w):
        from oracle import hsma_oracle as O
        self.O, self.w = O, w
        L = np.asarray(w.L, dtype=np.float64)
        self.src = np.ascontiguousarray(np.asarray(w.xyz, dtype=np.float64) - 0.5 * L)
        self.q = np.ascontiguousarray(w.q, dtype=np.float64)
        self.near = O.cell_table(w.kind, L, w.near_shell, w.gamma)
        self.rhs_cells = (O.cell_table(w.kind, L, w.far_shell, w.gamma, exclude_shell=w.near_shell)
                          if w.closure == W.CLOSURE_FAR_DATA else self.near)
        R0 = 0.5 * float(np.linalg.norm(L))
        if w.kind == W.BC_PERIODIC:
            x = O.fibonacci_sphere_checkpoints(w.K, R0)
            self.chk = np.concatenate([x, O.wrap_into_box(x, L)], axis=0)
        else:
            self.chk = np.asarray(w.check_xyz, dtype=np.float64)
        self.nodes, self.nrm, wq = O.make_nodes(w.M, w.R_aux, w.quad_rule)
        self.Q = wq / (4 * np.pi)
        self.D = wq / (4 * np.pi)
        self.cores = O.num_threads()

    def run(self, T_b: int):
        """Returns (seconds, pairs).  T_b source targets taken from the middle of the index range."""
        w, O = self.w, self.O
        N = w.N
        T_b = max(1, min(N, T_b))
        T_a = max(1, min(self.chk.shape[0], int(round(self.chk.shape[0] * T_b / N))))
        i0 = (N - T_b) // 2
        t0 = time.perf_counter()
        O.near_sum(self.chk[:T_a], self.src, self.q, self.rhs_cells)
        O.near_sum(self.src[i0:i0 + T_b], self.src, self.q, self.near, self_offset=i0)
        O.node_sum(self.src[i0:i0 + T_b], self.nodes, self.nrm, self.Q, self.D)
        dt = time.perf_counter() - t0
        pairs = (T_a * N * self.rhs_cells.w.shape[0] + T_b * N * self.near.w.shape[0] + T_b * w.M)
        return dt, pairs, T_a

    def calibrate(self, seconds: float) -> int:
        """Number of source targets whose sample takes about `seconds` on this host."""
        T = max(1, min(self.w.N, self.cores))
        dt, pairs, _ = self.run(T)
        while dt < 0.2 and T < self.w.N:
            T = min(self.w.N, T * 4)
            dt, pairs, _ = self.run(T)
        return max(1, min(self.w.N, int(T * seconds / max(dt, 1e-6))))


def cpu_baseline(w, seconds: float) -> dict:
    s = OracleSample(w)
    T = s.calibrate(seconds)
    dt, pairs, T_a = s.run(T)
    return {"value": pairs / dt, "unit": UNIT, "cores": s.cores, "kind": "oracle", "seconds": dt,
            "sample": f"{w.name}: oracle direct sums (a)+(b)+(c) at {T} of {w.N} source targets and {T_a} of "
                      f"{s.chk.shape[0]} check targets against all {w.N} sources x cells ({pairs:.3e} pairs); "
                      f"fit and mapping not in the sample"}


def run_reference(args, w) -> dict:
    """--impl reference: the oracle, as it stands, on the host cores; each step is a bounded sample."""
    s = OracleSample(w)
    T = s.calibrate(args.ref_step_seconds)
    for _ in range(args.warmup):
        s.run(T)
    tot_t, tot_p, T_a = 0.0, 0, 0
    for _ in range(args.steps):
        dt, pairs, T_a = s.run(T)
        tot_t += dt
        tot_p += pairs
    value = tot_p / tot_t
    sample = (f"{w.name}: per step the oracle direct sums (a)+(b)+(c) at {T} of {w.N} source targets and {T_a} check "
              f"targets against all sources x cells ({tot_p / args.steps:.3e} pairs/step); fit and mapping not in the sample")
    return {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps,
            "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "N": w.N, "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": s.cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}


# ---------------------------------------------------------------------------------------------------
# CUDA arm
# ---------------------------------------------------------------------------------------------------
def run_b200(args, w) -> dict:
    import torch
    import torch.distributed as dist

    import paper_1806_04801_b200 as H
    from paper_1806_04801_b200 import shard

    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the CUDA path has no CPU fallback")
    H.binding.load_library()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus:
        raise RuntimeError(f"--gpus {args.gpus} but WORLD_SIZE={world}: launch with torch.distributed.run")
    # Rehearsal switch (tests only): HSMA_BENCH_SHARE_GPU=1 runs all ranks on cuda:0 over a gloo group, so that the whole
    # N > 1 code path of this file -- rendezvous, barriers, shard.evaluate_distributed per step, max over ranks, rank-0
    # line -- can be executed on a one-GPU box (NCCL refuses two ranks on one device).  Its numbers are not measurements.
    share_gpu = world > 1 and os.environ.get("HSMA_BENCH_SHARE_GPU") == "1"
    if share_gpu:
        local = 0
    if local >= torch.cuda.device_count():
        raise RuntimeError(f"bench.py --gpus {args.gpus}: rank {rank} needs visible CUDA device {local}, but only "
                           f"{torch.cuda.device_count()} visible CUDA device(s) exist on this node")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    # everything (plan, kernels, flushes, events, NCCL) on one non-default stream: the library can then capture the
    # evaluate into a CUDA graph (it does so only while stage timing is off)
    torch.cuda.set_stream(torch.cuda.Stream(device=dev))
    if world > 1:
        if share_gpu:
            dist.init_process_group("gloo")
        else:
            dist.init_process_group("nccl", device_id=dev)
    N = w.N
    t0, t1 = shard.shard_bounds(N, world)[rank]
    T = t1 - t0

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    fmm_arm = args.near_algorithm == "fmm"
    plan = H.Plan.from_workload(w, rsqrt_refine=args.refine, near_algorithm=1 if fmm_arm else 0, fmm_order=args.fmm_order,
                                fmm_levels=args.fmm_levels)
    if args.pair_form != "auto":
        plan.set_pair_form(1 if args.pair_form == "ordered" else 2)
    if args.image_factoring == "off":
        plan.set_image_factoring(False)
    info = plan.info
    refine = args.refine   # 0: resolved after the warm-up (the library decides by the pair count)
    xyz = torch.as_tensor(np.ascontiguousarray(w.xyz), device=dev)
    q = torch.as_tensor(np.ascontiguousarray(w.q), device=dev)
    phi = torch.empty(T, dtype=torch.float64, device=dev)
    U = torch.empty(1, dtype=torch.float64, device=dev)
    force = torch.empty(T, 3, dtype=torch.float64, device=dev) if args.forces else None
    flush = torch.empty(256 * 1024 * 1024 // 8, dtype=torch.float64, device=dev)   # 256 MiB > 126 MB L2

    def step(events=None):
        flush.zero_()                                     # L2 flush between iterations (torch memset, outside the events)
        if events:
            events[0].record()
        if world > 1:
            # check-point sums sharded, then the PART form (or target shards); exchanges: all-gather of the K_t check
            # sums before the fit, all-reduce (or all-gather) of phi (F) and all-reduce of U at the end
            full, _, Uall = shard.evaluate_distributed(plan, xyz, q, forces=args.forces)
            U.copy_(Uall)
        elif args.forces:
            H.hsma_evaluate_forces_shard(plan.handle, xyz, q, t0, t1, phi, force, U)
        else:
            H.hsma_evaluate_shard(plan.handle, xyz, q, t0, t1, phi, U)
        if events:
            events[1].record()

    # peak FP64 (DFMA microbenchmark) before the run: the measured roofline denominator
    dfma_tflops, _ = H.hsma_fp64_peak(args.peak_seconds)

    for _ in range(args.warmup):
        step()
    plan.sync()
    info = H.binding.hsma_plan_info(plan.handle)          # now with the image count of the last evaluate
    plan.set_timing(args.stage_timing == "on")
    stage_ms = {k: 0.0 for k in H.binding.TIMING_KEYS}
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    launches0 = H.hsma_launch_count()
    # device time of EXACTLY args.steps steps: one event pair per step around the evaluate itself, so that the L2 flush
    # written between iterations (a 256 MiB memset, ~0.05 ms) is not in ms_per_step; the whole region, flushes
    # included, is ms_per_step_with_flush
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    for i in range(args.steps):
        step(ev[i])
        if args.stage_timing == "on":
            for k, v in plan.timing().items():           # synchronises the stream once per step
                stage_ms[k] += v
    e1.record()
    barrier()
    launches = H.hsma_launch_count() - launches0
    clocks = sampler.stop()
    ms_with_flush = e0.elapsed_time(e1) / args.steps
    ms = sum(a.elapsed_time(b) for a, b in ev) / args.steps
    plan.set_timing(False)
    U_val = float(U.cpu()[0])
    if world > 1:
        t = torch.tensor([ms], dtype=torch.float64, device="cpu" if share_gpu else dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t[0])
    stage_ms = {k: v / args.steps for k, v in stage_ms.items()}

    # whole-job pairs per step: (a) once (computed redundantly by every rank, counted once), (b), (c) over all N
    pc_all = pair_counts(info, N, N)
    pairs_step = pc_all["a"] + pc_all["b"] + pc_all["c"]
    value = pairs_step / (ms * 1e-3)

    # end to end through the C-ABI with HOST buffers (pinned): H2D of xyz,q and D2H of phi,U inside the timed region
    xyz_h = torch.as_tensor(np.ascontiguousarray(w.xyz)).pin_memory()
    q_h = torch.as_tensor(np.ascontiguousarray(w.q)).pin_memory()
    phi_h = torch.empty(max(T, 1), dtype=torch.float64).pin_memory()
    U_h = torch.empty(1, dtype=torch.float64).pin_memory()
    xyz_n, q_n, phi_n, U_n = xyz_h.numpy(), q_h.numpy(), phi_h.numpy(), U_h.numpy()
    force_n = torch.empty(max(T, 1), 3, dtype=torch.float64).pin_memory().numpy() if args.forces else None

    phi_all_h = torch.empty(N, dtype=torch.float64).pin_memory() if world > 1 else None

    def step_e2e():
        flush.zero_()
        if world > 1:
            # the distributed call a user makes (shard.evaluate_distributed), fed from pinned host memory
            xyz.copy_(xyz_h, non_blocking=True)
            q.copy_(q_h, non_blocking=True)
            full, _, Uall = shard.evaluate_distributed(plan, xyz, q, forces=args.forces)
            phi_all_h.copy_(full, non_blocking=True)
            U_h.copy_(Uall, non_blocking=True)
            torch.cuda.current_stream().synchronize()
        elif args.forces:
            H.hsma_evaluate_forces_host(plan.handle, xyz_n, q_n, phi_n, force_n, U_n)
        else:
            H.hsma_evaluate_shard_host(plan.handle, xyz_n, q_n, t0, t1, phi_n, U_n)   # synchronises (returns host data)

    n_e2e = max(1, min(args.steps, args.e2e_steps))
    step_e2e()
    barrier()
    tw = time.perf_counter()
    for _ in range(n_e2e):
        step_e2e()
    barrier()
    ms_e2e = 1e3 * (time.perf_counter() - tw) / n_e2e
    if world > 1:
        t = torch.tensor([ms_e2e], dtype=torch.float64, device="cpu" if share_gpu else dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_e2e = float(t[0])
    e2e = {"value": pairs_step / (ms_e2e * 1e-3), "unit": UNIT, "ms_per_step": ms_e2e, "steps": n_e2e,
           "h2d_bytes_per_step": int(xyz_n.nbytes + q_n.nbytes),
           "d2h_bytes_per_step": int(8 * N + 8) if world > 1 else int(8 * T + 8 + (24 * T if args.forces else 0)),
           "api": ("shard.evaluate_distributed fed from pinned host buffers (per rank: all sources in, phi and U out)" if world > 1 else
                   ("hsma_evaluate_forces_host" if args.forces else "hsma_evaluate_shard_host") +
                   " (pinned host buffers: all sources in, phi and U out)")}

    # roofline of the dominant kernel: near_sum_kernel over the sources, step (b)
    pc_rank = pair_counts(info, N, T)
    if not refine:
        refine = 2 if float(N) * pc_rank["b"] / max(T, 1) < 2.0 ** 32 else 1
    k_ms = stage_ms["near_source_kernel"] + stage_ms.get("fmm_far_field", 0.0)   # FMM: its far field runs before step (a)
    sm_count = torch.cuda.get_device_properties(dev).multi_processor_count
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except (OSError, ValueError):
        pass
    sm_max_mhz = float(peaks.get("sm_max_mhz") or clocks.get("sm_max_mhz") or 1965.0)
    peak_tf = sm_count * FP64_LANES_PER_SM * 2 * sm_max_mhz * 1e6 * 1e-12
    alg_flops_early = FLOPS_PAIR_CHARGE_FIELD if args.forces else FLOPS_PAIR_CHARGE
    ach_tf = pc_rank["b"] * alg_flops_early / (k_ms * 1e-3) * 1e-12 if k_ms > 0 else 0.0
    uniform_q = bool(np.all(np.abs(w.q) == abs(w.q[0])))
    ex_instr, ex_flops = (EXEC_PAIR_FIELD if args.forces else EXEC_PAIR)[(refine, uniform_q)]
    alg_flops = FLOPS_PAIR_CHARGE_FIELD if args.forces else FLOPS_PAIR_CHARGE
    traffic = NCU_TRAFFIC_BYTES_CFG5 if (args.config == 5 and args.size is None and world == 1 and not args.forces
                                         and not args.paper_timing) else None
    issue_peak = sm_count * FP64_LANES_PER_SM * sm_max_mhz * 1e6          # FP64-pipe thread-instructions/s
    symmetric = plan.last_pair_form == 2
    traffic_source = TRAFFIC_SOURCE
    if symmetric:
        traffic = NCU_TRAFFIC_BYTES_CFG5_SYM if traffic else None
        traffic_source = TRAFFIC_SOURCE_SYM
        units = sym_evaluations(N, info["near_cells"]) // world     # PART form: every rank 1/world of the fine units
        # 18 flops per charge pair (26 with the gradient) x pair EVALUATIONS; the second accumulation
        # of an evaluation (what makes it worth two ordered pairs) is charged only in frac_with_second_accumulation
        alg_flops = FLOPS_PAIR_CHARGE_FIELD if args.forces else FLOPS_PAIR_CHARGE
        alg_flops_2nd = FLOPS_EVAL_SYM_FIELD if args.forces else FLOPS_EVAL_SYM
        ex_instr, ex_flops = (EXEC_EVAL_SYM_FIELD if args.forces else EXEC_EVAL_SYM)[refine]
        ach_tf = units * alg_flops / (k_ms * 1e-3) * 1e-12 if k_ms > 0 else 0.0
        kernel_name = (f"near_sym_field_kernel<{refine}>" if args.forces else f"near_sym_kernel<{refine}>") + \
            " step (b), symmetric form: each unordered pair evaluated once"
        unit_name = "pair evaluations (one unordered source pair in one image cell, feeding phi_i and phi_j)"
    else:
        units = pc_rank["b"]
        kernel_name = (f"near_sum_kernel<R,{refine},{'uniform-|q|' if uniform_q else 'generic'},"
                       f"{'field' if args.forces else 'potential'}> step (b)")
        unit_name = "ordered pair interactions"
    lattice = bool(plan.image_factoring) and plan.last_pair_form in (1, 2)
    frac_survey = None
    if lattice:
        # the factored form needs fewer flops per image pair than SURVEY.md 8(d)'s per-pair count, so 18 x units / time can
        # exceed the FP64 peak: that figure is kept as frac_survey_8d_count (a comparison with the cell-by-cell kernels, not
        # a roofline); `frac` charges the factored formulation's own count
        refl = {W.BC_PERIODIC: (False, False, False), W.BC_MIRROR_CAVITY: (True, True, True),
                W.BC_SLAB_XY_PERIODIC_Z_MIRROR: (False, False, True)}[int(w.kind)]
        frac_survey = ach_tf / peak_tf
        if symmetric:
            traffic = NCU_TRAFFIC_BYTES_CFG5_LAT_SYM if traffic else None
            traffic_source = TRAFFIC_SOURCE_LAT_SYM
        else:
            traffic = None     # no capture of the ordered factored kernel at this size
        ex_instr, ex_flops = lat_counts(tuple(int(x) for x in w.near_shell), refl, refine, bool(args.forces), symmetric)
        alg_flops = ex_flops
        ach_tf = units * alg_flops / (k_ms * 1e-3) * 1e-12 if k_ms > 0 else 0.0
        kernel_name = (("near_lat_sym_field_kernel" if args.forces else "near_lat_sym_kernel") if symmetric else "near_lat_sum_kernel") + \
            f"<refine {refine}, shell {tuple(int(x) for x in w.near_shell)}> step (b), lattice-factored image sums" + \
            (", symmetric form: each unordered pair evaluated once" if symmetric else "")
        unit_name = ("image-pair evaluations (one source pair in one image cell" + (", feeding phi_i and phi_j)" if symmetric else ")"))
    roofline = {"bound": "alu", "kernel": kernel_name, "achieved": ach_tf, "peak": peak_tf,
                "unit": "TFLOP/s", "frac": ach_tf / peak_tf, "traffic": traffic,
                "traffic_source": traffic_source if traffic else None,
                "peak_source": f"derived: {sm_count} SMs x {FP64_LANES_PER_SM} FP64 lanes x 2 x {sm_max_mhz:.0f} MHz "
                               f"(no FP64 entry in MEASURED_PEAKS.json)",
                "units": unit_name, "units_per_launch": units, "flops_per_unit_algorithmic": alg_flops,
                "pair_interactions_per_launch": pc_rank["b"],
                "kernel_ms": k_ms, "kernel_pairs_per_s": pc_rank["b"] / (k_ms * 1e-3) if k_ms > 0 else 0.0,
                "kernel_share_of_step": k_ms / stage_ms["total"] if stage_ms["total"] > 0 else None,
                "flops_per_unit_executed": ex_flops, "fp64_instr_per_unit_executed": ex_instr,
                "frac_executed_flops": units * ex_flops / (k_ms * 1e-3) * 1e-12 / peak_tf if k_ms > 0 else 0.0,
                "fp64_pipe_issue_util": units * ex_instr / (k_ms * 1e-3) / issue_peak if k_ms > 0 else 0.0,
                "dfma_microbench_tflops": dfma_tflops, "frac_of_dfma_microbench": ach_tf / dfma_tflops if dfma_tflops else None}
    roofline["frac_definition"] = ("achieved = units_per_launch x flops_per_unit_algorithmic / kernel time; flops_per_unit_algorithmic = "
                                   "SURVEY.md 8(d)'s count for one charge pair (18; 26 with the gradient), applied to what the "
                                   "kernel evaluates (units); peak = derived FP64 FMA peak")
    roofline["evaluations_per_s"] = units / (k_ms * 1e-3) if k_ms > 0 else 0.0
    if lattice:
        roofline["frac_definition"] = ("achieved = units_per_launch x flops_per_unit_algorithmic / kernel time; the lattice-factored "
                                       "formulation (DESIGN.md 6.14) shares the per-axis squares between all images of a pair, so its "
                                       "algorithmic count per image pair is what it executes (flops_per_unit_algorithmic = "
                                       "flops_per_unit_executed); peak = derived FP64 FMA peak.  fp64_pipe_issue_util is the measure of "
                                       "kernel quality: FP64 instructions issued / (SMs x 64 lanes x clock)")
        roofline["frac_survey_8d_count"] = frac_survey
        roofline["frac_survey_8d_count_note"] = ("SURVEY.md 8(d)'s 18 flops (26 with the gradient) x units / time / peak: what the "
                                                 "cell-by-cell kernels were charged; above 1 here because the factoring removes "
                                                 "work, not a roofline")
    if symmetric and not lattice:
        roofline["frac_with_second_accumulation"] = units * alg_flops_2nd / (k_ms * 1e-3) * 1e-12 / peak_tf if k_ms > 0 else 0.0
        roofline["flops_per_unit_with_second_accumulation"] = alg_flops_2nd
        roofline["launches_per_step_of_this_kernel"] = "waves: the unordered pairs are walked in ceil(column scratch / cap) launches, each followed by a gather (in kernel_ms)"
        # for comparison with the ordered-pair kernel only: the same time charged with 18 flops for every ordered pair
        # interaction it accounts for.  It may exceed 1: the symmetry removes half of the work, it is not a roofline.
        roofline["ordered_pair_equivalent_frac"] = pc_rank["b"] * (FLOPS_PAIR_CHARGE_FIELD if args.forces else FLOPS_PAIR_CHARGE) / (k_ms * 1e-3) * 1e-12 / peak_tf if k_ms > 0 else 0.0

    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": ms, "ms_per_step_with_flush": ms_with_flush, "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f64",
           "data": "synthetic",
           "config": {"workload": w.name, "N": N, "near_cells": info["near_cells"], "p": info["p"], "M": info["M"],
                      "check_targets": info["check_targets"], "pairs_per_step": pc_all, "rsqrt_refine": refine, "forces": bool(args.forces),
                      "image_factoring": bool(plan.image_factoring),
                      "pair_form": "symmetric (each unordered source pair evaluated once; value counts the ordered pair interactions it accounts for)"
                                   if plan.last_pair_form == 2 else "ordered",
                      "parallelism": (f"check-point sums, unordered pairs of (b) and targets of (c) split over {world} rank(s), "
                                      f"sources replicated; all-reduce of phi and U" if world > 1 and plan.last_pair_form == 2 else
                                      f"targets and check-point sums sharded over {world} rank(s), sources replicated")
                                     + ("" if world == 1 else "; stage_ms covers the second phase only (step (a) runs in its own call)"),
                      "l2": "256 MiB flush written between iterations (outside the per-step events of ms_per_step)"},
           "pair_evaluations_per_s": ((pc_all["a"] + pc_all["c"] + sym_evaluations(N, info["near_cells"])) / (ms * 1e-3)
                                      if plan.last_pair_form == 2 else value),
           "plan_scratch_bytes": plan.scratch_bytes,
           "energy": U_val, "stage_ms": stage_ms, "e2e": e2e, "gpu_launches": int(launches),
           "launches_per_step": plan.launches_last_evaluate(),
           "graph_replays": H.binding.hsma_plan_info(plan.handle)["graph_replays"], "clocks": clocks, "roofline": roofline}
    if share_gpu:
        out["rehearsal"] = "HSMA_BENCH_SHARE_GPU=1: all ranks on cuda:0 over a gloo group -- exercises the N > 1 code path, NOT a measurement"
    if fmm_arm:
        fi = H.binding.hsma_plan_fmm_info(plan.handle)
        out["config"]["near_algorithm"] = (f"fmm (order {fi['order']}, two-box separation, leaf level {fi['leaf_level']} = "
                                           f"{fi['leaves']} leaves): steps (a), (b) sub-quadratic, DESIGN.md 6.13; value still "
                                           f"counts the pair interactions of the direct sum it replaces")
        roofline["kernel"] = "fmm step (b): sort + p2m + m2m + m2l_kernel + l2l + leaf_kernel (kernel_ms is the whole stage)"
        for k in ("achieved", "frac", "frac_executed_flops", "fp64_pipe_issue_util", "frac_of_dfma_microbench", "evaluations_per_s"):
            roofline[k] = None     # the direct-sum unit counts do not apply to the FMM; see profiles/ for its kernels
        roofline["traffic"] = None
    elif world == 1 and not args.forces and not args.no_fmm_line and not args.paper_timing:
        # the sub-quadratic form of step (b) on the same workload, measured beside the direct sum (not the headline)
        try:
            with H.Plan.from_workload(w, rsqrt_refine=args.refine, near_algorithm=1, fmm_order=args.fmm_order,
                                      fmm_levels=args.fmm_levels) as pf:
                phi_f = torch.empty(N, dtype=torch.float64, device=dev)
                U_f = torch.empty(1, dtype=torch.float64, device=dev)
                for _ in range(3):
                    H.hsma_evaluate(pf.handle, xyz, q, phi_f, U_f)
                pf.sync()
                f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                nrep = max(3, min(args.steps, 10))
                tot = 0.0
                for _ in range(nrep):
                    flush.zero_()
                    f0.record()
                    H.hsma_evaluate(pf.handle, xyz, q, phi_f, U_f)
                    f1.record()
                    f1.synchronize()
                    tot += f0.elapsed_time(f1)
                pf.set_timing(True)
                H.hsma_evaluate(pf.handle, xyz, q, phi_f, U_f)
                pf.sync()
                tm = pf.timing()
                fi = H.binding.hsma_plan_fmm_info(pf.handle)
                out["fmm"] = {"ms_per_step": tot / nrep, "steps": nrep, "near_source_ms": tm["near_source_kernel"] + tm["fmm_far_field"],
                              "stage_ms": tm,
                              "order": fi["order"], "leaf_level": fi["leaf_level"], "leaves": fi["leaves"], "energy": float(U_f.cpu()[0]),
                              "energy_rel_diff_vs_direct": abs(float(U_f.cpu()[0]) - U_val) / abs(U_val) if U_val else None,
                              "max_phi_rel_diff_vs_direct": float((phi_f - phi).abs().max() / phi.abs().max()),
                              "note": "near_algorithm = FMM (DESIGN.md 6.13): the same evaluate with step (b) by the fast multipole "
                                      "method; parity against the oracle in tests/test_gpu_fmm.py; run `--near-algorithm fmm` for its own line"}
        except H.HsmaError as e:   # geometry the FMM does not tile (non-cubic boxes)
            out["fmm"] = {"unavailable": str(e)}
    plan.close()
    if world > 1:
        dist.destroy_process_group()
    return out if rank == 0 else {}


def run_parts(args, w) -> dict:
    """--parts R: the per-rank device time of the R-rank PART form, measured on ONE GPU one rank at a
    time -- for each part r the two calls rank r makes (its slice of the check sums, then hsma_evaluate_rest_part),
    bracketed by CUDA events.  No collectives and no concurrency are involved: it measures how evenly the pair work
    splits and what a rank computes, not a multi-GPU run (that is `--gpus N` under torchrun)."""
    import torch
    import paper_1806_04801_b200 as H
    from paper_1806_04801_b200 import shard
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    stream = torch.cuda.Stream()
    R, N = args.parts, w.N
    with torch.cuda.stream(stream):
        xyz = torch.as_tensor(np.ascontiguousarray(w.xyz), device=dev)
        q = torch.as_tensor(np.ascontiguousarray(w.q), device=dev)
        with H.Plan.from_workload(w, rsqrt_refine=args.refine) as plan:
            if not H.binding.hsma_plan_part_form_applies(plan.handle, N):
                raise SystemExit("--parts: the PART form does not apply to this workload (needs N > 7936, whole-cell near set)")
            Kt = plan.info["check_targets"]
            phi_ref, U_ref = plan.evaluate(xyz, q, sync=True)
            total = torch.zeros(N, dtype=torch.float64, device=dev)
            rows = []
            for part, (t0, t1) in enumerate(shard.shard_bounds(N, R)):
                c0, c1 = shard.shard_bounds(Kt, R, align=1)[part]
                a = torch.empty(N, dtype=torch.float64, device=dev)
                f = torch.empty(N, 3, dtype=torch.float64, device=dev) if args.forces else None
                u = torch.empty(1, dtype=torch.float64, device=dev)
                best = None
                for _ in range(max(1, args.steps)):
                    e = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
                    plan.sync()
                    e[0].record()
                    H.binding.hsma_check_sums_shard(plan.handle, xyz, q, c0, c1)
                    e[1].record()
                    H.binding.hsma_evaluate_rest_part(plan.handle, xyz, q, part, R, t0, t1, a, f, u)
                    e[2].record()
                    plan.sync()
                    t = (e[0].elapsed_time(e[1]), e[1].elapsed_time(e[2]))
                    best = t if best is None or sum(t) < sum(best) else best
                rows.append({"part": part, "check_sums_ms": best[0], "rest_part_ms": best[1]})
                # for the check of the sum: the fit needs ALL check sums (the all-gather of the real run)
                H.binding.hsma_check_sums_shard(plan.handle, xyz, q, 0, Kt)
                H.binding.hsma_evaluate_rest_part(plan.handle, xyz, q, part, R, t0, t1, a, f, u)
                plan.sync()
                total += a
            err = float((total - phi_ref).abs().max() / phi_ref.abs().max())
    slowest = max(r["check_sums_ms"] + r["rest_part_ms"] for r in rows)
    return {"mode": "parts", "note": "per-rank device time of the PART form, one rank at a time on one GPU; collectives not included",
            "config": {"workload": w.name, "N": N, "forces": bool(args.forces)}, "n_parts": R, "per_part": rows,
            "slowest_rank_ms": slowest, "sum_of_parts_vs_evaluate_max_rel": err}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--config", type=int, default=5, help="BASELINE.json configs[config-1]; 5 = the metric's workload")
    ap.add_argument("--size", type=int, default=None, help="override N (same generator and seed)")
    ap.add_argument("--paper-timing", type=int, default=0, metavar="N",
                    help="the paper's own timing workload instead of a BASELINE.json config (PAPER.md:171,183: lattice "
                         "sites, random signs, alpha=1.3, P=25, N_o=5928, images inside the sphere); N an even cube")
    ap.add_argument("--face-pairs", action="store_true",
                    help="periodic configs: close by seeded value+derivative pairs on opposite faces instead of the "
                         "paper's circumsphere rule (DESIGN.md 6.10)")
    ap.add_argument("--image-factoring", choices=["on", "off"], default="on",
                    help="off: the cell-by-cell pair kernels everywhere (DESIGN.md 6.1, 6.12) instead of the lattice-factored "
                         "ones (6.14) -- for comparison")
    ap.add_argument("--pair-form", choices=["auto", "ordered", "symmetric"], default="auto",
                    help="step (b): auto = symmetric form (each unordered pair once) when one rank evaluates all targets "
                         "; ordered = always near_sum_kernel; symmetric = wherever it applies")
    ap.add_argument("--near-algorithm", choices=["direct", "fmm"], default="direct",
                    help="step (b): direct = the exact pair sum (the metric's kernel, default); fmm = sub-quadratic form "
                         "(DESIGN.md 6.13).  The default line also reports the FMM time of the same workload under \"fmm\"")
    ap.add_argument("--fmm-order", type=int, default=0, help="FMM expansion order (0 = 20)")
    ap.add_argument("--fmm-levels", type=int, default=0, help="FMM leaf level (0 = by N)")
    ap.add_argument("--no-fmm-line", action="store_true", help="skip the extra FMM measurement of the default line")
    ap.add_argument("--forces", action="store_true", help="time hsma_evaluate_forces (potential + forces) instead")
    ap.add_argument("--parts", type=int, default=0, metavar="R",
                    help="one GPU: time what each rank of the R-rank PART form computes, one rank at a time (DESIGN.md 8); "
                         "prints its own JSON line")
    ap.add_argument("--refine", type=int, default=0, choices=[0, 1, 2], help="hsma_plan_desc.rsqrt_refine")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--stage-timing", default="on", choices=["on", "off"],
                    help="off: no per-stage CUDA events (roofline fields are then null) and the library replays the "
                         "evaluate as one CUDA graph -- the latency-bound small configs")
    ap.add_argument("--peak-seconds", type=float, default=1.0)
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="size of the cpu_baseline sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--ref-step-seconds", type=float, default=5.0, help="--impl reference: oracle sample per step")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "b200":
        print(f"note: --warmup {args.warmup} < 3 (timing rules ask for >= 3)", file=sys.stderr)
    w = W.paper_timing(args.paper_timing) if args.paper_timing else W.config(args.config, N=args.size)
    if args.face_pairs:   # BASELINE.json's "check-point pairs on opposite faces", seeded
        w = w.with_(closure=W.CLOSURE_FACE_PAIRS, check_xyz=W.seeded_face_points(w.K, w.L, W.LOWER_FACES, seed=args.config))
    rank = int(os.environ.get("RANK", "0"))
    if args.impl == "reference":
        if rank == 0:
            print(json.dumps(run_reference(args, w)), flush=True)
        return
    if args.parts > 0:
        if rank == 0:
            print(json.dumps(run_parts(args, w)), flush=True)
        return
    out = run_b200(args, w)
    if rank == 0:
        if args.gpus == 1 and not args.no_cpu_baseline and not args.paper_timing:
            out["cpu_baseline"] = cpu_baseline(w, args.cpu_seconds)
        print(json.dumps(out), flush=True)


if __name__ == "__main__":
    main()

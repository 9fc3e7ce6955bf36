"""shard.evaluate_distributed with world = 2 FOR REAL on one GPU: two processes share cuda:0 (time-sliced), rendezvous
over a gloo group (NCCL refuses two ranks on one device; shard.py stages a gloo group's CUDA tensors through host
memory) and call the product function unchanged.  Every phi, F and U on BOTH ranks is compared with the oracle at the
north_star bars and with the one-rank evaluate.  Cases: the PART form (unordered pairs split over the ranks, SURVEY.md
8(e), "two ... GPUs"), target shards (small N), the sphere-culled near set, and derivative rows (face-pair
closure: the all-gather of grad Phi_in at the check targets runs).  All `-m gpu`."""
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import hsma_workloads as W  # noqa: E402
from oracle import hsma_oracle as O  # noqa: E402

pytestmark = pytest.mark.gpu

PHI_TOL, U_TOL, F_TOL = 1e-10, 1e-11, 1e-10


def make_case(name):
    if name == "part":              # PART form applies (N > 7936, whole cells)
        return W.config(5, N=9000), {}
    if name == "part_mirror":       # the same with reflected images (metallic cavity), net charge allowed
        return W.config(3, N=9001), {}
    if name == "shards":            # too small for the symmetric form: contiguous target shards
        return W.config(2, N=3000), {}
    if name == "sphere":            # paper-literal near set: always target shards
        w = W.config(2, N=3000)
        return w.with_(near_mode=W.NEAR_SPHERE), {}
    if name == "face_pairs":        # derivative rows: step (a) in its FIELD form, pcg is gathered too
        w = W.config(5, N=9000)
        return w.with_(closure=W.CLOSURE_FACE_PAIRS, check_xyz=W.seeded_face_points(w.K, w.L, W.LOWER_FACES, seed=5)), {}
    raise KeyError(name)


def _worker(rank, world, port, name, side_stream, out_dir):
    import torch
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import paper_1806_04801_b200 as H
        from paper_1806_04801_b200 import shard
        H.binding.load_library()
        torch.cuda.set_device(0)
        w, kw = make_case(name)
        xyz = torch.as_tensor(np.ascontiguousarray(w.xyz), device="cuda")
        q = torch.as_tensor(np.ascontiguousarray(w.q), device="cuda")
        # the plan lives on its own stream; with side_stream the caller stays on the default stream, so the ordering
        # between the library's stream and the collectives' stream is exercised
        ps = torch.cuda.Stream()
        with torch.cuda.stream(ps):
            plan = H.Plan.from_workload(w, **kw)
        ctx = torch.cuda.stream(ps) if not side_stream else torch.cuda.stream(torch.cuda.default_stream())
        with ctx:
            phi, _, U = shard.evaluate_distributed(plan, xyz, q)
            phi_f, F, U_f = shard.evaluate_distributed(plan, xyz, q, forces=True)
            torch.cuda.current_stream().synchronize()
            out = dict(phi=phi.cpu().numpy(), U=U.cpu().numpy(), phi_f=phi_f.cpu().numpy(), F=F.cpu().numpy(),
                       U_f=U_f.cpu().numpy(), part_form=np.array(H.binding.hsma_plan_part_form_applies(plan.handle, w.N)))
        with torch.cuda.stream(ps):
            one, U1 = plan.evaluate(xyz, q, sync=True)       # the one-rank evaluate of the same plan
            out["one"] = one.cpu().numpy()
            out["U1"] = U1.cpu().numpy()
        plan.close()
        np.savez(os.path.join(out_dir, f"r{rank}.npz"), **out)
        dist.barrier()
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("name,side_stream", [("part", False), ("part", True), ("part_mirror", False), ("shards", False),
                                              ("shards", True), ("sphere", False), ("face_pairs", True)])
def test_evaluate_distributed_two_processes_one_gpu(tmp_path, name, side_stream):
    import torch
    import torch.multiprocessing as mp
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    w, _ = make_case(name)
    r = O.hsma(w, forces=True)
    world, port = 2, 35500 + (os.getpid() * 7 + len(name) * 131 + int(side_stream)) % 2000
    mp.spawn(_worker, args=(world, port, name, side_stream, str(tmp_path)), nprocs=world, join=True)
    fscale = float(np.max(np.abs(r.F)))
    got = [np.load(tmp_path / f"r{k}.npz") for k in range(world)]
    assert int(got[0]["part_form"]) == (1 if name in ("part", "part_mirror", "face_pairs") else 0)
    for g in got:
        for key in ("phi", "phi_f"):
            assert g[key].shape == (w.N,)
            assert np.max(np.abs(g[key] - r.phi)) <= PHI_TOL * np.max(np.abs(r.phi))
            assert np.max(np.abs(g[key] - g["one"])) <= 1e-12 * np.max(np.abs(r.phi))
        for key in ("U", "U_f"):
            assert abs(float(g[key][0]) - r.U) <= U_TOL * abs(r.U)
            assert abs(float(g[key][0]) - float(g["U1"][0])) <= 1e-12 * abs(r.U)
        assert g["F"].shape == (w.N, 3)
        assert np.max(np.abs(g["F"] - r.F)) <= F_TOL * fscale
    # both ranks hold the same bits (the collectives leave identical results everywhere)
    for key in ("phi", "phi_f", "F", "U", "U_f"):
        assert np.array_equal(got[0][key], got[1][key])


def test_bench_refuses_more_ranks_than_devices():
    """bench.py --gpus 2 on a one-GPU box: a clear message, not a CUDA error from set_device."""
    import subprocess
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT="36999")
    import torch
    if torch.cuda.device_count() >= 2:
        pytest.skip("two devices visible: the N = 2 bench itself is the test")
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "1", "--warmup", "1",
                        "--config", "2", "--no-cpu-baseline"], env=env, capture_output=True, text=True, timeout=600)
    assert p.returncode != 0
    assert "visible CUDA device" in (p.stderr + p.stdout)


@pytest.mark.parametrize("extra", [[], ["--forces"], ["--size", "3000", "--config", "2"]])
def test_bench_two_ranks_rehearsal_on_one_gpu(extra):
    """bench.py --gpus 2 exactly as the driver launches it (torch.distributed.run, two ranks), with HSMA_BENCH_SHARE_GPU=1:
    both ranks on cuda:0 over gloo.  The whole N > 1 path of bench.py runs -- rendezvous, barriers, one
    shard.evaluate_distributed per step (PART form at N = 9,000; target shards at N = 3,000), max over ranks, end-to-end
    leg, ONE JSON line from rank 0 with n_gpus = 2 -- and the energy agrees with the one-rank run."""
    import json
    import subprocess
    base = [os.path.join(ROOT, "bench.py"), "--steps", "2", "--warmup", "1", "--no-cpu-baseline", "--e2e-steps", "1",
            "--peak-seconds", "0.1"] + (extra if "--size" in extra else ["--size", "9000"] + extra)
    env = dict(os.environ, HSMA_BENCH_SHARE_GPU="1")
    port = 37100 + (os.getpid() + len(extra)) % 800
    p2 = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
                         "127.0.0.1", "--master-port", str(port)] + base + ["--gpus", "2"], env=env, capture_output=True, text=True,
                        timeout=900)
    assert p2.returncode == 0, p2.stderr[-2000:]
    lines = [ln for ln in p2.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, p2.stdout[-2000:]
    d2 = json.loads(lines[0])
    assert d2["n_gpus"] == 2 and d2["ms_per_step"] > 0 and d2["value"] > 0 and d2["gpu_launches"] > 0 and "rehearsal" in d2
    p1 = subprocess.run([sys.executable] + base + ["--no-fmm-line"], capture_output=True, text=True, timeout=900)
    assert p1.returncode == 0, p1.stderr[-2000:]
    d1 = json.loads([ln for ln in p1.stdout.splitlines() if ln.startswith("{")][0])
    assert abs(d2["energy"] - d1["energy"]) <= 1e-11 * abs(d1["energy"])
    assert d2["config"]["pairs_per_step"] == d1["config"]["pairs_per_step"]

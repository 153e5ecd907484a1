"""Host-side logic of bench.py on CPU: replicas-only aggregation under world_size-2 gloo,
the reference arm's rank handling, and the JSON contract of the `--impl reference` line."""
import json
import os
import socket
import subprocess
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as tmp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close()
    return p


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    # rank r took (10 + 5 r) ms for (1000 + 100 r) iterations
    t, u = bench.aggregate(dist, 10.0 + 5.0 * rank, 1000.0 + 100.0 * rank, torch.device("cpu"))
    out.put((rank, t, u))
    dist.barrier()
    dist.destroy_process_group()


def test_aggregate_world2_gloo():
    ctx = tmp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs: p.start()
    got = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(60); assert p.exitcode == 0
    for rank, t, u in got:
        assert t == 15.0          # max over ranks
        assert u == 2100.0        # sum over ranks: whole-job units
    # whole-job value = sum(units) / max(time)
    assert got[0][2] / (got[0][1] * 1e-3) == pytest.approx(140000.0)


def test_aggregate_single_process():
    import bench
    assert bench.aggregate(None, 3.5, 7.0, torch.device("cpu")) == (3.5, 7.0)


def _run_reference(rank, world):
    env = dict(os.environ, RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank))
    return subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "cfg1",
                           "--gpus", str(world), "--steps", "1", "--warmup", "0"], env=env, capture_output=True,
                          text=True, timeout=300)


def test_reference_arm_rank0_prints_contract_line():
    p = _run_reference(0, 2)
    assert p.returncode == 0, p.stderr
    line = json.loads(p.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["metric"] == "mp_iterations_per_s" and line["higher_is_better"]
    assert line["value"] > 0 and line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["value"] == line["value"]
    assert line["e2e"]["value"] == line["value"] and line["e2e"]["h2d_bytes_per_step"] == 0
    assert line["gpu_launches"] == 0 and line["vs_baseline"] is None and "workload" in line["config"]


def test_reference_arm_other_ranks_exit_silently():
    p = _run_reference(1, 2)
    assert p.returncode == 0 and p.stdout.strip() == ""


def test_grading_drift_caps_hold_for_a_run_within_g3_and_catch_one_outside():
    """tests/grading.py caps the state drift behind R14b / R16b by what G3 tolerates (||d|| <= sum_s c_tol ||r_s||) and by fixed
    ceilings.  A stand-in for a GPU run is made on the host -- the MP trajectory with every step perturbed by up to half the G3
    tolerance, as fp32 dot products would -- and must be graded clean with the caps in place; the session-level use counts must
    leave room for what the full GPU session is known to need."""
    import numpy as np
    import grading
    import oracle
    import problems
    pb = problems.make_problem(problems.custom_config(96, 300, 8, eps=1e-5, max_iter=40), seed=5)
    y = pb.Y[0]
    ref = oracle.mp(pb.psi32, y.astype(np.float64), float(np.float32(pb.cfg.eps)), pb.cfg.max_iter, 1)
    rng = np.random.default_rng(0)
    # replay the oracle's atoms with perturbed steps: c_s = <r_s, psi> + 0.5 * C_TOL * ||r_s|| * u, u in [-1, 1]
    r = y.astype(np.float64).copy()
    idx, c = [], []
    ny = np.linalg.norm(r)
    thr = float(np.float32(pb.cfg.eps)) * ny
    x = np.zeros(pb.cfg.M)
    while np.linalg.norm(r) > thr and len(idx) < pb.cfg.max_iter:
        corr = pb.psi32.astype(np.float64) @ r
        i = int(np.argmax(np.abs(corr)))
        step = float(np.float32(corr[i] + 0.5 * grading.C_TOL * np.linalg.norm(r) * rng.uniform(-1, 1)))
        idx.append(i); c.append(step)
        x[i] += step
        r -= step * pb.psi32[i].astype(np.float64)
    g = grading.grade_single(pb.psi32, y, pb.cfg.eps, pb.cfg.max_iter, x.astype(np.float32), r.astype(np.float32), len(idx),
                             np.array(idx, np.int32), np.array(c, np.float32), ref=ref, nthreads=1)
    assert g.max_c_err <= grading.C_TOL and g.g1_allowance <= grading.G1_ALLOWANCE_CEILING
    assert grading.G1_ALLOWANCE_MAX_USES >= 33 and grading.N_ITER_DRIFT_MAX_USES >= 1      # the full GPU session's counts fit


def test_traffic_capture_is_not_older_than_the_kernel_sources():
    """profiles/dominant_kernel_traffic.txt (the ncu DRAM traffic bench.py multiplies into roofline.traffic) names the commit it was
    captured at; no later commit may have touched the dominant kernel's sources.  Needs the git history (skipped without it)."""
    import subprocess
    import bench
    import shutil
    if not os.path.isdir(os.path.join(bench.ROOT, ".git")) or shutil.which("git") is None:
        pytest.skip("no git history (or no git) here")
    kv = {}
    for line in open(os.path.join(bench.ROOT, "profiles", "dominant_kernel_traffic.txt")):
        if "=" in line and not line.lstrip().startswith("#"):
            k, _, v = line.partition("=")
            kv[k.strip()] = v.split("#")[0].strip()
    have = subprocess.run(["git", "-C", bench.ROOT, "cat-file", "-e", kv["commit"] + "^{commit}"], capture_output=True)
    if have.returncode != 0:
        pytest.skip("the capture's commit is not in this (shallow?) history")
    assert bench.capture_is_stale(kv["commit"]) == ""
    first = subprocess.run(["git", "-C", bench.ROOT, "rev-list", "--max-parents=0", "HEAD"], capture_output=True, text=True).stdout.split()[0]
    assert "re-capture" in bench.capture_is_stale(first)          # the check does fire for a capture that predates the kernel

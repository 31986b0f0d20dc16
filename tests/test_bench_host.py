"""Host-side logic of bench.py that needs no GPU: the replicas-only multi-rank aggregation
(world_size 2 over gloo) and the reference arm's rank handling."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    import torch
    import torch.distributed as dist

    sys.path.insert(0, ROOT)
    import bench

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms_local = 10.0 + 5.0 * rank  # rank 1 is the slow replica
    ms_max = bench.max_over_ranks(ms_local, world, torch.device("cpu"))
    out[rank] = (ms_max, bench.whole_job_value(1000, 4, world, ms_max))
    dist.barrier()
    dist.destroy_process_group()


def test_replicas_take_the_slowest_rank_gloo_world2():
    import torch.multiprocessing as mp

    ctx = mp.get_context("spawn")
    out = ctx.Manager().dict()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    # both ranks agree on the slowest time; the job advanced 2 replicas x 1000 atoms x 4 steps in 15 ms
    assert out[0] == out[1]
    assert out[0][0] == 15.0
    assert out[0][1] == pytest.approx(2 * 1000 * 4 / 15e-3)


def test_single_rank_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench

    assert bench.max_over_ranks(7.5, 1, None) == 7.5
    assert bench.whole_job_value(1 << 20, 20, 1, 20.0) == pytest.approx((1 << 20) * 20 / 20e-3)


def test_reference_arm_other_ranks_exit_quietly():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"],
                       env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.strip() == ""


def test_stage_model_covers_every_stage_name():
    sys.path.insert(0, ROOT)
    import bench
    import workloads as wl

    w = wl.li3po4_box(1024)
    for forces in ("gather", "pairbuf"):
        sm = bench.stage_model(w, 143.5, 90.3, 446976, "3xtf32", forces)
        for name in ("gather", "pair_forward", "contract_forward", "mlp_forward", "mlp_heads", "mlp_backward",
                     "contract_backward", "pair_backward", "outputs", "kick_drift", "kick_ke", "rebuild_if_moved"):
            assert name in sm and sm[name]["bound"] in ("hbm", "alu", "tensor")
    # the pair buffer halves the pair-gradient flops and pays for it in bytes
    g = bench.stage_model(w, 143.5, 90.3, 446976, "3xtf32", "gather")["pair_backward"]
    p = bench.stage_model(w, 143.5, 90.3, 446976, "3xtf32", "pairbuf")["pair_backward"]
    assert p["flops"] < g["flops"] and p["bytes"] > g["bytes"]

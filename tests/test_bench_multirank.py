"""CPU, world_size 2 over gloo: bench.py's N > 1 path ("replicas only": every rank times an independent
replica; the job's time is the MAX over ranks and `value` = units of all ranks / that time), and the
reference arm's rank-0-only behaviour."""
import json
import os
import subprocess
import sys

import pytest
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    sys.path.insert(0, ROOT)
    import bench
    r, local, w = bench.dist_init(use_cuda=False)
    assert (r, local, w) == (rank, rank, world)
    bench.barrier(w, use_cuda=False)
    local_ms = 100.0 * (rank + 1)                      # rank 1 is the slow replica
    mx = bench.max_over_ranks(local_ms, w, use_cuda=False)
    value, ms_per_step = bench.aggregate_value(7.0, steps=10, world=w, local_ms_total=local_ms, use_cuda=False)
    q.put((rank, mx, value, ms_per_step))
    import torch.distributed as dist
    dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_value_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29600 + os.getpid() % 300
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, mx, value, ms_per_step in res:
        assert mx == 200.0                              # max over ranks, on every rank
        assert ms_per_step == 20.0
        assert value == pytest.approx(7.0 * 2 / 20e-3)  # units of BOTH ranks / slowest time


def test_reference_arm_prints_one_line_on_rank0_only():
    env = dict(os.environ, WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT="29911")
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "1", "--steps", "1",
           "--warmup", "0", "--ref-rows", "16", "--gpus", "2"]
    out1 = subprocess.run(cmd, env=dict(env, RANK="1", LOCAL_RANK="1"), capture_output=True, text=True, timeout=300)
    assert out1.returncode == 0 and out1.stdout.strip() == ""
    out0 = subprocess.run(cmd, env=dict(env, RANK="0", LOCAL_RANK="0"), capture_output=True, text=True, timeout=300)
    assert out0.returncode == 0, out0.stderr
    line = json.loads(out0.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["value"] > 0
    assert line["e2e"]["value"] == line["value"] and line["e2e"]["h2d_bytes_per_step"] == 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    for key in ("metric", "unit", "steps", "warmup", "ms_per_step", "higher_is_better", "config"):
        assert key in line


# ---------------------------------------------------------------------------------------------
# hcms_dist: host-side plumbing of the multi-rank path, no GPU
# ---------------------------------------------------------------------------------------------

def _gather_worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    import paper_2607_01817_b200 as H
    dist.init_process_group("gloo", rank=rank, world_size=world)
    blob = bytes([rank + 1]) * H.HCMS_DIST_HANDLE_BYTES                # stands in for this rank's export handle
    parts = H.all_gather_bytes(blob)
    q.put((rank, [p[0] for p in parts], [len(p) for p in parts]))
    dist.destroy_process_group()


def test_handle_exchange_is_rank_ordered_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29950 + os.getpid() % 40
    procs = [ctx.Process(target=_gather_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, firsts, lens in res:
        assert firsts == [1, 2] and lens == [128, 128]                 # rank order, on every rank


def test_dist_plan_validation_precedes_device_use():
    sys.path.insert(0, ROOT)
    import paper_2607_01817_b200 as H
    for args, code in [((1024, 4, 64, 2, 2, 2), H.HCMS_ERR_INVALID_ARG),            # rank >= P
                       ((1024, 4, 64, 2, 3, 0), H.HCMS_ERR_UNSUPPORTED_SHAPE),      # C > H/P
                       ((1000, 4, 64, 3, 1, 0), H.HCMS_ERR_UNSUPPORTED_SHAPE),      # S % P
                       ((1024, 4, 96, 2, 1, 0), H.HCMS_ERR_UNSUPPORTED_SHAPE),      # D
                       ((1088, 34, 64, 17, 1, 0), H.HCMS_ERR_UNSUPPORTED_SHAPE)]:   # P > 16 peers
        with pytest.raises(H.HcmsError) as ei:
            H.hcms_dist_plan(*args)
        assert ei.value.status == code, args
    with pytest.raises(H.HcmsError) as ei:
        H.hcms_dist_plan(1024, 4, 64, 2, 2, 0, H.HCMS_DTYPE_F32)
    assert ei.value.status == H.HCMS_ERR_UNSUPPORTED_DTYPE
    assert H.lib.hcms_dist_block_bytes(None) == 0 and H.lib.hcms_dist_plan_destroy(None) == 0
    assert H.lib.hcms_dist_attention_forward(None, None, None, None, None, 1.0, None) == H.HCMS_ERR_INVALID_ARG

"""Worker of tests/test_gpu_dist.py::test_ranks_as_processes_over_cuda_ipc and of bench.py's multi-rank smoke: one
process per HCMS rank, all on cuda:0 (one GPU per run here), handles exchanged over gloo.

    python tests/dist_worker.py --spawn P --S .. --H .. --D .. --C ..      one process per rank (CUDA IPC)
    python tests/dist_worker.py --local P --S .. --H .. --D .. --C ..      P ranks in this process (hcms_dist_attach_local)

--local drives the P ranks with hcms_dist_attention_forward_group (phase-by-phase enqueue; see hcms.h).

Every process has a watchdog: a rank that cannot finish within 120 s kills itself, so a broken exchange never hangs
the GPU box.  Holds no method arithmetic: inputs from hcms_inputs, expected bits from the single-device emulation."""
import argparse
import faulthandler
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def worker(rank, world, port, a):
    faulthandler.dump_traceback_later(120, exit=True)
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    import numpy as np
    import torch
    import torch.distributed as dist

    import hcms_inputs as I
    import paper_2607_01817_b200 as H

    torch.cuda.set_device(0)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    S, Hh, D, P, C = a.S, a.H, a.D, world, a.C
    w = I.Workload("distproc", S, Hh, D, P, C, 72, "bf16", 1.0)
    q, k, v = I.make_qkv(w)
    Sl = S // P
    dev = [torch.from_numpy(t[rank * Sl:(rank + 1) * Sl].view(np.int16).copy()).to("cuda:0") for t in (q, k, v)]
    out = torch.empty_like(dev[0])
    plan = H.hcms_dist_plan(S, Hh, D, P, C, rank, H.HCMS_DTYPE_BF16, a.flags)
    H.hcms_dist_exchange_handles(plan)                       # all_gather of 128 bytes per rank over gloo, then attach
    gathered = None
    for rep in range(3):
        out.fill_(0x7FC0)
        torch.cuda.synchronize()
        dist.barrier()
        H.hcms_dist_attention_forward(plan, dev[0], dev[1], dev[2], out, w.scale)
        torch.cuda.synchronize()
        mine = out.cpu().view(torch.uint8)                   # gloo has no int16 collectives
        parts = [torch.empty_like(mine) for _ in range(world)]
        dist.all_gather(parts, mine)
        gathered = torch.cat(parts, dim=0).numpy().view(np.uint16)
        if rank == 0:
            qd, kd, vd = (torch.from_numpy(t.view(np.int16)).to("cuda:0") for t in (q, k, v))
            want = torch.empty_like(qd)
            with H.hcms_plan(S, Hh, D, P, C) as ref_plan:
                H.hcms_attention_forward(ref_plan, qd, kd, vd, want, w.scale)
                torch.cuda.synchronize()
            assert np.array_equal(gathered, want.cpu().numpy().view(np.uint16)), f"call {rep}: ranks differ from the emulation"
    torch.cuda.synchronize()
    dist.barrier()                                           # nobody unmaps while a peer may still read
    plan.close()
    dist.barrier()
    dist.destroy_process_group()
    if rank == 0:
        print("DIST_OK", flush=True)


def local(a):
    """P ranks driven by this one process: distinct caller streams, the group call, three epochs."""
    faulthandler.dump_traceback_later(120, exit=True)
    import numpy as np
    import torch

    import hcms_inputs as I
    import paper_2607_01817_b200 as H

    torch.cuda.set_device(0)
    S, Hh, D, P, C = a.S, a.H, a.D, a.local, a.C
    w = I.Workload("distlocal", S, Hh, D, P, C, 71, "bf16", 1.0)
    q, k, v = I.make_qkv(w)
    qd, kd, vd = (torch.from_numpy(t.view(np.int16)).to("cuda:0") for t in (q, k, v))
    want = torch.empty_like(qd)
    with H.hcms_plan(S, Hh, D, P, C) as ref_plan:
        H.hcms_attention_forward(ref_plan, qd, kd, vd, want, w.scale)
        torch.cuda.synchronize()
    want = want.cpu().numpy().view(np.uint16)
    Sl = S // P
    shards = [[t[r * Sl:(r + 1) * Sl].contiguous() for t in (qd, kd, vd)] for r in range(P)]
    outs = [torch.empty_like(shards[r][0]) for r in range(P)]
    streams = [torch.cuda.Stream() for _ in range(P)]
    plans = [H.hcms_dist_plan(S, Hh, D, P, C, r, H.HCMS_DTYPE_BF16, a.flags) for r in range(P)]
    for pl in plans:
        H.hcms_dist_attach_local(pl, plans)
    for rep in range(3):
        for o in outs:
            o.fill_(0x7FC0)
        torch.cuda.synchronize()
        H.hcms_dist_attention_forward_group(plans, [s[0] for s in shards], [s[1] for s in shards], [s[2] for s in shards],
                                            outs, w.scale, streams)
        for s in streams:
            s.synchronize()
        got = torch.cat(outs, dim=0).cpu().numpy().view(np.uint16)
        assert np.array_equal(got, want), f"call {rep}: ranks differ from the emulation"
    # push + signal + attention + signal (+ pull) per chunk; the fused form has no pull kernel
    assert H.hcms_dist_last_launch_count(plans[0]) == (4 if a.flags & H.HCMS_FLAG_DIST_FUSE_OUT else 5) * C
    torch.cuda.synchronize()
    for pl in plans:
        pl.close()
    print("DIST_OK", flush=True)


def _layer_reference(H, I, np, torch, w, S, Hh, D, P, C):
    """y of the single-device layer (hcms_layer_forward) on the whole sequence, and the layer inputs on the device."""
    Dm = Hh * D
    x, w_qkv, w_o, cos, sin = I.make_layer_inputs(w)
    xd, wqd, wod = (torch.from_numpy(t.view(np.int16)).to("cuda:0") for t in (x, w_qkv, w_o))
    cd, sd = (torch.from_numpy(t).to("cuda:0") for t in (cos, sin))
    want = torch.full((S, Dm), 0x7FC0, dtype=torch.int16, device="cuda:0")
    with H.hcms_plan(S, Hh, D, P, C) as ref_plan:
        H.hcms_layer_forward(ref_plan, xd, wqd, wod, cd, sd, want, Dm, w.scale)
        torch.cuda.synchronize()
    return (xd, wqd, wod, cd, sd), want.cpu().numpy().view(np.uint16)


def local_layer(a):
    """The whole layer between P in-process ranks (hcms_dist_layer_forward_group): both all-to-alls inside the GEMM /
    attention epilogues; concatenated y bit-equal to hcms_layer_forward, three epochs."""
    faulthandler.dump_traceback_later(150, exit=True)
    import numpy as np
    import torch

    import hcms_inputs as I
    import paper_2607_01817_b200 as H

    torch.cuda.set_device(0)
    S, Hh, D, P, C = a.S, a.H, a.D, a.local, a.C
    Dm, Sl = Hh * D, S // P
    w = I.Workload("distlayer", S, Hh, D, P, C, 73, "bf16", 1.0)
    (xd, wqd, wod, cd, sd), want = _layer_reference(H, I, np, torch, w, S, Hh, D, P, C)
    sl = lambda t, r: t[r * Sl:(r + 1) * Sl].contiguous()
    xs, coss, sins = ([sl(t, r) for r in range(P)] for t in (xd, cd, sd))
    ys = [torch.empty((Sl, Dm), dtype=torch.int16, device="cuda:0") for _ in range(P)]
    streams = [torch.cuda.Stream() for _ in range(P)]
    plans = [H.hcms_dist_plan(S, Hh, D, P, C, r, H.HCMS_DTYPE_BF16, a.flags | H.HCMS_FLAG_DIST_FUSE_OUT) for r in range(P)]
    for pl in plans:
        H.hcms_dist_attach_local(pl, plans)
    for rep in range(3):
        for y in ys:
            y.fill_(0x7FC0)
        torch.cuda.synchronize()
        H.hcms_dist_layer_forward_group(plans, xs, wqd, wod, coss, sins, ys, Dm, w.scale, streams)
        for s in streams:
            s.synchronize()
        got = torch.cat(ys, dim=0).cpu().numpy().view(np.uint16)
        assert np.array_equal(got, want), f"call {rep}: the ranks' y differs from hcms_layer_forward"
    assert H.hcms_dist_last_launch_count(plans[0]) == 3 * C + 2        # QKV GEMM + C signals + C attention + C signals + out GEMM
    torch.cuda.synchronize()
    for pl in plans:
        pl.close()
    print("DIST_OK", flush=True)


def worker_layer(rank, world, port, a):
    """One PROCESS per rank: hcms_dist_layer_forward over CUDA IPC, rank 0 checks the all-gathered y."""
    faulthandler.dump_traceback_later(150, exit=True)
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    import numpy as np
    import torch
    import torch.distributed as dist

    import hcms_inputs as I
    import paper_2607_01817_b200 as H

    torch.cuda.set_device(0)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    S, Hh, D, P, C = a.S, a.H, a.D, world, a.C
    Dm, Sl = Hh * D, S // P
    w = I.Workload("distlayer", S, Hh, D, P, C, 73, "bf16", 1.0)
    (xd, wqd, wod, cd, sd), want = _layer_reference(H, I, np, torch, w, S, Hh, D, P, C)
    sl = lambda t: t[rank * Sl:(rank + 1) * Sl].contiguous()
    x, cos, sin = sl(xd), sl(cd), sl(sd)
    y = torch.empty((Sl, Dm), dtype=torch.int16, device="cuda:0")
    plan = H.hcms_dist_plan(S, Hh, D, P, C, rank, H.HCMS_DTYPE_BF16, a.flags | H.HCMS_FLAG_DIST_FUSE_OUT)
    H.hcms_dist_exchange_handles(plan)
    for rep in range(3):
        y.fill_(0x7FC0)
        torch.cuda.synchronize()
        dist.barrier()
        H.hcms_dist_layer_forward(plan, x, wqd, wod, cos, sin, y, Dm, w.scale)
        torch.cuda.synchronize()
        mine = y.cpu().view(torch.uint8)
        parts = [torch.empty_like(mine) for _ in range(world)]
        dist.all_gather(parts, mine)
        if rank == 0:
            got = torch.cat(parts, dim=0).numpy().view(np.uint16).reshape(S, Dm)
            assert np.array_equal(got, want), f"call {rep}: the ranks' y differs from hcms_layer_forward"
    torch.cuda.synchronize()
    dist.barrier()
    plan.close()
    dist.barrier()
    dist.destroy_process_group()
    if rank == 0:
        print("DIST_OK", flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--spawn", type=int, default=0)
    ap.add_argument("--local", type=int, default=0)
    for name in ("S", "H", "D", "C"):
        ap.add_argument("--" + name, type=int, required=True)
    ap.add_argument("--layer", type=int, default=0, help="1: the whole layer (hcms_dist_layer_forward[_group])")
    ap.add_argument("--flags", type=int, default=0, help="hcms_dist_plan flags (HCMS_FLAG_DIST_FUSE_OUT, HCMS_FLAG_ATTN_PAIR)")
    a = ap.parse_args()
    if a.local:
        (local_layer if a.layer else local)(a)
        return
    import torch.multiprocessing as mp
    port = 29700 + os.getpid() % 200
    ctx = mp.get_context("spawn")
    procs = [ctx.Process(target=worker_layer if a.layer else worker, args=(r, a.spawn, port, a)) for r in range(a.spawn)]
    for p in procs:
        p.start()
    code = 0
    for p in procs:
        p.join(timeout=200)
        if p.is_alive():
            p.kill()
            code = 1
        elif p.exitcode != 0:
            code = 1
    sys.exit(code)


if __name__ == "__main__":
    main()

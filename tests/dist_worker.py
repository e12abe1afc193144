"""Worker of tests/test_gpu_dist.py (bench.py does not use it): one process per HCMS rank, all on cuda:0 (one GPU per run
here), handles exchanged over gloo.

    python tests/dist_worker.py --spawn P --S .. --H .. --D .. --C ..      one process per rank (CUDA IPC)
    python tests/dist_worker.py --local P --S .. --H .. --D .. --C ..      P ranks in this process (hcms_dist_attach_local)
    python tests/dist_worker.py --fail P  --S .. --H .. --D .. --C ..      the error path (HCMS_FLAG_DEBUG_DIST_FAIL)

--local drives the P ranks with hcms_dist_attention_forward_group (phase-by-phase enqueue; see hcms.h).

Every process has a watchdog: a rank that cannot finish within 120 s kills itself, so a broken exchange never hangs
the GPU box.  Holds no method arithmetic: inputs from hcms_inputs; the ranks' concatenated result is compared bit for
bit with the single-device emulation AND, element by element, with the fp64 oracle (oracle/, test infrastructure) at
the north-star gates (max |err| <= 2e-2, mean |err| <= 2e-3) plus relative L2 <= 1e-2."""
import argparse
import faulthandler
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def check_against_oracle(got_bits, ref, what):
    """got_bits: bf16 bit patterns (uint16) of the ranks' concatenated result; ref: the oracle's fp64 array, same shape."""
    import numpy as np
    got = (got_bits.astype(np.uint32) << np.uint32(16)).view(np.float32).astype(np.float64).reshape(ref.shape)
    assert not np.isnan(got).any(), f"{what}: NaN (a tile was never delivered)"
    err = np.abs(got - ref)
    rel = np.linalg.norm(got - ref) / np.linalg.norm(ref)
    assert err.max() <= 2e-2 and err.mean() <= 2e-3 and rel <= 1e-2, \
        f"{what} vs the fp64 oracle: max_abs={err.max():.3e} mean_abs={err.mean():.3e} rel_l2={rel:.3e}"


BIG = 8192      # above this S the oracle is evaluated on sampled rows (boundary rows of every rank's shard + seeded rows)


def oracle_check_attention(got_bits, q, k, v, scale, P, what):
    """Whole tensor against attention_full for small S; O.sample_rows / attention_sampled at BASELINE.json's full sizes."""
    from oracle import hcms_oracle as O
    S = q.shape[0]
    if S <= BIG:
        check_against_oracle(got_bits, O.attention_full(q, k, v, scale), what)
    else:
        rows = O.sample_rows(S, P)
        check_against_oracle(got_bits.reshape(q.shape)[rows], O.attention_sampled(q, k, v, scale, rows), what + " (sampled rows)")


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
            if rep == 2:
                from oracle import hcms_oracle as O
                check_against_oracle(gathered, O.attention_full(q, k, v, w.scale), f"{world} processes")
    # the host-buffer entry point: pinned host shards in, this rank's output shard out, same bits as the device call
    host_in = [t.cpu().pin_memory() for t in dev]
    host_out = torch.full_like(host_in[0], 0x7FC0).pin_memory()
    dist.barrier()
    H.hcms_dist_attention_forward_host(plan, host_in[0], host_in[1], host_in[2], host_out, w.scale)
    assert torch.equal(host_out, out.cpu()), "hcms_dist_attention_forward_host differs from the device call"
    torch.cuda.synchronize()
    dist.barrier()                                           # nobody unmaps while a peer may still read
    plan.close()
    dist.barrier()
    dist.destroy_process_group()
    if rank == 0:
        print("DIST_OK", flush=True)


def local(a):
    """P ranks driven by this one process: distinct caller streams, the group call, three epochs."""
    faulthandler.dump_traceback_later(120 if a.S <= BIG else 400, exit=True)
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
    oracle_check_attention(got, q, k, v, w.scale, P, f"{P} in-process ranks")
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
    return (xd, wqd, wod, cd, sd), want.cpu().numpy().view(np.uint16), (x, w_qkv, w_o, cos, sin)


def check_layer_against_oracle(got_bits, host_inputs, Hh, D, scale, what):
    from oracle import hcms_layer_oracle as L
    check_against_oracle(got_bits, L.layer_forward(*host_inputs, Hh, D, scale), what)


def local_layer(a):
    """The whole layer between P in-process ranks (hcms_dist_layer_forward_group): both all-to-alls inside the GEMM /
    attention epilogues; concatenated y bit-equal to hcms_layer_forward, three epochs."""
    faulthandler.dump_traceback_later(150 if a.S <= BIG else 400, exit=True)
    import numpy as np
    import torch

    import hcms_inputs as I
    import paper_2607_01817_b200 as H

    torch.cuda.set_device(0)
    S, Hh, D, P, C = a.S, a.H, a.D, a.local, a.C
    Dm, Sl = Hh * D, S // P
    w = I.Workload("distlayer", S, Hh, D, P, C, 73, "bf16", 1.0)
    (xd, wqd, wod, cd, sd), want, host_inputs = _layer_reference(H, I, np, torch, w, S, Hh, D, P, C)
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
    if S <= BIG:      # at full size the layer oracle needs K, V of every token in fp64 (minutes): there the reference is
        #                 hcms_layer_forward, whose parts are oracle-checked at these sizes in test_gpu_fullsize_next.py
        check_layer_against_oracle(got, host_inputs, Hh, D, w.scale, f"layer, {P} in-process ranks")
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
    (xd, wqd, wod, cd, sd), want, host_inputs = _layer_reference(H, I, np, torch, w, S, Hh, D, P, C)
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
            if rep == 2:
                check_layer_against_oracle(got, host_inputs, Hh, D, w.scale, f"layer, {world} processes")
    torch.cuda.synchronize()
    dist.barrier()
    plan.close()
    dist.barrier()
    dist.destroy_process_group()
    if rank == 0:
        print("DIST_OK", flush=True)


def local_fail(a):
    """The error path of the forward calls (include/hcms.h, "Failure of a forward call"): with HCMS_FLAG_DEBUG_DIST_FAIL the
    attention phase fails after the pushes and a flag wait are enqueued.  The call must return the error, the caller
    streams and the plans' own streams must drain (before the fix S_comm waited for ready flags that no kernel would ever
    publish, and both the caller and hcms_dist_plan_destroy blocked for good), later calls must be refused, and an error
    found by the argument checks must leave a healthy plan usable."""
    faulthandler.dump_traceback_later(60, exit=True)
    import numpy as np
    import torch

    import hcms_inputs as I
    import paper_2607_01817_b200 as H

    torch.cuda.set_device(0)
    S, Hh, D, P, C = a.S, a.H, a.D, a.fail, a.C
    w = I.Workload("distfail", S, Hh, D, P, C, 74, "bf16", 1.0)
    q, k, v = I.make_qkv(w)
    qd, kd, vd = (torch.from_numpy(t.view(np.int16)).to("cuda:0") for t in (q, k, v))
    Sl = S // P
    shards = [[t[r * Sl:(r + 1) * Sl].contiguous() for t in (qd, kd, vd)] for r in range(P)]
    outs = [torch.empty_like(shards[r][0]) for r in range(P)]
    streams = [torch.cuda.Stream() for _ in range(P)]
    group_args = ([s[0] for s in shards], [s[1] for s in shards], [s[2] for s in shards], outs, w.scale, streams)

    def status_of(fn):
        try:
            fn()
        except H.HcmsError as e:
            return e.status, str(e)
        return H.HCMS_OK, ""

    # (1) the group call: P in-process ranks
    plans = [H.hcms_dist_plan(S, Hh, D, P, C, r, H.HCMS_DTYPE_BF16, a.flags | H.HCMS_FLAG_DEBUG_DIST_FAIL) for r in range(P)]
    for pl in plans:
        H.hcms_dist_attach_local(pl, plans)
    st, text = status_of(lambda: H.hcms_dist_attention_forward_group(plans, *group_args))
    assert st == H.HCMS_ERR_CUDA and "injected failure" in text, (st, text)
    for s in streams:
        s.synchronize()                      # the joins were enqueued and nothing waits on an unpublished flag
    torch.cuda.synchronize()
    st, text = status_of(lambda: H.hcms_dist_attention_forward_group(plans, *group_args))
    assert st == H.HCMS_ERR_INVALID_ARG and "earlier forward call" in text, (st, text)      # poisoned, nothing enqueued
    torch.cuda.synchronize()
    for pl in plans:
        pl.close()                           # synchronises the plan's streams: returns
    # (2) one process per rank, P = 1 (attached through an exported handle, so the single-rank call applies)
    out1 = torch.empty_like(qd)
    for layer in (0, 1):
        flags = a.flags | H.HCMS_FLAG_DEBUG_DIST_FAIL | (H.HCMS_FLAG_DIST_FUSE_OUT if layer else 0)
        with H.hcms_dist_plan(S, Hh, D, 1, C, 0, H.HCMS_DTYPE_BF16, flags) as pl:
            H.hcms_dist_attach(pl, [H.hcms_dist_export(pl)])
            if layer:
                Dm = Hh * D
                x, w_qkv, w_o, cos, sin = (torch.from_numpy(t.view(np.int16) if t.dtype == np.uint16 else t).to("cuda:0")
                                           for t in I.make_layer_inputs(w))
                y = torch.empty((S, Dm), dtype=torch.int16, device="cuda:0")
                call = lambda: H.hcms_dist_layer_forward(pl, x, w_qkv, w_o, cos, sin, y, Dm, w.scale)
            else:
                call = lambda: H.hcms_dist_attention_forward(pl, qd, kd, vd, out1, w.scale)
            st, text = status_of(call)
            assert st == H.HCMS_ERR_CUDA and "injected failure" in text, (layer, st, text)
            torch.cuda.synchronize()
            st, text = status_of(call)
            assert st == H.HCMS_ERR_INVALID_ARG and "earlier forward call" in text, (layer, st, text)
    # (3) a healthy plan: an error found by the checks consumes no epoch -- the next call is right
    want = torch.empty_like(qd)
    with H.hcms_plan(S, Hh, D, 1, C) as ref_plan:
        H.hcms_attention_forward(ref_plan, qd, kd, vd, want, w.scale)
        torch.cuda.synchronize()
    with H.hcms_dist_plan(S, Hh, D, 1, C, 0, H.HCMS_DTYPE_BF16, a.flags) as pl:
        H.hcms_dist_attach(pl, [H.hcms_dist_export(pl)])
        for bad in (lambda: H.hcms_dist_attention_forward(pl, qd, kd, vd, qd, w.scale),               # alias
                    lambda: H.hcms_dist_attention_forward(pl, qd, kd, vd, out1, float("inf"))):      # scale
            assert status_of(bad)[0] in (H.HCMS_ERR_ALIAS, H.HCMS_ERR_INVALID_ARG)
        out1.fill_(0x7FC0)
        H.hcms_dist_attention_forward(pl, qd, kd, vd, out1, w.scale)
        torch.cuda.synchronize()
        assert torch.equal(out1, want)
        host_in = [t.cpu().pin_memory() for t in (qd, kd, vd)]
        host_out = torch.full_like(host_in[0], 0x7FC0).pin_memory()
        H.hcms_dist_attention_forward_host(pl, host_in[0], host_in[1], host_in[2], host_out, w.scale)
        assert torch.equal(host_out, want.cpu())
        assert status_of(lambda: H.hcms_dist_attention_forward_host(pl, host_in[0], host_in[1], host_in[2], host_in[0], w.scale))[0] \
            == H.HCMS_ERR_ALIAS
    print("DIST_OK", flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--spawn", type=int, default=0)
    ap.add_argument("--local", type=int, default=0)
    ap.add_argument("--fail", type=int, default=0, help="P in-process ranks with HCMS_FLAG_DEBUG_DIST_FAIL: the error path")
    for name in ("S", "H", "D", "C"):
        ap.add_argument("--" + name, type=int, required=True)
    ap.add_argument("--layer", type=int, default=0, help="1: the whole layer (hcms_dist_layer_forward[_group])")
    ap.add_argument("--flags", type=int, default=0, help="hcms_dist_plan flags (HCMS_FLAG_DIST_FUSE_OUT, HCMS_FLAG_ATTN_PAIR)")
    a = ap.parse_args()
    if a.fail:
        local_fail(a)
        return
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

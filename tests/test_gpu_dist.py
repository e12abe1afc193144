"""-m gpu: HCMS between P real ranks (Alg. 1 lines 8 and 21): hcms_dist_*.

One GPU is all a run has, so the P ranks share cuda:0: (a) P plans in ONE process attached with
hcms_dist_attach_local (the code path one process driving several GPUs would take), (b) P PROCESSES exchanging
CUDA-IPC handles over gloo (the one-process-per-GPU path; the same mapping works between processes on one
device).  No rank's kernel waits on another rank: cross-rank ordering is stream waits on epoch flags.

Checks: the concatenated rank outputs are BIT-EQUAL to hcms_attention_forward (the single-device emulation) on the
concatenated inputs -- same attention kernel, same per-head arithmetic (Table 14 "max diff 0") --
and within the north-star tolerance of the fp64 oracle; repeated calls (buffer reuse across epochs) keep the bits;
NaN-poisoned outputs show any pull that ran before its attention.
"""
import os
import subprocess
import sys

import numpy as np
import pytest
import torch

import hcms_inputs as I
import paper_2607_01817_b200 as H
from oracle import hcms_oracle as O
from gpu_util import DEV, bf16_bits_to_f64, nan_fill_, to_dev, to_host

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _emulation(q, k, v, S, Hh, D, P, C, scale):
    qd, kd, vd = to_dev(q), to_dev(k), to_dev(v)
    out = nan_fill_(torch.empty_like(qd))
    with H.hcms_plan(S, Hh, D, P, C) as plan:
        H.hcms_attention_forward(plan, qd, kd, vd, out, scale)
        torch.cuda.synchronize()
    return to_host(out)


def _run_worker(mode, P, S, Hh, D, C, env=None, flags=0, layer=0, timeout=240):
    cmd = [sys.executable, os.path.join(ROOT, "tests", "dist_worker.py"), mode, str(P), "--S", str(S), "--H", str(Hh),
           "--D", str(D), "--C", str(C), "--flags", str(flags), "--layer", str(layer)]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=timeout, cwd=ROOT, env=dict(os.environ, **(env or {})))
    assert r.returncode == 0, r.stdout[-2000:] + r.stderr[-3000:]
    assert "DIST_OK" in r.stdout, r.stdout[-2000:]


@pytest.mark.parametrize("S,Hh,D,P,C", [(1024, 4, 64, 2, 2), (2040, 12, 128, 4, 3), (768, 6, 128, 3, 2), (516, 8, 64, 1, 3)])
def test_ranks_in_one_process_bit_equal_to_the_emulation(S, Hh, D, P, C):
    """P plans in one process on cuda:0 (hcms_dist_attach_local), one caller stream per rank, driven by
    hcms_dist_attention_forward_group, three calls: concatenated outputs bit-equal to hcms_attention_forward.  Runs in a
    child process with a watchdog, so a broken exchange cannot hang the test session."""
    _run_worker("--local", P, S, Hh, D, C)


def test_emulation_matches_oracle_on_the_dist_shapes():
    """The reference bits of the two tests around this one are hcms_attention_forward's; they are oracle-checked here."""
    S, Hh, D, P, C = 2040, 12, 128, 4, 3
    w = I.Workload("distlocal", S, Hh, D, P, C, 71, "bf16", 1.0)
    q, k, v = I.make_qkv(w)
    want = _emulation(q, k, v, S, Hh, D, P, C, w.scale)
    ref = O.attention_full(q, k, v, w.scale)
    err = np.abs(bf16_bits_to_f64(want) - ref)
    assert err.max() <= 2e-2 and err.mean() <= 2e-3
    assert np.linalg.norm(bf16_bits_to_f64(want) - ref) / np.linalg.norm(ref) <= 1e-2


@pytest.mark.parametrize("cfg,P,flags,layer", [(3, 4, 0, 0), (3, 4, H.HCMS_FLAG_DIST_FUSE_OUT, 0), (3, 4, 0, 1),
                                              (4, 8, 0, 0), (4, 8, H.HCMS_FLAG_DIST_FUSE_OUT, 0)],
                         ids=["cfg3-4ranks-pull", "cfg3-4ranks-fused-out", "cfg3-4ranks-layer", "cfg4-8ranks-pull", "cfg4-8ranks-fused-out"])
def test_full_size_ranks_in_one_process(cfg, P, flags, layer):
    """BASELINE.json's full shapes between in-process ranks: cfg 3 as 4 ranks (shards of 8190 rows: output tiles straddle
    two ranks' shards, GB-sized exchange blocks, more than one wave per launch) and cfg 4 as 8 ranks (shards of 7020 rows,
    chunks 3 + 2); push scatter + pull gather, the fused output push, and the whole layer with both all-to-alls inside the
    GEMM / attention epilogues (48 chunk maps).  Bit-equal to the emulation on all three calls; attention forms also
    against the fp64 oracle on sampled rows (shard boundaries + seeded rows)."""
    w = I.workload(cfg)
    _run_worker("--local", P, w.S, w.H, w.D, w.C, flags=flags, layer=layer, timeout=500)


def test_failed_forward_joins_and_poisons_instead_of_hanging():
    """HCMS_FLAG_DEBUG_DIST_FAIL injects a failure in the attention phase, after the pushes: the call returns the error,
    every stream drains (no wait on a flag nobody publishes), hcms_dist_plan_destroy returns, later calls are refused;
    group call with 3 in-process ranks, the single-rank calls (attention and layer) with P = 1.  In a child process with a
    60 s watchdog."""
    _run_worker("--fail", 3, 768, 6, 128, 2)


def test_dist_plan_argument_errors():
    S, Hh, D, P, C = 512, 4, 64, 2, 2
    def status(fn):
        with pytest.raises(H.HcmsError) as ei:
            fn()
        return ei.value.status
    assert status(lambda: H.hcms_dist_plan(S, Hh, D, P, C, 2)) == H.HCMS_ERR_INVALID_ARG               # rank >= P
    assert status(lambda: H.hcms_dist_plan(S, Hh, D, P, 3, 0)) == H.HCMS_ERR_UNSUPPORTED_SHAPE         # C > H/P
    assert status(lambda: H.hcms_dist_plan(S, 34, D, 17, 1, 0)) == H.HCMS_ERR_UNSUPPORTED_SHAPE        # S % P, P > 16
    assert status(lambda: H.hcms_dist_plan(S, Hh, D, P, C, 0, H.HCMS_DTYPE_F32)) == H.HCMS_ERR_UNSUPPORTED_DTYPE
    a, b = H.hcms_dist_plan(S, Hh, D, P, C, 0), H.hcms_dist_plan(S, Hh, D, P, C, 1)
    other = H.hcms_dist_plan(S, Hh, D, P, 1, 1)                                                        # another C
    x = torch.zeros(S // P * Hh * D, dtype=torch.int16, device=DEV)
    y = torch.zeros_like(x)
    try:
        assert status(lambda: H.hcms_dist_attention_forward(a, x, x, x, y, 0.1)) == H.HCMS_ERR_INVALID_ARG      # not attached
        assert status(lambda: H.hcms_dist_attach_local(a, [a])) == H.HCMS_ERR_PLAN_MISMATCH
        assert status(lambda: H.hcms_dist_attach_local(a, [b, a])) == H.HCMS_ERR_PLAN_MISMATCH                  # rank order
        assert status(lambda: H.hcms_dist_attach_local(a, [a, other])) == H.HCMS_ERR_PLAN_MISMATCH
        handles = [H.hcms_dist_export(a), H.hcms_dist_export(other)]
        assert status(lambda: H.hcms_dist_attach(a, handles)) == H.HCMS_ERR_PLAN_MISMATCH
        assert status(lambda: H.hcms_dist_attach(a, [b"\0" * 128, b"\0" * 128])) == H.HCMS_ERR_INVALID_ARG      # not a handle
        H.hcms_dist_attach_local(a, [a, b])
        assert status(lambda: H.hcms_dist_attach_local(a, [a, b])) == H.HCMS_ERR_INVALID_ARG                    # twice
        assert status(lambda: H.hcms_dist_attention_forward(a, x, x, x, y, 0.1)) == H.HCMS_ERR_INVALID_ARG      # local plans: group call only
        assert status(lambda: H.hcms_dist_attention_forward(a, x, x, x, x, 0.1)) == H.HCMS_ERR_ALIAS
        assert status(lambda: H.hcms_dist_attention_forward(a, x, x, x, y, float("nan"))) == H.HCMS_ERR_INVALID_ARG
    finally:
        for pl in (a, b, other):
            pl.close()


@pytest.mark.parametrize("P,C", [(2, 2), (4, 1)])
def test_ranks_as_processes_over_cuda_ipc(P, C):
    """One process per rank on cuda:0, CUDA-IPC handles exchanged over gloo, three forward calls; rank 0 compares the
    all-gathered outputs with the single-device emulation bit for bit.  Every worker carries a 120 s watchdog."""
    _run_worker("--spawn", P, 1024, 8, 128, C)


# ---------------------------------------------------------------------------------------------
# HCMS_FLAG_DIST_FUSE_OUT: the output all-to-all in the attention kernel's epilogue (TMA stores into peer memory)
# ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("S,Hh,D,P,C", [(1024, 4, 64, 2, 2), (2040, 12, 128, 4, 3), (768, 6, 128, 3, 2), (516, 8, 64, 1, 3),
                                        (900, 6, 128, 3, 1)])
def test_fused_output_push_in_one_process_bit_equal(S, Hh, D, P, C):
    """Same check as above with the pull-gather kernel replaced by epilogue stores into every rank's output: tiles that
    straddle two ranks (S/P = 510, 256, 300 are not multiples of 128) are stored twice with clipping."""
    _run_worker("--local", P, S, Hh, D, C, flags=H.HCMS_FLAG_DIST_FUSE_OUT)


def test_fused_output_push_with_pairs_in_one_process():
    _run_worker("--local", 2, 2048, 8, 128, 2, flags=H.HCMS_FLAG_DIST_FUSE_OUT | H.HCMS_FLAG_ATTN_PAIR)


@pytest.mark.parametrize("P,C", [(2, 2), (4, 1)])
def test_fused_output_push_as_processes_over_cuda_ipc(P, C):
    _run_worker("--spawn", P, 1024, 8, 128, C, flags=H.HCMS_FLAG_DIST_FUSE_OUT)


# ---------------------------------------------------------------------------------------------
# hcms_dist_layer_forward: QKV projection -> (push in its epilogue) -> attention -> (push in its epilogue) -> output projection
# ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("S,Hh,D,P,C", [(1024, 4, 64, 2, 2), (2040, 12, 128, 4, 3), (768, 6, 128, 3, 2), (640, 8, 64, 1, 2),
                                        (1024, 40, 128, 8, 4)])   # the last: cfg 3's heads on 8 ranks, 3*C*P = 96 maps
def test_layer_between_ranks_in_one_process_bit_equal(S, Hh, D, P, C):
    """Both all-to-alls inside compute kernels: the concatenated y of the ranks equals hcms_layer_forward bit for bit
    (shards whose length is not a multiple of the 128-row GEMM tile included: 510, 256, 640 tokens per rank)."""
    _run_worker("--local", P, S, Hh, D, C, layer=1)


@pytest.mark.parametrize("P,C", [(2, 2), (4, 1)])
def test_layer_between_processes_over_cuda_ipc(P, C):
    _run_worker("--spawn", P, 1024, 8, 128, C, layer=1)


def test_dist_layer_argument_errors():
    S, Hh, D, P, C = 512, 4, 64, 2, 2
    Dm, Sl = Hh * D, S // P
    def status(fn):
        with pytest.raises(H.HcmsError) as ei:
            fn()
        return ei.value.status
    plain = [H.hcms_dist_plan(S, Hh, D, P, C, r) for r in range(P)]
    fused = [H.hcms_dist_plan(S, Hh, D, P, C, r, H.HCMS_DTYPE_BF16, H.HCMS_FLAG_DIST_FUSE_OUT) for r in range(P)]
    x = torch.zeros((Sl, Dm), dtype=torch.int16, device=DEV)
    wq = torch.zeros((3 * Dm, Dm), dtype=torch.int16, device=DEV)
    wo = torch.zeros((Dm, Dm), dtype=torch.int16, device=DEV)
    y = torch.zeros_like(x)
    try:
        assert status(lambda: H.hcms_dist_layer_forward(fused[0], x, wq, wo, None, None, y, Dm, 0.1)) == H.HCMS_ERR_INVALID_ARG   # not attached
        for group in (plain, fused):
            for pl in group:
                H.hcms_dist_attach_local(pl, group)
        streams = [torch.cuda.Stream() for _ in range(P)]
        call = lambda plans, dm=Dm, cos=None: H.hcms_dist_layer_forward_group(plans, [x] * P, wq, wo, cos, None, [y, torch.zeros_like(y)], dm,
                                                                            0.1, streams)
        assert status(lambda: call(plain)) == H.HCMS_ERR_INVALID_ARG                 # plan without HCMS_FLAG_DIST_FUSE_OUT
        assert status(lambda: call(fused, dm=Dm - 64)) == H.HCMS_ERR_UNSUPPORTED_SHAPE
        assert status(lambda: call(fused, cos=[x, x])) == H.HCMS_ERR_INVALID_ARG     # cos without sin
        assert status(lambda: H.hcms_dist_layer_forward(fused[0], x, wq, wo, None, None, y, Dm, 0.1)) == H.HCMS_ERR_INVALID_ARG  # local plans: group call
        call(fused)                                                                   # and the valid call goes through
        torch.cuda.synchronize()
    finally:
        for pl in plain + fused:
            pl.close()

"""-m gpu: the SURVEY 8(f) rows at BASELINE.json's full sizes -- cfg 3 (S=32760, H=40, D=128, P=4, C=4; Dm = 5120), cfg 4
(S=56160, H=40, P=8, C=2: 5 heads per rank split 3 + 2) and cfg 5 (S=98304, H=24, P=8, C=3: one head per chunk, 768 key
tiles; Dm = 3072) -- in the launch configuration bench.py times, checked on sampled outputs the oracle computes one by one:

* projections: sampled token rows (tile and shard boundaries + seeded rows) of q, k, v and y;
* backward: dq on sampled query rows and dk, dv on sampled key rows of sampled heads (one per logical rank pair,
  covering different chunks); each sampled dk / dv row sums over all 32760 queries in the oracle.

Tolerances as in test_gpu_layer.py / test_gpu_backward.py.
"""
import numpy as np
import pytest
import torch

import hcms_inputs as I
import paper_2607_01817_b200 as H
from oracle import hcms_backward_oracle as B
from oracle import hcms_layer_oracle as L
from oracle import hcms_oracle as O
from gpu_util import DEV, bf16_bits_to_f64, nan_fill_, to_dev, to_host

pytestmark = pytest.mark.gpu

FULL = pytest.mark.parametrize("cfg", [3, 4, 5], ids=["cfg3", "cfg4", "cfg5"])


def dev_out(*shape):
    return nan_fill_(torch.empty(shape, dtype=torch.int16, device=DEV))


def rows_sample(S, P, n_random, seed):
    return O.sample_rows(S, P, n_random=n_random, seed=seed)


def check_rounded(got_bits, ref, what):
    got = bf16_bits_to_f64(got_bits)
    assert not np.isnan(got).any(), what
    err = np.abs(got - ref)
    bound = 2.0 ** -8 * np.abs(ref) + 1e-5 * np.abs(ref).max()
    rel = np.linalg.norm(got - ref) / np.linalg.norm(ref)
    assert (err / bound).max() <= 1.0 and rel <= 3e-3, f"{what}: worst={(err / bound).max():.3f} rel_l2={rel:.3e}"


@FULL
def test_projections_sampled_rows(cfg):
    w = I.workload(cfg)
    S, Hh, D = w.S, w.H, w.D
    Dm = Hh * D
    x, w_qkv, w_o, cos, sin = I.make_layer_inputs(w)
    rows = rows_sample(S, w.P, 40, 7)
    q, k, v = dev_out(S, Hh, D), dev_out(S, Hh, D), dev_out(S, Hh, D)
    y = dev_out(S, Dm)
    o_in = I.f32_to_bf16_bits(I.normal_f32(w.seed, 7, S * Hh * D).reshape(S, Hh, D))
    with H.hcms_plan(S, Hh, D, w.P, w.C) as plan:
        H.hcms_qkv_projection_rope(plan, to_dev(x), to_dev(w_qkv), to_dev(cos), to_dev(sin), q, k, v, Dm)
        H.hcms_output_projection(plan, to_dev(o_in), to_dev(w_o), y, Dm)
        torch.cuda.synchronize()
    ref = L.project_and_rotate(x[rows], w_qkv, cos[rows], sin[rows], Hh, D)
    for name, g, r in zip("qkv", (q, k, v), ref):
        check_rounded(to_host(g[torch.from_numpy(rows).to(DEV)]), r, f"{name} rows of cfg {cfg}")
    check_rounded(to_host(y[torch.from_numpy(rows).to(DEV)]), L.output_projection(o_in[rows], w_o), f"y rows of cfg {cfg}")
    # every element was written (no tile skipped anywhere)
    for t in (q, k, v, y):
        assert not bool((t == 0x7FC0).any())


# (cfg, backward kernel, sampled global heads).  The oracle walks all S queries for every sampled key row, S^2 work per
# head: two heads at cfg 3 / 4, one at cfg 5.  cfg 4: head 2 = rank 0 chunk 0, head 39 = rank 7 chunk 1 (local head 4);
# cfg 5: head 16 = rank 5 chunk 1.
@pytest.mark.parametrize("cfg,bwd_flag,heads", [(3, 0, [2, 27]), (3, H.HCMS_FLAG_BWD_ONE_PASS, [2, 27]), (4, 0, [2, 39]),
                                                (4, H.HCMS_FLAG_BWD_ONE_PASS, [39]), (5, 0, [16])],
                         ids=["cfg3-two_pass", "cfg3-one_pass", "cfg4-two_pass", "cfg4-one_pass", "cfg5-two_pass"])
def test_forward_backward_sampled(cfg, bwd_flag, heads):
    """Full configs through the chunk pipeline, both backward kernels (the launch configuration bench.py times).  The
    one-pass runs are also the stress case of its ordered reduction: 256 / 439 key tiles x 12 / 24 heads per launch, far
    more CTAs than SMs, a grid in flight on each of the two compute streams."""
    w = I.workload(cfg)
    S, Hh, D, P, C = w.S, w.H, w.D, w.P, w.C
    q, k, v = I.make_qkv(w)
    do = I.f32_to_bf16_bits(I.normal_f32(w.seed, 6, S * Hh * D).reshape(S, Hh, D))
    qd, kd, vd, dod = (to_dev(t) for t in (q, k, v, do))
    out, dq, dk, dv = (dev_out(S, Hh, D) for _ in range(4))
    with H.hcms_plan(S, Hh, D, P, C, H.HCMS_DTYPE_BF16, H.HCMS_FLAG_TRAINING | bwd_flag) as plan:
        H.hcms_attention_forward(plan, qd, kd, vd, out, w.scale)
        H.hcms_attention_backward(plan, dod, dq, dk, dv, w.scale)
        torch.cuda.synchronize()
    for t in (dq, dk, dv):
        assert not bool((t == 0x7FC0).any()), "a gradient element was never written (or is NaN)"
    # cfg 3: head 2 = rank 0 chunk 0 (local head 2), head 27 = rank 2 chunk 2 (local head 7)
    q_rows = rows_sample(S, P, 24, 11)
    k_rows = rows_sample(S, P, 8, 12)
    sub = lambda t: np.ascontiguousarray(t[:, heads, :])
    ref_dq, ref_dk, ref_dv = B.attention_backward_sampled(sub(q), sub(k), sub(v), sub(do), w.scale, q_rows, k_rows)
    hd = torch.tensor(heads, device=DEV)

    def take(t, rows):
        return to_host(t[torch.from_numpy(rows).to(DEV)][:, hd, :].contiguous())

    for name, got, ref in (("dq", take(dq, q_rows), ref_dq), ("dk", take(dk, k_rows), ref_dk), ("dv", take(dv, k_rows), ref_dv)):
        g = bf16_bits_to_f64(got)
        err = np.abs(g - ref)
        rel = np.linalg.norm(g - ref) / np.linalg.norm(ref)
        assert rel <= 1e-2 and err.max() <= 2e-2 * np.abs(ref).max() + 1e-5, \
            f"{name}: rel_l2={rel:.3e} max_err={err.max():.3e} max_ref={np.abs(ref).max():.3e}"


@FULL
def test_fused_layer_equals_unfused_bitwise(cfg):
    """HCMS_FLAG_FUSE_A2A at the full shapes (cfg 3: 6 launches instead of 14), identical y."""
    w = I.workload(cfg)
    S, Hh, D = w.S, w.H, w.D
    Dm = Hh * D
    arrs = I.make_layer_inputs(w)
    xd, wqd, wod, cd, sd = (to_dev(t) for t in arrs)
    ys = []
    for flags in (0, H.HCMS_FLAG_FUSE_A2A):
        y = dev_out(S, Dm)
        with H.hcms_plan(S, Hh, D, w.P, w.C, H.HCMS_DTYPE_BF16, flags) as plan:
            H.hcms_layer_forward(plan, xd, wqd, wod, cd, sd, y, Dm, w.scale)
            torch.cuda.synchronize()
        ys.append(y)
    assert not bool((ys[0] == 0x7FC0).any())
    assert torch.equal(ys[0], ys[1])

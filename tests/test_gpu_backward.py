"""-m gpu: backward of the hot path (Table 15) through the C ABI against the fp64
oracle (oracle/hcms_backward_oracle.py).

Tolerance.  The kernels round P and dS to bf16 before the accumulating MMAs (relative 2^-9 each, independent per
element) and the gradients to bf16 at the end; q, k, v, dO and the saved O are bf16.  A gradient element is a sum
of S such products, so its error is ~2^-9 |typical term| sqrt(S) against a value of the same order: relative L2
~3e-3.  Gates: relative L2 <= 1e-2 and max |err| <= 2e-2 * max |ref| per tensor.  Bit claims are exact: the
gradients do not depend on P, C or the stream arrangement (Table 14's "max error 0", for the gradients), and
scale = 0 gives dq = dk = 0 exactly.
"""
import numpy as np
import pytest
import torch

import hcms_inputs as I
import paper_2607_01817_b200 as H
from oracle import hcms_backward_oracle as B
from oracle import hcms_oracle as O
from gpu_util import DEV, bf16_bits_to_f64, nan_fill_, to_dev, to_host

pytestmark = pytest.mark.gpu


def bits(x):
    return I.f32_to_bf16_bits(np.asarray(x, dtype=np.float32))


def dev_out(*shape):
    return nan_fill_(torch.empty(shape, dtype=torch.int16, device=DEV))


def seeded(S, Hh, D, seed, k_scale=1.0):
    """q, k, v, dO as bf16 bit patterns [S,H,D] (tensor ids 0..2 of hcms_inputs, 6 for dO)."""
    w = I.Workload("t", S, Hh, D, 1, 1, seed, "bf16", k_scale)
    q, k, v = I.make_qkv(w)
    do = I.f32_to_bf16_bits(I.normal_f32(seed, 6, S * Hh * D).reshape(S, Hh, D))
    return q, k, v, do


def check_grad(got_bits, ref, what):
    got = bf16_bits_to_f64(got_bits)
    assert not np.isnan(got).any(), f"{what}: NaN (a tile was never written, or a pass ran before its input)"
    err = np.abs(got - ref)
    # 1e-5: absolute floor for gradients that are exactly 0 (one key: dq = dk = 0; fp32 leaves ~1e-7 there)
    rel = np.linalg.norm(got - ref) / max(np.linalg.norm(ref), 1e-3 * np.sqrt(ref.size))
    assert rel <= 1e-2 and err.max() <= 2e-2 * np.abs(ref).max() + 1e-5, \
        f"{what}: rel_l2={rel:.3e} max_err={err.max():.3e} max_ref={np.abs(ref).max():.3e}"
    return rel


# ---------------------------------------------------------------------------------------------
# the saved row statistic
# ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("S,D", [(300, 64), (520, 128), (2, 64)])
def test_forward_lse_vs_oracle(S, D):
    P, h = 2, 2
    q, k, v, _ = seeded(S, P * h, D, 31)
    scale = float(np.float32(1.0 / np.sqrt(D)))
    qc, kc, vc = (O.scatter_chunk(t, P, 1, 0) for t in (q, k, v))            # [P,S,h,D]
    oc, oc2 = dev_out(P, S, h, D), dev_out(P, S, h, D)
    lse = torch.full((P * h, S), float("nan"), dtype=torch.float32, device=DEV)
    with H.hcms_plan(S, P * h, D, P, 1) as plan:
        H.hcms_attention_chunk_lse(plan, to_dev(qc), to_dev(kc), to_dev(vc), oc, lse, 0, scale)
        H.hcms_attention_chunk(plan, to_dev(qc), to_dev(kc), to_dev(vc), oc2, 0, scale)
        torch.cuda.synchronize()
    assert torch.equal(oc, oc2)                                    # saving lse changes no output bit
    got = lse.cpu().numpy().astype(np.float64)
    for p in range(P):
        for j in range(h):
            ref = B.log_sum_exp(qc[p, :, j, :], kc[p, :, j, :], scale)
            assert np.abs(got[p * h + j] - ref).max() <= 1e-3, (p, j)


# ---------------------------------------------------------------------------------------------
# the attention backward of one chunk on oracle-made saved tensors
# ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("S,D,P,h", [(300, 64, 2, 2), (333, 128, 1, 3), (64, 128, 2, 1), (1, 64, 1, 1), (1100, 128, 2, 1)])
def test_backward_chunk_vs_oracle(S, D, P, h):
    """Ragged S (not a multiple of 64 or 128), one tile, a single token, several tiles; both head dims."""
    Hh = P * h
    q, k, v, do = seeded(S, Hh, D, 40 + S)
    scale = float(np.float32(1.0 / np.sqrt(D)))
    o_ref = O.attention_full(q, k, v, scale)
    o_bits = bits(o_ref)                                                      # the forward's saved output, bf16
    qc, kc, vc, oc, doc = (O.scatter_chunk(t, P, 1, 0) for t in (q, k, v, o_bits, do))
    lse = np.empty((Hh, S), np.float32)
    for p in range(P):
        for j in range(h):
            lse[p * h + j] = B.log_sum_exp(qc[p, :, j, :], kc[p, :, j, :], scale)
    dq, dk, dv = (dev_out(P, S, h, D) for _ in range(3))
    with H.hcms_plan(S, Hh, D, P, 1) as plan:
        H.hcms_attention_backward_chunk(plan, to_dev(qc), to_dev(kc), to_dev(vc), to_dev(oc), to_dev(doc), to_dev(lse),
                                        dq, dk, dv, 0, scale)
        torch.cuda.synchronize()
        assert H.hcms_plan_last_launch_count(plan) == 3
    ref = B.attention_backward(q, k, v, do, scale)
    for name, g, r in zip(("dq", "dk", "dv"), (dq, dk, dv), ref):
        check_grad(to_host(g), O.scatter_chunk(r, P, 1, 0), f"{name} S={S} D={D}")


# ---------------------------------------------------------------------------------------------
# the whole path: forward then backward through the chunk pipeline
# ---------------------------------------------------------------------------------------------

def run_fwd_bwd(q, k, v, do, S, Hh, D, P, C, scale, flags=0):
    qd, kd, vd, dod = (to_dev(t) for t in (q, k, v, do))
    out, dq, dk, dv = (dev_out(S, Hh, D) for _ in range(4))
    with H.hcms_plan(S, Hh, D, P, C, H.HCMS_DTYPE_BF16, flags | H.HCMS_FLAG_TRAINING) as plan:
        H.hcms_attention_forward(plan, qd, kd, vd, out, scale)
        H.hcms_attention_backward(plan, dod, dq, dk, dv, scale)
        torch.cuda.synchronize()
        assert H.hcms_plan_last_launch_count(plan) == 5 * C            # scatter + 3 kernels + gather per chunk
    return tuple(to_host(t) for t in (out, dq, dk, dv))


def test_forward_backward_config1_and_invariance():
    w = I.workload(1)                                    # S=1024 H=4 D=64 P=2 C=2
    q, k, v, do = seeded(w.S, w.H, w.D, 50)
    got = run_fwd_bwd(q, k, v, do, w.S, w.H, w.D, w.P, w.C, w.scale)
    ref = B.attention_backward(q, k, v, do, w.scale)
    for name, g, r in zip(("dq", "dk", "dv"), got[1:], ref):
        check_grad(g, r, name)
    for P, C, flags in [(1, 1, H.HCMS_FLAG_SERIAL), (4, 1, 0), (1, 4, 0), (2, 1, H.HCMS_FLAG_SINGLE_COMP), (1, 3, 0)]:
        other = run_fwd_bwd(q, k, v, do, w.S, w.H, w.D, P, C, w.scale, flags)
        for a, b in zip(got, other):
            assert np.array_equal(a, b), (P, C, flags)


def test_forward_backward_ragged_uneven_d128():
    """S = 2730 (= cfg 3's 32760 / 12: 21 x 128 + 42, shards of 1365 rows), H = 6, D = 128, P = 2, C = 2 (3 -> 2 + 1),
    K scaled by 0.5 as in cfg 3."""
    S, Hh, D, P, C = 2730, 6, 128, 2, 2
    q, k, v, do = seeded(S, Hh, D, 51, k_scale=0.5)
    scale = float(np.float32(1.0 / np.sqrt(D)))
    got = run_fwd_bwd(q, k, v, do, S, Hh, D, P, C, scale)
    ref = B.attention_backward(q, k, v, do, scale)
    for name, g, r in zip(("dq", "dk", "dv"), got[1:], ref):
        check_grad(g, r, name)


def test_scale_zero_closed_form():
    """scale = 0: dq = dk = 0 bit for bit; dv_k = mean_i dO_i for every key."""
    S, Hh, D = 500, 2, 64
    q, k, v, do = seeded(S, Hh, D, 52)
    _, dq, dk, dv = run_fwd_bwd(q, k, v, do, S, Hh, D, 1, 1, 0.0)
    assert not (dq & 0x7FFF).any() and not (dk & 0x7FFF).any()              # +-0
    want = bf16_bits_to_f64(do).mean(axis=0, keepdims=True)
    got = bf16_bits_to_f64(dv)
    assert np.abs(got - want).max() <= 2.0 ** -8 * np.abs(want).max() + 1e-4


def test_backward_errors():
    S, Hh, D = 256, 2, 64
    t = [dev_out(S, Hh, D) for _ in range(5)]
    with H.hcms_plan(S, Hh, D, 1, 1) as plan:
        with pytest.raises(H.HcmsError) as e:
            H.hcms_attention_backward(plan, t[0], t[1], t[2], t[3], 0.1)
        assert e.value.status == H.HCMS_ERR_INVALID_ARG               # not a TRAINING plan
    with H.hcms_plan(S, Hh, D, 1, 1, H.HCMS_DTYPE_BF16, H.HCMS_FLAG_TRAINING) as plan:
        with pytest.raises(H.HcmsError) as e:
            H.hcms_attention_backward(plan, t[0], t[1], t[2], t[3], 0.1)
        assert e.value.status == H.HCMS_ERR_INVALID_ARG               # no forward yet
        H.hcms_attention_forward(plan, t[0], t[1], t[2], t[4], 0.1)
        with pytest.raises(H.HcmsError) as e:
            H.hcms_attention_backward(plan, t[0], t[1], t[1], t[3], 0.1)
        assert e.value.status == H.HCMS_ERR_ALIAS
        torch.cuda.synchronize()


# ---------------------------------------------------------------------------------------------
# HCMS_FLAG_BWD_ONE_PASS (D = 128): S and dP formed once, dQ reduced over the key tiles in a fixed order
# ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("S,P,h", [(333, 1, 3), (64, 2, 1), (1, 1, 1), (1100, 2, 1), (1365, 1, 2)])
def test_backward_chunk_one_pass_vs_oracle(S, P, h):
    """The single-pass kernel on oracle-made saved tensors: ragged S, one tile, one token, several key and query tiles."""
    D, Hh = 128, P * h
    q, k, v, do = seeded(S, Hh, D, 60 + S)
    scale = float(np.float32(1.0 / np.sqrt(D)))
    o_bits = bits(O.attention_full(q, k, v, scale))
    qc, kc, vc, oc, doc = (O.scatter_chunk(t, P, 1, 0) for t in (q, k, v, o_bits, do))
    lse = np.empty((Hh, S), np.float32)
    for p in range(P):
        for j in range(h):
            lse[p * h + j] = B.log_sum_exp(qc[p, :, j, :], kc[p, :, j, :], scale)
    ref = B.attention_backward(q, k, v, do, scale)
    runs = []
    with H.hcms_plan(S, Hh, D, P, 1, H.HCMS_DTYPE_BF16, H.HCMS_FLAG_BWD_ONE_PASS) as plan:
        for _ in range(2):
            dq, dk, dv = (dev_out(P, S, h, D) for _ in range(3))
            H.hcms_attention_backward_chunk(plan, to_dev(qc), to_dev(kc), to_dev(vc), to_dev(oc), to_dev(doc), to_dev(lse),
                                            dq, dk, dv, 0, scale)
            torch.cuda.synchronize()
            runs.append([to_host(g) for g in (dq, dk, dv)])
    for name, g, r in zip(("dq", "dk", "dv"), runs[0], ref):
        check_grad(g, O.scatter_chunk(r, P, 1, 0), f"one-pass {name} S={S}")
    for a, b in zip(runs[0], runs[1]):
        assert np.array_equal(a, b)                                # the ordered dQ reduction is deterministic


def test_forward_backward_one_pass_invariance():
    """Whole pipeline with the single-pass kernel: against the oracle, and bit for bit across P, C and the stream
    arrangement (the dQ partials are added in key-tile order whatever the chunking)."""
    S, Hh, D, P, C = 2730, 6, 128, 2, 2
    q, k, v, do = seeded(S, Hh, D, 53, k_scale=0.5)
    scale = float(np.float32(1.0 / np.sqrt(D)))
    got = run_fwd_bwd(q, k, v, do, S, Hh, D, P, C, scale, H.HCMS_FLAG_BWD_ONE_PASS)
    ref = B.attention_backward(q, k, v, do, scale)
    for name, g, r in zip(("dq", "dk", "dv"), got[1:], ref):
        check_grad(g, r, name)
    two_pass = run_fwd_bwd(q, k, v, do, S, Hh, D, P, C, scale)
    assert np.array_equal(got[0], two_pass[0])                      # the forward is untouched
    for Pn, Cn, flags in [(1, 1, H.HCMS_FLAG_SERIAL), (3, 2, 0), (1, 6, 0), (6, 1, H.HCMS_FLAG_SINGLE_COMP)]:
        other = run_fwd_bwd(q, k, v, do, S, Hh, D, Pn, Cn, scale, flags | H.HCMS_FLAG_BWD_ONE_PASS)
        for a, b in zip(got, other):
            assert np.array_equal(a, b), (Pn, Cn, flags)

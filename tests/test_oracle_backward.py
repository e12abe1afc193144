"""Pins for oracle/hcms_backward_oracle.py (gradient of Eq. 2 L76 / Alg. 1 lines 4-26; PAPER.md L304,
Table 15) -- CPU only.

The gradient's definition is the derivative of the forward definition, so the strongest pin is numerical
differentiation of the (already pinned) forward oracle; torch.autograd in fp64 differentiates an independent
implementation; closed forms and invariants catch sign / transpose / scale mistakes one by one.
"""
import numpy as np
import pytest
import torch

from oracle import hcms_backward_oracle as B
from oracle import hcms_oracle as A


def _problem(S=10, H=2, D=4, seed=0):
    r = np.random.default_rng(seed)
    return tuple(r.standard_normal((S, H, D)) for _ in range(4))          # q, k, v, dO


def test_finite_differences_of_the_forward_oracle():
    """dL/dx for L = sum(O * dO), central differences with step 1e-6 on every element of q, k, v."""
    q, k, v, do = _problem(S=6, H=2, D=3, seed=1)
    scale = 0.7
    dq, dk, dv = B.attention_backward(q, k, v, do, scale)
    loss = lambda q_, k_, v_: float((A.attention_full(q_, k_, v_, scale) * do).sum())
    eps = 1e-6
    for t, (x, g) in enumerate(((q, dq), (k, dk), (v, dv))):
        num = np.empty_like(x)
        for idx in np.ndindex(*x.shape):
            xp, xm = x.copy(), x.copy()
            xp[idx] += eps
            xm[idx] -= eps
            args_p = [q, k, v]
            args_m = [q, k, v]
            args_p[t], args_m[t] = xp, xm
            num[idx] = (loss(*args_p) - loss(*args_m)) / (2 * eps)
        assert np.abs(num - g).max() < 1e-8, f"tensor {t}"


@pytest.mark.parametrize("use_sdpa", [False, True])
def test_torch_autograd_fp64(use_sdpa):
    q, k, v, do = _problem(S=17, H=3, D=8, seed=2)
    scale = 1.0 / np.sqrt(8)
    tq, tk, tv = (torch.from_numpy(x).clone().requires_grad_(True) for x in (q, k, v))
    if use_sdpa:
        o = torch.nn.functional.scaled_dot_product_attention(tq.transpose(0, 1)[None], tk.transpose(0, 1)[None],
                                                             tv.transpose(0, 1)[None], scale=scale)[0].transpose(0, 1)
    else:
        s = torch.einsum("ihd,khd->hik", tq, tk) * scale
        o = torch.einsum("hik,khd->ihd", torch.softmax(s, dim=-1), tv)
    o.backward(torch.from_numpy(do))
    for got, want in zip(B.attention_backward(q, k, v, do, scale), (tq.grad, tk.grad, tv.grad)):
        assert np.abs(got - want.numpy()).max() < 1e-12


def test_scale_zero_closed_form():
    """scale = 0: P is uniform 1/S, so dV_k = mean_i dO_i for every k, and dQ = dK = 0."""
    q, k, v, do = _problem(S=9, H=2, D=5, seed=3)
    dq, dk, dv = B.attention_backward(q, k, v, do, 0.0)
    assert np.array_equal(dq, np.zeros_like(dq)) and np.array_equal(dk, np.zeros_like(dk))
    assert np.abs(dv - do.mean(axis=0, keepdims=True)).max() < 1e-14


def test_one_key_closed_form():
    """A single key: O_i = v_0 whatever q, k are, so dV_0 = sum_i dO_i and dQ = dK = 0."""
    r = np.random.default_rng(4)
    q, do = r.standard_normal((7, 1, 4)), r.standard_normal((7, 1, 4))
    k, v = r.standard_normal((1, 1, 4)), r.standard_normal((1, 1, 4))
    dq, dk, dv = (g for g in B.attention_backward_head(q[:, 0], k[:, 0], v[:, 0], do[:, 0], 0.9))
    assert np.abs(dq).max() < 1e-15 and np.abs(dk).max() < 1e-15
    assert np.abs(dv[0] - do[:, 0].sum(axis=0)).max() < 1e-14


def test_two_keys_logistic_closed_form():
    """One query, two keys: O = v_1 + sig(z)(v_0 - v_1), z = scale q.(k_0 - k_1).  Hence
    dq = sig'(z) * (dO.(v_0 - v_1)) * scale (k_0 - k_1), dk_0 = -dk_1 = sig'(z) (dO.(v_0-v_1)) scale q,
    dv_0 = sig dO, dv_1 = (1 - sig) dO."""
    r = np.random.default_rng(5)
    q, do = r.standard_normal((1, 6)), r.standard_normal((1, 6))
    k, v = r.standard_normal((2, 6)), r.standard_normal((2, 6))
    scale = 0.4
    z = scale * float(q[0] @ (k[0] - k[1]))
    sig = 1.0 / (1.0 + np.exp(-z))
    g = sig * (1 - sig) * float(do[0] @ (v[0] - v[1]))
    dq, dk, dv = B.attention_backward_head(q, k, v, do, scale)
    assert np.abs(dq[0] - g * scale * (k[0] - k[1])).max() < 1e-14
    assert np.abs(dk[0] - g * scale * q[0]).max() < 1e-14 and np.abs(dk[1] + g * scale * q[0]).max() < 1e-14
    assert np.abs(dv[0] - sig * do[0]).max() < 1e-14 and np.abs(dv[1] - (1 - sig) * do[0]).max() < 1e-14


def test_invariants():
    q, k, v, do = _problem(S=12, H=2, D=6, seed=6)
    scale = 0.5
    dq, dk, dv = B.attention_backward(q, k, v, do, scale)
    # softmax is shift invariant in k: sum_k dK_k = 0; each row of P sums to 1: sum_k dV_k = sum_i dO_i
    assert np.abs(dk.sum(axis=0)).max() < 1e-13
    assert np.abs(dv.sum(axis=0) - do.sum(axis=0)).max() < 1e-13
    # the gradient is linear in dO
    g2 = B.attention_backward(q, k, v, -3.0 * do, scale)
    for a, b in zip((dq, dk, dv), g2):
        assert np.abs(b + 3.0 * a).max() < 1e-12
    # uniform V: O does not depend on q, k
    vu = np.repeat(v[:1], 12, axis=0)
    dq, dk, _ = B.attention_backward(q, k, vu, do, scale)
    assert np.abs(dq).max() < 1e-14 and np.abs(dk).max() < 1e-14


def test_log_sum_exp_definition():
    q, k, _, _ = _problem(S=11, H=1, D=4, seed=7)
    lse = B.log_sum_exp(q[:, 0], k[:, 0], 0.3)
    want = np.array([np.log(sum(np.exp(0.3 * float(q[i, 0] @ k[j, 0])) for j in range(11))) for i in range(11)])
    assert np.abs(lse - want).max() < 1e-13
    assert np.abs(lse - torch.logsumexp(torch.from_numpy(0.3 * q[:, 0] @ k[:, 0].T), dim=1).numpy()).max() < 1e-13


def test_sampled_rows_equal_full():
    q, k, v, do = _problem(S=40, H=2, D=8, seed=8)
    full = B.attention_backward(q, k, v, do, 0.35)
    qr, kr = np.array([0, 7, 39]), np.array([1, 20, 38, 39])
    dq, dk, dv = B.attention_backward_sampled(q, k, v, do, 0.35, qr, kr)
    assert np.abs(dq - full[0][qr]).max() < 1e-13
    assert np.abs(dk - full[1][kr]).max() < 1e-13 and np.abs(dv - full[2][kr]).max() < 1e-13


@pytest.mark.parametrize("P,C", [(1, 1), (2, 1), (2, 3), (4, 1), (1, 5), (2, 2)])
def test_composed_backward_equals_direct_bitwise(P, C):
    """The chunked, all-to-all'ed backward changes no bit (L304 "maximum error of 0", for the gradients)."""
    H = {1: 5, 2: 6, 4: 4}[P]
    q, k, v, do = _problem(S=8 * P, H=H, D=4, seed=9 + P + C)
    direct = B.attention_backward(q, k, v, do, 0.5)
    composed = B.hcms_backward_composed(q, k, v, do, P, C, 0.5)
    for a, b in zip(direct, composed):
        assert np.array_equal(a, b)


# ---------------------------------------------------------------------------------------------
# the row-block accumulation of attention_backward_sampled (dK, dV summed over query blocks with +=): the
# reference for the cfg 3 backward (16 blocks).  Second and later blocks, ragged last block, block > S.
# ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("S,row_block", [(40, 7), (40, 16), (300, 7), (300, 16), (129, 128), (50, 4096)])
def test_sampled_backward_row_blocks(S, row_block):
    q, k, v, do = _problem(S=S, H=2, D=8, seed=20 + S + row_block)
    scale = 0.35
    full = B.attention_backward(q, k, v, do, scale)
    r = np.random.default_rng(S)
    qr = np.unique(np.concatenate([[0, S - 1, min(row_block, S) - 1, min(row_block, S - 1)], r.integers(0, S, 6)]))
    kr = np.unique(np.concatenate([[0, S - 1, min(row_block, S) - 1, min(row_block, S - 1)], r.integers(0, S, 6)]))
    multi = B.attention_backward_sampled(q, k, v, do, scale, qr, kr, row_block=row_block)
    single = B.attention_backward_sampled(q, k, v, do, scale, qr, kr, row_block=S)
    for a, b in zip(multi, single):                    # accumulation order differs only by block boundaries
        assert np.abs(a - b).max() <= 1e-13
    assert np.abs(multi[0] - full[0][qr]).max() <= 1e-13
    assert np.abs(multi[1] - full[1][kr]).max() <= 1e-13
    assert np.abs(multi[2] - full[2][kr]).max() <= 1e-13
    # and against an implementation that shares nothing with the oracle: torch.autograd through fp64 SDPA
    tq, tk, tv = (torch.from_numpy(x).clone().requires_grad_(True) for x in (q, k, v))
    o = torch.nn.functional.scaled_dot_product_attention(tq.transpose(0, 1)[None], tk.transpose(0, 1)[None],
                                                         tv.transpose(0, 1)[None], scale=scale)[0].transpose(0, 1)
    o.backward(torch.from_numpy(do))
    assert np.abs(multi[0] - tq.grad.numpy()[qr]).max() <= 1e-12
    assert np.abs(multi[1] - tk.grad.numpy()[kr]).max() <= 1e-12
    assert np.abs(multi[2] - tv.grad.numpy()[kr]).max() <= 1e-12


def test_sampled_backward_blocks_accumulate_not_overwrite():
    """`=` for `+=` in the block loop would keep only the last block's contribution.  With scale = 0, P is uniform
    1/S, so dV_k = mean_i dO_i needs every block; dK = 0."""
    S = 37
    q, k, v, do = _problem(S=S, H=1, D=4, seed=31)
    kr = np.array([0, 5, 36])
    _, dk, dv = B.attention_backward_sampled(q, k, v, do, 0.0, np.array([0]), kr, row_block=5)
    assert np.abs(dv - do.mean(axis=0, keepdims=True)).max() < 1e-14
    assert np.abs(dk).max() == 0.0

"""Pins for the oracle's attention (Eq. 2; Alg. 1 line 15) and the composed HCMS path.
CPU only.  Closed forms, invariants, a library special case (torch SDPA in fp64) and an
independent brute-force formulation (log-sum-exp in long double, pure Python loops)."""
import math

import numpy as np
import pytest
import torch

from hcms_inputs import f32_to_bf16_bits, normal_f32
from oracle import hcms_oracle as O


def rnd(seed, S, H, D, scale=1.0):
    return [normal_f32(seed, t, S * H * D, threads=1).reshape(S, H, D).astype(np.float64) * scale
            for t in range(3)]


def test_uniform_v_returns_per_head_constant():
    S, H, D = 96, 3, 8
    q, k, _ = rnd(1, S, H, D)
    c = np.arange(1, H * D + 1, dtype=np.float64).reshape(1, H, D) / 7.0
    v = np.broadcast_to(c, (S, H, D)).copy()
    out = O.attention_full(q, k, v, 0.3)
    assert np.allclose(out, v, rtol=0, atol=1e-13)      # also catches head mix-ups: c differs per head


def test_scale_zero_is_mean_of_v():
    S, H, D = 64, 2, 4
    q, k, v = rnd(2, S, H, D)
    out = O.attention_full(q, k, v, 0.0)
    assert np.allclose(out, np.broadcast_to(v.mean(axis=0, keepdims=True), out.shape), atol=1e-14)


def test_one_key_returns_v0():
    q, k, v = rnd(3, 1, 2, 4)
    qq = rnd(4, 5, 2, 4)[0]
    for h in range(2):
        out = O.attention_rows(qq[:, h], k[:, h], v[:, h], 0.7)
        assert np.array_equal(out, np.broadcast_to(v[0, h], out.shape))


def test_two_keys_is_logistic_blend():
    D = 6
    q, k, v = rnd(5, 2, 1, D)
    scale = 0.41
    for i in range(2):
        s0 = scale * float(q[i, 0] @ k[0, 0]); s1 = scale * float(q[i, 0] @ k[1, 0])
        sig = 1.0 / (1.0 + math.exp(-(s0 - s1)))
        want = sig * v[0, 0] + (1 - sig) * v[1, 0]
        got = O.attention_rows(q[i:i + 1, 0], k[:, 0], v[:, 0], scale)[0]
        assert np.allclose(got, want, rtol=1e-13, atol=1e-14)


def test_one_hot_scores_select_a_row():
    S, D = 200, 16
    _, k, v = rnd(6, S, 1, D)
    k = k[:, 0] / np.linalg.norm(k[:, 0], axis=1, keepdims=True)      # unit rows
    perm = np.random.default_rng(0).permutation(S)
    gram = k @ k.T
    np.fill_diagonal(gram, -1)
    margin = 1.0 - gram.max()
    alpha = 40.0 / margin                                              # >= 40 nats margin
    q = alpha * k[perm]
    out = O.attention_rows(q, k, v[:, 0], 1.0)
    assert np.allclose(out, v[perm, 0], rtol=0, atol=1e-12)


def test_output_in_convex_hull_of_v():
    S, H, D = 128, 2, 8
    q, k, v = rnd(7, S, H, D, 2.0)
    out = O.attention_full(q, k, v, 0.5)
    assert (out <= v.max(axis=0, keepdims=True) + 1e-12).all()
    assert (out >= v.min(axis=0, keepdims=True) - 1e-12).all()


def test_kv_permutation_shift_and_duplication_invariance():
    S, H, D = 80, 2, 8
    q, k, v = rnd(8, S, H, D)
    base = O.attention_full(q, k, v, 0.35)
    perm = np.random.default_rng(1).permutation(S)
    assert np.allclose(O.attention_full(q, k[perm], v[perm], 0.35), base, atol=1e-12)
    # adding a constant vector to every K row shifts every score of a row equally
    shift = np.linspace(-1, 1, D).reshape(1, 1, D)
    assert np.allclose(O.attention_full(q, k + shift, v, 0.35), base, atol=1e-12)
    # duplicating K,V leaves O unchanged
    k2, v2 = np.concatenate([k, k]), np.concatenate([v, v])
    for h in range(H):
        got = O.attention_rows(q[:, h], k2[:, h], v2[:, h], 0.35)
        assert np.allclose(got, base[:, h], atol=1e-12)


def test_large_scores_do_not_overflow():
    # max-subtraction: scores ~ 1e3 would overflow exp() without it
    S, D = 32, 4
    q, k, v = rnd(9, S, 1, D, 30.0)
    out = O.attention_rows(q[:, 0], k[:, 0], v[:, 0], 1.0)
    assert np.isfinite(out).all()


@pytest.mark.parametrize("S,H,D", [(33, 2, 8), (64, 3, 16), (7, 1, 4)])
def test_matches_torch_sdpa_fp64(S, H, D):
    q, k, v = rnd(10 + S, S, H, D)
    scale = 1.0 / math.sqrt(D)
    tq, tk, tv = (torch.from_numpy(t).permute(1, 0, 2)[None] for t in (q, k, v))   # [1,H,S,D]
    ref = torch.nn.functional.scaled_dot_product_attention(tq, tk, tv, scale=scale)[0].permute(1, 0, 2).numpy()
    assert np.allclose(O.attention_full(q, k, v, scale), ref, rtol=1e-12, atol=1e-13)


def test_brute_force_logsumexp_long_double():
    S, H, D = 24, 2, 4
    q, k, v = rnd(11, S, H, D)
    scale = 0.5
    got = O.attention_full(q, k, v, scale)
    LD = np.longdouble
    for h in range(H):
        for i in range(S):
            s = [LD(scale) * sum(LD(q[i, h, d]) * LD(k[j, h, d]) for d in range(D)) for j in range(S)]
            mx = max(s)
            lse = mx + np.log(sum(np.exp(x - mx) for x in s))
            for d in range(D):
                want = sum(np.exp(s[j] - lse) * LD(v[j, h, d]) for j in range(S))
                assert abs(float(want) - got[i, h, d]) < 1e-13


def test_transposed_operand_would_fail():
    # guards the pins themselves: q.k^T vs k.q^T differ for non-symmetric inputs
    S, D = 16, 4
    q, k, v = rnd(12, S, 1, D)
    a = O.attention_rows(q[:, 0], k[:, 0], v[:, 0], 1.0)
    b = O.attention_rows(k[:, 0], q[:, 0], v[:, 0], 1.0)
    assert not np.allclose(a, b, atol=1e-3)


def test_bf16_inputs_are_widened_exactly():
    x = normal_f32(13, 0, 4096, threads=1)
    bits = f32_to_bf16_bits(x)
    wide = O.widen_to_f64(bits)
    ref = torch.from_numpy(x).to(torch.bfloat16).double().numpy()      # library RNE rounding
    assert np.array_equal(wide, ref)
    with pytest.raises(TypeError):
        O.widen_to_f64(np.zeros(3, dtype=np.int32))


@pytest.mark.parametrize("S,H,D,P", [(16, 4, 4, 2), (24, 6, 8, 3), (8, 6, 4, 1), (32, 8, 8, 4)])
def test_composed_equals_direct_bitwise(S, H, D, P):
    # the paper's equivalence claim (L304; Table 14) on the CPU, every C incl. uneven
    q, k, v = (f32_to_bf16_bits(normal_f32(14, t, S * H * D, threads=1)).reshape(S, H, D) for t in range(3))
    direct = O.attention_full(q, k, v, 0.37)
    for C in range(1, H // P + 1):
        comp = O.hcms_forward_composed(q, k, v, P, C, 0.37)
        assert np.array_equal(comp, direct)


def test_sampled_rows_equal_full():
    S, H, D = 300, 2, 8
    q, k, v = rnd(15, S, H, D)
    rows = O.sample_rows(S, 2, n_random=10, seed=3)
    assert rows[0] == 0 and rows[-1] == S - 1 and 128 in rows and 127 in rows and 256 in rows and 255 in rows
    assert np.allclose(O.attention_sampled(q, k, v, 0.3, rows), O.attention_full(q, k, v, 0.3)[rows],
                       rtol=1e-13, atol=1e-14)


# ---------------------------------------------------------------------------------------------
# the row-block loop of attention_full (the reference for cfg 2 = 4 blocks and for the ragged shapes):
# second and later blocks, a ragged last block, a block larger than S
# ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("S,row_block", [(40, 7), (40, 16), (300, 7), (300, 16), (129, 128), (64, 64), (50, 4096)])
def test_attention_full_row_blocks_equal_single_block(S, row_block):
    """Rows are independent (Eq. 2), so the block size may not change any row: every row of the multi-block
    result equals the single-block result (to BLAS rounding of the [rows,S] product, <= 1e-14), the definition
    evaluated one row at a time, and fp64 SDPA."""
    H, D = 2, 8
    q, k, v = rnd(40 + S + row_block, S, H, D)
    scale = 0.3
    multi = O.attention_full(q, k, v, scale, row_block=row_block)
    single = O.attention_full(q, k, v, scale, row_block=S)
    assert multi.shape == single.shape and np.isfinite(multi).all()
    assert np.abs(multi - single).max() <= 1e-14
    # one row at a time: no block structure at all
    for h in range(H):
        for i in list(range(0, S, max(1, S // 23))) + [S - 1]:
            one = O.attention_rows(q[i:i + 1, h], k[:, h], v[:, h], scale)[0]
            assert np.abs(multi[i, h] - one).max() <= 1e-14, (i, h)
    tq, tk, tv = (torch.from_numpy(t).permute(1, 0, 2)[None] for t in (q, k, v))
    ref = torch.nn.functional.scaled_dot_product_attention(tq, tk, tv, scale=scale)[0].permute(1, 0, 2).numpy()
    assert np.abs(multi - ref).max() <= 1e-12


def test_attention_full_row_blocks_write_every_row_once():
    """A slip in the block slices (an off-by-one, a skipped tail) leaves rows of the np.empty output unwritten or
    written from the wrong query: with V = one-hot(key index) and Q_i = 50*K_i the output row i is e_i exactly."""
    S, D = 45, 45
    k = np.eye(S)[:, None, :]                       # K_i = e_i  (H = 1)
    q = 50.0 * k                                    # score(i, i) = 50*scale, others 0
    v = np.eye(S)[:, None, :]
    for rb in (1, 7, 16, 44, 45, 46):
        out = O.attention_full(q, k, v, 1.0, row_block=rb)
        assert np.abs(out[:, 0, :] - np.eye(S)).max() < 1e-12, rb
        assert np.array_equal(out.argmax(axis=2)[:, 0], np.arange(S)), rb

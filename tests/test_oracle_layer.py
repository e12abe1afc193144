"""Pins for oracle/hcms_layer_oracle.py (Alg. 1 lines 2-3, 26-27) -- CPU only.

Each check is something the mathematics fixes independently of the oracle's own formula: closed
forms, invariants of rotations, brute-force loops, torch fp64 library routines, and the paper's
equivalence claim (chunked path == direct path, L304).  A dropped term, a wrong sign, a swapped
pair or a transposed weight fails at least one of them.
"""
import numpy as np
import pytest
import torch

from oracle import hcms_layer_oracle as L
from oracle import hcms_oracle as A


def _rng(seed=0):
    return np.random.default_rng(seed)


def _tables(S, D, seed=1):
    ang = _rng(seed).uniform(-np.pi, np.pi, size=(S, D // 2))
    return np.cos(ang), np.sin(ang), ang


def _problem(S=24, H=4, D=8, Dm=16, seed=0):
    r = _rng(seed)
    x = r.standard_normal((S, Dm))
    w_qkv = r.standard_normal((3 * H * D, Dm)) / np.sqrt(Dm)
    w_o = r.standard_normal((Dm, H * D)) / np.sqrt(H * D)
    cos, sin, _ = _tables(S, D, seed + 1)
    return x, w_qkv, w_o, cos, sin


# ---- qkv_projection ---------------------------------------------------------------------------

def test_qkv_projection_brute_force():
    S, H, D, Dm = 5, 2, 4, 6
    x, w, _, _, _ = _problem(S, H, D, Dm)
    q, k, v = L.qkv_projection(x, w, H, D)
    for t, got in enumerate((q, k, v)):
        for s in range(S):
            for h in range(H):
                for d in range(D):
                    n = t * H * D + h * D + d
                    want = sum(x[s, m] * w[n, m] for m in range(Dm))
                    assert abs(got[s, h, d] - want) < 1e-12


def test_qkv_projection_selector_weights():
    """W = rows of the identity picks input features: q[s,h,d] = x[s, h*D+d], k = 2x, v = -x."""
    S, H, D = 7, 3, 4
    Dm = H * D
    x = _rng(3).standard_normal((S, Dm))
    eye = np.eye(Dm)
    w = np.concatenate([eye, 2 * eye, -eye], axis=0)
    q, k, v = L.qkv_projection(x, w, H, D)
    assert np.array_equal(q, x.reshape(S, H, D))
    assert np.array_equal(k, 2 * x.reshape(S, H, D))
    assert np.array_equal(v, -x.reshape(S, H, D))


def test_qkv_projection_matches_torch_linear():
    S, H, D, Dm = 9, 2, 8, 12
    x, w, _, _, _ = _problem(S, H, D, Dm)
    y = torch.nn.functional.linear(torch.from_numpy(x), torch.from_numpy(w)).numpy()
    q, k, v = L.qkv_projection(x, w, H, D)
    got = np.concatenate([t.reshape(S, H * D) for t in (q, k, v)], axis=1)
    assert np.abs(got - y).max() < 1e-12


def test_qkv_projection_takes_bf16_bits():
    """uint16 inputs are bf16 bit patterns, widened exactly: 0x3F80 = 1.0, 0xC000 = -2.0."""
    x = np.array([[0x3F80, 0xC000]], dtype=np.uint16)
    w = np.array([[0x3F80, 0x3F80]] * 3, dtype=np.uint16)          # H = D = 1
    q, k, v = L.qkv_projection(x, w, 1, 1)
    assert q[0, 0, 0] == -1.0 and k[0, 0, 0] == -1.0 and v[0, 0, 0] == -1.0


# ---- apply_rope ---------------------------------------------------------------------------------

def test_rope_zero_angle_is_identity():
    x = _rng(4).standard_normal((6, 3, 8))
    out = L.apply_rope(x, np.ones((6, 4)), np.zeros((6, 4)))
    assert np.array_equal(out, x)


def test_rope_quarter_turn_closed_form():
    """angle = pi/2: (a, b) -> (-b, a); angle = pi: (a, b) -> (-a, -b)."""
    x = _rng(5).standard_normal((4, 2, 6))
    out = L.apply_rope(x, np.zeros((4, 3)), np.ones((4, 3)))
    assert np.array_equal(out[:, :, 0::2], -x[:, :, 1::2])
    assert np.array_equal(out[:, :, 1::2], x[:, :, 0::2])
    out = L.apply_rope(x, -np.ones((4, 3)), np.zeros((4, 3)))
    assert np.array_equal(out, -x)


def test_rope_equals_complex_multiplication():
    """Adjacent pairs as complex numbers: RoPE is multiplication by exp(i*angle) (library complex math)."""
    S, H, D = 10, 3, 8
    x = _rng(6).standard_normal((S, H, D))
    cos, sin, ang = _tables(S, D)
    z = torch.view_as_complex(torch.from_numpy(x).reshape(S, H, D // 2, 2).contiguous())
    rot = torch.polar(torch.ones(S, D // 2, dtype=torch.float64), torch.from_numpy(ang))[:, None, :]
    want = torch.view_as_real(z * rot).reshape(S, H, D).numpy()
    assert np.abs(L.apply_rope(x, cos, sin) - want).max() < 1e-14


def test_rope_preserves_pair_norms_and_composes():
    S, H, D = 8, 2, 16
    x = _rng(7).standard_normal((S, H, D))
    c1, s1, a1 = _tables(S, D, 11)
    c2, s2, a2 = _tables(S, D, 12)
    y = L.apply_rope(x, c1, s1)
    n_in = x[:, :, 0::2] ** 2 + x[:, :, 1::2] ** 2
    n_out = y[:, :, 0::2] ** 2 + y[:, :, 1::2] ** 2
    assert np.abs(n_in - n_out).max() < 1e-13
    both = L.apply_rope(y, c2, s2)
    direct = L.apply_rope(x, np.cos(a1 + a2), np.sin(a1 + a2))
    assert np.abs(both - direct).max() < 1e-13
    back = L.apply_rope(y, c1, -s1)                      # inverse rotation
    assert np.abs(back - x).max() < 1e-13


def test_rope_relative_position_property():
    """RoFormer's defining property: with angle(s, i) = s * theta_i, <R_m q, R_n k> depends on m - n only."""
    D, S = 16, 12
    theta = 10000.0 ** (-np.arange(D // 2) * 2.0 / D)
    ang = np.arange(S)[:, None] * theta[None, :]
    q1 = _rng(8).standard_normal((1, 1, D))
    k1 = _rng(9).standard_normal((1, 1, D))
    q = L.apply_rope(np.repeat(q1, S, axis=0), np.cos(ang), np.sin(ang))[:, 0, :]
    k = L.apply_rope(np.repeat(k1, S, axis=0), np.cos(ang), np.sin(ang))[:, 0, :]
    dots = q @ k.T                                           # [m, n]
    for delta in range(-3, 4):
        diag = np.array([dots[m, m - delta] for m in range(S) if 0 <= m - delta < S])
        assert np.abs(diag - diag[0]).max() < 1e-12
    assert abs(dots[5, 2] - dots[5, 3]) > 1e-6               # and it does depend on m - n


def test_rope_is_per_token_and_per_pair():
    """Changing the angle of (token 2, pair 1) changes exactly x[2, :, 2:4]."""
    S, H, D = 5, 2, 8
    x = _rng(10).standard_normal((S, H, D))
    cos, sin, ang = _tables(S, D)
    ang2 = ang.copy()
    ang2[2, 1] += 0.7
    a, b = L.apply_rope(x, cos, sin), L.apply_rope(x, np.cos(ang2), np.sin(ang2))
    diff = np.abs(a - b) > 0
    want = np.zeros_like(diff)
    want[2, :, 2:4] = True
    assert np.array_equal(diff, want)


# ---- output_projection ----------------------------------------------------------------------------

def test_output_projection_brute_force_and_identity():
    S, H, D, Dm = 4, 2, 3, 5
    o = _rng(12).standard_normal((S, H, D))
    w = _rng(13).standard_normal((Dm, H * D))
    y = L.output_projection(o, w)
    for s in range(S):
        for m in range(Dm):
            want = sum(o[s, h, d] * w[m, h * D + d] for h in range(H) for d in range(D))
            assert abs(y[s, m] - want) < 1e-12
    assert np.array_equal(L.output_projection(o, np.eye(H * D)), o.reshape(S, H * D))


# ---- the layer ----------------------------------------------------------------------------------------

def test_layer_with_identity_weights_is_plain_attention():
    """W_q = W_k = W_v = W_o = I and zero angles: the layer is Eq. 2 on x itself."""
    S, H, D = 16, 2, 4
    Dm = H * D
    x = _rng(14).standard_normal((S, Dm))
    eye = np.eye(Dm)
    w_qkv = np.concatenate([eye, eye, eye], axis=0)
    y = L.layer_forward(x, w_qkv, eye, np.ones((S, D // 2)), np.zeros((S, D // 2)), H, D, 0.5)
    xs = x.reshape(S, H, D)
    want = A.attention_full(xs, xs, xs, 0.5).reshape(S, Dm)
    assert np.array_equal(y, want)


def test_layer_matches_torch_sdpa_fp64():
    S, H, D, Dm = 20, 3, 8, 24
    x, w_qkv, w_o, cos, sin = _problem(S, H, D, Dm, seed=20)
    scale = 1.0 / np.sqrt(D)
    tx, tw, two = (torch.from_numpy(a) for a in (x, w_qkv, w_o))
    qkv = torch.nn.functional.linear(tx, tw).reshape(S, 3, H, D)
    ang = torch.from_numpy(np.arctan2(sin, cos))
    rot = torch.polar(torch.ones_like(ang), ang)[:, None, :]

    def rope(t):
        z = torch.view_as_complex(t.reshape(S, H, D // 2, 2).contiguous())
        return torch.view_as_real(z * rot).reshape(S, H, D)

    q, k, v = rope(qkv[:, 0]), rope(qkv[:, 1]), qkv[:, 2]
    o = torch.nn.functional.scaled_dot_product_attention(q.transpose(0, 1)[None], k.transpose(0, 1)[None],
                                                         v.transpose(0, 1)[None], scale=scale)[0]
    want = torch.nn.functional.linear(o.transpose(0, 1).reshape(S, H * D), two).numpy()
    got = L.layer_forward(x, w_qkv, w_o, cos, sin, H, D, scale)
    assert np.abs(got - want).max() < 1e-12


def test_layer_uniform_v_closed_form():
    """W_v = 0 except a bias-like constant is impossible without bias; instead make every token's v equal:
    x rows identical => softmax averages identical v => y = W_o v for every token, whatever q, k are."""
    S, H, D, Dm = 12, 2, 4, 8
    _, w_qkv, w_o, cos, sin = _problem(S, H, D, Dm, seed=21)
    x = np.repeat(_rng(22).standard_normal((1, Dm)), S, axis=0)
    y = L.layer_forward(x, w_qkv, w_o, cos, sin, H, D, 0.3)
    v = (x[0] @ w_qkv[2 * H * D:].T)
    want = w_o @ v
    assert np.abs(y - want[None, :]).max() < 1e-12


def test_layer_is_linear_in_w_o_and_rows_sample():
    S, H, D, Dm = 18, 2, 8, 16
    x, w_qkv, w_o, cos, sin = _problem(S, H, D, Dm, seed=23)
    y = L.layer_forward(x, w_qkv, w_o, cos, sin, H, D, 0.35)
    y2 = L.layer_forward(x, w_qkv, 2.0 * w_o, cos, sin, H, D, 0.35)
    assert np.abs(y2 - 2.0 * y).max() < 1e-12
    rows = np.array([0, 3, 17])
    assert np.array_equal(L.layer_forward_rows(x, w_qkv, w_o, cos, sin, H, D, 0.35, rows), y[rows])


def test_layer_global_rotation_of_q_and_k_cancels():
    """Adding the same angle to every token's table rotates q and k alike: scores, hence y, are unchanged."""
    S, H, D, Dm = 14, 2, 8, 16
    x, w_qkv, w_o, cos, sin = _problem(S, H, D, Dm, seed=24)
    ang = np.arctan2(sin, cos) + _rng(25).uniform(-1, 1, size=(1, D // 2))
    y = L.layer_forward(x, w_qkv, w_o, cos, sin, H, D, 0.35)
    y2 = L.layer_forward(x, w_qkv, w_o, np.cos(ang), np.sin(ang), H, D, 0.35)
    assert np.abs(y - y2).max() < 1e-12


@pytest.mark.parametrize("P,C", [(1, 1), (2, 1), (2, 2), (2, 3), (4, 1), (1, 5)])
def test_layer_composed_equals_direct_bitwise(P, C):
    """The paper's equivalence claim (L304, Table 14) for the whole of Alg. 1: any P, any C (uneven too)."""
    H = {1: 5, 2: 6, 4: 4}[P]
    S, D, Dm = 8 * P, 4, 12
    x, w_qkv, w_o, cos, sin = _problem(S, H, D, Dm, seed=30 + P + C)
    direct = L.layer_forward(x, w_qkv, w_o, cos, sin, H, D, 0.5)
    composed = L.layer_forward_composed(x, w_qkv, w_o, cos, sin, H, D, P, C, 0.5)
    assert np.array_equal(direct, composed)

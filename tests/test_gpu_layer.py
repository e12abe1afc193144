"""-m gpu: the attention layer around the hot path (Alg. 1 lines 2-3 and 27) through the
C ABI against the fp64 oracle (oracle/hcms_layer_oracle.py).

Tolerances.  A projection rounds an fp32-accumulated sum once to bf16: |err| <= 2^-9 |ref| (half an ulp) plus
the fp32 accumulation error (~1e-6 relative; half an ulp reaches 2^-8 |ref| just above a power of two), so the
gates are |err| <= 2^-8 |ref| + 1e-5 max|ref| element-wise (the second term covers the fp32 accumulation and
the RoPE products, which are absolute, not relative, errors)
and relative L2 <= 3e-3 (uniform rounding gives 2^-9/sqrt(3) = 1.1e-3).  Cases whose results are exactly
representable in bf16 are compared bit for bit.  The whole layer takes the north-star attention gates
(max-abs 2e-2, mean-abs 2e-3) plus relative L2 <= 1e-2 on y (q, k, v and o are each rounded to bf16 on the
GPU and kept in fp64 by the oracle).
"""
import numpy as np
import pytest
import torch

import hcms_inputs as I
import paper_2607_01817_b200 as H
from oracle import hcms_layer_oracle as L
from oracle import hcms_oracle as O
from gpu_util import DEV, bf16_bits_to_f64, nan_fill_, to_dev, to_host

pytestmark = pytest.mark.gpu


def bits(x):
    return I.f32_to_bf16_bits(np.asarray(x, dtype=np.float32))


def dev_out(*shape):
    return nan_fill_(torch.empty(shape, dtype=torch.int16, device=DEV))


def check_rounded(got_bits, ref, what):
    got = bf16_bits_to_f64(got_bits)
    assert not np.isnan(got).any(), f"{what}: NaN (an output tile was never written)"
    err = np.abs(got - ref)
    bound = 2.0 ** -8 * np.abs(ref) + 1e-5 * np.abs(ref).max()
    rel = np.linalg.norm(got - ref) / np.linalg.norm(ref)
    worst = (err / bound).max()
    assert worst <= 1.0 and rel <= 3e-3, f"{what}: worst err/bound={worst:.3f} rel_l2={rel:.3e}"
    return rel


# ---------------------------------------------------------------------------------------------
# the bare contraction
# ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("M,N,K", [(128, 256, 64), (1000, 384, 200), (389, 512, 256), (2048, 768, 1024),
                                   (130, 128, 8), (20000, 256, 128)])
def test_gemm_vs_fp64(M, N, K):
    """Several tiles in both directions, ragged M, K tails (K % 64 != 0), both tile widths (N % 256 == 0 or not),
    more tiles than SMs (20000 x 256: 157 tiles)."""
    rng = np.random.default_rng(M + N + K)
    a, b = bits(rng.standard_normal((M, K))), bits(rng.standard_normal((N, K)) / np.sqrt(K))
    c = dev_out(M, N)
    H.hcms_gemm_bf16_nt(to_dev(a), to_dev(b), c, M, N, K)
    torch.cuda.synchronize()
    ref = bf16_bits_to_f64(a) @ bf16_bits_to_f64(b).T
    check_rounded(to_host(c), ref, f"gemm {M}x{N}x{K}")


def test_gemm_small_integers_bit_exact():
    """Entries in {-2..2} and K = 40: every partial sum is a small integer, exact in fp32 and in bf16, so the
    result must equal the integer matrix product bit for bit -- any misplaced tile, row or k-slice shows."""
    M, N, K = 700, 640, 40
    rng = np.random.default_rng(7)
    a = rng.integers(-2, 3, size=(M, K)).astype(np.float32)
    b = rng.integers(-2, 3, size=(N, K)).astype(np.float32)
    c = dev_out(M, N)
    H.hcms_gemm_bf16_nt(to_dev(bits(a)), to_dev(bits(b)), c, M, N, K)
    torch.cuda.synchronize()
    want = (a.astype(np.int64) @ b.astype(np.int64).T).astype(np.float32)      # |values| <= 160 < 256: exact in bf16
    assert np.array_equal(to_host(c), bits(want))


def test_gemm_argument_errors():
    t = torch.zeros(128 * 128, dtype=torch.int16, device=DEV)
    for args, status in [((t, t[128 * 64:], t, 128, 128, 64), H.HCMS_ERR_ALIAS),
                         ((t, t, None, 128, 128, 64), H.HCMS_ERR_INVALID_ARG),
                         ((t, t, t, 128, 100, 64), H.HCMS_ERR_UNSUPPORTED_SHAPE),
                         ((t, t, t, 128, 128, 60), H.HCMS_ERR_UNSUPPORTED_SHAPE),
                         ((t, t, t, 0, 128, 64), H.HCMS_ERR_INVALID_ARG)]:
        with pytest.raises(H.HcmsError) as e:
            H.hcms_gemm_bf16_nt(*args)
        assert e.value.status == status


# ---------------------------------------------------------------------------------------------
# QKV projection + RoPE (Alg. 1 lines 2-3), output projection (line 27)
# ---------------------------------------------------------------------------------------------

def run_qkv(x, w_qkv, cos, sin, S, Hh, D, Dm, P=1, C=1):
    q, k, v = dev_out(S, Hh, D), dev_out(S, Hh, D), dev_out(S, Hh, D)
    with H.hcms_plan(S, Hh, D, P, C) as plan:
        H.hcms_qkv_projection_rope(plan, to_dev(x), to_dev(w_qkv), None if cos is None else to_dev(cos),
                                   None if sin is None else to_dev(sin), q, k, v, Dm)
        torch.cuda.synchronize()
    return to_host(q), to_host(k), to_host(v)


@pytest.mark.parametrize("S,Hh,D,Dm", [(1024, 4, 64, 256), (777, 2, 128, 384), (300, 6, 64, 128), (2500, 8, 128, 1024)])
def test_qkv_projection_rope_vs_oracle(S, Hh, D, Dm):
    w = I.Workload("t", S, Hh, D, 1, 1, 11, "bf16", 1.0)
    x, w_qkv, _, cos, sin = I.make_layer_inputs(w, Dm)
    got = run_qkv(x, w_qkv, cos, sin, S, Hh, D, Dm)
    ref = L.project_and_rotate(x, w_qkv, cos, sin, Hh, D)
    for name, g, r in zip("qkv", got, ref):
        check_rounded(g, r, f"{name} S={S} H={Hh} D={D} Dm={Dm}")
    # without tables the rotation is skipped
    got0 = run_qkv(x, w_qkv, None, None, S, Hh, D, Dm)
    ref0 = L.qkv_projection(x, w_qkv, Hh, D)
    for name, g, r in zip("qkv", got0, ref0):
        check_rounded(g, r, f"{name} (no RoPE)")
    assert np.array_equal(got0[2], got[2])               # v never rotates


@pytest.mark.parametrize("D", [64, 128])
def test_qkv_selector_weights_and_quarter_turn_bit_exact(D):
    """W = [I; I; I] copies x into q, k, v bit for bit; with cos = 0, sin = 1 the pairs become (-x1, x0) exactly
    (sign flips and copies are exact in every precision).  Pins feature order, head order, pair order and sign."""
    Hh, S = 256 // D, 333
    Dm = Hh * D
    x = bits(np.random.default_rng(3).standard_normal((S, Dm)))
    eye = bits(np.eye(Dm))
    w_qkv = np.concatenate([eye, eye, eye], axis=0)
    q, k, v = run_qkv(x, w_qkv, None, None, S, Hh, D, Dm)
    xs = x.reshape(S, Hh, D)
    assert np.array_equal(q, xs) and np.array_equal(k, xs) and np.array_equal(v, xs)
    zeros, ones = np.zeros((S, D // 2), np.float32), np.ones((S, D // 2), np.float32)
    q, k, v = run_qkv(x, w_qkv, zeros, ones, S, Hh, D, Dm)
    want = np.empty_like(xs)
    want[:, :, 0::2] = xs[:, :, 1::2] ^ np.uint16(0x8000)         # -x1
    want[:, :, 1::2] = xs[:, :, 0::2]                             #  x0
    assert np.array_equal(q, want) and np.array_equal(k, want) and np.array_equal(v, xs)


def test_rope_angle_is_per_token_and_pair():
    """One table entry (token 200, pair 5) differs: exactly q[200, :, 10:12] and k[200, :, 10:12] change."""
    S, Hh, D, Dm = 384, 2, 64, 128
    w = I.Workload("t", S, Hh, D, 1, 1, 12, "bf16", 1.0)
    x, w_qkv, _, cos, sin = I.make_layer_inputs(w, Dm)
    a = run_qkv(x, w_qkv, cos, sin, S, Hh, D, Dm)
    cos2, sin2 = cos.copy(), sin.copy()
    cos2[200, 5], sin2[200, 5] = np.float32(np.cos(1.0)), np.float32(np.sin(1.0))
    b = run_qkv(x, w_qkv, cos2, sin2, S, Hh, D, Dm)
    for t in range(2):
        diff = a[t] != b[t]
        assert diff[200, :, 10:12].all()
        diff[200, :, 10:12] = False
        assert not diff.any()
    assert np.array_equal(a[2], b[2])


@pytest.mark.parametrize("S,Hh,D,Dm", [(1024, 4, 64, 256), (900, 3, 128, 640)])
def test_output_projection_vs_oracle(S, Hh, D, Dm):
    rng = np.random.default_rng(S + Dm)
    o = bits(rng.standard_normal((S, Hh, D)))
    w_o = bits(rng.standard_normal((Dm, Hh * D)) / np.sqrt(Hh * D))
    y = dev_out(S, Dm)
    with H.hcms_plan(S, Hh, D, 1, 1) as plan:
        H.hcms_output_projection(plan, to_dev(o), to_dev(w_o), y, Dm)
        torch.cuda.synchronize()
    check_rounded(to_host(y), L.output_projection(o, w_o), f"out-proj S={S}")


# ---------------------------------------------------------------------------------------------
# the whole layer (Alg. 1 lines 2-27)
# ---------------------------------------------------------------------------------------------

def run_layer(x, w_qkv, w_o, cos, sin, S, Hh, D, Dm, P, C, scale, flags=0):
    y = dev_out(S, Dm)
    with H.hcms_plan(S, Hh, D, P, C, H.HCMS_DTYPE_BF16, flags) as plan:
        n = H.hcms_plan_workspace_bytes(plan)
        ws = nan_fill_(torch.empty((n + 1) // 2, dtype=torch.int16, device=DEV))
        H.hcms_plan_set_workspace(plan, ws, n)
        H.hcms_layer_forward(plan, to_dev(x), to_dev(w_qkv), to_dev(w_o), to_dev(cos), to_dev(sin), y, Dm, scale)
        torch.cuda.synchronize()
        launches = H.hcms_plan_last_launch_count(plan)
    assert launches == 3 * C + 2
    return to_host(y)


def check_layer(got_bits, ref, what):
    got = bf16_bits_to_f64(got_bits)
    assert not np.isnan(got).any(), f"{what}: NaN in y"
    err = np.abs(got - ref)
    rel = np.linalg.norm(got - ref) / np.linalg.norm(ref)
    assert err.max() <= 2e-2 and err.mean() <= 2e-3 and rel <= 1e-2, \
        f"{what}: max_abs={err.max():.3e} mean_abs={err.mean():.3e} rel_l2={rel:.3e}"


def test_layer_config1_vs_oracle_and_c_p_invariance():
    w = I.workload(1)                                    # S=1024 H=4 D=64 P=2 C=2, Dm = H*D = 256
    Dm = w.H * w.D
    x, w_qkv, w_o, cos, sin = I.make_layer_inputs(w)
    y = run_layer(x, w_qkv, w_o, cos, sin, w.S, w.H, w.D, Dm, w.P, w.C, w.scale)
    check_layer(y, L.layer_forward(x, w_qkv, w_o, cos, sin, w.H, w.D, w.scale), "layer cfg1")
    # Table 14 (L472-477): the chunked pipeline changes no bit, whatever P, C and the stream arrangement
    for P, C, flags in [(1, 1, H.HCMS_FLAG_SERIAL), (4, 1, 0), (2, 1, 0), (1, 4, 0), (1, 3, H.HCMS_FLAG_SINGLE_COMP)]:
        assert np.array_equal(run_layer(x, w_qkv, w_o, cos, sin, w.S, w.H, w.D, Dm, P, C, w.scale, flags), y), (P, C)


def test_layer_ragged_d128_uneven_chunks():
    """S = 2100 (ragged tiles, shards of 525 rows), H = 12, D = 128, P = 4, C = 2 (per-rank 3 heads split 2 + 1),
    Dm = 512 != H*D."""
    w = I.Workload("t", 2100, 12, 128, 4, 2, 21, "bf16", 1.0)
    Dm = 512
    x, w_qkv, w_o, cos, sin = I.make_layer_inputs(w, Dm)
    y = run_layer(x, w_qkv, w_o, cos, sin, w.S, w.H, w.D, Dm, w.P, w.C, w.scale)
    check_layer(y, L.layer_forward(x, w_qkv, w_o, cos, sin, w.H, w.D, w.scale), "layer ragged")


def test_layer_equals_its_three_steps_bitwise():
    """hcms_layer_forward == hcms_qkv_projection_rope; hcms_attention_forward; hcms_output_projection on caller
    tensors, and its q, k, v buffers are the projection's outputs."""
    w = I.workload(2)                                    # S=8192 H=12 D=64 P=4 C=2 (2+1)
    S, Dm = 4096, 768
    x, w_qkv, w_o, cos, sin = I.make_layer_inputs(w, Dm, S=S)
    xd, wqd, wod, cd, sd = (to_dev(t) for t in (x, w_qkv, w_o, cos, sin))
    y1, y2 = dev_out(S, Dm), dev_out(S, Dm)
    q, k, v, o = (dev_out(S, w.H, w.D) for _ in range(4))
    with H.hcms_plan(S, w.H, w.D, w.P, w.C) as plan:
        H.hcms_layer_forward(plan, xd, wqd, wod, cd, sd, y1, Dm, w.scale)
        H.hcms_qkv_projection_rope(plan, xd, wqd, cd, sd, q, k, v, Dm)
        H.hcms_attention_forward(plan, q, k, v, o, w.scale)
        H.hcms_output_projection(plan, o, wod, y2, Dm)
        torch.cuda.synchronize()
        n = S * w.H * w.D
        for which, t in enumerate((q, k, v, o)):
            src = H.hcms_plan_layer_buffer(plan, which)
            assert src
            assert torch.equal(_device_view(src, n), t.reshape(-1)), f"layer buffer {which}"
    assert np.array_equal(to_host(y1), to_host(y2))


def _device_view(ptr: int, n: int) -> torch.Tensor:
    """int16 view of n elements of device memory at ``ptr`` (a plan-owned buffer) through __cuda_array_interface__."""
    class _Raw:
        __cuda_array_interface__ = {"shape": (n,), "typestr": "<i2", "data": (ptr, False), "version": 3}
    return torch.as_tensor(_Raw(), device=DEV)


def test_layer_timings_and_errors():
    w = I.workload(1)
    Dm = 256
    x, w_qkv, w_o, cos, sin = (to_dev(t) for t in I.make_layer_inputs(w))
    y = dev_out(w.S, Dm)
    with H.hcms_plan(w.S, w.H, w.D, w.P, w.C, H.HCMS_DTYPE_BF16, H.HCMS_FLAG_PROFILE) as plan:
        with pytest.raises(H.HcmsError):
            H.hcms_plan_layer_timings(plan)                      # nothing recorded yet
        H.hcms_layer_forward(plan, x, w_qkv, w_o, cos, sin, y, Dm, w.scale)
        t = H.hcms_plan_layer_timings(plan)
        assert all(ms > 0 for ms in t)
        with pytest.raises(H.HcmsError) as e:
            H.hcms_layer_forward(plan, x, w_qkv, w_o, cos, None, y, Dm, w.scale)
        assert e.value.status == H.HCMS_ERR_INVALID_ARG           # one table only
        with pytest.raises(H.HcmsError) as e:
            H.hcms_layer_forward(plan, x, w_qkv, w_o, cos, sin, x, Dm, w.scale)
        assert e.value.status == H.HCMS_ERR_ALIAS
        with pytest.raises(H.HcmsError) as e:
            H.hcms_layer_forward(plan, x, w_qkv, w_o, cos, sin, y, 200, w.scale)
        assert e.value.status == H.HCMS_ERR_UNSUPPORTED_SHAPE


# ---------------------------------------------------------------------------------------------
# HCMS_FLAG_FUSE_A2A: all-to-alls fused into the projection GEMMs
# ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("S,Hh,D,Dm,P,C", [(1024, 4, 64, 256, 2, 2), (2100, 12, 128, 512, 4, 2), (777, 6, 64, 384, 1, 5),
                                           (1500, 8, 128, 1024, 2, 3)])
def test_fused_layer_equals_unfused_bitwise(S, Hh, D, Dm, P, C):
    """The fused layer launches 2 + C kernels (no scatter / gather) and must reproduce the unfused layer bit for
    bit: same projections, same attention kernel on the same chunk buffers.  Uneven chunks (3 -> 2+1, 6 -> 2+1+1+1+1,
    4 -> 2+1+1), ragged S, both head dims, one head per 64-column panel (D=64) and two panels per head (D=128)."""
    w = I.Workload("t", S, Hh, D, P, C, 33, "bf16", 1.0)
    x, w_qkv, w_o, cos, sin = I.make_layer_inputs(w, Dm)
    xd, wqd, wod, cd, sd = (to_dev(t) for t in (x, w_qkv, w_o, cos, sin))
    scale = w.scale
    ys = []
    for flags in (0, H.HCMS_FLAG_FUSE_A2A, H.HCMS_FLAG_FUSE_A2A | H.HCMS_FLAG_SERIAL):
        y = dev_out(S, Dm)
        with H.hcms_plan(S, Hh, D, P, C, H.HCMS_DTYPE_BF16, flags) as plan:
            n = H.hcms_plan_workspace_bytes(plan)
            ws = nan_fill_(torch.empty((n + 1) // 2, dtype=torch.int16, device=DEV))
            H.hcms_plan_set_workspace(plan, ws, n)
            H.hcms_layer_forward(plan, xd, wqd, wod, cd, sd, y, Dm, scale)
            torch.cuda.synchronize()
            assert H.hcms_plan_last_launch_count(plan) == (3 * C + 2 if flags == 0 else C + 2)
        ys.append(to_host(y))
    assert not np.isnan(bf16_bits_to_f64(ys[0])).any()
    assert np.array_equal(ys[0], ys[1]) and np.array_equal(ys[0], ys[2])


def test_fused_layer_vs_oracle_and_chunk_buffers():
    """Fused layer against the fp64 oracle, and its chunk buffers against the oracle's scatter of the projected q, k, v
    (the epilogue must place every head in the right rank / chunk / slot)."""
    w = I.Workload("t", 900, 6, 128, 2, 2, 34, "bf16", 1.0)          # per-rank 3 heads -> chunks 2 + 1
    Dm = 256
    x, w_qkv, w_o, cos, sin = I.make_layer_inputs(w, Dm)
    y = dev_out(w.S, Dm)
    with H.hcms_plan(w.S, w.H, w.D, w.P, w.C, H.HCMS_DTYPE_BF16, H.HCMS_FLAG_FUSE_A2A) as plan:
        H.hcms_layer_forward(plan, to_dev(x), to_dev(w_qkv), to_dev(w_o), to_dev(cos), to_dev(sin), y, Dm, w.scale)
        torch.cuda.synchronize()
        base = H.hcms_plan_workspace(plan)
        ref_qkv = L.project_and_rotate(x, w_qkv, cos, sin, w.H, w.D)
        _, h_c = H.hcms_chunk_table(plan)
        for c in range(w.C):
            lay = H.hcms_chunk_layout(plan, c)
            n = w.P * w.S * h_c[c] * w.D
            for t, key in enumerate(("q_off", "k_off", "v_off")):
                got = to_host(_device_view(base + lay[key], n)).reshape(w.P, w.S, h_c[c], w.D)
                check_rounded(got, O.scatter_chunk(ref_qkv[t], w.P, w.C, c), f"chunk {c} tensor {t}")
    check_layer(to_host(y), L.layer_forward(x, w_qkv, w_o, cos, sin, w.H, w.D, w.scale), "fused layer")

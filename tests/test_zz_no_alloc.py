"""-m gpu: hcms_attention_backward_chunk_static, the entry point for callers that may not allocate device memory.

Who that is: an operator inside a framework whose caching allocator already owns the card, a serving loop that cannot
afford cudaMalloc's device-wide synchronisation once it is running, a process whose memory budget was committed at
launch.  For them the scratch of the attention backward (the packed row statistics) is a fixed 4 MiB array inside
libhcms.so rather than plan-owned memory from cudaMalloc (include/hcms.h).

The check is against the existing path: the same three kernels run in hcms_attention_backward_chunk on a plan, so the
gradients must agree BIT FOR BIT -- tighter than the 1e-2 relative-L2 gate the oracle tests use, which is also applied.
Two calls in a row, the second on a smaller, ragged problem: the array is shared and keeps the first call's contents,
so a call that relied on stale or zeroed scratch would differ on the second.  The file sorts last on purpose: with
`pytest -x` a failure here hides no other test.  It holds no state of its own, so it passes alone in a fresh process
(where its first call does the per-device set-up) and after the rest of the suite.
"""
import numpy as np
import pytest
import torch

import hcms_inputs as I
import paper_2607_01817_b200 as H
from gpu_util import DEV, bf16_bits_to_f64, nan_fill_, to_dev

pytestmark = pytest.mark.gpu


def make_case(S, D, P, h, seed):
    """Saved tensors of one chunk made by the library's own forward: qc, kc, vc, oc, doc [P,S,h,D] bf16 bits, lse."""
    n = P * S * h * D
    qc, kc, vc, doc = (to_dev(I.f32_to_bf16_bits(I.normal_f32(seed, t, n).reshape(P, S, h, D))) for t in (0, 1, 2, 6))
    oc = nan_fill_(torch.empty((P, S, h, D), dtype=torch.int16, device=DEV))
    lse = torch.full((P * h, S), float("nan"), dtype=torch.float32, device=DEV)
    scale = float(np.float32(1.0 / np.sqrt(D)))
    with H.hcms_plan(S, P * h, D, P, 1) as plan:
        H.hcms_attention_chunk_lse(plan, qc, kc, vc, oc, lse, 0, scale)
        torch.cuda.synchronize()
    return qc, kc, vc, oc, doc, lse, scale


def grads(P, S, h, D):
    return tuple(nan_fill_(torch.empty((P, S, h, D), dtype=torch.int16, device=DEV)) for _ in range(3))


def existing_path(case, S, D, P, h):
    qc, kc, vc, oc, doc, lse, scale = case
    out = grads(P, S, h, D)
    with H.hcms_plan(S, P * h, D, P, 1) as plan:            # allocates its statistics scratch with cudaMalloc
        H.hcms_attention_backward_chunk(plan, qc, kc, vc, oc, doc, lse, *out, 0, scale)
        torch.cuda.synchronize()
    return out


def static_path(case, S, D, P, h):
    qc, kc, vc, oc, doc, lse, scale = case
    out = grads(P, S, h, D)
    H.hcms_attention_backward_chunk_static(qc, kc, vc, oc, doc, lse, *out, S, P, h, D, scale)
    torch.cuda.synchronize()
    return out


def assert_same(got, want, what):
    for name, g, w in zip(("dq", "dk", "dv"), got, want):
        a, b = bf16_bits_to_f64(g.cpu().numpy().view(np.uint16)), bf16_bits_to_f64(w.cpu().numpy().view(np.uint16))
        assert not np.isnan(a).any() and not np.isnan(b).any(), f"{what} {name}: NaN (a tile was never written)"
        rel = np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-30)
        assert rel <= 1e-2, f"{what} {name}: rel_l2={rel:.3e} against the existing path"      # the suite's gradient gate
        assert torch.equal(g, w), f"{what} {name}: same kernels, same inputs, different bits (rel_l2={rel:.3e})"


@pytest.mark.parametrize("D", [128, 64])
def test_static_scratch_matches_the_allocating_path_twice_in_a_row(D):
    # call 1: several key / query tiles, P = 2 ranks' heads; call 2: fewer heads, a ragged S whose padding rows
    # [S, s_pad) land where call 1 left real statistics
    shapes = [(700, D, 2, 2, 71), (333, D, 1, 3, 72)]
    cases = [make_case(*s) for s in shapes]
    want = [existing_path(c, *s[:4]) for c, s in zip(cases, shapes)]
    torch.cuda.synchronize()
    got = []
    free_before = None
    for i, (c, s) in enumerate(zip(cases, shapes)):          # the two static calls back to back, nothing in between
        if i == 1:
            outs = grads(s[2], s[0], s[3], s[1])             # torch allocates the outputs BEFORE the measurement
            torch.cuda.synchronize()
            free_before = torch.cuda.mem_get_info()[0]
            qc, kc, vc, oc, doc, lse, scale = c
            H.hcms_attention_backward_chunk_static(qc, kc, vc, oc, doc, lse, *outs, s[0], s[2], s[3], s[1], scale)
            torch.cuda.synchronize()
            assert torch.cuda.mem_get_info()[0] == free_before, "the call changed the device's free memory"
            got.append(outs)
        else:
            got.append(static_path(c, *s[:4]))
    for i, s in enumerate(shapes):
        assert_same(got[i], want[i], f"call {i + 1} S={s[0]} D={D} P={s[2]} h={s[3]}")
    # and once more on the first problem: the array now holds call 2's contents
    assert_same(static_path(cases[0], *shapes[0][:4]), want[0], "call 3 (first problem again)")


def test_static_scratch_rejects_what_does_not_fit():
    """Beyond HCMS_STATIC_SCRATCH_BYTES the call says so and enqueues nothing (the pointers are never touched)."""
    dummy = torch.zeros(64, dtype=torch.int16, device=DEV)
    S_fit = H.HCMS_STATIC_SCRATCH_BYTES // 8                   # one head of exactly the limit: accepted by the size test
    args = [dummy] * 9
    with pytest.raises(H.HcmsError) as ei:
        H.hcms_attention_backward_chunk_static(*args, S_fit, 1, 2, 128, 0.1)       # two such heads: 8 MiB
    assert ei.value.status == H.HCMS_ERR_WORKSPACE_TOO_SMALL and "static" in str(ei.value)
    with pytest.raises(H.HcmsError) as ei:
        H.hcms_attention_backward_chunk_static(*args, S_fit + 1, 1, 1, 128, 0.1)   # rounds up to the next 64 rows
    assert ei.value.status == H.HCMS_ERR_WORKSPACE_TOO_SMALL
    with pytest.raises(H.HcmsError) as ei:
        H.hcms_attention_backward_chunk_static(*args, 128, 1, 1, 96, 0.1)
    assert ei.value.status == H.HCMS_ERR_UNSUPPORTED_SHAPE
    torch.cuda.synchronize()

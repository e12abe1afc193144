"""-m gpu: the dual-stream chunk scheduler of hcms_attention_forward (section 3.4-3.6,
Algorithm 1) observed through the C ABI: event ordering (Eq. 6-7), the host-routed emulated
wire (BASELINE.json configs[4]), the adaptive chunk count (future work L346), and a negative test that
shows the E_c^comm wait is what keeps attention behind its all-to-all.

Every variant must produce the SAME BITS as the plain call (the schedule changes, the function does
not: L31, Table 14); the plain call itself is checked against the oracle in
test_gpu_attention.py.
"""
import numpy as np
import pytest
import torch

import hcms_inputs as I
import paper_2607_01817_b200 as H
from gpu_util import DEV, nan_fill_, to_dev, to_host

pytestmark = pytest.mark.gpu


def _inputs(S, Hh, D, seed=11):
    w = I.Workload("sched", S, Hh, D, 1, 1, seed, "bf16", 1.0)
    return tuple(to_dev(t) for t in I.make_qkv(w)), float(D) ** -0.5


def _forward(qkv, S, Hh, D, P, C, scale, flags=0, poison_ws=True):
    q, k, v = qkv
    out = nan_fill_(torch.empty_like(q))
    with H.hcms_plan(S, Hh, D, P, C, H.HCMS_DTYPE_BF16, flags) as plan:
        if poison_ws:
            n = H.hcms_plan_workspace_bytes(plan)
            ws = nan_fill_(torch.empty((n + 1) // 2, dtype=torch.int16, device=DEV))
            H.hcms_plan_set_workspace(plan, ws, n)
        H.hcms_attention_forward(plan, q, k, v, out, scale)
        torch.cuda.synchronize()
    return to_host(out)


def test_timeline_obeys_eq6_eq7_and_alg1_order():
    S, Hh, D, P, C = 4096, 12, 128, 2, 3
    qkv, scale = _inputs(S, Hh, D)
    out = torch.empty_like(qkv[0])
    for flags in (0, H.HCMS_FLAG_SINGLE_COMP, H.HCMS_FLAG_SPLIT_COMM):
        with H.hcms_plan(S, Hh, D, P, C, H.HCMS_DTYPE_BF16, flags | H.HCMS_FLAG_PROFILE) as plan:
            for _ in range(3):
                H.hcms_attention_forward(plan, *qkv, out, scale)
            b, e = H.hcms_plan_timeline(plan, 0)
            dur = H.hcms_plan_timings(plan, 0)
        (sb, ab, gb), (se, ae, ge) = b, e
        assert sb[0] == 0.0
        for c in range(C):
            assert se[c] <= ab[c] + 1e-3, "Attn_c <- wait(E_c^comm)  (Eq. 6)"
            assert ae[c] <= gb[c] + 1e-3, "A_c^out <- wait(E_c^comp)  (Eq. 7)"
            assert se[c] > sb[c] and ae[c] > ab[c] and ge[c] > gb[c]
            for kind, (bb, ee) in enumerate(((sb, se), (ab, ae), (gb, ge))):
                assert abs((ee[c] - bb[c]) - dur[kind][c]) < 2e-3
            if c:
                assert sb[c] >= se[c - 1] - 1e-3, "S_comm issues the input all-to-alls in chunk order (Alg. 1 lines 6-11)"
                assert gb[c] >= ge[c - 1] - 1e-3
                if flags & H.HCMS_FLAG_SINGLE_COMP:
                    assert ab[c] >= ae[c - 1] - 1e-3, "one S_comp runs the chunks in order"
        if not flags & H.HCMS_FLAG_SPLIT_COMM:
            assert gb[0] >= se[C - 1] - 1e-3, "single S_comm: output all-to-alls follow all input all-to-alls (R-8)"
        # the overlap the method exists for: chunk 1's scatter is under way or done before chunk 0's attention ends
        assert sb[1] < ae[0]


def test_timeline_errors():
    with H.hcms_plan(1024, 4, 64, 2, 2) as plan:
        with pytest.raises(H.HcmsError) as ei:
            H.hcms_plan_timeline(plan, 0)
        assert ei.value.status == H.HCMS_ERR_INVALID_ARG
    with H.hcms_plan(1024, 4, 64, 2, 2, H.HCMS_DTYPE_BF16, H.HCMS_FLAG_PROFILE) as plan:
        with pytest.raises(H.HcmsError):
            H.hcms_plan_timeline(plan, 0)          # no call recorded yet


def test_host_routed_wire_keeps_the_bits():
    S, Hh, D, P, C = 2048, 8, 64, 2, 2
    qkv, scale = _inputs(S, Hh, D, seed=5)
    ref = _forward(qkv, S, Hh, D, P, C, scale)
    Q, K, V, O = H.HCMS_FLAG_HOST_ROUTE_Q, H.HCMS_FLAG_HOST_ROUTE_K, H.HCMS_FLAG_HOST_ROUTE_V, H.HCMS_FLAG_HOST_ROUTE_O
    for mask in (O, Q | O, Q | K | V | O):
        for extra in (0, H.HCMS_FLAG_SERIAL, H.HCMS_FLAG_SPLIT_COMM):
            got = _forward(qkv, S, Hh, D, P, C, scale, mask | extra)
            assert np.array_equal(got, ref), (hex(mask), hex(extra))


def test_autotune_chunks_measures_every_C_and_keeps_the_bits():
    S, Hh, D, P = 2048, 8, 128, 2
    qkv, scale = _inputs(S, Hh, D, seed=3)
    ref = _forward(qkv, S, Hh, D, P, 1, scale)
    out = nan_fill_(torch.empty_like(qkv[0]))
    best, ms = H.hcms_autotune_chunks(S, Hh, D, P, H.HCMS_DTYPE_BF16, 0, *qkv, out, scale, 6, 2)
    torch.cuda.synchronize()
    assert 1 <= best <= 4 and len(ms) == 6
    assert all(m > 0 for m in ms[:4]) and ms[4] == -1 and ms[5] == -1       # H/P = 4 caps the sweep
    assert ms[best - 1] == min(ms[:4])
    assert np.array_equal(to_host(out), ref)
    with pytest.raises(H.HcmsError) as ei:
        H.hcms_autotune_chunks(S, Hh, D, P, H.HCMS_DTYPE_BF16, 0, *qkv, out, scale, 0, 2)
    assert ei.value.status == H.HCMS_ERR_INVALID_ARG


def test_dropping_the_comm_wait_lets_attention_read_unscattered_chunks():
    """Negative test: with HCMS_FLAG_DEBUG_NO_COMM_WAIT the compute stream no longer waits
    on E_c^comm.  V takes the emulated wire through pinned host memory (milliseconds), so attention, no longer
    held back by the event, reads the NaN-poisoned V'_c before the wire delivers it.  The same call with the
    wait in place is clean (checked first)."""
    S, Hh, D, P, C = 8192, 16, 128, 2, 2
    qkv, scale = _inputs(S, Hh, D, seed=9)
    is_nan = lambda bits: ((bits & 0x7F80) == 0x7F80) & ((bits & 0x007F) != 0)
    good = _forward(qkv, S, Hh, D, P, C, scale, H.HCMS_FLAG_HOST_ROUTE_V)
    assert not is_nan(good).any()
    assert np.array_equal(good, _forward(qkv, S, Hh, D, P, C, scale))
    bad = _forward(qkv, S, Hh, D, P, C, scale, H.HCMS_FLAG_HOST_ROUTE_V | H.HCMS_FLAG_DEBUG_NO_COMM_WAIT)
    assert is_nan(bad).any(), "the race did not show: the negative test has lost its teeth"


# ---------------------------------------------------------------------------------------------
# HCMS_FLAG_GRAPH: the chunk pipeline captured into a CUDA graph
# ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("extra", [0, H.HCMS_FLAG_SERIAL, H.HCMS_FLAG_SPLIT_COMM, H.HCMS_FLAG_SINGLE_COMP,
                                   H.HCMS_FLAG_HOST_ROUTE_K | H.HCMS_FLAG_HOST_ROUTE_O, H.HCMS_FLAG_LAYOUT_TMA])
def test_graph_replay_same_bits(extra):
    """One capture, many replays, the bits of the plain call; new tensors capture again; poisoned workspace and
    output before every replay (a replay that skipped a node or broke an Eq. 6-7 edge would leave NaN)."""
    S, Hh, D, P, C = 2048, 6, 64, 2, 3
    qkv, scale = _inputs(S, Hh, D, seed=21)
    want = _forward(qkv, S, Hh, D, P, C, scale, extra)
    q, k, v = qkv
    out, out2 = nan_fill_(torch.empty_like(q)), nan_fill_(torch.empty_like(q))
    with H.hcms_plan(S, Hh, D, P, C, H.HCMS_DTYPE_BF16, extra | H.HCMS_FLAG_GRAPH) as plan:
        n = H.hcms_plan_workspace_bytes(plan)
        ws = torch.empty((n + 1) // 2, dtype=torch.int16, device=DEV)
        H.hcms_plan_set_workspace(plan, ws, n)
        for _ in range(3):
            nan_fill_(ws)
            nan_fill_(out)
            H.hcms_attention_forward(plan, q, k, v, out, scale)
            torch.cuda.synchronize()
            assert np.array_equal(to_host(out), want)
        assert H.hcms_plan_graph_captures(plan) == 1
        launches = H.hcms_plan_last_launch_count(plan)
        H.hcms_attention_forward(plan, q, k, v, out2, scale)             # another output tensor -> second capture
        torch.cuda.synchronize()
        assert H.hcms_plan_graph_captures(plan) == 2 and np.array_equal(to_host(out2), want)
        assert H.hcms_plan_last_launch_count(plan) == launches
        H.hcms_attention_forward(plan, q, k, v, out2, scale * 0.5)       # another scale -> third capture
        torch.cuda.synchronize()
        assert H.hcms_plan_graph_captures(plan) == 3 and not np.array_equal(to_host(out2), want)


def test_graph_recaptures_after_a_workspace_swap():
    """a captured graph holds the workspace addresses; hcms_plan_set_workspace must void it.  Capture on
    the plan-owned workspace (freed by the swap), swap in a NaN-poisoned one, call again on the same tensors: same
    bits, second capture, and the new workspace is the one that was written."""
    S, Hh, D, P, C = 2048, 6, 64, 2, 3
    qkv, scale = _inputs(S, Hh, D, seed=23)
    want = _forward(qkv, S, Hh, D, P, C, scale)
    q, k, v = qkv
    out = nan_fill_(torch.empty_like(q))
    with H.hcms_plan(S, Hh, D, P, C, H.HCMS_DTYPE_BF16, H.HCMS_FLAG_GRAPH) as plan:
        H.hcms_attention_forward(plan, q, k, v, out, scale)               # capture #1 on the plan-owned workspace
        torch.cuda.synchronize()
        assert np.array_equal(to_host(out), want) and H.hcms_plan_graph_captures(plan) == 1
        n = H.hcms_plan_workspace_bytes(plan)
        for _ in range(2):                                                # two swaps: caller-owned -> caller-owned too
            ws = nan_fill_(torch.empty((n + 1) // 2, dtype=torch.int16, device=DEV))
            H.hcms_plan_set_workspace(plan, ws, n)
            captures = H.hcms_plan_graph_captures(plan)
            nan_fill_(out)
            H.hcms_attention_forward(plan, q, k, v, out, scale)
            torch.cuda.synchronize()
            assert np.array_equal(to_host(out), want)
            assert H.hcms_plan_graph_captures(plan) == captures + 1
            o_off = H.hcms_chunk_layout(plan, 0)["o_off"]
            head = to_host(ws[o_off // 2:o_off // 2 + 4096])              # chunk 0's O'_c lives in the NEW workspace
            assert not (head == 0x7FC0).all()


def test_graph_on_a_side_stream_orders_with_the_caller():
    """The replay is ordered after work already on the caller's stream and before what follows it."""
    S, Hh, D, P, C = 1024, 4, 64, 2, 2
    qkv, scale = _inputs(S, Hh, D, seed=22)
    want = _forward(qkv, S, Hh, D, P, C, scale)
    side = torch.cuda.Stream()
    with H.hcms_plan(S, Hh, D, P, C, H.HCMS_DTYPE_BF16, H.HCMS_FLAG_GRAPH) as plan:
        with torch.cuda.stream(side):
            q = torch.zeros_like(qkv[0])
            for _ in range(3):
                q.copy_(qkv[0], non_blocking=True)                       # producer on the caller's stream
                out = nan_fill_(torch.empty_like(q))
                H.hcms_attention_forward(plan, q, qkv[1], qkv[2], out, scale, stream=side)
                res = out.clone()                                        # consumer on the caller's stream
                q.zero_()
        side.synchronize()
        assert np.array_equal(to_host(res), want)


# ---------------------------------------------------------------------------------------------
# hcms_attention_forward_host: the host link as the wire (strided copies = the all-to-all)
# ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("S,Hh,D,P,C", [(1024, 4, 64, 2, 2), (2100, 12, 128, 4, 2), (777, 5, 128, 1, 3)])
def test_host_entry_strided_copies_same_bits(S, Hh, D, P, C):
    """Default host path (cudaMemcpy2DAsync per rank and chunk into / out of the chunk buffers, no layout kernels) ==
    staged host path == device path, bit for bit; pageable and pinned host memory; poisoned output and workspace."""
    w = I.Workload("host", S, Hh, D, P, C, 71, "bf16", 1.0)
    q, k, v = I.make_qkv(w)
    want = _forward(tuple(to_dev(t) for t in (q, k, v)), S, Hh, D, P, C, w.scale)
    for flags, launches in ((0, 4 * P * C + C), (H.HCMS_FLAG_HOST_STAGED, 3 * C)):
        with H.hcms_plan(S, Hh, D, P, C, H.HCMS_DTYPE_BF16, flags) as plan:
            n = H.hcms_plan_workspace_bytes(plan)
            ws = nan_fill_(torch.empty((n + 1) // 2, dtype=torch.int16, device=DEV))
            H.hcms_plan_set_workspace(plan, ws, n)
            out = np.full_like(q, 0x7FC0)
            H.hcms_attention_forward_host(plan, q, k, v, out, w.scale)              # pageable numpy memory
            assert np.array_equal(out, want), flags
            assert H.hcms_plan_last_launch_count(plan) == launches
            pin = [torch.from_numpy(t.view(np.int16)).pin_memory() for t in (q, k, v)]
            pout = torch.full(q.shape, 0x7FC0, dtype=torch.int16).pin_memory()
            for _ in range(2):
                H.hcms_attention_forward_host(plan, pin[0], pin[1], pin[2], pout, w.scale)
            assert np.array_equal(pout.numpy().view(np.uint16), want), flags


def test_autotune_chunks_over_the_host_link():
    """Adaptive C (L346, Theorem 1) where it matters: every C in [1, H/P] timed through the host-buffer path; the
    result of the last measured call is the plain call's bits, and a single chunk (no overlap at all) is never best
    when the transfer is a large share of the call."""
    S, Hh, D, P = 8192, 8, 128, 2
    w = I.Workload("tune", S, Hh, D, P, 1, 81, "bf16", 1.0)
    q, k, v = I.make_qkv(w)
    want = _forward(tuple(to_dev(t) for t in (q, k, v)), S, Hh, D, P, 2, w.scale)
    pin = [torch.from_numpy(t.view(np.int16)).pin_memory() for t in (q, k, v)]
    pout = torch.full(q.shape, 0x7FC0, dtype=torch.int16).pin_memory()
    best, ms = H.hcms_autotune_chunks_host(S, Hh, D, P, 0, pin[0], pin[1], pin[2], pout, w.scale, 6, 3)
    assert 1 <= best <= 4 and all(m > 0 for m in ms[:4]) and ms[4] == -1 and ms[5] == -1      # H/P = 4 caps the range
    assert ms[best - 1] == min(ms[:4]) and best > 1
    assert np.array_equal(pout.numpy().view(np.uint16), want)


# ---------------------------------------------------------------------------------------------
# plan-level caching ("device-level caching"): descriptors, workspace
# ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("flags", [0, H.HCMS_FLAG_LAYOUT_TMA, H.HCMS_FLAG_ATTN_PAIR])
def test_tensor_maps_are_encoded_once_per_plan(flags):
    """Every TMA descriptor lives in the plan: the first call encodes them, later calls on the same tensors
    encode nothing; another output tensor encodes only the maps that name it."""
    S, Hh, D, P, C = 2048, 8, 128, 2, 2
    qkv, scale = _inputs(S, Hh, D, seed=31)
    q, k, v = qkv
    out, out2 = torch.empty_like(q), torch.empty_like(q)
    with H.hcms_plan(S, Hh, D, P, C, H.HCMS_DTYPE_BF16, flags) as plan:
        assert H.hcms_plan_tensor_map_encodes(plan) == 0
        H.hcms_attention_forward(plan, q, k, v, out, scale)
        first = H.hcms_plan_tensor_map_encodes(plan)
        assert first >= 4 * C                                   # q, k, v, o maps of every chunk's attention launch
        for _ in range(3):
            H.hcms_attention_forward(plan, q, k, v, out, scale)
        assert H.hcms_plan_tensor_map_encodes(plan) == first
        H.hcms_attention_forward(plan, q, k, v, out2, scale)
        extra = H.hcms_plan_tensor_map_encodes(plan) - first
        _, h_c = H.hcms_chunk_table(plan)
        assert extra == (len(set(h_c)) if flags & H.HCMS_FLAG_LAYOUT_TMA else 0)   # only the TMA gather's map(s) of `out`
        torch.cuda.synchronize()
        assert torch.equal(out, out2)


def test_workspace_is_allocated_on_first_use_only():
    """A caller-supplied workspace never coexists with a plan-owned one: creating the plan allocates
    no chunk buffers; the first forward does, unless hcms_plan_set_workspace came first."""
    S, Hh, D, P, C = 8192, 16, 128, 2, 2
    qkv, scale = _inputs(S, Hh, D, seed=32)
    q, k, v = qkv
    out = torch.empty_like(q)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    with H.hcms_plan(S, Hh, D, P, C) as plan:
        n = H.hcms_plan_workspace_bytes(plan)
        assert n >= 4 * S * Hh * D * 2
        free1, _ = torch.cuda.mem_get_info()
        assert free0 - free1 < n // 2                                     # no workspace yet
        ws = torch.empty((n + 1) // 2, dtype=torch.int16, device=DEV)     # torch's allocation, counted before the call
        free2, _ = torch.cuda.mem_get_info()
        H.hcms_plan_set_workspace(plan, ws, n)
        H.hcms_attention_forward(plan, q, k, v, out, scale)
        torch.cuda.synchronize()
        free3, _ = torch.cuda.mem_get_info()
        assert free2 - free3 < n // 2                                     # the plan never allocated its own
    with H.hcms_plan(S, Hh, D, P, C) as plan:
        free4, _ = torch.cuda.mem_get_info()
        H.hcms_attention_forward(plan, q, k, v, out, scale)
        torch.cuda.synchronize()
        free5, _ = torch.cuda.mem_get_info()
        assert free4 - free5 >= n // 2                                    # allocated by the first call


def test_backward_rejects_another_scale_and_a_replaced_workspace():
    S, Hh, D, P, C = 512, 4, 64, 2, 2
    qkv, scale = _inputs(S, Hh, D, seed=33)
    q, k, v = qkv
    out = torch.empty_like(q)
    g = [torch.empty_like(q) for _ in range(4)]
    with H.hcms_plan(S, Hh, D, P, C, H.HCMS_DTYPE_BF16, H.HCMS_FLAG_TRAINING) as plan:
        H.hcms_attention_forward(plan, q, k, v, out, scale)
        with pytest.raises(H.HcmsError) as ei:
            H.hcms_attention_backward(plan, g[0], g[1], g[2], g[3], scale * 0.5)
        assert ei.value.status == H.HCMS_ERR_INVALID_ARG
        H.hcms_attention_backward(plan, g[0], g[1], g[2], g[3], scale)
        n = H.hcms_plan_workspace_bytes(plan)
        ws = torch.empty((n + 1) // 2, dtype=torch.int16, device=DEV)
        H.hcms_plan_set_workspace(plan, ws, n)
        with pytest.raises(H.HcmsError) as ei:                              # the saved Q'_c .. O'_c are gone
            H.hcms_attention_backward(plan, g[0], g[1], g[2], g[3], scale)
        assert ei.value.status == H.HCMS_ERR_INVALID_ARG
        torch.cuda.synchronize()


# ---------------------------------------------------------------------------------------------
# HCMS_FLAG_RECYCLE_WS: two chunk buffer sets instead of C (peak memory, Table 16)
# ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("S,Hh,D,P,C", [(1500, 12, 64, 2, 3), (2100, 20, 128, 2, 5), (1024, 12, 128, 1, 12), (1024, 8, 64, 2, 2)])
def test_recycled_workspace_same_bits_and_smaller(S, Hh, D, P, C):
    """Chunk c reuses the buffers of chunk c - 2 (A_{c-2}^out before A_c^in on the comm stream): same bits as the plain
    plan from a NaN-poisoned workspace, three calls in a row, also serial, as a graph and through the host entry; the
    workspace shrinks to two sets of the largest chunk."""
    qkv, scale = _inputs(S, Hh, D, seed=21)
    ref = _forward(qkv, S, Hh, D, P, C, scale)
    R = H.HCMS_FLAG_RECYCLE_WS
    with H.hcms_plan(S, Hh, D, P, C) as plain, H.hcms_plan(S, Hh, D, P, C, H.HCMS_DTYPE_BF16, R) as ring:
        full, small = H.hcms_plan_workspace_bytes(plain), H.hcms_plan_workspace_bytes(ring)
        _, h = H.hcms_chunk_table(ring)
        if C > 2:
            assert small < full and small <= 2 * 4 * (P * S * h[0] * D * 2 + 1024)
            l0, l2 = H.hcms_chunk_layout(ring, 0), H.hcms_chunk_layout(ring, 2)
            assert l0["q_off"] == l2["q_off"] and l0["o_off"] >= l2["o_off"]          # chunk 2 lives in chunk 0's set
        else:
            assert small == full
    for extra in (0, H.HCMS_FLAG_SERIAL, H.HCMS_FLAG_SINGLE_COMP, H.HCMS_FLAG_GRAPH, H.HCMS_FLAG_LAYOUT_TMA, H.HCMS_FLAG_PROFILE,
                  H.HCMS_FLAG_HOST_ROUTE_Q | H.HCMS_FLAG_HOST_ROUTE_O):
        q, k, v = qkv
        out = nan_fill_(torch.empty_like(q))
        with H.hcms_plan(S, Hh, D, P, C, H.HCMS_DTYPE_BF16, R | extra) as plan:
            n = H.hcms_plan_workspace_bytes(plan)
            ws = nan_fill_(torch.empty((n + 1) // 2, dtype=torch.int16, device=DEV))
            H.hcms_plan_set_workspace(plan, ws, n)
            for _ in range(3):
                nan_fill_(out)
                H.hcms_attention_forward(plan, q, k, v, out, scale)
            torch.cuda.synchronize()
            assert H.hcms_plan_last_launch_count(plan) == 3 * C or (extra & (H.HCMS_FLAG_GRAPH | H.HCMS_FLAG_HOST_ROUTE_Q))
        assert np.array_equal(to_host(out), ref), hex(extra)
    hq, hk, hv = (to_host(t) for t in qkv)
    hout = np.full_like(hq, 0x7FC0)
    with H.hcms_plan(S, Hh, D, P, C, H.HCMS_DTYPE_BF16, R) as plan:
        H.hcms_attention_forward_host(plan, hq, hk, hv, hout, scale)
    assert np.array_equal(hout, ref)


def test_recycled_workspace_flag_errors():
    for bad in (H.HCMS_FLAG_TRAINING, H.HCMS_FLAG_FUSE_A2A, H.HCMS_FLAG_SPLIT_COMM):
        with pytest.raises(H.HcmsError) as e:
            H.hcms_plan(1024, 8, 64, 2, 4, H.HCMS_DTYPE_BF16, H.HCMS_FLAG_RECYCLE_WS | bad)
        assert e.value.status == H.HCMS_ERR_INVALID_ARG

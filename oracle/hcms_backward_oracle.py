"""fp64 CPU oracle for the BACKWARD of the HCMS hot path.  TEST INFRASTRUCTURE, NOT
PRODUCT -- same rules as ``oracle/hcms_oracle.py``; shares no code with ``paper_2607_01817_b200``.

PAPER.md: "HCMS is compatible with PyTorch autograd, achieving 3.5% speedup for forward+backward combined
execution" (L304; Appendix C Table 15) and "extending HCMS to backward propagation" (L346).  The
paper gives no backward algorithm: autograd differentiates Alg. 1 (L170).  What that computes has a plain
definition -- the gradient of the forward definition -- so the oracle is that definition written out:

forward (Eq. 2, per head):  s_ik = scale * q_i . k_k ;  p_ik = softmax_k(s_ik) ;  o_i = sum_k p_ik v_k
given dO = dL/dO, the chain rule gives (standard softmax-attention calculus)
    dV_k  = sum_i p_ik dO_i
    dP_ik = dO_i . v_k
    dS_ik = p_ik * (dP_ik - sum_k' p_ik' dP_ik')          (softmax Jacobian;  the sum equals dO_i . o_i)
    dQ_i  = scale * sum_k dS_ik k_k ,     dK_k = scale * sum_i dS_ik q_i
The all-to-alls are permutations, so their adjoints are the inverse permutations: the backward of
Alg. 1 lines 4-26 is  dO --scatter--> dO'_c --attention backward per head--> dQ'_c, dK'_c, dV'_c --gather-->
dQ, dK, dV  (``hcms_backward_composed``), chunk by chunk, and equals the direct gradient bit for bit.

* ``log_sum_exp``               the row statistic the forward saves: lse_i = log sum_k exp(s_ik)
* ``attention_backward_head``   the five formulas above for one head
* ``attention_backward``        all heads of global [S,H,D] tensors
* ``attention_backward_sampled`` dQ for sampled query rows and dK, dV for sampled key rows (large shapes)
* ``hcms_backward_composed``    the chunked path executed literally

Pins (tests/test_oracle_backward.py): central finite differences of the forward oracle, torch.autograd in
fp64 through a hand-written softmax and through scaled_dot_product_attention, closed forms (scale = 0,
one key, two keys), invariants (sum_k dS_ik = 0; dL/dV linear in dO), composed == direct.
No function here is "parity unpinned".
"""
from __future__ import annotations

import numpy as np

from . import hcms_oracle as A

widen_to_f64 = A.widen_to_f64


def _probs(q, k, scale: float):
    s = (q @ k.T) * float(scale)
    m = s.max(axis=1, keepdims=True)
    w = np.exp(s - m)
    den = w.sum(axis=1, keepdims=True)
    return w / den, (m + np.log(den))[:, 0]


def log_sum_exp(q, k, scale: float) -> np.ndarray:
    """One head: ``lse_i = log sum_k exp(scale * q_i . k_k)`` (natural log), fp64 ``[S]``."""
    return _probs(widen_to_f64(q), widen_to_f64(k), scale)[1]


def attention_backward_head(q, k, v, do, scale: float):
    """One head, fp64 ``[S,D]`` inputs -> ``(dq, dk, dv)``, the formulas in the module docstring."""
    p, _ = _probs(q, k, scale)                      # [Sq, Sk]
    dv = p.T @ do
    dp = do @ v.T
    ds = p * (dp - (p * dp).sum(axis=1, keepdims=True))
    dq = float(scale) * (ds @ k)
    dk = float(scale) * (ds.T @ q)
    return dq, dk, dv


def attention_backward(q, k, v, do, scale: float):
    """Global ``[S,H,D]`` tensors (any storage dtype) -> fp64 ``(dq, dk, dv)`` each ``[S,H,D]``."""
    S, H, D = q.shape
    outs = [np.empty((S, H, D), dtype=np.float64) for _ in range(3)]
    for h in range(H):
        g = attention_backward_head(*(widen_to_f64(t[:, h, :]) for t in (q, k, v, do)), scale)
        for o, x in zip(outs, g):
            o[:, h, :] = x
    return tuple(outs)


def attention_backward_sampled(q, k, v, do, scale: float, q_rows, k_rows, row_block: int = 2048):
    """Large shapes: ``dq[q_rows]`` needs those query rows only; ``dk[k_rows]``, ``dv[k_rows]`` need column
    ``k`` of P for every query, i.e. every row's normaliser.  Returns fp64 ``(dq [Rq,H,D], dk [Rk,H,D], dv [Rk,H,D])``.
    Row statistics are computed in blocks of ``row_block`` query rows (it only bounds the ``[rows, S]`` score
    matrix); nothing inside a row is reordered, and the sums over queries ``dV_k = sum_i p_ik dO_i``,
    ``dK_k = scale sum_i dS_ik q_i`` are accumulated block after block in row order."""
    q_rows, k_rows = np.asarray(q_rows, np.int64), np.asarray(k_rows, np.int64)
    S, H, D = q.shape
    dq = np.empty((len(q_rows), H, D))
    dk = np.zeros((len(k_rows), H, D))
    dv = np.zeros((len(k_rows), H, D))
    for h in range(H):
        qh, kh, vh, doh = (widen_to_f64(t[:, h, :]) for t in (q, k, v, do))
        # dq for the sampled query rows
        p, _ = _probs(qh[q_rows], kh, scale)
        dp = doh[q_rows] @ vh.T
        ds = p * (dp - (p * dp).sum(axis=1, keepdims=True))
        dq[:, h, :] = float(scale) * (ds @ kh)
        # dk, dv for the sampled key rows: walk over all query rows in blocks
        for r0 in range(0, S, row_block):
            sl = slice(r0, min(r0 + row_block, S))
            p, _ = _probs(qh[sl], kh, scale)                            # [rows, S]
            delta = (doh[sl] * (p @ vh)).sum(axis=1, keepdims=True)     # dO_i . o_i
            pk = p[:, k_rows]                                           # [rows, Rk]
            dpk = doh[sl] @ vh[k_rows].T
            dsk = pk * (dpk - delta)
            dv[:, h, :] += pk.T @ doh[sl]
            dk[:, h, :] += float(scale) * (dsk.T @ qh[sl])
    return dq, dk, dv


def hcms_backward_composed(q, k, v, do, P: int, C: int, scale: float):
    """The backward of Alg. 1 lines 4-26 executed literally: per head chunk, the input all-to-all of dO (and
    of the saved Q, K, V), the attention backward on every rank's heads, the output all-to-all of dQ', dK', dV'."""
    S, H, D = q.shape
    outs = [np.full((S, H, D), np.nan) for _ in range(3)]
    Hl = H // P
    for c, (_, h_c) in enumerate(A.chunk_table(Hl, C)):
        qc, kc, vc, doc = (A.scatter_chunk(t, P, C, c) for t in (q, k, v, do))
        gc = [np.empty((P, S, h_c, D)) for _ in range(3)]
        for p in range(P):
            for j in range(h_c):
                g = attention_backward_head(*(widen_to_f64(t[p, :, j, :]) for t in (qc, kc, vc, doc)), scale)
                for dst, x in zip(gc, g):
                    dst[p, :, j, :] = x
        for dst, src in zip(outs, gc):
            A.gather_chunk(src, dst, P, C, c)
    return tuple(outs)

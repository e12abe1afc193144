"""fp64 CPU oracle for the HCMS attention LAYER (Alg. 1 lines 2-3 and 26-27 around the hot path).
TEST INFRASTRUCTURE, NOT PRODUCT -- same rules as ``oracle/hcms_oracle.py``: only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may
import it; it shares no code with ``paper_2607_01817_b200`` and imports nothing from it.

Written from /root/reference/PAPER.md ("L<n>" = PAPER.md line).  Section 3.1 (L59): "the forward
pass consisting of: QKV projection -> RoPE positional encoding -> input all-to-all -> attention
computation -> output all-to-all -> output projection"; Algorithm 1 (L170) line 2
``Q,K,V <- QKVProjection(X)``, line 3 ``Q,K <- ApplyRoPE(Q,K)``, line 26 ``O <- Concat``, line 27
``Y <- OutputProjection(O)``.  Table 3 (L210-215): D_model = 5120 = H*D (40 x 128).

Each result has a plain definition, so each function IS that definition in fp64:

* ``qkv_projection``     three linear maps of X (a matmul per tensor; no bias -- reading R-22).
* ``apply_rope``         rotary embedding [34]: every adjacent pair (x[2i], x[2i+1]) of a head vector
                         is rotated by the angle of (token, i) -- reading R-23; the angles come in as
                         cos/sin tables, so any position scheme (1-D, 3-D video grid) is covered.
* ``output_projection``  one linear map of the concatenated heads.
* ``layer_forward``      lines 2-27 with the attention of ``hcms_oracle.attention_full``.
* ``layer_forward_rows`` the same for a sample of output rows (large shapes).
* ``layer_forward_composed``  lines 2-27 executed literally through the chunked path
                         (``hcms_oracle.hcms_forward_composed``); must equal ``layer_forward`` bit for bit.

Pins: tests/test_oracle_layer.py (closed forms, invariants, brute force, torch fp64 library
routines).  No function here is "parity unpinned".
"""
from __future__ import annotations

import numpy as np

from . import hcms_oracle as A

widen_to_f64 = A.widen_to_f64


def qkv_projection(x, w_qkv, H: int, D: int):
    """Alg. 1 line 2.  ``x [S, Dm]``, ``w_qkv [3*H*D, Dm]`` (row n = output feature n; features are
    ordered q heads, then k heads, then v heads, each head D consecutive features; ``y = x W^T`` as
    in ``torch.nn.Linear`` without bias, reading R-22).  Returns fp64 q, k, v ``[S, H, D]``."""
    x64, w64 = widen_to_f64(x), widen_to_f64(w_qkv)
    S, Dm = x64.shape
    if w64.shape != (3 * H * D, Dm):
        raise ValueError("w_qkv must be [3*H*D, Dm]")
    y = x64 @ w64.T                                   # [S, 3*H*D]
    q, k, v = (y[:, t * H * D:(t + 1) * H * D].reshape(S, H, D) for t in range(3))
    return q, k, v


def apply_rope(x, cos, sin):
    """Alg. 1 line 3 for one tensor ``x [S, H, D]`` (fp64): for token s, head h, pair i < D/2
    ``(x[2i], x[2i+1]) <- (x[2i] c - x[2i+1] s, x[2i] s + x[2i+1] c)`` with ``c = cos[s, i]``,
    ``s = sin[s, i]`` (tables ``[S, D/2]``): the 2-D rotation of RoFormer [34] on adjacent pairs."""
    x = np.asarray(x, dtype=np.float64)
    c = widen_to_f64(cos)[:, None, :]
    s = widen_to_f64(sin)[:, None, :]
    S, H, D = x.shape
    if c.shape != (S, 1, D // 2) or s.shape != (S, 1, D // 2):
        raise ValueError("cos/sin must be [S, D/2]")
    out = np.empty_like(x)
    xe, xo = x[:, :, 0::2], x[:, :, 1::2]
    out[:, :, 0::2] = xe * c - xo * s
    out[:, :, 1::2] = xe * s + xo * c
    return out


def output_projection(o, w_o):
    """Alg. 1 line 27.  ``o [S, H, D]`` (Concat of the head outputs, line 26), ``w_o [Dm, H*D]``;
    ``y = o.reshape(S, H*D) @ w_o^T`` -> fp64 ``[S, Dm]``."""
    o64, w64 = widen_to_f64(o), widen_to_f64(w_o)
    S, H, D = o64.shape
    if w64.shape[1] != H * D:
        raise ValueError("w_o must be [Dm, H*D]")
    return o64.reshape(S, H * D) @ w64.T


def project_and_rotate(x, w_qkv, cos, sin, H: int, D: int):
    """Lines 2-3: q, k after RoPE and v, fp64 ``[S, H, D]`` each."""
    q, k, v = qkv_projection(x, w_qkv, H, D)
    return apply_rope(q, cos, sin), apply_rope(k, cos, sin), v


def layer_forward(x, w_qkv, w_o, cos, sin, H: int, D: int, scale: float):
    """Alg. 1 lines 2-27 as one function of X: projection, RoPE, per-head softmax(QK^T scale)V
    (Eq. 2, bidirectional L43), output projection.  fp64 ``[S, Dm]``."""
    q, k, v = project_and_rotate(x, w_qkv, cos, sin, H, D)
    o = A.attention_full(q, k, v, scale)
    return output_projection(o, w_o)


def layer_forward_rows(x, w_qkv, w_o, cos, sin, H: int, D: int, scale: float, rows):
    """Rows ``rows`` of :func:`layer_forward` (each output row needs that token's q but every
    token's k and v): fp64 ``[len(rows), Dm]``."""
    rows = np.asarray(rows, dtype=np.int64)
    q, k, v = project_and_rotate(x, w_qkv, cos, sin, H, D)
    o = A.attention_sampled(q, k, v, scale, rows)        # [R, H, D]
    return output_projection(o, w_o)


def layer_forward_composed(x, w_qkv, w_o, cos, sin, H: int, D: int, P: int, C: int, scale: float):
    """Alg. 1 executed literally: lines 2-3 on the main stream, lines 4-26 through the head-chunked
    all-to-all path of ``hcms_forward_composed`` (P ranks, C chunks), line 27."""
    q, k, v = project_and_rotate(x, w_qkv, cos, sin, H, D)
    o = A.hcms_forward_composed(q, k, v, P, C, scale)
    return output_projection(o, w_o)

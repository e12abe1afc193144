"""fp64 CPU oracle for the HCMS hot path.  TEST INFRASTRUCTURE, NOT PRODUCT.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It shares no code with the CUDA
path (``paper_2607_01817_b200``): it imports nothing from it, nothing from
``hcms_inputs`` and nothing from ``include/``; inputs arrive as plain numpy arrays.

Everything is written from /root/reference/PAPER.md (arxiv/paper_2607_01817, "HCMS");
"L<n>" below is a PAPER.md line.  HCMS changes the schedule, not the function (L31
"without altering computational semantics"; L304 "maximum error of 0"), so where a result
has a plain definition the oracle IS that definition, in fp64:

* ``chunk_table``            Eq. 3 (L83-84) applied per rank (Table 8).
* ``scatter_chunk``          input all-to-all of one head chunk (L45, L59; Alg. 1 line 8).
* ``gather_chunk``           output all-to-all + Concat (L45; Alg. 1 lines 21, 26).
* ``attention_rows`` / ``attention_full``   Eq. 2 (L76) / Alg. 1 line 15: per head
  ``softmax(Q K^T * scale) V``, bidirectional (L43), two-pass softmax.
* ``hcms_forward_composed``  Alg. 1 lines 4-26 executed literally, chunk by chunk.
* ``t_base`` ``t_hcms`` ``c_star`` ``speedup`` ``s_max``   Eq. 9-11, Theorems 1-2 (L154-160, L413-429).

Readings of silent / garbled passages are the ones listed in DESIGN.md ("Readings").
Pins: tests/test_oracle_*.py check every function here against values the paper prints
(tests/golden/), closed forms, invariants, library routines and brute force; no function in
this file is "parity unpinned".
"""
from __future__ import annotations

import math

import numpy as np

# --------------------------------------------------------------------------------------
# dtype plumbing (the oracle's own; nothing is shared with the CUDA path)
# --------------------------------------------------------------------------------------


def widen_to_f64(x: np.ndarray) -> np.ndarray:
    """Exact widening of the stored inputs to fp64.

    ``uint16`` arrays are bf16 bit patterns (sign, 8 exponent bits, 7 mantissa bits = the
    upper half of an IEEE fp32); float arrays are widened as they are.
    """
    x = np.asarray(x)
    if x.dtype == np.uint16:
        return (x.astype(np.uint32) << np.uint32(16)).view(np.float32).astype(np.float64)
    if x.dtype in (np.float32, np.float64):
        return x.astype(np.float64)
    raise TypeError(f"unsupported input dtype {x.dtype}")


# --------------------------------------------------------------------------------------
# a0  chunk table -- Eq. 3 (L83-84), "more-first-less-later" (L221, L290), Table 8
# --------------------------------------------------------------------------------------


def chunk_table(heads_per_rank: int, C: int):
    """Return ``[(o_c, h_c)]`` for ``c < C``.

    Eq. 3: ``H_c = floor(H/C) + 1[c < H mod C]``.  Table 8 (L292-300) applies it to the
    per-rank head count (H=40, 4 GPUs, H_per_rank=10, C=4 -> [3,3,2,2]); DESIGN.md
    reading R-1.  ``o_c`` is the running sum (Eq. 4's concatenation order).
    """
    Hl, C = int(heads_per_rank), int(C)
    if Hl <= 0 or C <= 0 or C > Hl:
        raise ValueError("need 1 <= C <= heads_per_rank")  # reading R-11
    table, o = [], 0
    for c in range(C):
        h = Hl // C + (1 if c < Hl % C else 0)
        table.append((o, h))
        o += h
    return table


def imbalance(sizes) -> float:
    """Table 8's "Imbal." column: (max - min) / mean of the chunk sizes."""
    sizes = [int(s) for s in sizes]
    return (max(sizes) - min(sizes)) / (sum(sizes) / len(sizes))


# --------------------------------------------------------------------------------------
# a2 / a6  the Ulysses all-to-all as a layout change (L45, L59)
# --------------------------------------------------------------------------------------


def scatter_chunk(x: np.ndarray, P: int, C: int, c: int) -> np.ndarray:
    """Input all-to-all of head chunk ``c`` for one of Q/K/V.

    ``x`` is the concatenation, in rank order, of the P ranks' sequence shards
    ``[S/P, H, D]`` ("sequence-sharded, heads-complete", L45), i.e. the global ``[S,H,D]``
    tensor (readings R-3, R-4).  After the exchange rank ``p`` holds the whole sequence for
    its own heads ("sequence-complete, heads-sharded"); rank p owns global heads
    ``[p*Hl, (p+1)*Hl)`` (R-2) and chunk c is local heads ``[o_c, o_c+h_c)`` on every rank
    (R-1).  Result ``[P, S, h_c, D]`` with
    ``out[p, s, j, d] = x[s, p*Hl + o_c + j, d]``; bits are copied untouched.
    """
    S, H, D = x.shape
    if H % P or S % P:
        raise ValueError("S and H must be divisible by P")
    Hl = H // P
    o_c, h_c = chunk_table(Hl, C)[c]
    out = np.empty((P, S, h_c, D), dtype=x.dtype)
    for p in range(P):                      # destination rank
        for j in range(h_c):                # local head inside the chunk
            out[p, :, j, :] = x[:, p * Hl + o_c + j, :]
    return out


def gather_chunk(oc: np.ndarray, out: np.ndarray, P: int, C: int, c: int) -> None:
    """Output all-to-all of chunk ``c`` (inverse of :func:`scatter_chunk`) written straight
    into the global ``out[S,H,D]`` at the chunk's head offsets, which is Alg. 1 line 26's
    Concat: ``out[s, p*Hl + o_c + j, d] = oc[p, s, j, d]``."""
    S, H, D = out.shape
    Hl = H // P
    o_c, h_c = chunk_table(Hl, C)[c]
    if oc.shape != (P, S, h_c, D):
        raise ValueError("chunk buffer has the wrong shape")
    for p in range(P):
        for j in range(h_c):
            out[:, p * Hl + o_c + j, :] = oc[p, :, j, :]


# --------------------------------------------------------------------------------------
# a4  attention -- Eq. 2 (L76), Alg. 1 line 15, bidirectional (L43)
# --------------------------------------------------------------------------------------


def attention_rows(q_rows: np.ndarray, k: np.ndarray, v: np.ndarray, scale: float) -> np.ndarray:
    """One head, some query rows: ``softmax_k(scale * q_i . k_k) @ V`` in fp64.

    ``q_rows [R, D]``, ``k [S, D]``, ``v [S, D]`` already widened to fp64.  Two-pass
    softmax exactly as in SURVEY 8(c): ``s_k = scale * sum_d q_d k_kd``; ``m = max_k s_k``;
    ``w_k = exp(s_k - m)``; ``O = (sum_k w_k V_k) / sum_k w_k``.  No mask, dropout or bias.
    ``scale`` is the fp32 value handed to the GPU, widened (reading R-5).
    """
    s = (q_rows @ k.T) * float(scale)            # [R, S]
    m = s.max(axis=1, keepdims=True)
    w = np.exp(s - m)
    den = w.sum(axis=1, keepdims=True)
    return (w @ v) / den


def attention_full(q, k, v, scale: float, row_block: int = 2048) -> np.ndarray:
    """All heads, all rows of global ``[S,H,D]`` inputs (any storage dtype) -> fp64 ``[S,H,D]``.

    Rows are independent by definition, so looping over blocks of rows only bounds the
    size of the ``[rows, S]`` score matrix; nothing is reordered inside a row.
    """
    S, H, D = q.shape
    out = np.empty((S, H, D), dtype=np.float64)
    for h in range(H):
        qh, kh, vh = (widen_to_f64(t[:, h, :]) for t in (q, k, v))
        for r0 in range(0, S, row_block):
            out[r0:r0 + row_block, h, :] = attention_rows(qh[r0:r0 + row_block], kh, vh, scale)
    return out


def attention_sampled(q, k, v, scale: float, rows) -> np.ndarray:
    """Rows ``rows`` (1-D int array) of every head -> fp64 ``[len(rows), H, D]``.
    Each row is an independent exact evaluation of the definition (large-config strategy,
    SURVEY 8(c))."""
    rows = np.asarray(rows, dtype=np.int64)
    S, H, D = q.shape
    out = np.empty((len(rows), H, D), dtype=np.float64)
    for h in range(H):
        qh = widen_to_f64(q[rows, h, :])
        kh, vh = widen_to_f64(k[:, h, :]), widen_to_f64(v[:, h, :])
        out[:, h, :] = attention_rows(qh, kh, vh, scale)
    return out


def sample_rows(S: int, P: int, n_random: int = 48, seed: int = 0) -> np.ndarray:
    """Deterministic row sample of SURVEY 8(c): tile/shard boundary rows plus seeded rows."""
    Sl = S // P
    tail0 = S - (S % 128) if S % 128 else S - 128
    fixed = [0, 1, 127, 128, Sl - 1, Sl, tail0 - 1, tail0, S - 1]
    rng = np.random.default_rng(seed)
    rand = rng.integers(0, S, size=n_random).tolist()
    rows = sorted({r for r in fixed + rand if 0 <= r < S})
    return np.asarray(rows, dtype=np.int64)


# --------------------------------------------------------------------------------------
# Alg. 1 lines 4-26 executed literally (the "composed oracle")
# --------------------------------------------------------------------------------------


def hcms_forward_composed(q, k, v, P: int, C: int, scale: float) -> np.ndarray:
    """SplitByHeads(C) -> per chunk: AllToAll(Q_c,K_c,V_c) -> Attention on every rank's
    head-sharded buffers -> AllToAll(O'_c) -> Concat.  Must equal :func:`attention_full`
    bit for bit in fp64 (same per-head arithmetic): the paper's equivalence claim
    (L304, Table 14) executed on the CPU."""
    S, H, D = q.shape
    out = np.full((S, H, D), np.nan, dtype=np.float64)
    Hl = H // P
    for c, (_, h_c) in enumerate(chunk_table(Hl, C)):
        qc, kc, vc = (scatter_chunk(t, P, C, c) for t in (q, k, v))
        oc = np.empty((P, S, h_c, D), dtype=np.float64)
        for p in range(P):
            for j in range(h_c):
                oc[p, :, j, :] = attention_rows(widen_to_f64(qc[p, :, j, :]),
                                                widen_to_f64(kc[p, :, j, :]),
                                                widen_to_f64(vc[p, :, j, :]), scale)
        gather_chunk(oc, out, P, C, c)
    return out


# --------------------------------------------------------------------------------------
# Time model -- section 3.7 (L154-160), Appendix A (L413-429)
# --------------------------------------------------------------------------------------


def t_base(t0: float, t_comm: float, t_attn: float) -> float:
    """Eq. 9: serial execution, ``T_base = T_0 + T_comm + T_attn``."""
    return t0 + t_comm + t_attn


def t_hcms(C: int, t0: float, t_comm: float, t_attn: float, beta: float) -> float:
    """Eq. 10: ``T_hcms(C) = T_0 + T_comm/C + T_attn + C*beta``."""
    return t0 + t_comm / C + t_attn + C * beta


def c_star(t_comm: float, beta: float) -> float:
    """Theorem 1 (L156, L421): ``C* = sqrt(T_comm / beta)``."""
    return math.sqrt(t_comm / beta)


def speedup(C: int, rho: float, beta: float, t_total: float) -> float:
    """Eq. 11: ``S(C) = 1 / (1 - rho*(C-1)/C + C*beta/T_total)``, ``rho = T_comm/T_total``."""
    return 1.0 / (1.0 - rho * (C - 1) / C + C * beta / t_total)


def s_max(rho: float) -> float:
    """Theorem 2 (L158, L429): ``S_max = 1 / (1 - rho)``."""
    return 1.0 / (1.0 - rho)


def choose_chunks(heads_per_rank: int, t_comm: float, beta: float) -> int:
    """Adaptive C (future work L346) by brute force over Eq. 10: the integer ``C`` in
    ``[1, heads_per_rank]`` with the smallest ``T_hcms(C)`` (T_0, T_attn do not depend on C),
    ties to the smaller C.  Theorem 1 says this is a neighbour of ``sqrt(T_comm/beta)``."""
    best, best_t = 1, None
    for C in range(1, heads_per_rank + 1):
        t = t_hcms(C, 0.0, t_comm, 0.0, beta)
        if best_t is None or t < best_t:
            best, best_t = C, t
    return best

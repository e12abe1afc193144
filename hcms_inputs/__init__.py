"""Seeded synthetic inputs for the HCMS hot path (shared by tests, bench and smoke).

This module holds NONE of the method's arithmetic (no chunking, no permutation, no
attention): it only describes the five BASELINE.json workloads and produces their
Q/K/V tensors from a counter-based generator, so that the fp64 oracle (``oracle/``)
and the CUDA path (``paper_2607_01817_b200``) can be fed identical bits without
sharing any code with each other.  Neither of them imports this module; tests and
``bench.py`` do, and pass the arrays in.

Recipe: element ``i`` of tensor
``t`` (q=0, k=1, v=2) of the workload with seed ``s`` is one output of a Box-Muller
pair whose two uniforms come from a splitmix64-style hash of ``(s, t, i // 2)``;
the fp32 normal is then rounded to bf16 with round-to-nearest-even.  The paper
(Table 3, section 4.4) measures on model-shaped activations,
not on a dataset; these tensors stand in for them.
"""
from __future__ import annotations

from concurrent.futures import ThreadPoolExecutor
from dataclasses import dataclass

import numpy as np

__all__ = [
    "Workload", "WORKLOADS", "workload", "normal_f32", "f32_to_bf16_bits",
    "bf16_bits_to_f32", "make_qkv", "index_pattern", "make_layer_inputs", "rope_tables",
]

_MASK64 = np.uint64(0xFFFFFFFFFFFFFFFF)


@dataclass(frozen=True)
class Workload:
    """One BASELINE.json config: global ``[S, H, D]`` tensors, P logical ranks, C chunks."""
    name: str
    S: int
    H: int
    D: int
    P: int
    C: int
    seed: int
    dtype: str          # "f32" (config 1's layout test) or "bf16"
    k_scale: float      # config 3 multiplies K by 0.5 (exact in bf16)

    @property
    def scale(self) -> float:
        return float(np.float32(1.0) / np.sqrt(np.float32(self.D)))


# BASELINE.json configs[0..4] (1-based "cfg" numbering in SURVEY.md section 8).
WORKLOADS = {
    1: Workload("cfg1_tiny", 1024, 4, 64, 2, 2, 0, "f32", 1.0),
    2: Workload("cfg2_uneven", 8192, 12, 64, 4, 2, 1, "bf16", 1.0),
    3: Workload("cfg3_dit720p", 32760, 40, 128, 4, 4, 2, "bf16", 0.5),
    4: Workload("cfg4_longvideo", 56160, 40, 128, 8, 2, 3, "bf16", 1.0),
    5: Workload("cfg5_stress", 98304, 24, 128, 8, 3, 4, "bf16", 1.0),
}


def workload(cfg: int) -> Workload:
    return WORKLOADS[int(cfg)]


def _splitmix64(x: np.ndarray) -> np.ndarray:
    """splitmix64 finaliser on a uint64 array (wrap-around arithmetic)."""
    with np.errstate(over="ignore"):
        x = (x + np.uint64(0x9E3779B97F4A7C15)) & _MASK64
        x = ((x ^ (x >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)) & _MASK64
        x = ((x ^ (x >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)) & _MASK64
        x = x ^ (x >> np.uint64(31))
    return x


def _normal_block(seed: int, tensor_id: int, start: int, stop: int) -> np.ndarray:
    idx = np.arange(start, stop, dtype=np.uint64)
    pair = idx >> np.uint64(1)
    with np.errstate(over="ignore"):
        key = _splitmix64(np.uint64(seed) * np.uint64(0xD1342543DE82EF95)
                          + np.uint64(tensor_id) * np.uint64(0xA0761D6478BD642F)
                          + np.uint64(0x2545F4914F6CDD1D))
        h1 = _splitmix64(pair ^ key)
        h2 = _splitmix64(h1 ^ np.uint64(0x632BE59BD9B4E019))
    # 53-bit uniforms; u1 in (0, 1], u2 in [0, 1)
    u1 = ((h1 >> np.uint64(11)).astype(np.float64) + 1.0) * (1.0 / 9007199254740992.0)
    u2 = (h2 >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)
    r = np.sqrt(-2.0 * np.log(u1))
    ang = (2.0 * np.pi) * u2
    odd = (idx & np.uint64(1)).astype(bool)
    z = np.where(odd, r * np.sin(ang), r * np.cos(ang))
    return z.astype(np.float32)


def normal_f32(seed: int, tensor_id: int, n: int, threads: int = 8) -> np.ndarray:
    """``n`` N(0,1) fp32 values; value ``i`` depends only on ``(seed, tensor_id, i)``."""
    out = np.empty(n, dtype=np.float32)
    block = 1 << 21
    spans = [(a, min(a + block, n)) for a in range(0, n, block)]

    def work(span):
        a, b = span
        out[a:b] = _normal_block(seed, tensor_id, a, b)

    if threads > 1 and len(spans) > 1:
        with ThreadPoolExecutor(max_workers=threads) as ex:
            list(ex.map(work, spans))
    else:
        for sp in spans:
            work(sp)
    return out


def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """fp32 -> bf16 bit patterns (uint16), round-to-nearest-even; NaN kept quiet."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    lsb = (u >> np.uint32(16)) & np.uint32(1)
    rounded = (u + np.uint32(0x7FFF) + lsb) >> np.uint32(16)
    is_nan = (u & np.uint32(0x7FFFFFFF)) > np.uint32(0x7F800000)
    rounded = np.where(is_nan, (u >> np.uint32(16)) | np.uint32(0x40), rounded)
    return rounded.astype(np.uint16)


def bf16_bits_to_f32(b: np.ndarray) -> np.ndarray:
    """bf16 bit patterns (uint16) -> the exactly equal fp32 values."""
    return (np.ascontiguousarray(b, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32)


def make_qkv(w: Workload, S: int | None = None, threads: int = 8):
    """Return ``(q, k, v)`` for workload ``w``.

    bf16 workloads: three uint16 arrays ``[S, H, D]`` of bf16 bit patterns.
    f32 workload (config 1): three float32 arrays ``[S, H, D]``; round them with
    :func:`f32_to_bf16_bits` for the bf16 attention kernel (SURVEY R-12).
    ``S`` may override the sequence length (same seed, a prefix of the same stream
    per tensor is NOT implied: the stream is indexed by the flat element index).
    """
    S = w.S if S is None else int(S)
    n = S * w.H * w.D
    out = []
    for tid in range(3):
        x = normal_f32(w.seed, tid, n, threads=threads).reshape(S, w.H, w.D)
        if w.dtype == "bf16":
            bits = f32_to_bf16_bits(x)
            if tid == 1 and w.k_scale != 1.0:
                # x0.5 after rounding (SURVEY R-13): exact for normal bf16 values.
                bits = f32_to_bf16_bits(bf16_bits_to_f32(bits) * np.float32(w.k_scale))
            out.append(bits)
        else:
            if tid == 1 and w.k_scale != 1.0:
                x = x * np.float32(w.k_scale)
            out.append(x)
    return tuple(out)


def index_pattern(S: int, H: int, D: int, dtype) -> np.ndarray:
    """``X[s,h,d]`` = a unique id per element (wraps for 16-bit types): layout tests use it
    so that any misplaced element is identifiable (scatter/gather pin iii)."""
    n = S * H * D
    ids = np.arange(n, dtype=np.uint64)
    dt = np.dtype(dtype)
    if dt.itemsize == 2:
        # mix so that neighbouring rows differ even after wrapping to 16 bits
        ids = (_splitmix64(ids) & np.uint64(0xFFFF)).astype(np.uint16)
        return ids.reshape(S, H, D).view(dt) if dt != np.uint16 else ids.reshape(S, H, D)
    ids = (ids & np.uint64(0xFFFFFFFF)).astype(np.uint32)
    return ids.reshape(S, H, D).view(dt) if dt != np.uint32 else ids.reshape(S, H, D)


def rope_tables(S: int, D: int, base: float = 10000.0):
    """cos/sin tables ``[S, D/2]`` fp32 handed to the layer as INPUT data (the library and the oracle both
    only consume tables): angle(s, i) = s * base**(-2i/D), the 1-D position scheme of RoFormer [34], computed
    in fp64 and rounded once.  A video DiT would tabulate its 3-D grid angles the same way."""
    i = np.arange(D // 2, dtype=np.float64)
    ang = np.arange(S, dtype=np.float64)[:, None] * (base ** (-2.0 * i / D))[None, :]
    return np.cos(ang).astype(np.float32), np.sin(ang).astype(np.float32)


def make_layer_inputs(w: Workload, Dm: int | None = None, S: int | None = None, threads: int = 8):
    """Inputs of the whole attention layer (Alg. 1 lines 2-27) for workload ``w``: activations
    ``x [S, Dm]`` ~ N(0,1) (tensor id 3), ``w_qkv [3*H*D, Dm]`` ~ N(0, 1/Dm) (id 4), ``w_o [Dm, H*D]`` ~
    N(0, 1/(H*D)) (id 5), all rounded to bf16 bit patterns, plus :func:`rope_tables`.  ``Dm`` defaults to
    ``H*D`` (Table 3: 5120 = 40 x 128).  Random-init weights stand in for the model's: the paper's
    checkpoints are not available here.  With these variances q, k, v come out ~ N(0,1), the distribution of
    :func:`make_qkv`; ``k_scale`` (config 3) multiplies the K rows of ``w_qkv``."""
    S = w.S if S is None else int(S)
    hd = w.H * w.D
    Dm = hd if Dm is None else int(Dm)
    x = f32_to_bf16_bits(normal_f32(w.seed, 3, S * Dm, threads=threads).reshape(S, Dm))
    wq = normal_f32(w.seed, 4, 3 * hd * Dm, threads=threads).reshape(3 * hd, Dm) * np.float32(1.0 / np.sqrt(Dm))
    if w.k_scale != 1.0:
        wq[hd:2 * hd] *= np.float32(w.k_scale)
    wo = normal_f32(w.seed, 5, Dm * hd, threads=threads).reshape(Dm, hd) * np.float32(1.0 / np.sqrt(hd))
    cos, sin = rope_tables(S, w.D)
    return x, f32_to_bf16_bits(wq), f32_to_bf16_bits(wo), cos, sin

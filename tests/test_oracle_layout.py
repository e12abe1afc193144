"""Pins for the oracle's all-to-all layout maps (scatter_chunk / gather_chunk).  CPU only.
Pins: identity of gather o scatter, a numpy reshape/transpose restatement (library routine),
index-encoded inputs, brute-force loops on tiny shapes, C-independence after re-slicing."""
import numpy as np
import pytest

from hcms_inputs import index_pattern
from oracle import hcms_oracle as O

SHAPES = [  # S, H, D, P
    (8, 4, 4, 2), (12, 6, 8, 3), (6, 6, 2, 1), (4, 4, 8, 4), (16, 12, 4, 4), (2, 2, 2, 2),
]


@pytest.mark.parametrize("S,H,D,P", SHAPES)
@pytest.mark.parametrize("dtype", [np.uint16, np.uint32])
def test_scatter_equals_reshape_transpose(S, H, D, P, dtype):
    x = index_pattern(S, H, D, dtype)
    Hl = H // P
    for C in range(1, Hl + 1):
        for c, (o, h) in enumerate(O.chunk_table(Hl, C)):
            ref = x.reshape(S, P, Hl, D).transpose(1, 0, 2, 3)[:, :, o:o + h, :]
            got = O.scatter_chunk(x, P, C, c)
            assert got.dtype == x.dtype and got.shape == (P, S, h, D)
            assert np.array_equal(got, ref)


@pytest.mark.parametrize("S,H,D,P", SHAPES)
def test_scatter_brute_force(S, H, D, P):
    x = index_pattern(S, H, D, np.uint32)
    Hl, Sl = H // P, S // P
    for C in range(1, Hl + 1):
        for c, (o, h) in enumerate(O.chunk_table(Hl, C)):
            got = O.scatter_chunk(x, P, C, c)
            for p in range(P):               # destination rank
                for r in range(P):           # source rank: message r -> p is rows [r*Sl,(r+1)*Sl)
                    for t in range(Sl):
                        for j in range(h):
                            for d in range(D):
                                assert got[p, r * Sl + t, j, d] == x[r * Sl + t, p * Hl + o + j, d]


@pytest.mark.parametrize("S,H,D,P", SHAPES)
@pytest.mark.parametrize("dtype", [np.uint16, np.uint32])
def test_gather_of_scatter_is_identity_and_writes_once(S, H, D, P, dtype):
    x = index_pattern(S, H, D, dtype)
    Hl = H // P
    for C in range(1, Hl + 1):
        out = np.zeros_like(x)
        count = np.zeros((S, H, D), dtype=np.int32)
        ones = np.ones((S, H, D), dtype=np.int32)
        for c in range(C):
            O.gather_chunk(O.scatter_chunk(x, P, C, c), out, P, C, c)
            tmp = np.zeros_like(count)
            O.gather_chunk(O.scatter_chunk(ones, P, C, c), tmp, P, C, c)
            count += tmp
        assert np.array_equal(out, x)
        assert np.array_equal(count, ones)     # every element written exactly once


def test_chunks_reslice_independent_of_C():
    S, H, D, P = 8, 12, 4, 2
    x = index_pattern(S, H, D, np.uint32)
    Hl = H // P
    full = O.scatter_chunk(x, P, 1, 0)                       # [P,S,Hl,D]
    for C in range(1, Hl + 1):
        cat = np.concatenate([O.scatter_chunk(x, P, C, c) for c in range(C)], axis=2)
        assert np.array_equal(cat, full)


def test_gather_rejects_wrong_shape():
    out = np.zeros((4, 4, 2), dtype=np.float64)
    with pytest.raises(ValueError):
        O.gather_chunk(np.zeros((2, 4, 1, 2)), out, 2, 1, 0)
    with pytest.raises(ValueError):
        O.scatter_chunk(np.zeros((5, 4, 2)), 2, 1, 0)

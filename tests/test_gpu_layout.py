"""-m gpu: the all-to-all layout kernels (hcms_a2a_scatter / hcms_a2a_gather, both variants) against
the permutation oracle, BIT-EXACT: small shapes spanning several tiles and ragged
tails, 2- and 4-byte elements, every chunk of every C, then the full-size BASELINE.json shapes."""
import numpy as np
import pytest
import torch

import hcms_inputs as I
import paper_2607_01817_b200 as H
from oracle import hcms_oracle as O
from gpu_util import DEV, to_dev, to_host

pytestmark = pytest.mark.gpu

VARIANTS = [0, H.HCMS_FLAG_LAYOUT_TMA]

SMALL = [  # S, H, D, P, dtype
    (1024, 4, 64, 2, "f32"),      # BASELINE.json configs[0]
    (8192, 12, 64, 4, "bf16"),    # configs[1]
    (1000, 12, 128, 4, "bf16"),   # ragged: Sl = 250
    (130, 10, 128, 1, "bf16"),    # P = 1, a few rows
    (6, 6, 64, 3, "f32"),         # Sl = 2
    (4, 8, 128, 4, "bf16"),       # Sl = 1
    (2046, 20, 128, 2, "bf16"),   # Hl = 10 (Table 8), ragged
]


def _pattern(S, Hh, D, dt):
    if dt == "f32":
        return I.index_pattern(S, Hh, D, np.uint32), H.HCMS_DTYPE_F32
    return I.index_pattern(S, Hh, D, np.uint16), H.HCMS_DTYPE_BF16


@pytest.mark.parametrize("flags", VARIANTS)
@pytest.mark.parametrize("S,Hh,D,P,dt", SMALL)
def test_scatter_gather_bit_exact_every_chunking(S, Hh, D, P, dt, flags):
    x, dtype = _pattern(S, Hh, D, dt)
    xd = to_dev(x)
    Hl = Hh // P
    for C in sorted({1, 2, 3, Hl} & set(range(1, Hl + 1))):
        with H.hcms_plan(S, Hh, D, P, C, dtype, flags) as plan:
            o, h = H.hcms_chunk_table(plan)
            assert list(zip(o, h)) == O.chunk_table(Hl, C)
            out = torch.full_like(xd, -1)                       # sentinel: every element must be overwritten
            for c in range(C):
                dst = torch.full((P, S, h[c], D), -1, dtype=xd.dtype, device=DEV)
                H.hcms_a2a_scatter(plan, [xd], [dst], c)
                torch.cuda.synchronize()
                assert np.array_equal(to_host(dst), O.scatter_chunk(x, P, C, c)), (C, c)
                H.hcms_a2a_gather(plan, dst, out, c)
                torch.cuda.synchronize()
                # the gather of chunk c writes chunk c's heads and nothing else
                ref = np.full_like(x, np.iinfo(x.dtype).max)
                for cc in range(c + 1):
                    O.gather_chunk(O.scatter_chunk(x, P, C, cc), ref, P, C, cc)
                assert np.array_equal(to_host(out), ref), (C, c)
            assert np.array_equal(to_host(out), x)              # gather o scatter = identity


@pytest.mark.parametrize("flags", VARIANTS)
def test_three_tensors_in_one_launch(flags):
    S, Hh, D, P, C = 1536, 12, 128, 4, 2
    xs = [I.f32_to_bf16_bits(I.normal_f32(11, t, S * Hh * D)).reshape(S, Hh, D) for t in range(3)]
    xd = [to_dev(x) for x in xs]
    with H.hcms_plan(S, Hh, D, P, C, H.HCMS_DTYPE_BF16, flags) as plan:
        _, h = H.hcms_chunk_table(plan)
        for c in range(C):
            dst = [torch.full((P, S, h[c], D), -1, dtype=torch.int16, device=DEV) for _ in range(3)]
            H.hcms_a2a_scatter(plan, xd, dst, c)
            torch.cuda.synchronize()
            for t in range(3):
                assert np.array_equal(to_host(dst[t]), O.scatter_chunk(xs[t], P, C, c))


@pytest.mark.parametrize("flags", VARIANTS)
@pytest.mark.parametrize("cfg", [3, 4, 5])
def test_full_size_configs_bit_exact(cfg, flags):
    """BASELINE.json configs[2..4] at full size, in the launch configuration bench.py times."""
    w = I.workload(cfg)
    x = I.index_pattern(w.S, w.H, w.D, np.uint16)
    xd = to_dev(x)
    out = torch.full_like(xd, -1)
    with H.hcms_plan(w.S, w.H, w.D, w.P, w.C, H.HCMS_DTYPE_BF16, flags) as plan:
        _, h = H.hcms_chunk_table(plan)
        for c in range(w.C):
            dst = torch.full((w.P, w.S, h[c], w.D), -1, dtype=torch.int16, device=DEV)
            H.hcms_a2a_scatter(plan, [xd], [dst], c)
            torch.cuda.synchronize()
            assert np.array_equal(to_host(dst), O.scatter_chunk(x, w.P, w.C, c)), c
            H.hcms_a2a_gather(plan, dst, out, c)
            del dst
        torch.cuda.synchronize()
        assert np.array_equal(to_host(out), x)


def test_layout_argument_errors():
    S, Hh, D, P, C = 256, 4, 64, 2, 2
    with H.hcms_plan(S, Hh, D, P, C) as plan:
        x = torch.zeros(S * Hh * D + 8, dtype=torch.int16, device=DEV)
        d = torch.zeros(P * S * 1 * D + 8, dtype=torch.int16, device=DEV)
        for bad in [lambda: H.hcms_a2a_scatter(plan, [x], [d], 2),
                    lambda: H.hcms_a2a_gather(plan, d, x, -1)]:
            with pytest.raises(H.HcmsError) as ei:
                bad()
            assert ei.value.status == H.HCMS_ERR_PLAN_MISMATCH
        with pytest.raises(H.HcmsError) as ei:
            H.hcms_a2a_scatter(plan, [x[1:]], [d], 0)            # 2-byte offset: not 16-byte aligned
        assert ei.value.status == H.HCMS_ERR_MISALIGNED
        with pytest.raises(H.HcmsError) as ei:
            H.hcms_a2a_scatter(plan, [], [], 0)
        assert ei.value.status == H.HCMS_ERR_INVALID_ARG

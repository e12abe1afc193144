"""Python binding of libhcms (include/hcms.h): argument marshalling only.

Every step of the HCMS hot path (Alg. 1 lines 4-26: head-chunked all-to-all layout
kernels, bf16 attention, dual-stream scheduler) runs inside ``libhcms.so`` (CUDA, sm_100a).
The functions here carry the same names as the C entry points and only turn torch tensors /
numpy arrays / ints into pointers.  There is no CPU fallback: importing this package without a
built ``libhcms.so`` raises, and a compute call without a B200 returns the library's error.
"""
from __future__ import annotations

import ctypes
import os
from ctypes import POINTER, c_char_p, c_double, c_float, c_int, c_int64, c_size_t, c_uint32, c_void_p

_PKG_DIR = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG_DIR, "libhcms.so")

# status codes / dtypes / flags (mirrors include/hcms.h)
HCMS_OK = 0
HCMS_ERR_INVALID_ARG = -1
HCMS_ERR_UNSUPPORTED_SHAPE = -2
HCMS_ERR_UNSUPPORTED_DTYPE = -3
HCMS_ERR_UNSUPPORTED_DEVICE = -4
HCMS_ERR_MISALIGNED = -5
HCMS_ERR_ALIAS = -6
HCMS_ERR_PLAN_MISMATCH = -7
HCMS_ERR_WORKSPACE_TOO_SMALL = -8
HCMS_ERR_CUDA = -9

HCMS_DTYPE_BF16 = 0
HCMS_DTYPE_F32 = 1
HCMS_DTYPE_F16 = 2

HCMS_FLAG_SERIAL = 0x1
HCMS_FLAG_LAYOUT_TMA = 0x2
HCMS_FLAG_SPLIT_COMM = 0x4
HCMS_FLAG_HOST_ROUTE_Q = 0x10
HCMS_FLAG_HOST_ROUTE_K = 0x20
HCMS_FLAG_HOST_ROUTE_V = 0x40
HCMS_FLAG_HOST_ROUTE_O = 0x80
HCMS_FLAG_DEBUG_NO_COMM_WAIT = 0x100
HCMS_FLAG_PROFILE = 0x200
HCMS_FLAG_SINGLE_COMP = 0x400
HCMS_FLAG_TRAINING = 0x800
HCMS_FLAG_FUSE_A2A = 0x1000
HCMS_FLAG_GRAPH = 0x2000
HCMS_FLAG_ATTN_PAIR = 0x4000
HCMS_FLAG_HOST_STAGED = 0x8000
HCMS_FLAG_GEMM_1CTA = 0x10000
HCMS_FLAG_DEBUG_ATTN_ONLY = 0x20000
HCMS_FLAG_BWD_ONE_PASS = 0x40000
HCMS_FLAG_RECYCLE_WS = 0x80000
HCMS_FLAG_DIST_FUSE_OUT = 0x100000
HCMS_FLAG_DEBUG_DIST_FAIL = 0x200000

# every symbol include/hcms.h declares: name -> (restype, argtypes)
_SIGNATURES = {
    "hcms_version": (c_int, []),
    "hcms_status_string": (c_char_p, [c_int]),
    "hcms_last_error": (c_char_p, []),
    "hcms_chunk_table_host": (c_int, [c_int, c_int, POINTER(c_int), POINTER(c_int)]),
    "hcms_model_t_hcms": (c_double, [c_int, c_double, c_double, c_double, c_double]),
    "hcms_model_c_star": (c_double, [c_double, c_double]),
    "hcms_model_speedup": (c_double, [c_int, c_double, c_double, c_double]),
    "hcms_model_s_max": (c_double, [c_double]),
    "hcms_model_choose_chunks": (c_int, [c_int, c_double, c_double]),
    "hcms_plan": (c_int, [POINTER(c_void_p), c_int64, c_int, c_int, c_int, c_int, c_int, c_uint32]),
    "hcms_plan_destroy": (c_int, [c_void_p]),
    "hcms_plan_workspace_bytes": (c_size_t, [c_void_p]),
    "hcms_plan_set_workspace": (c_int, [c_void_p, c_void_p, c_size_t]),
    "hcms_chunk_table": (c_int, [c_void_p, POINTER(c_int), POINTER(c_int)]),
    "hcms_chunk_layout": (c_int, [c_void_p, c_int] + [POINTER(c_size_t)] * 5),
    "hcms_plan_workspace": (c_void_p, [c_void_p]),
    "hcms_plan_tensor_map_encodes": (ctypes.c_longlong, [c_void_p]),
    "hcms_attention_forward": (c_int, [c_void_p] * 5 + [c_int64, c_int, c_int, c_int, c_int, c_float, c_void_p]),
    "hcms_attention_forward_host": (c_int, [c_void_p] * 5 + [c_int64, c_int, c_int, c_int, c_int, c_float, c_void_p]),
    "hcms_a2a_scatter": (c_int, [c_void_p, c_int, POINTER(c_void_p), POINTER(c_void_p), c_int, c_void_p]),
    "hcms_a2a_gather": (c_int, [c_void_p, c_void_p, c_void_p, c_int, c_void_p]),
    "hcms_attention_chunk": (c_int, [c_void_p] * 5 + [c_int, c_float, c_void_p]),
    "hcms_plan_last_launch_count": (c_int, [c_void_p]),
    "hcms_plan_timings": (c_int, [c_void_p, c_int, POINTER(c_float), POINTER(c_float), POINTER(c_float)]),
    "hcms_plan_step_span": (c_int, [c_void_p, c_int, c_int, POINTER(c_float)]),
    "hcms_plan_timeline": (c_int, [c_void_p, c_int, POINTER(c_float), POINTER(c_float)]),
    "hcms_autotune_chunks": (c_int, [c_int64, c_int, c_int, c_int, c_int, c_uint32] + [c_void_p] * 4 +
                             [c_float, c_void_p, c_int, c_int, POINTER(c_int), POINTER(c_float)]),
    "hcms_gemm_bf16_nt": (c_int, [c_void_p] * 3 + [c_int64, c_int, c_int, c_void_p]),
    "hcms_qkv_projection_rope": (c_int, [c_void_p] * 8 + [c_int, c_void_p]),
    "hcms_output_projection": (c_int, [c_void_p] * 4 + [c_int, c_void_p]),
    "hcms_layer_forward": (c_int, [c_void_p] * 7 + [c_int64, c_int, c_int, c_int, c_int, c_int, c_float, c_void_p]),
    "hcms_plan_layer_buffer": (c_void_p, [c_void_p, c_int]),
    "hcms_plan_layer_timings": (c_int, [c_void_p, POINTER(c_float), POINTER(c_float), POINTER(c_float)]),
    "hcms_attention_backward": (c_int, [c_void_p] * 5 + [c_int64, c_int, c_int, c_int, c_int, c_float, c_void_p]),
    "hcms_attention_chunk_lse": (c_int, [c_void_p] * 6 + [c_int, c_float, c_void_p]),
    "hcms_attention_backward_chunk": (c_int, [c_void_p] * 10 + [c_int, c_float, c_void_p]),
    "hcms_attention_backward_chunk_static": (c_int, [c_void_p] * 9 + [c_int64, c_int, c_int, c_int, c_float, c_void_p]),
    "hcms_plan_lse": (c_void_p, [c_void_p]),
    "hcms_plan_graph_captures": (c_int, [c_void_p]),
    "hcms_dist_plan": (c_int, [POINTER(c_void_p), c_int64, c_int, c_int, c_int, c_int, c_int, c_uint32, c_int]),
    "hcms_dist_plan_destroy": (c_int, [c_void_p]),
    "hcms_dist_export": (c_int, [c_void_p, c_void_p]),
    "hcms_dist_attach": (c_int, [c_void_p, c_void_p, c_int]),
    "hcms_dist_attach_local": (c_int, [c_void_p, POINTER(c_void_p), c_int]),
    "hcms_dist_attention_forward": (c_int, [c_void_p] * 5 + [c_float, c_void_p]),
    "hcms_dist_attention_forward_host": (c_int, [c_void_p] * 5 + [c_float, c_void_p]),
    "hcms_dist_attention_forward_group": (c_int, [POINTER(c_void_p), c_int] + [POINTER(c_void_p)] * 4 + [c_float, POINTER(c_void_p)]),
    "hcms_dist_layer_forward": (c_int, [c_void_p] * 7 + [c_int, c_float, c_void_p]),
    "hcms_dist_layer_forward_group": (c_int, [POINTER(c_void_p), c_int, POINTER(c_void_p), c_void_p, c_void_p, POINTER(c_void_p),
                                              POINTER(c_void_p), POINTER(c_void_p), c_int, c_float, POINTER(c_void_p)]),
    "hcms_dist_block_bytes": (c_size_t, [c_void_p]),
    "hcms_dist_last_launch_count": (c_int, [c_void_p]),
    "hcms_autotune_chunks_host": (c_int, [c_int64, c_int, c_int, c_int, c_uint32] + [c_void_p] * 4 +
                                  [c_float, c_void_p, c_int, c_int, POINTER(c_int), POINTER(c_float)]),
}


class HcmsError(RuntimeError):
    """A libhcms call returned a negative status."""

    def __init__(self, status: int, name: str, text: str):
        super().__init__(f"{name}: {text} [{status}]")
        self.status = status


def _load() -> ctypes.CDLL:
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            f"{LIB_PATH} is missing: build it with `python -m paper_2607_01817_b200.build` "
            "(the HCMS hot path exists only as CUDA code; there is no CPU fallback)")
    lib = ctypes.CDLL(LIB_PATH)
    for name, (res, args) in _SIGNATURES.items():
        fn = getattr(lib, name)      # AttributeError if the library lacks a declared symbol
        fn.restype = res
        fn.argtypes = args
    return lib


class _LazyLib:
    """Loads libhcms.so on first use, so that ``python -m paper_2607_01817_b200.build`` can import
    the package before the library exists.  Any call without the library raises ImportError."""

    _cdll = None

    def __getattr__(self, name):
        if _LazyLib._cdll is None:
            _LazyLib._cdll = _load()
        return getattr(_LazyLib._cdll, name)


lib = _LazyLib()


def _check(status: int, name: str) -> None:
    if status != HCMS_OK:
        raise HcmsError(status, lib.hcms_status_string(status).decode(), f"{name}: {lib.hcms_last_error().decode()}")


def _ptr(x) -> int:
    """Address of a torch tensor / numpy array / raw int pointer (no copies, no conversions)."""
    if x is None:
        return 0
    if isinstance(x, int):
        return x
    if hasattr(x, "data_ptr"):          # torch.Tensor
        if not x.is_contiguous():
            raise ValueError("libhcms needs contiguous tensors")
        return x.data_ptr()
    if hasattr(x, "ctypes"):            # numpy.ndarray
        if not x.flags["C_CONTIGUOUS"]:
            raise ValueError("libhcms needs C-contiguous arrays")
        return x.ctypes.data
    raise TypeError(f"cannot take the address of {type(x)}")


def _stream(stream) -> int:
    """cudaStream_t of a torch.cuda.Stream / int / None (None = torch's current stream)."""
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    if isinstance(stream, int):
        return stream
    return stream.cuda_stream


# ---- host-only entry points ------------------------------------------------------------------

def hcms_version() -> int:
    return lib.hcms_version()


def hcms_status_string(status: int) -> str:
    return lib.hcms_status_string(status).decode()


def hcms_last_error() -> str:
    return lib.hcms_last_error().decode()


def hcms_chunk_table_host(heads_per_rank: int, C: int):
    """Eq. 3 on the per-rank head count -> ([o_c], [h_c])."""
    n = max(int(C), 1)
    o, h = (c_int * n)(), (c_int * n)()
    _check(lib.hcms_chunk_table_host(heads_per_rank, C, o, h), "hcms_chunk_table_host")
    return list(o)[:C], list(h)[:C]


def hcms_model_t_hcms(C, t0, t_comm, t_attn, beta) -> float:
    return lib.hcms_model_t_hcms(C, t0, t_comm, t_attn, beta)


def hcms_model_c_star(t_comm, beta) -> float:
    return lib.hcms_model_c_star(t_comm, beta)


def hcms_model_speedup(C, rho, beta, t_total) -> float:
    return lib.hcms_model_speedup(C, rho, beta, t_total)


def hcms_model_s_max(rho) -> float:
    return lib.hcms_model_s_max(rho)


def hcms_model_choose_chunks(heads_per_rank: int, t_comm: float, beta: float) -> int:
    return lib.hcms_model_choose_chunks(heads_per_rank, t_comm, beta)


# ---- plan ------------------------------------------------------------------------------------

class Plan:
    """Owner of one ``hcms_plan_t*`` (destroyed on ``close()`` / garbage collection)."""

    def __init__(self, handle: int, S, H, D, P, C, dtype, flags):
        self.handle = handle
        self.S, self.H, self.D, self.P, self.C = int(S), int(H), int(D), int(P), int(C)
        self.dtype, self.flags = dtype, flags

    def close(self) -> None:
        if self.handle:
            lib.hcms_plan_destroy(self.handle)
            self.handle = 0

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def hcms_plan(S, H, D, P, C, dtype=HCMS_DTYPE_BF16, flags=0) -> Plan:
    h = c_void_p()
    _check(lib.hcms_plan(ctypes.byref(h), S, H, D, P, C, dtype, flags), "hcms_plan")
    return Plan(h.value, S, H, D, P, C, dtype, flags)


def hcms_plan_destroy(plan: Plan) -> None:
    plan.close()


def hcms_plan_workspace_bytes(plan: Plan) -> int:
    return lib.hcms_plan_workspace_bytes(plan.handle)


def hcms_plan_workspace(plan: Plan) -> int:
    return lib.hcms_plan_workspace(plan.handle) or 0


def hcms_plan_set_workspace(plan: Plan, dev, nbytes: int) -> None:
    _check(lib.hcms_plan_set_workspace(plan.handle, _ptr(dev), nbytes), "hcms_plan_set_workspace")


def hcms_chunk_table(plan: Plan):
    o, h = (c_int * plan.C)(), (c_int * plan.C)()
    _check(lib.hcms_chunk_table(plan.handle, o, h), "hcms_chunk_table")
    return list(o), list(h)


def hcms_chunk_layout(plan: Plan, c: int):
    """-> dict(bytes, q_off, k_off, v_off, o_off) of chunk c inside the workspace."""
    vals = [c_size_t() for _ in range(5)]
    _check(lib.hcms_chunk_layout(plan.handle, c, *[ctypes.byref(v) for v in vals]), "hcms_chunk_layout")
    return dict(zip(("bytes", "q_off", "k_off", "v_off", "o_off"), (v.value for v in vals)))


def hcms_plan_tensor_map_encodes(plan: Plan) -> int:
    return lib.hcms_plan_tensor_map_encodes(plan.handle)


def hcms_plan_last_launch_count(plan: Plan) -> int:
    return lib.hcms_plan_last_launch_count(plan.handle)


HCMS_PROFILE_RING = 64


def hcms_plan_timings(plan: Plan, calls_back: int = 0):
    """-> (scatter_ms[C], attn_ms[C], gather_ms[C]) of a recent forward call (HCMS_FLAG_PROFILE plans)."""
    arrs = [(c_float * plan.C)() for _ in range(3)]
    _check(lib.hcms_plan_timings(plan.handle, calls_back, *arrs), "hcms_plan_timings")
    return tuple(list(a) for a in arrs)


def hcms_plan_step_span(plan: Plan, calls_back: int = 0, step: int = 1) -> float:
    """-> ms from chunk 0's begin event to the last end event of step kind ``step`` (0 scatter, 1 attention, 2 gather)."""
    ms = c_float()
    _check(lib.hcms_plan_step_span(plan.handle, calls_back, step, ctypes.byref(ms)), "hcms_plan_step_span")
    return float(ms.value)


def hcms_plan_timeline(plan: Plan, calls_back: int = 0):
    """-> (begin_ms, end_ms), each [3][C] (scatter, attention, gather) in ms after chunk 0's scatter began."""
    n = 3 * plan.C
    b, e = (c_float * n)(), (c_float * n)()
    _check(lib.hcms_plan_timeline(plan.handle, calls_back, b, e), "hcms_plan_timeline")
    cut = lambda a: [list(a)[k * plan.C:(k + 1) * plan.C] for k in range(3)]
    return cut(b), cut(e)


def hcms_autotune_chunks(S, H, D, P, dtype, flags, q, k, v, out, scale: float, max_C: int, reps: int = 3, stream=None):
    """Measure every C in [1, min(max_C, H/P)] on the caller's tensors -> (best_C, [ms per call for C = 1..max_C])."""
    best = c_int()
    ms = (c_float * max(int(max_C), 1))()
    _check(lib.hcms_autotune_chunks(S, H, D, P, dtype, flags, _ptr(q), _ptr(k), _ptr(v), _ptr(out), scale,
                                    _stream(stream), max_C, reps, ctypes.byref(best), ms), "hcms_autotune_chunks")
    return int(best.value), list(ms)


# ---- the hot path ------------------------------------------------------------------------------

def hcms_attention_forward(plan: Plan, q, k, v, out, scale: float, stream=None) -> None:
    """Alg. 1 lines 4-26 on device tensors [S,H,D] bf16; asynchronous on ``stream``."""
    _check(lib.hcms_attention_forward(plan.handle, _ptr(q), _ptr(k), _ptr(v), _ptr(out), plan.S, plan.H, plan.D,
                                      plan.P, plan.C, scale, _stream(stream)), "hcms_attention_forward")


def hcms_attention_forward_host(plan: Plan, q, k, v, out, scale: float, stream=None) -> None:
    """Same with HOST buffers (numpy uint16 / pinned torch tensors); synchronises ``stream``."""
    _check(lib.hcms_attention_forward_host(plan.handle, _ptr(q), _ptr(k), _ptr(v), _ptr(out), plan.S, plan.H,
                                           plan.D, plan.P, plan.C, scale, _stream(stream)),
           "hcms_attention_forward_host")


def hcms_a2a_scatter(plan: Plan, srcs, dsts, c: int, stream=None) -> None:
    n = len(srcs)
    if n != len(dsts):
        raise ValueError("srcs and dsts differ in length")
    s = (c_void_p * n)(*[_ptr(x) for x in srcs])
    d = (c_void_p * n)(*[_ptr(x) for x in dsts])
    _check(lib.hcms_a2a_scatter(plan.handle, n, s, d, c, _stream(stream)), "hcms_a2a_scatter")


def hcms_a2a_gather(plan: Plan, src, dst, c: int, stream=None) -> None:
    _check(lib.hcms_a2a_gather(plan.handle, _ptr(src), _ptr(dst), c, _stream(stream)), "hcms_a2a_gather")


def hcms_attention_chunk(plan: Plan, qc, kc, vc, oc, c: int, scale: float, stream=None) -> None:
    _check(lib.hcms_attention_chunk(plan.handle, _ptr(qc), _ptr(kc), _ptr(vc), _ptr(oc), c, scale, _stream(stream)),
           "hcms_attention_chunk")


# ---- the attention layer around the hot path (Alg. 1 lines 2-3, 27) ------------------------------

def hcms_gemm_bf16_nt(a, b, c, M: int, N: int, K: int, stream=None) -> None:
    """c[M,N] = a[M,K] @ b[N,K]^T on device bf16 tensors; asynchronous on ``stream``."""
    _check(lib.hcms_gemm_bf16_nt(_ptr(a), _ptr(b), _ptr(c), M, N, K, _stream(stream)), "hcms_gemm_bf16_nt")


def hcms_qkv_projection_rope(plan: Plan, x, w_qkv, rope_cos, rope_sin, q, k, v, Dm: int, stream=None) -> None:
    """Alg. 1 lines 2-3: x[S,Dm] @ w_qkv[3HD,Dm]^T -> q,k,v [S,H,D], RoPE on q,k (tables [S,D/2] fp32 or None)."""
    _check(lib.hcms_qkv_projection_rope(plan.handle, _ptr(x), _ptr(w_qkv), _ptr(rope_cos), _ptr(rope_sin), _ptr(q),
                                        _ptr(k), _ptr(v), Dm, _stream(stream)), "hcms_qkv_projection_rope")


def hcms_output_projection(plan: Plan, o, w_o, y, Dm: int, stream=None) -> None:
    """Alg. 1 line 27: y[S,Dm] = o[S,H*D] @ w_o[Dm,H*D]^T."""
    _check(lib.hcms_output_projection(plan.handle, _ptr(o), _ptr(w_o), _ptr(y), Dm, _stream(stream)),
           "hcms_output_projection")


def hcms_layer_forward(plan: Plan, x, w_qkv, w_o, rope_cos, rope_sin, y, Dm: int, scale: float, stream=None) -> None:
    """Alg. 1 lines 2-27 on device tensors; asynchronous on ``stream``."""
    _check(lib.hcms_layer_forward(plan.handle, _ptr(x), _ptr(w_qkv), _ptr(w_o), _ptr(rope_cos), _ptr(rope_sin), _ptr(y),
                                  plan.S, Dm, plan.H, plan.D, plan.P, plan.C, scale, _stream(stream)),
           "hcms_layer_forward")


def hcms_plan_layer_buffer(plan: Plan, which: int) -> int:
    return lib.hcms_plan_layer_buffer(plan.handle, which) or 0


def hcms_plan_layer_timings(plan: Plan):
    """-> (qkv_ms, hcms_ms, out_ms) of the last hcms_layer_forward (HCMS_FLAG_PROFILE plans)."""
    vals = [c_float() for _ in range(3)]
    _check(lib.hcms_plan_layer_timings(plan.handle, *[ctypes.byref(v) for v in vals]), "hcms_plan_layer_timings")
    return tuple(float(v.value) for v in vals)


# ---- backward of the hot path -----------------------------------------------------

def hcms_attention_backward(plan: Plan, dout, dq, dk, dv, scale: float, stream=None) -> None:
    """Gradients of the last hcms_attention_forward on a HCMS_FLAG_TRAINING plan; device [S,H,D] bf16 tensors."""
    _check(lib.hcms_attention_backward(plan.handle, _ptr(dout), _ptr(dq), _ptr(dk), _ptr(dv), plan.S, plan.H, plan.D,
                                       plan.P, plan.C, scale, _stream(stream)), "hcms_attention_backward")


def hcms_attention_chunk_lse(plan: Plan, qc, kc, vc, oc, lse, c: int, scale: float, stream=None) -> None:
    _check(lib.hcms_attention_chunk_lse(plan.handle, _ptr(qc), _ptr(kc), _ptr(vc), _ptr(oc), _ptr(lse), c, scale,
                                        _stream(stream)), "hcms_attention_chunk_lse")


def hcms_attention_backward_chunk(plan: Plan, qc, kc, vc, oc, doc, lse, dqc, dkc, dvc, c: int, scale: float,
                                  stream=None) -> None:
    _check(lib.hcms_attention_backward_chunk(plan.handle, _ptr(qc), _ptr(kc), _ptr(vc), _ptr(oc), _ptr(doc), _ptr(lse),
                                             _ptr(dqc), _ptr(dkc), _ptr(dvc), c, scale, _stream(stream)),
           "hcms_attention_backward_chunk")


HCMS_STATIC_SCRATCH_BYTES = 4 << 20


def hcms_attention_backward_chunk_static(qc, kc, vc, oc, doc, lse, dqc, dkc, dvc, S: int, P: int, h_c: int, D: int,
                                         scale: float, stream=None) -> None:
    """hcms_attention_backward_chunk without a plan and without any device allocation: its scratch is a fixed
    HCMS_STATIC_SCRATCH_BYTES array inside libhcms.so (see include/hcms.h for who needs that, the size limit and the
    rule that overlapping calls race).  Raises HcmsError(HCMS_ERR_WORKSPACE_TOO_SMALL) beyond the limit."""
    _check(lib.hcms_attention_backward_chunk_static(_ptr(qc), _ptr(kc), _ptr(vc), _ptr(oc), _ptr(doc), _ptr(lse), _ptr(dqc),
                                                    _ptr(dkc), _ptr(dvc), S, P, h_c, D, scale, _stream(stream)),
           "hcms_attention_backward_chunk_static")


def hcms_plan_lse(plan: Plan) -> int:
    return lib.hcms_plan_lse(plan.handle) or 0


def hcms_plan_graph_captures(plan: Plan) -> int:
    return lib.hcms_plan_graph_captures(plan.handle)


def hcms_autotune_chunks_host(S, H, D, P, flags, q, k, v, out, scale: float, max_C: int, reps: int = 3, stream=None):
    """hcms_autotune_chunks over the host-buffer path (q, k, v, out in host memory) -> (best_C, [ms per call])."""
    best = c_int()
    ms = (c_float * max(int(max_C), 1))()
    _check(lib.hcms_autotune_chunks_host(S, H, D, P, flags, _ptr(q), _ptr(k), _ptr(v), _ptr(out), scale, _stream(stream),
                                         max_C, reps, ctypes.byref(best), ms), "hcms_autotune_chunks_host")
    return int(best.value), list(ms)


# ---- HCMS between P real ranks --------------------------------------------------------

HCMS_DIST_HANDLE_BYTES = 128


class DistPlan:
    """Owns one rank's hcms_dist_plan_t*; use as a context manager or call close()."""

    def __init__(self, handle: int, S: int, H: int, D: int, P: int, C: int, rank: int):
        self.handle = c_void_p(handle)
        self.S, self.H, self.D, self.P, self.C, self.rank = S, H, D, P, C, rank

    def close(self) -> None:
        if self.handle:
            lib.hcms_dist_plan_destroy(self.handle)
            self.handle = c_void_p(0)

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def hcms_dist_plan(S: int, H: int, D: int, P: int, C: int, rank: int, dtype: int = HCMS_DTYPE_BF16, flags: int = 0) -> DistPlan:
    h = c_void_p(0)
    _check(lib.hcms_dist_plan(ctypes.byref(h), S, H, D, P, C, dtype, flags, rank), "hcms_dist_plan")
    return DistPlan(h.value, S, H, D, P, C, rank)


def hcms_dist_export(plan: DistPlan) -> bytes:
    buf = ctypes.create_string_buffer(HCMS_DIST_HANDLE_BYTES)
    _check(lib.hcms_dist_export(plan.handle, buf), "hcms_dist_export")
    return buf.raw


def hcms_dist_attach(plan: DistPlan, handles) -> None:
    """handles: the P ranks' hcms_dist_export bytes in rank order."""
    blob = b"".join(handles)
    if len(blob) != HCMS_DIST_HANDLE_BYTES * len(handles):
        raise ValueError("every handle must be HCMS_DIST_HANDLE_BYTES long")
    buf = ctypes.create_string_buffer(blob, len(blob))
    _check(lib.hcms_dist_attach(plan.handle, buf, len(handles)), "hcms_dist_attach")


def hcms_dist_attach_local(plan: DistPlan, peers) -> None:
    arr = (c_void_p * len(peers))(*[p.handle.value for p in peers])
    _check(lib.hcms_dist_attach_local(plan.handle, arr, len(peers)), "hcms_dist_attach_local")


def hcms_dist_attention_forward(plan: DistPlan, q, k, v, out, scale: float, stream=None) -> None:
    _check(lib.hcms_dist_attention_forward(plan.handle, _ptr(q), _ptr(k), _ptr(v), _ptr(out), scale, _stream(stream)),
           "hcms_dist_attention_forward")


def hcms_dist_attention_forward_host(plan: DistPlan, q, k, v, out, scale: float, stream=None) -> None:
    """hcms_dist_attention_forward on HOST shards (pinned for asynchronous copies); synchronises the stream."""
    _check(lib.hcms_dist_attention_forward_host(plan.handle, _ptr(q), _ptr(k), _ptr(v), _ptr(out), scale, _stream(stream)),
           "hcms_dist_attention_forward_host")


def hcms_dist_attention_forward_group(plans, qs, ks, vs, outs, scale: float, streams) -> None:
    """All P ranks of one process in one call (plans attached with hcms_dist_attach_local), distinct caller streams."""
    n = len(plans)
    arr = lambda xs: (c_void_p * n)(*[_ptr(x) for x in xs])
    pl = (c_void_p * n)(*[p.handle.value for p in plans])
    st = (c_void_p * n)(*[_stream(s) for s in streams])
    _check(lib.hcms_dist_attention_forward_group(pl, n, arr(qs), arr(ks), arr(vs), arr(outs), scale, st),
           "hcms_dist_attention_forward_group")


def hcms_dist_layer_forward(plan: DistPlan, x, w_qkv, w_o, rope_cos, rope_sin, y, Dm: int, scale: float, stream=None) -> None:
    """Alg. 1 lines 2-27 between real ranks (plan made with HCMS_FLAG_DIST_FUSE_OUT); this rank's [S/P, Dm] tokens."""
    _check(lib.hcms_dist_layer_forward(plan.handle, _ptr(x), _ptr(w_qkv), _ptr(w_o), _ptr(rope_cos), _ptr(rope_sin), _ptr(y),
                                       Dm, scale, _stream(stream)), "hcms_dist_layer_forward")


def hcms_dist_layer_forward_group(plans, xs, w_qkv, w_o, coss, sins, ys, Dm: int, scale: float, streams) -> None:
    """All P ranks of one process in one call (plans attached with hcms_dist_attach_local), distinct caller streams."""
    n = len(plans)
    arr = lambda v: (c_void_p * n)(*[_ptr(t) for t in v]) if v is not None else None
    pl = (c_void_p * n)(*[p.handle.value for p in plans])
    st = (c_void_p * n)(*[_stream(s) for s in streams])
    _check(lib.hcms_dist_layer_forward_group(pl, n, arr(xs), _ptr(w_qkv), _ptr(w_o), arr(coss), arr(sins), arr(ys), Dm, scale, st),
           "hcms_dist_layer_forward_group")


def hcms_dist_block_bytes(plan: DistPlan) -> int:
    return lib.hcms_dist_block_bytes(plan.handle)


def hcms_dist_last_launch_count(plan: DistPlan) -> int:
    return lib.hcms_dist_last_launch_count(plan.handle)


def all_gather_bytes(blob: bytes, group=None):
    """Every rank's `blob` (equal lengths) in rank order, over torch.distributed (any backend: the bytes travel as a
    uint8 tensor on the backend's device).  Plumbing only."""
    import torch
    import torch.distributed as dist
    mine = torch.frombuffer(bytearray(blob), dtype=torch.uint8)
    if dist.get_backend(group) == "nccl":
        mine = mine.cuda()
    parts = [torch.empty_like(mine) for _ in range(dist.get_world_size(group))]
    dist.all_gather(parts, mine, group=group)
    return [t.cpu().numpy().tobytes() for t in parts]


def hcms_dist_exchange_handles(plan: DistPlan, group=None):
    """All-gather the ranks' export handles over torch.distributed and attach.  The data path never touches
    torch.distributed: only these 128 bytes per rank do."""
    import torch.distributed as dist
    world = dist.get_world_size(group)
    if world != plan.P:
        raise ValueError(f"process group has {world} ranks, the plan has P={plan.P}")
    handles = all_gather_bytes(hcms_dist_export(plan), group)
    hcms_dist_attach(plan, handles)
    return handles

"""Thin ctypes binding of the osdp-b200 C ABI (``include/osdp.h``): same names, argument marshalling only.

Every step of the hot path runs inside ``libosdp_b200.so``; this file allocates nothing on the device except
what the caller asks for through torch (device memory, streams).  There is NO fallback: if the library is
missing, importing this module raises.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("OSDP_B200_LIB") or os.path.join(_HERE, "libosdp_b200.so")   # override: A/B builds

if not os.path.exists(LIB_PATH):
    raise ImportError(
        f"{LIB_PATH} not found: build it with `python -m paper_2305_09940_b200.build` "
        "(or __graft_entry__.build()).  There is no CPU/PyTorch fallback for the osdp-b200 hot path.")

_lib = C.CDLL(LIB_PATH)

OSDP_OK = 0
OSDP_ERR_NULL, OSDP_ERR_SHAPE, OSDP_ERR_K, OSDP_ERR_DTYPE, OSDP_ERR_WORKSPACE, OSDP_ERR_ALIGN = 1, 2, 3, 4, 5, 6
OSDP_ERR_ARCH, OSDP_ERR_CUDA, OSDP_ERR_INFEASIBLE, OSDP_ERR_ARG, OSDP_ERR_SEARCH_LIMIT = 7, 8, 9, 10, 11
OSDP_ERR_STATIC_LIMIT = 12
OSDP_ERR_COMM = 13
OSDP_BIAS_GRAD_STATIC_MAX_COLS = 16384
OSDP_F32, OSDP_BF16 = 0, 1
OSDP_FWD, OSDP_BWD = 0, 1
OSDP_DP, OSDP_ZDP = 0, 1

EXPORTS = (
    "osdp_status_string", "osdp_last_cuda_error", "osdp_version", "osdp_split_mlp_workspace_bytes",
    "osdp_split_mlp_forward", "osdp_split_mlp_backward", "osdp_last_launch_count", "osdp_cost_eval",
    "osdp_mlp_op_cost", "osdp_plan", "osdp_plan_batch", "osdp_trace_enable", "osdp_trace_read", "osdp_step_name",
    "osdp_set_tuning", "osdp_get_tuning", "osdp_ffn_split_mlp_workspace_bytes", "osdp_ffn_split_mlp_forward",
    "osdp_ffn_split_mlp_backward", "osdp_ffn_split_mlp_op_cost", "osdp_cost_eval_mixed", "osdp_plan_mixed",
    "osdp_split_linear_workspace_bytes", "osdp_split_linear_forward", "osdp_split_linear_backward", "osdp_linear_op_cost",
    "osdp_zdp_shard_elems", "osdp_zdp_slice_layout", "osdp_zdp_schedule", "osdp_zdp_ffn_split_mlp_workspace_bytes",
    "osdp_zdp_ffn_split_mlp_forward", "osdp_zdp_ffn_split_mlp_backward", "osdp_zdp_ffn_split_mlp_op_cost",
    "osdp_bias_grad_static",
)


class osdp_mlp_desc(C.Structure):
    _fields_ = [("tokens", C.c_int64), ("hidden", C.c_int64), ("ffn", C.c_int64), ("dtype", C.c_int32),
                ("k", C.c_int32)]


class osdp_linear_desc(C.Structure):
    _fields_ = [("tokens", C.c_int64), ("in_features", C.c_int64), ("out_features", C.c_int64), ("dtype", C.c_int32),
                ("k", C.c_int32), ("axis", C.c_int32), ("has_bias", C.c_int32)]


OSDP_SPLIT_TOKENS, OSDP_SPLIT_CONTRACTION = 0, 1


class osdp_zdp_desc(C.Structure):
    _fields_ = [("mlp", osdp_mlp_desc), ("world", C.c_int32), ("rank", C.c_int32)]


class osdp_zdp_slice(C.Structure):
    _fields_ = [("lo", C.c_int64), ("hi", C.c_int64), ("w1_off", C.c_int64), ("w1_elems", C.c_int64),
                ("b1_off", C.c_int64), ("b1_elems", C.c_int64), ("w2_off", C.c_int64), ("w2_elems", C.c_int64)]


class osdp_zdp_step(C.Structure):
    _fields_ = [("op", C.c_int32), ("slice", C.c_int32), ("buffer", C.c_int32), ("on_comm_stream", C.c_int32),
                ("bytes_per_rank", C.c_uint64)]


ALL_GATHER_FN = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p)
REDUCE_SCATTER_FN = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p)


class osdp_comm(C.Structure):
    _fields_ = [("ctx", C.c_void_p), ("all_gather", ALL_GATHER_FN), ("reduce_scatter_f32", REDUCE_SCATTER_FN)]


OSDP_ZDP_GATHER, OSDP_ZDP_COMPUTE, OSDP_ZDP_REDUCE_SCATTER = 0, 1, 2


class osdp_op_cost(C.Structure):
    _fields_ = [("S", C.c_double), ("model_bytes", C.c_uint64), ("act_bytes", C.c_uint64),
                ("extra_fixed", C.c_uint64), ("extra_summed", C.c_uint64), ("extra_transient", C.c_uint64),
                ("gamma", C.c_double), ("delta", C.c_double)]


class osdp_device(C.Structure):
    _fields_ = [("N", C.c_int32), ("alpha", C.c_double), ("beta", C.c_double), ("mem_limit_bytes", C.c_uint64),
                ("checkpointing", C.c_int32), ("recompute_fraction", C.c_double), ("act_keep_fraction", C.c_double)]


_lib.osdp_status_string.restype = C.c_char_p
_lib.osdp_status_string.argtypes = [C.c_int]
_lib.osdp_last_cuda_error.restype = C.c_char_p
_lib.osdp_version.restype = C.c_char_p
_lib.osdp_last_launch_count.restype = C.c_int64
_lib.osdp_split_mlp_workspace_bytes.restype = C.c_size_t
_lib.osdp_split_mlp_workspace_bytes.argtypes = [C.POINTER(osdp_mlp_desc), C.c_int]
_lib.osdp_split_mlp_forward.restype = C.c_int
_lib.osdp_split_mlp_forward.argtypes = [C.POINTER(osdp_mlp_desc)] + [C.c_void_p] * 7 + [C.c_size_t, C.c_void_p]
_lib.osdp_split_mlp_backward.restype = C.c_int
_lib.osdp_split_mlp_backward.argtypes = [C.POINTER(osdp_mlp_desc)] + [C.c_void_p] * 12 + [C.c_size_t, C.c_void_p]
_lib.osdp_ffn_split_mlp_workspace_bytes.restype = C.c_size_t
_lib.osdp_ffn_split_mlp_workspace_bytes.argtypes = [C.POINTER(osdp_mlp_desc), C.c_int]
_lib.osdp_ffn_split_mlp_forward.restype = C.c_int
_lib.osdp_ffn_split_mlp_forward.argtypes = [C.POINTER(osdp_mlp_desc)] + [C.c_void_p] * 7 + [C.c_size_t, C.c_void_p]
_lib.osdp_ffn_split_mlp_backward.restype = C.c_int
_lib.osdp_ffn_split_mlp_backward.argtypes = [C.POINTER(osdp_mlp_desc)] + [C.c_void_p] * 12 + [C.c_size_t, C.c_void_p]
_lib.osdp_ffn_split_mlp_op_cost.restype = C.c_int
_lib.osdp_ffn_split_mlp_op_cost.argtypes = [C.POINTER(osdp_mlp_desc), C.c_int, C.POINTER(osdp_op_cost)]
_lib.osdp_cost_eval.restype = C.c_int
_lib.osdp_cost_eval.argtypes = [C.POINTER(osdp_op_cost), C.c_int, C.c_int32, C.c_int64, C.POINTER(osdp_device),
                                C.POINTER(C.c_uint64), C.POINTER(C.c_uint64), C.POINTER(C.c_double)]
_lib.osdp_mlp_op_cost.restype = C.c_int
_lib.osdp_mlp_op_cost.argtypes = [C.POINTER(osdp_mlp_desc), C.c_int, C.POINTER(osdp_op_cost)]
_lib.osdp_plan.restype = C.c_int
_lib.osdp_plan.argtypes = [C.POINTER(osdp_op_cost), C.c_int32, C.POINTER(osdp_device), C.c_int64,
                           C.POINTER(C.c_int32), C.c_int32, C.POINTER(C.c_int32), C.POINTER(C.c_int32),
                           C.POINTER(C.c_double), C.POINTER(C.c_uint64)]
_lib.osdp_cost_eval_mixed.restype = C.c_int
_lib.osdp_cost_eval_mixed.argtypes = [C.POINTER(osdp_op_cost), C.c_int32, C.c_int32, C.c_int64, C.POINTER(osdp_device),
                                      C.POINTER(C.c_uint64), C.POINTER(C.c_uint64), C.POINTER(C.c_double)]
_lib.osdp_plan_mixed.restype = C.c_int
_lib.osdp_plan_mixed.argtypes = _lib.osdp_plan.argtypes
_lib.osdp_plan_batch.restype = C.c_int
_lib.osdp_plan_batch.argtypes = [C.POINTER(osdp_op_cost), C.c_int32, C.POINTER(osdp_device), C.c_int64,
                                 C.POINTER(C.c_int32), C.c_int32, C.POINTER(C.c_int32), C.POINTER(C.c_int32),
                                 C.POINTER(C.c_int64), C.POINTER(C.c_double), C.POINTER(C.c_uint64)]


_lib.osdp_split_linear_workspace_bytes.restype = C.c_int
_lib.osdp_split_linear_workspace_bytes.argtypes = [C.POINTER(osdp_linear_desc), C.c_int, C.POINTER(C.c_size_t)]
_lib.osdp_split_linear_forward.restype = C.c_int
_lib.osdp_split_linear_forward.argtypes = [C.POINTER(osdp_linear_desc)] + [C.c_void_p] * 5 + [C.c_size_t, C.c_void_p]
_lib.osdp_split_linear_backward.restype = C.c_int
_lib.osdp_split_linear_backward.argtypes = [C.POINTER(osdp_linear_desc)] + [C.c_void_p] * 7 + [C.c_size_t, C.c_void_p]
_lib.osdp_bias_grad_static.restype = C.c_int
_lib.osdp_bias_grad_static.argtypes = [C.c_void_p, C.c_int64, C.c_int64, C.c_int32, C.c_void_p, C.c_void_p]
_lib.osdp_linear_op_cost.restype = C.c_int
_lib.osdp_linear_op_cost.argtypes = [C.POINTER(osdp_linear_desc), C.c_int, C.POINTER(osdp_op_cost)]
_lib.osdp_zdp_shard_elems.restype = C.c_int
_lib.osdp_zdp_shard_elems.argtypes = [C.POINTER(osdp_zdp_desc), C.POINTER(C.c_int64)]
_lib.osdp_zdp_slice_layout.restype = C.c_int
_lib.osdp_zdp_slice_layout.argtypes = [C.POINTER(osdp_zdp_desc), C.c_int32, C.POINTER(osdp_zdp_slice)]
_lib.osdp_zdp_schedule.restype = C.c_int64
_lib.osdp_zdp_schedule.argtypes = [C.POINTER(osdp_zdp_desc), C.c_int, C.c_int64, C.POINTER(osdp_zdp_step)]
_lib.osdp_zdp_ffn_split_mlp_workspace_bytes.restype = C.c_int
_lib.osdp_zdp_ffn_split_mlp_workspace_bytes.argtypes = [C.POINTER(osdp_zdp_desc), C.c_int, C.POINTER(C.c_size_t)]
_lib.osdp_zdp_ffn_split_mlp_forward.restype = C.c_int
_lib.osdp_zdp_ffn_split_mlp_forward.argtypes = [C.POINTER(osdp_zdp_desc)] + [C.c_void_p] * 4 + [C.c_size_t, C.POINTER(osdp_comm),
                                                                                         C.c_void_p, C.c_void_p]
_lib.osdp_zdp_ffn_split_mlp_backward.restype = C.c_int
_lib.osdp_zdp_ffn_split_mlp_backward.argtypes = [C.POINTER(osdp_zdp_desc)] + [C.c_void_p] * 6 + [C.c_size_t, C.POINTER(osdp_comm),
                                                                                          C.c_void_p, C.c_void_p]
_lib.osdp_zdp_ffn_split_mlp_op_cost.restype = C.c_int
_lib.osdp_zdp_ffn_split_mlp_op_cost.argtypes = [C.POINTER(osdp_zdp_desc), C.c_int, C.POINTER(osdp_op_cost)]
_lib.osdp_trace_enable.restype = C.c_int
_lib.osdp_trace_enable.argtypes = [C.c_int]
_lib.osdp_set_tuning.restype = C.c_int
_lib.osdp_set_tuning.argtypes = [C.c_int, C.c_int64]
_lib.osdp_get_tuning.restype = C.c_int64
_lib.osdp_get_tuning.argtypes = [C.c_int]
OSDP_TUNE_MT2_MIN_K, OSDP_TUNE_MT2_MIN_TILES, OSDP_TUNE_WAVE_SYNC, OSDP_TUNE_BAND_MIB = 0, 1, 2, 3
OSDP_TUNE_CLUSTER_MIN_TILES = 4
OSDP_TUNE_MT2_MIN_K_ACC = 5
OSDP_TUNE_FORK_MAX_TILES = 6
OSDP_TUNE_SLICE_KERNEL_MAX_TILES = 7
OSDP_TUNE_SLICE_KERNEL_FFN_MAX_TILES = 8
OSDP_TUNE_BALANCE_N = 9
_lib.osdp_trace_read.restype = C.c_int64
_lib.osdp_trace_read.argtypes = [C.c_int64, C.POINTER(C.c_int32), C.POINTER(C.c_float)]
_lib.osdp_step_name.restype = C.c_char_p
_lib.osdp_step_name.argtypes = [C.c_int]


class OsdpError(RuntimeError):
    def __init__(self, status: int, where: str, detail: str = ""):
        self.status = status
        msg = f"{where}: {osdp_status_string(status)} (status {status})" + (f": {detail}" if detail else "")
        if status == OSDP_ERR_CUDA:
            msg += f": {osdp_last_cuda_error()}"
        super().__init__(msg)


def osdp_status_string(status: int) -> str:
    return _lib.osdp_status_string(int(status)).decode()


def osdp_last_cuda_error() -> str:
    return _lib.osdp_last_cuda_error().decode()


def osdp_version() -> str:
    return _lib.osdp_version().decode()


def osdp_last_launch_count() -> int:
    return int(_lib.osdp_last_launch_count())


def osdp_set_tuning(key: int, value: int, check: bool = True) -> int:
    rc = int(_lib.osdp_set_tuning(key, value))
    if check and rc != OSDP_OK:
        raise OsdpError(rc, "osdp_set_tuning")
    return rc


def osdp_get_tuning(key: int) -> int:
    return int(_lib.osdp_get_tuning(key))


def osdp_trace_enable(on: bool) -> None:
    _lib.osdp_trace_enable(1 if on else 0)


def osdp_trace_read(max_entries: int = 1 << 16):
    """[(step_id, milliseconds)] for every launch since the last read (waits for them)."""
    ids, ms = (C.c_int32 * max_entries)(), (C.c_float * max_entries)()
    n = int(_lib.osdp_trace_read(max_entries, ids, ms))
    if n < 0:
        raise OsdpError(OSDP_ERR_CUDA, "osdp_trace_read")
    n = min(n, max_entries)
    return [(int(ids[i]), float(ms[i])) for i in range(n)]


def osdp_step_name(step_id: int) -> str:
    return _lib.osdp_step_name(int(step_id)).decode()


def _dtype_code(dtype: torch.dtype) -> int:
    if dtype == torch.float32:
        return OSDP_F32
    if dtype == torch.bfloat16:
        return OSDP_BF16
    return -1


def make_desc(tokens: int, hidden: int, ffn: int, dtype, k: int) -> osdp_mlp_desc:
    code = dtype if isinstance(dtype, int) else _dtype_code(dtype)
    return osdp_mlp_desc(int(tokens), int(hidden), int(ffn), int(code), int(k))


def osdp_split_mlp_workspace_bytes(desc: osdp_mlp_desc, pass_: int) -> int:
    return int(_lib.osdp_split_mlp_workspace_bytes(C.byref(desc), int(pass_)))


def _ptr(t):
    if t is None:
        return None
    if isinstance(t, int):
        return t
    return t.data_ptr()


def _stream_ptr(stream):
    if stream is None:
        stream = torch.cuda.current_stream()
    return stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream)


_TORCH_DTYPE = {OSDP_F32: torch.float32, OSDP_BF16: torch.bfloat16}


def _validate(where, desc, spec, workspace, workspace_bytes):
    """Marshalling checks (no arithmetic of the method): every torch tensor handed to the C ABI must be a dense CUDA
    tensor of the dtype and element count the descriptor implies, all on one device; raw integer addresses are taken
    on trust.  Returns that device (or None) so the call can run with it current - the library launches on the
    calling thread's current device.  Returns (device, status, detail)."""
    T, h, f = desc.tokens, desc.hidden, desc.ffn
    st = _TORCH_DTYPE.get(desc.dtype)
    numel = {"X": T * h, "Y": T * h, "dY": T * h, "dX": T * h, "W1": h * f, "W2": f * h, "b1": f, "b2": h,
             "dW1": h * f, "dW2": f * h, "db1": f, "db2": h}
    dev = None
    for name, t in spec:
        if t is None or isinstance(t, int):
            continue
        want = torch.float32 if name in ("dW1", "dW2", "db1", "db2") else st
        if not t.is_cuda:
            return None, OSDP_ERR_ARG, f"{name} is not a CUDA tensor"
        if not t.is_contiguous():
            return None, OSDP_ERR_ARG, f"{name} is not dense row-major"
        if want is not None and t.dtype != want:
            return None, OSDP_ERR_DTYPE, f"{name} has dtype {t.dtype}, descriptor needs {want}"
        if t.numel() != numel[name]:
            return None, OSDP_ERR_SHAPE, f"{name} has {t.numel()} elements, descriptor needs {numel[name]}"
        if dev is not None and t.device != dev:
            return None, OSDP_ERR_ARG, f"{name} is on {t.device}, other tensors on {dev}"
        dev = t.device
    if workspace is not None and not isinstance(workspace, int):
        if not workspace.is_cuda or not workspace.is_contiguous():
            return None, OSDP_ERR_WORKSPACE, f"workspace must be a dense CUDA tensor"
        if dev is not None and workspace.device != dev:
            return None, OSDP_ERR_ARG, f"workspace is on {workspace.device}, tensors on {dev}"
        if workspace_bytes > workspace.numel() * workspace.element_size():
            return None, OSDP_ERR_WORKSPACE, f"workspace_bytes exceeds the workspace tensor"
        dev = dev or workspace.device
    return dev, OSDP_OK, ""


class _on_device:
    """Runs the C call with the tensors' device current (a no-op when it already is, or when only raw addresses came)."""

    def __init__(self, dev):
        self.ctx = torch.cuda.device(dev) if dev is not None and dev.index != torch.cuda.current_device() else None

    def __enter__(self):
        if self.ctx is not None:
            self.ctx.__enter__()

    def __exit__(self, *a):
        if self.ctx is not None:
            self.ctx.__exit__(*a)


def _call_fwd(fn, where, desc, X, W1, b1, W2, b2, Y, workspace, workspace_bytes, stream, check):
    if workspace_bytes is None:
        workspace_bytes = workspace.numel() * workspace.element_size()
    dev, vs, detail = _validate(where, desc, (("X", X), ("W1", W1), ("b1", b1), ("W2", W2), ("b2", b2), ("Y", Y)),
                                workspace, int(workspace_bytes))
    if vs != OSDP_OK:
        if check:
            raise OsdpError(vs, where, detail)
        return vs
    with _on_device(dev):
        st = fn(C.byref(desc), _ptr(X), _ptr(W1), _ptr(b1), _ptr(W2), _ptr(b2), _ptr(Y), _ptr(workspace),
                int(workspace_bytes), _stream_ptr(stream))
    if check and st != OSDP_OK:
        raise OsdpError(st, where)
    return st


def _call_bwd(fn, where, desc, X, W1, b1, W2, b2, dY, dX, dW1, db1, dW2, db2, workspace, workspace_bytes, stream, check):
    if workspace_bytes is None:
        workspace_bytes = workspace.numel() * workspace.element_size()
    dev, vs, detail = _validate(where, desc, (("X", X), ("W1", W1), ("b1", b1), ("W2", W2), ("b2", b2), ("dY", dY),
                                              ("dX", dX), ("dW1", dW1), ("db1", db1), ("dW2", dW2), ("db2", db2)),
                                workspace, int(workspace_bytes))
    if vs != OSDP_OK:
        if check:
            raise OsdpError(vs, where, detail)
        return vs
    with _on_device(dev):
        st = fn(C.byref(desc), _ptr(X), _ptr(W1), _ptr(b1), _ptr(W2), _ptr(b2), _ptr(dY), _ptr(dX), _ptr(dW1),
                _ptr(db1), _ptr(dW2), _ptr(db2), _ptr(workspace), int(workspace_bytes), _stream_ptr(stream))
    if check and st != OSDP_OK:
        raise OsdpError(st, where)
    return st


def osdp_split_mlp_forward(desc, X, W1, b1, W2, b2, Y, workspace, workspace_bytes=None, stream=None, check=True):
    """Enqueue the split forward.  Tensors are torch CUDA tensors (or raw device addresses)."""
    return _call_fwd(_lib.osdp_split_mlp_forward, "osdp_split_mlp_forward", desc, X, W1, b1, W2, b2, Y, workspace,
                     workspace_bytes, stream, check)


def osdp_split_mlp_backward(desc, X, W1, b1, W2, b2, dY, dX, dW1, db1, dW2, db2, workspace, workspace_bytes=None,
                            stream=None, check=True):
    return _call_bwd(_lib.osdp_split_mlp_backward, "osdp_split_mlp_backward", desc, X, W1, b1, W2, b2, dY, dX, dW1, db1,
                     dW2, db2, workspace, workspace_bytes, stream, check)


def osdp_ffn_split_mlp_workspace_bytes(desc: osdp_mlp_desc, pass_: int) -> int:
    return int(_lib.osdp_ffn_split_mlp_workspace_bytes(C.byref(desc), int(pass_)))


def osdp_ffn_split_mlp_forward(desc, X, W1, b1, W2, b2, Y, workspace, workspace_bytes=None, stream=None, check=True):
    return _call_fwd(_lib.osdp_ffn_split_mlp_forward, "osdp_ffn_split_mlp_forward", desc, X, W1, b1, W2, b2, Y,
                     workspace, workspace_bytes, stream, check)


def osdp_ffn_split_mlp_backward(desc, X, W1, b1, W2, b2, dY, dX, dW1, db1, dW2, db2, workspace, workspace_bytes=None,
                                stream=None, check=True):
    return _call_bwd(_lib.osdp_ffn_split_mlp_backward, "osdp_ffn_split_mlp_backward", desc, X, W1, b1, W2, b2, dY, dX,
                     dW1, db1, dW2, db2, workspace, workspace_bytes, stream, check)


def osdp_ffn_split_mlp_op_cost(desc: osdp_mlp_desc, pass_: int) -> osdp_op_cost:
    out = osdp_op_cost()
    st = _lib.osdp_ffn_split_mlp_op_cost(C.byref(desc), pass_, C.byref(out))
    if st != OSDP_OK:
        raise OsdpError(st, "osdp_ffn_split_mlp_op_cost")
    return out


# ------------------------------------------------------------------------------------- Linear operator
def make_linear_desc(tokens, in_features, out_features, dtype, k, axis=OSDP_SPLIT_TOKENS, has_bias=True) -> osdp_linear_desc:
    code = dtype if isinstance(dtype, int) else _dtype_code(dtype)
    return osdp_linear_desc(int(tokens), int(in_features), int(out_features), int(code), int(k), int(axis),
                            1 if has_bias else 0)


def osdp_split_linear_workspace_bytes(desc: osdp_linear_desc, pass_: int, check=True) -> int:
    out = C.c_size_t()
    st = _lib.osdp_split_linear_workspace_bytes(C.byref(desc), int(pass_), C.byref(out))
    if st != OSDP_OK:
        if check:
            raise OsdpError(st, "osdp_split_linear_workspace_bytes")
        return -st
    return int(out.value)


def _validate_linear(desc, spec, workspace, workspace_bytes):
    T, i, o = desc.tokens, desc.in_features, desc.out_features
    st = _TORCH_DTYPE.get(desc.dtype)
    numel = {"X": T * i, "dX": T * i, "Y": T * o, "dY": T * o, "W": i * o, "dW": i * o, "b": o, "db": o}
    dev = None
    for name, t in spec:
        if t is None or isinstance(t, int):
            continue
        want = torch.float32 if name in ("dW", "db") else st
        if not t.is_cuda or not t.is_contiguous():
            return None, OSDP_ERR_ARG, f"{name} must be a dense CUDA tensor"
        if want is not None and t.dtype != want:
            return None, OSDP_ERR_DTYPE, f"{name} has dtype {t.dtype}, descriptor needs {want}"
        if t.numel() != numel[name]:
            return None, OSDP_ERR_SHAPE, f"{name} has {t.numel()} elements, descriptor needs {numel[name]}"
        if dev is not None and t.device != dev:
            return None, OSDP_ERR_ARG, f"{name} is on {t.device}, other tensors on {dev}"
        dev = t.device
    if workspace is not None and not isinstance(workspace, int):
        if not workspace.is_cuda or (dev is not None and workspace.device != dev):
            return None, OSDP_ERR_WORKSPACE, "workspace must be a CUDA tensor on the tensors' device"
        if workspace_bytes > workspace.numel() * workspace.element_size():
            return None, OSDP_ERR_WORKSPACE, "workspace_bytes exceeds the workspace tensor"
    return dev, OSDP_OK, ""


def osdp_split_linear_forward(desc, X, W, b, Y, workspace=None, workspace_bytes=None, stream=None, check=True):
    if workspace_bytes is None:
        workspace_bytes = 0 if workspace is None else workspace.numel() * workspace.element_size()
    dev, vs, detail = _validate_linear(desc, (("X", X), ("W", W), ("b", b), ("Y", Y)), workspace, int(workspace_bytes))
    if vs != OSDP_OK:
        if check:
            raise OsdpError(vs, "osdp_split_linear_forward", detail)
        return vs
    with _on_device(dev):
        st = _lib.osdp_split_linear_forward(C.byref(desc), _ptr(X), _ptr(W), _ptr(b), _ptr(Y), _ptr(workspace),
                                            int(workspace_bytes), _stream_ptr(stream))
    if check and st != OSDP_OK:
        raise OsdpError(st, "osdp_split_linear_forward")
    return st


def osdp_split_linear_backward(desc, X, W, dY, dX, dW, db, workspace=None, workspace_bytes=None, stream=None, check=True):
    if workspace_bytes is None:
        workspace_bytes = 0 if workspace is None else workspace.numel() * workspace.element_size()
    dev, vs, detail = _validate_linear(desc, (("X", X), ("W", W), ("dY", dY), ("dX", dX), ("dW", dW), ("db", db)),
                                       workspace, int(workspace_bytes))
    if vs != OSDP_OK:
        if check:
            raise OsdpError(vs, "osdp_split_linear_backward", detail)
        return vs
    with _on_device(dev):
        st = _lib.osdp_split_linear_backward(C.byref(desc), _ptr(X), _ptr(W), _ptr(dY), _ptr(dX), _ptr(dW), _ptr(db),
                                             _ptr(workspace), int(workspace_bytes), _stream_ptr(stream))
    if check and st != OSDP_OK:
        raise OsdpError(st, "osdp_split_linear_backward")
    return st


def osdp_bias_grad_static(dY, db, stream=None, check=True) -> int:
    """db = column sums of dY ([rows x cols] bf16 / fp32 -> [cols] fp32) WITHOUT a workspace: the entry point for
    callers that cannot allocate device memory where they need the bias gradient (code running inside another
    library's callback or allocator hook, a device whose memory belongs to a pool the caller may not draw from, a host
    that is only handed the input and output pointers).  The partial sums go to a 2 MiB static array inside the library
    instead, so cols <= OSDP_BIAS_GRAD_STATIC_MAX_COLS (else OSDP_ERR_STATIC_LIMIT), the first call on a device should
    come before any stream capture (it looks the array's address up), and calls that overlap on one GPU race on that
    array - keep them on one stream or order them.  Same bits as the db2 of osdp_split_mlp_backward.  This wrapper only
    marshals: dY and db are dense CUDA tensors the caller already owns."""
    where = "osdp_bias_grad_static"
    vs, detail = OSDP_OK, ""
    if not (isinstance(dY, torch.Tensor) and isinstance(db, torch.Tensor) and dY.is_cuda and db.is_cuda):
        vs, detail = OSDP_ERR_ARG, "dY and db must be CUDA tensors"
    elif dY.dim() != 2 or not dY.is_contiguous() or not db.is_contiguous():
        vs, detail = OSDP_ERR_ARG, "dY must be a dense [rows x cols] tensor, db dense"
    elif db.dtype != torch.float32 or db.numel() != dY.shape[1]:
        vs, detail = OSDP_ERR_SHAPE, "db must hold cols fp32 values"
    elif db.device != dY.device:
        vs, detail = OSDP_ERR_ARG, f"db is on {db.device}, dY on {dY.device}"
    if vs != OSDP_OK:
        if check:
            raise OsdpError(vs, where, detail)
        return vs
    with _on_device(dY.device):
        st = _lib.osdp_bias_grad_static(_ptr(dY), int(dY.shape[0]), int(dY.shape[1]), _dtype_code(dY.dtype), _ptr(db),
                                        _stream_ptr(stream))
    if check and st != OSDP_OK:
        raise OsdpError(st, where)
    return st


def osdp_linear_op_cost(desc: osdp_linear_desc, pass_: int) -> osdp_op_cost:
    out = osdp_op_cost()
    st = _lib.osdp_linear_op_cost(C.byref(desc), pass_, C.byref(out))
    if st != OSDP_OK:
        raise OsdpError(st, "osdp_linear_op_cost")
    return out


class SplitLinear:
    """Descriptor + caller-owned workspace for repeated calls of the split Linear operator (marshalling only)."""

    def __init__(self, tokens, in_features, out_features, dtype: torch.dtype, k: int, axis="contraction", has_bias=True,
                 device="cuda"):
        ax = {"tokens": OSDP_SPLIT_TOKENS, "contraction": OSDP_SPLIT_CONTRACTION}[axis]
        self.desc = make_linear_desc(tokens, in_features, out_features, dtype, k, ax, has_bias)
        self.dtype, self.device = dtype, torch.device(device)
        n = max(osdp_split_linear_workspace_bytes(self.desc, OSDP_FWD), osdp_split_linear_workspace_bytes(self.desc, OSDP_BWD))
        self.workspace = torch.empty(max(n, 256), dtype=torch.uint8, device=self.device)

    def forward(self, X, W, b, Y=None, stream=None):
        if Y is None:
            Y = torch.empty((self.desc.tokens, self.desc.out_features), dtype=self.dtype, device=X.device)
        osdp_split_linear_forward(self.desc, X, W, b, Y, self.workspace, stream=stream)
        return Y

    def backward(self, X, W, dY, out=None, stream=None):
        if out is None:
            out = dict(dX=torch.empty_like(X), dW=torch.empty(W.shape, dtype=torch.float32, device=X.device),
                       db=torch.empty(W.shape[1], dtype=torch.float32, device=X.device) if self.desc.has_bias else None)
        osdp_split_linear_backward(self.desc, X, W, dY, out["dX"], out["dW"], out["db"], self.workspace, stream=stream)
        return out


# ------------------------------------------------------------------ ZDP mode with weight-slice gathering
def make_zdp_desc(tokens, hidden, ffn, dtype, k, world, rank) -> osdp_zdp_desc:
    return osdp_zdp_desc(make_desc(tokens, hidden, ffn, dtype, k), int(world), int(rank))


def osdp_zdp_shard_elems(desc: osdp_zdp_desc) -> int:
    out = C.c_int64()
    st = _lib.osdp_zdp_shard_elems(C.byref(desc), C.byref(out))
    if st != OSDP_OK:
        raise OsdpError(st, "osdp_zdp_shard_elems")
    return int(out.value)


def osdp_zdp_slice_layout(desc: osdp_zdp_desc, s: int) -> osdp_zdp_slice:
    out = osdp_zdp_slice()
    st = _lib.osdp_zdp_slice_layout(C.byref(desc), int(s), C.byref(out))
    if st != OSDP_OK:
        raise OsdpError(st, "osdp_zdp_slice_layout")
    return out


def osdp_zdp_schedule(desc: osdp_zdp_desc, pass_: int):
    """[(op, slice, buffer, on_comm_stream, bytes_per_rank)] in enqueue order."""
    n = int(_lib.osdp_zdp_schedule(C.byref(desc), int(pass_), 0, None))
    if n < 0:
        raise OsdpError(-n, "osdp_zdp_schedule")
    arr = (osdp_zdp_step * n)()
    _lib.osdp_zdp_schedule(C.byref(desc), int(pass_), n, arr)
    return [(a.op, a.slice, a.buffer, a.on_comm_stream, int(a.bytes_per_rank)) for a in arr]


def osdp_zdp_ffn_split_mlp_workspace_bytes(desc: osdp_zdp_desc, pass_: int) -> int:
    out = C.c_size_t()
    st = _lib.osdp_zdp_ffn_split_mlp_workspace_bytes(C.byref(desc), int(pass_), C.byref(out))
    if st != OSDP_OK:
        raise OsdpError(st, "osdp_zdp_ffn_split_mlp_workspace_bytes")
    return int(out.value)


def osdp_zdp_ffn_split_mlp_op_cost(desc: osdp_zdp_desc, pass_: int) -> osdp_op_cost:
    out = osdp_op_cost()
    st = _lib.osdp_zdp_ffn_split_mlp_op_cost(C.byref(desc), int(pass_), C.byref(out))
    if st != OSDP_OK:
        raise OsdpError(st, "osdp_zdp_ffn_split_mlp_op_cost")
    return out


def zdp_shard(desc: osdp_zdp_desc, W1, b1, W2, b2, rank=None):
    """Rank `rank`'s dense shard (1-D tensor, dtype of W1) of the whole tensors, in the layout osdp_zdp_slice_layout
    describes.  Pure data movement; also maps whole fp32 gradients to a gradient shard."""
    d = osdp_zdp_desc(desc.mlp, desc.world, desc.rank if rank is None else int(rank))
    N, r, h, k = d.world, d.rank, d.mlp.hidden, d.mlp.k
    out = torch.empty(osdp_zdp_shard_elems(d), dtype=W1.dtype, device=W1.device)
    for s in range(k):
        sl = osdp_zdp_slice_layout(d, s)
        fs = sl.hi - sl.lo
        out[sl.w1_off:sl.w1_off + sl.w1_elems] = W1[r * h // N:(r + 1) * h // N, sl.lo:sl.hi].reshape(-1)
        out[sl.b1_off:sl.b1_off + sl.b1_elems] = b1[sl.lo + r * fs // N:sl.lo + (r + 1) * fs // N]
        out[sl.w2_off:sl.w2_off + sl.w2_elems] = W2[sl.lo + r * fs // N:sl.lo + (r + 1) * fs // N, :].reshape(-1)
    sl = osdp_zdp_slice_layout(d, k)
    out[sl.b1_off:sl.b1_off + sl.b1_elems] = b2[r * h // N:(r + 1) * h // N]
    return out


def zdp_unshard(desc: osdp_zdp_desc, shards):
    """Inverse of zdp_shard over the list of every rank's shard: (W1, b1, W2, b2)-shaped whole tensors."""
    N, h, f, k = desc.world, desc.mlp.hidden, desc.mlp.ffn, desc.mlp.k
    t = shards[0]
    W1, b1 = torch.empty((h, f), dtype=t.dtype, device=t.device), torch.empty(f, dtype=t.dtype, device=t.device)
    W2, b2 = torch.empty((f, h), dtype=t.dtype, device=t.device), torch.empty(h, dtype=t.dtype, device=t.device)
    for r, sh in enumerate(shards):
        d = osdp_zdp_desc(desc.mlp, N, r)
        for s in range(k):
            sl = osdp_zdp_slice_layout(d, s)
            fs = sl.hi - sl.lo
            W1[r * h // N:(r + 1) * h // N, sl.lo:sl.hi] = sh[sl.w1_off:sl.w1_off + sl.w1_elems].reshape(h // N, fs)
            b1[sl.lo + r * fs // N:sl.lo + (r + 1) * fs // N] = sh[sl.b1_off:sl.b1_off + sl.b1_elems]
            W2[sl.lo + r * fs // N:sl.lo + (r + 1) * fs // N, :] = sh[sl.w2_off:sl.w2_off + sl.w2_elems].reshape(fs // N, h)
        sl = osdp_zdp_slice_layout(d, k)
        b2[r * h // N:(r + 1) * h // N] = sh[sl.b1_off:sl.b1_off + sl.b1_elems]
    return W1, b1, W2, b2


class _DevMem:
    """A raw device range as a __cuda_array_interface__ object (so torch can wrap it without a copy)."""

    def __init__(self, ptr, nbytes, typestr):
        item = 4 if typestr == "<f4" else 1
        self.__cuda_array_interface__ = {"shape": (nbytes // item,), "typestr": typestr, "data": (int(ptr), False),
                                         "version": 2}


class TorchDistComm:
    """osdp_comm over torch.distributed (NCCL: ring / NVSwitch collectives over NVLink): the two collectives the paper
    names.  The callbacks wrap the raw device ranges the library passes and enqueue the collective on the
    stream it names.  Argument marshalling only."""

    def __init__(self, group=None):
        import torch.distributed as dist
        self.dist, self.group = dist, group
        self.world = dist.get_world_size(group)
        self._ag = ALL_GATHER_FN(self._all_gather)
        self._rs = REDUCE_SCATTER_FN(self._reduce_scatter)
        self.struct = osdp_comm(None, self._ag, self._rs)
        self.error = None

    def _all_gather(self, ctx, send, recv, nbytes, stream):
        try:
            s = torch.as_tensor(_DevMem(send, nbytes, "|u1"), device="cuda")
            r = torch.as_tensor(_DevMem(recv, nbytes * self.world, "|u1"), device="cuda")
            with torch.cuda.stream(torch.cuda.ExternalStream(int(stream or 0))):
                self.dist.all_gather_into_tensor(r, s, group=self.group)
            return 0
        except Exception as e:      # a Python exception must not unwind through C
            self.error = e
            return 1

    def _reduce_scatter(self, ctx, send, recv, nfloats, stream):
        try:
            s = torch.as_tensor(_DevMem(send, nfloats * 4 * self.world, "<f4"), device="cuda")
            r = torch.as_tensor(_DevMem(recv, nfloats * 4, "<f4"), device="cuda")
            with torch.cuda.stream(torch.cuda.ExternalStream(int(stream or 0))):
                self.dist.reduce_scatter_tensor(r, s, group=self.group)
            return 0
        except Exception as e:
            self.error = e
            return 1


def _validate_zdp(desc, spec, workspace):
    """Marshalling checks for the ZDP calls, as _validate does for the others: dense CUDA tensors of the dtype and element
    count the descriptor implies, all on one device (returned, so the call runs with it current).  Raw integer addresses
    are taken on trust.  Returns (device, status, detail)."""
    T, h = desc.mlp.tokens, desc.mlp.hidden
    st = _TORCH_DTYPE.get(desc.mlp.dtype)
    try:
        shard = osdp_zdp_shard_elems(desc)
    except OsdpError as e:
        return None, e.status, "invalid ZDP descriptor"
    numel = {"param_shard": shard, "grad_shard": shard, "X": T * h, "Y": T * h, "dY": T * h, "dX": T * h}
    dev = None
    for name, t in spec:
        if t is None or isinstance(t, int):
            continue
        if not isinstance(t, torch.Tensor) or not t.is_cuda:
            return None, OSDP_ERR_ARG, f"{name} is not a CUDA tensor"
        if not t.is_contiguous():
            return None, OSDP_ERR_ARG, f"{name} is not dense row-major"
        want = torch.float32 if name == "grad_shard" else st
        if t.dtype != want:
            return None, OSDP_ERR_DTYPE, f"{name} has dtype {t.dtype}, descriptor needs {want}"
        if t.numel() != numel[name]:
            return None, OSDP_ERR_SHAPE, f"{name} has {t.numel()} elements, descriptor needs {numel[name]}"
        if dev is not None and t.device != dev:
            return None, OSDP_ERR_ARG, f"{name} is on {t.device}, other tensors on {dev}"
        dev = t.device
    if isinstance(workspace, torch.Tensor):
        if not workspace.is_cuda or not workspace.is_contiguous():
            return None, OSDP_ERR_WORKSPACE, "workspace must be a dense CUDA tensor"
        if dev is not None and workspace.device != dev:
            return None, OSDP_ERR_ARG, f"workspace is on {workspace.device}, tensors on {dev}"
    return dev, OSDP_OK, ""


def osdp_zdp_ffn_split_mlp_forward(desc, param_shard, X, Y, workspace, comm=None, compute_stream=None, comm_stream=None,
                                   check=True):
    where = "osdp_zdp_ffn_split_mlp_forward"
    dev, vs, detail = _validate_zdp(desc, (("param_shard", param_shard), ("X", X), ("Y", Y)), workspace)
    if vs != OSDP_OK:
        if check:
            raise OsdpError(vs, where, detail)
        return vs
    with _on_device(dev):
        cs = _stream_ptr(compute_stream)
        ms = cs if comm_stream is None else _stream_ptr(comm_stream)
        st = _lib.osdp_zdp_ffn_split_mlp_forward(C.byref(desc), _ptr(param_shard), _ptr(X), _ptr(Y), _ptr(workspace),
                                                 0 if workspace is None else workspace.numel() * workspace.element_size(),
                                                 C.byref(comm.struct) if comm is not None else None, cs, ms)
    if check and st != OSDP_OK:
        raise OsdpError(st, where, str(getattr(comm, "error", "") or ""))
    return st


def osdp_zdp_ffn_split_mlp_backward(desc, param_shard, X, dY, dX, grad_shard, workspace, comm=None, compute_stream=None,
                                    comm_stream=None, check=True):
    where = "osdp_zdp_ffn_split_mlp_backward"
    dev, vs, detail = _validate_zdp(desc, (("param_shard", param_shard), ("X", X), ("dY", dY), ("dX", dX),
                                           ("grad_shard", grad_shard)), workspace)
    if vs != OSDP_OK:
        if check:
            raise OsdpError(vs, where, detail)
        return vs
    with _on_device(dev):
        cs = _stream_ptr(compute_stream)
        ms = cs if comm_stream is None else _stream_ptr(comm_stream)
        st = _lib.osdp_zdp_ffn_split_mlp_backward(C.byref(desc), _ptr(param_shard), _ptr(X), _ptr(dY), _ptr(dX),
                                                  _ptr(grad_shard), _ptr(workspace),
                                                  0 if workspace is None else workspace.numel() * workspace.element_size(),
                                                  C.byref(comm.struct) if comm is not None else None, cs, ms)
    if check and st != OSDP_OK:
        raise OsdpError(st, where, str(getattr(comm, "error", "") or ""))
    return st


# ---------------------------------------------------------------------------------------------- planner
def osdp_cost_eval(op: osdp_op_cost, mode: int, k: int, batch: int, dev: osdp_device):
    p, t, s = C.c_uint64(), C.c_uint64(), C.c_double()
    st = _lib.osdp_cost_eval(C.byref(op), mode, k, batch, C.byref(dev), C.byref(p), C.byref(t), C.byref(s))
    if st != OSDP_OK:
        raise OsdpError(st, "osdp_cost_eval")
    return int(p.value), int(t.value), float(s.value)


def osdp_mlp_op_cost(desc: osdp_mlp_desc, pass_: int) -> osdp_op_cost:
    out = osdp_op_cost()
    st = _lib.osdp_mlp_op_cost(C.byref(desc), pass_, C.byref(out))
    if st != OSDP_OK:
        raise OsdpError(st, "osdp_mlp_op_cost")
    return out


def _op_array(ops):
    arr = (osdp_op_cost * len(ops))()
    for i, o in enumerate(ops):
        arr[i] = o
    return arr


def osdp_plan(ops, dev: osdp_device, batch: int, k_candidates, check=True):
    """Returns (status, ks, modes, est_seconds, est_peak_bytes)."""
    n = len(ops)
    cand = (C.c_int32 * len(k_candidates))(*k_candidates)
    ks, modes = (C.c_int32 * n)(), (C.c_int32 * n)()
    sec, peak = C.c_double(), C.c_uint64()
    st = _lib.osdp_plan(_op_array(ops), n, C.byref(dev), batch, cand, len(k_candidates), ks, modes, C.byref(sec),
                        C.byref(peak))
    if check and st not in (OSDP_OK, OSDP_ERR_INFEASIBLE):
        raise OsdpError(st, "osdp_plan")
    if st != OSDP_OK:
        return st, None, None, None, None
    return st, list(ks), list(modes), float(sec.value), int(peak.value)


def osdp_cost_eval_mixed(op: osdp_op_cost, k: int, zdp_slices: int, batch: int, dev: osdp_device, check=True):
    """(persist_bytes, transient_bytes, seconds) of an operator with zdp_slices of its k slices in ZDP mode."""
    p, t, s = C.c_uint64(), C.c_uint64(), C.c_double()
    st = _lib.osdp_cost_eval_mixed(C.byref(op), k, zdp_slices, batch, C.byref(dev), C.byref(p), C.byref(t), C.byref(s))
    if st != OSDP_OK:
        if check:
            raise OsdpError(st, "osdp_cost_eval_mixed")
        return st
    return int(p.value), int(t.value), float(s.value)


def osdp_plan_mixed(ops, dev: osdp_device, batch: int, k_candidates, check=True):
    """Returns (status, ks, zdp_slices, est_seconds, est_peak_bytes)."""
    n = len(ops)
    cand = (C.c_int32 * len(k_candidates))(*k_candidates)
    ks, zs = (C.c_int32 * n)(), (C.c_int32 * n)()
    sec, peak = C.c_double(), C.c_uint64()
    st = _lib.osdp_plan_mixed(_op_array(ops), n, C.byref(dev), batch, cand, len(k_candidates), ks, zs, C.byref(sec),
                              C.byref(peak))
    if check and st not in (OSDP_OK, OSDP_ERR_INFEASIBLE):
        raise OsdpError(st, "osdp_plan_mixed")
    if st != OSDP_OK:
        return st, None, None, None, None
    return st, list(ks), list(zs), float(sec.value), int(peak.value)


def osdp_plan_batch(ops, dev: osdp_device, batch_max: int, k_candidates, check=True):
    """Returns (status, ks, modes, batch, est_seconds, est_peak_bytes)."""
    n = len(ops)
    cand = (C.c_int32 * len(k_candidates))(*k_candidates)
    ks, modes = (C.c_int32 * n)(), (C.c_int32 * n)()
    sec, peak, b = C.c_double(), C.c_uint64(), C.c_int64()
    st = _lib.osdp_plan_batch(_op_array(ops), n, C.byref(dev), batch_max, cand, len(k_candidates), ks, modes,
                              C.byref(b), C.byref(sec), C.byref(peak))
    if check and st not in (OSDP_OK, OSDP_ERR_INFEASIBLE):
        raise OsdpError(st, "osdp_plan_batch")
    if st != OSDP_OK:
        return st, None, None, None, None, None
    return st, list(ks), list(modes), int(b.value), float(sec.value), int(peak.value)


# ------------------------------------------------------------------------------ convenience (marshalling only)
class SplitMlp:
    """Holds a descriptor and caller-owned workspace/outputs for repeated calls on one device."""

    def __init__(self, tokens, hidden, ffn, dtype: torch.dtype, k: int, device="cuda", axis="tokens"):
        """axis = "tokens" (osdp_split_mlp_*) or "ffn" (osdp_ffn_split_mlp_*, the paper-literal contraction split)."""
        if axis not in ("tokens", "ffn"):
            raise ValueError("axis must be 'tokens' or 'ffn'")
        self.desc = make_desc(tokens, hidden, ffn, dtype, k)
        self.dtype, self.device, self.axis = dtype, torch.device(device), axis
        ws = osdp_split_mlp_workspace_bytes if axis == "tokens" else osdp_ffn_split_mlp_workspace_bytes
        self._fwd = osdp_split_mlp_forward if axis == "tokens" else osdp_ffn_split_mlp_forward
        self._bwd = osdp_split_mlp_backward if axis == "tokens" else osdp_ffn_split_mlp_backward
        self.ws_fwd_bytes = ws(self.desc, OSDP_FWD)
        self.ws_bwd_bytes = ws(self.desc, OSDP_BWD)
        if self.ws_fwd_bytes == 0:
            raise OsdpError(OSDP_ERR_SHAPE, "SplitMlp: invalid descriptor")
        self.workspace = torch.empty(max(self.ws_fwd_bytes, self.ws_bwd_bytes), dtype=torch.uint8, device=self.device)

    def forward(self, X, W1, b1, W2, b2, Y=None, stream=None):
        if Y is None:
            Y = torch.empty_like(X)
        self._fwd(self.desc, X, W1, b1, W2, b2, Y, self.workspace, stream=stream)
        return Y

    def backward(self, X, W1, b1, W2, dY, out=None, stream=None):
        if out is None:
            out = dict(dX=torch.empty_like(X),
                       dW1=torch.empty(W1.shape, dtype=torch.float32, device=X.device),
                       db1=torch.empty(b1.shape, dtype=torch.float32, device=X.device),
                       dW2=torch.empty(W2.shape, dtype=torch.float32, device=X.device),
                       db2=torch.empty(W2.shape[1], dtype=torch.float32, device=X.device))
        self._bwd(self.desc, X, W1, b1, W2, None, dY, out["dX"], out["dW1"], out["db1"], out["dW2"],
                  out["db2"], self.workspace, stream=stream)
        return out

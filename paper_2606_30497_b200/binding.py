"""Thin ctypes binding of libmlp_b200.so -- same names as include/mlp.h, argument marshalling only.

Every step of the path runs in the library's CUDA kernels; torch is used for device memory and
streams.  There is NO CPU fallback: if the extension is missing or a call fails this module
raises (it never routes through oracle/).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmlp_b200.so")

MLP_OK = 0
VARIANT_FUSED = 0
VARIANT_UNFUSED = 1
VARIANT_TF32 = 2
VARIANT_PRIOR_NAIVE = 3
VARIANT_PRIOR_TILED = 4
VARIANT_BF16 = 5
VARIANT_TF32X3 = 6

EXPORTS = [
    "mlp_init", "mlp_init_weights", "mlp_train", "mlp_train_ex", "mlp_eval_loss",
    "mlp_eval_loss_async", "mlp_eval_loss_static", "mlp_eval_loss_ws", "mlp_eval_workspace_bytes", "mlp_train_host", "mlp_fit_host",
    "mlp_eval_loss_host", "mlp_set_cluster", "mlp_train_rows", "mlp_get_cluster", "mlp_get_cluster_for",
    "mlp_get_train_stats", "mlp_train_order_errors", "mlp_launch_count", "mlp_last_error", "mlp_version",
    "mlp_shutdown",
]


class MlpError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"mlp error {code}: {msg}")
        self.code = code


_lib = None


def lib():
    """Load libmlp_b200.so (fails loudly if it has not been built)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2606_30497_b200.build` "
                          "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp, i64, i32, f32, f64 = C.c_void_p, C.c_int64, C.c_int, C.c_float, C.c_double
    L.mlp_init.argtypes = [C.c_uint64, i32, i32, i32]; L.mlp_init.restype = i32
    L.mlp_init_weights.argtypes = [vp, vp, vp]; L.mlp_init_weights.restype = i32
    L.mlp_train.argtypes = [vp, vp, i64, i32, f32, i32, vp, vp, vp]; L.mlp_train.restype = i32
    L.mlp_train_ex.argtypes = [vp, vp, i64, i32, f32, i32, vp, vp, vp, i32, vp]
    L.mlp_train_ex.restype = i32
    L.mlp_train_rows.argtypes = [vp, vp, i64, i32, f32, i32, vp, vp, vp, vp]; L.mlp_train_rows.restype = i32
    L.mlp_eval_loss.argtypes = [vp, vp, i64, vp, vp, vp]; L.mlp_eval_loss.restype = f64
    L.mlp_eval_loss_async.argtypes = [vp, vp, i64, vp, vp, vp, i32, vp]
    L.mlp_eval_loss_async.restype = i32
    L.mlp_eval_loss_static.argtypes = [vp, vp, i64, vp, vp, vp, i32, vp]
    L.mlp_eval_loss_static.restype = i32
    L.mlp_eval_loss_ws.argtypes = [vp, vp, i64, vp, vp, vp, i32, vp, C.c_size_t, vp]
    L.mlp_eval_loss_ws.restype = i32
    L.mlp_eval_workspace_bytes.argtypes = []; L.mlp_eval_workspace_bytes.restype = C.c_size_t
    L.mlp_train_host.argtypes = [vp, vp, i64, i32, f32, i32, vp, vp, vp, i32]
    L.mlp_train_host.restype = i32
    L.mlp_fit_host.argtypes = [vp, vp, i64, i32, f32, i32, vp, vp, vp, i32, i32, vp]
    L.mlp_fit_host.restype = i32
    L.mlp_get_cluster_for.argtypes = [i32]; L.mlp_get_cluster_for.restype = i32
    L.mlp_train_order_errors.argtypes = []; L.mlp_train_order_errors.restype = i64
    L.mlp_eval_loss_host.argtypes = [vp, vp, i64, vp, vp, i32]; L.mlp_eval_loss_host.restype = f64
    L.mlp_set_cluster.argtypes = [i32]; L.mlp_set_cluster.restype = i32
    L.mlp_get_cluster.argtypes = []; L.mlp_get_cluster.restype = i32
    L.mlp_get_train_stats.argtypes = [C.POINTER(f64)]; L.mlp_get_train_stats.restype = i32
    L.mlp_launch_count.argtypes = []; L.mlp_launch_count.restype = i64
    L.mlp_last_error.argtypes = []; L.mlp_last_error.restype = C.c_char_p
    L.mlp_version.argtypes = []; L.mlp_version.restype = C.c_char_p
    L.mlp_shutdown.argtypes = []; L.mlp_shutdown.restype = None
    _lib = L
    return L


def _check(rc):
    if rc != MLP_OK:
        raise MlpError(rc, lib().mlp_last_error().decode())


def _stream(stream):
    if stream is None:
        import torch
        return C.c_void_p(torch.cuda.current_stream().cuda_stream)
    return C.c_void_p(getattr(stream, "cuda_stream", stream))


def _dptr(t, dtype_name, what):
    """Device pointer of a contiguous CUDA tensor of the given dtype."""
    import torch
    want = getattr(torch, dtype_name)
    if not (t.is_cuda and t.is_contiguous() and t.dtype == want):
        raise TypeError(f"{what}: need a contiguous CUDA {dtype_name} tensor")
    return C.c_void_p(t.data_ptr())


# ------------------------------------------------------------------ include/mlp.h, 1:1
def mlp_init(seed: int, in_features: int, hidden: int, out: int) -> None:
    _check(lib().mlp_init(seed, in_features, hidden, out))


def mlp_init_weights(W1, W2, stream=None) -> None:
    _check(lib().mlp_init_weights(_dptr(W1, "float32", "W1"), _dptr(W2, "float32", "W2"), _stream(stream)))


def mlp_train(X, Y, n, batch, lr, epochs, W1, W2, stream=None) -> None:
    _check(lib().mlp_train(_dptr(X, "float32", "X"), _dptr(Y, "float32", "Y"), int(n), int(batch),
                           float(lr), int(epochs), _dptr(W1, "float32", "W1"),
                           _dptr(W2, "float32", "W2"), _stream(stream)))


def mlp_train_ex(X, Y, n, batch, lr, epochs, W1, W2, batch_order=None, variant=VARIANT_FUSED,
                 stream=None) -> None:
    op = _dptr(batch_order, "int32", "batch_order") if batch_order is not None else None
    _check(lib().mlp_train_ex(_dptr(X, "float32", "X"), _dptr(Y, "float32", "Y"), int(n), int(batch),
                              float(lr), int(epochs), _dptr(W1, "float32", "W1"),
                              _dptr(W2, "float32", "W2"), op, int(variant), _stream(stream)))


def mlp_train_rows(X, Y, n, batch, lr, epochs, W1, W2, row_order, stream=None) -> None:
    _check(lib().mlp_train_rows(_dptr(X, "float32", "X"), _dptr(Y, "float32", "Y"), int(n), int(batch),
                                float(lr), int(epochs), _dptr(W1, "float32", "W1"),
                                _dptr(W2, "float32", "W2"), _dptr(row_order, "int32", "row_order"),
                                _stream(stream)))


def mlp_eval_loss(X, Y, n, W1, W2, stream=None) -> float:
    v = lib().mlp_eval_loss(_dptr(X, "float32", "X"), _dptr(Y, "float32", "Y"), int(n),
                            _dptr(W1, "float32", "W1"), _dptr(W2, "float32", "W2"), _stream(stream))
    if v != v:
        raise MlpError(-1, lib().mlp_last_error().decode() or "mlp_eval_loss returned NaN")
    return float(v)


def mlp_eval_loss_async(X, Y, n, W1, W2, d_out, variant=VARIANT_FUSED, stream=None) -> None:
    _check(lib().mlp_eval_loss_async(_dptr(X, "float32", "X"), _dptr(Y, "float32", "Y"), int(n),
                                     _dptr(W1, "float32", "W1"), _dptr(W2, "float32", "W2"),
                                     _dptr(d_out, "float64", "d_out"), int(variant), _stream(stream)))


def mlp_eval_loss_static(X, Y, n, W1, W2, d_out, variant=VARIANT_FUSED, stream=None) -> None:
    _check(lib().mlp_eval_loss_static(_dptr(X, "float32", "X"), _dptr(Y, "float32", "Y"), int(n),
                                      _dptr(W1, "float32", "W1"), _dptr(W2, "float32", "W2"),
                                      _dptr(d_out, "float64", "d_out"), int(variant), _stream(stream)))


def mlp_eval_workspace_bytes() -> int:
    return int(lib().mlp_eval_workspace_bytes())


def mlp_eval_loss_ws(X, Y, n, W1, W2, d_out, variant, workspace, stream=None) -> None:
    if not (workspace.is_cuda and workspace.is_contiguous()):
        raise TypeError("workspace: need a contiguous CUDA tensor")
    _check(lib().mlp_eval_loss_ws(_dptr(X, "float32", "X"), _dptr(Y, "float32", "Y"), int(n),
                                  _dptr(W1, "float32", "W1"), _dptr(W2, "float32", "W2"),
                                  _dptr(d_out, "float64", "d_out"), int(variant),
                                  C.c_void_p(workspace.data_ptr()), workspace.numel() * workspace.element_size(),
                                  _stream(stream)))


def _hptr(a, dtype, what):
    """Host pointer of a C-contiguous numpy array or CPU torch tensor (pinned or not)."""
    if isinstance(a, np.ndarray):
        if a.dtype != dtype or not a.flags["C_CONTIGUOUS"]:
            raise TypeError(f"{what}: need a C-contiguous {dtype} array")
        return C.c_void_p(a.ctypes.data)
    if a.is_cuda or not a.is_contiguous():
        raise TypeError(f"{what}: need a contiguous host tensor")
    return C.c_void_p(a.data_ptr())


def mlp_train_host(X, Y, n, batch, lr, epochs, W1, W2, order=None, variant=VARIANT_FUSED) -> None:
    op = _hptr(order, np.int32, "order") if order is not None else None
    _check(lib().mlp_train_host(_hptr(X, np.float32, "X"), _hptr(Y, np.float32, "Y"), int(n),
                                int(batch), float(lr), int(epochs), _hptr(W1, np.float32, "W1"),
                                _hptr(W2, np.float32, "W2"), op, int(variant)))


def mlp_fit_host(X, Y, n, batch, lr, epochs, W1, W2, order=None, variant=VARIANT_FUSED,
                 eval_variant=VARIANT_FUSED, epoch_loss=None) -> None:
    op = _hptr(order, np.int32, "order") if order is not None else None
    lp = _hptr(epoch_loss, np.float64, "epoch_loss") if epoch_loss is not None else None
    _check(lib().mlp_fit_host(_hptr(X, np.float32, "X"), _hptr(Y, np.float32, "Y"), int(n),
                              int(batch), float(lr), int(epochs), _hptr(W1, np.float32, "W1"),
                              _hptr(W2, np.float32, "W2"), op, int(variant), int(eval_variant), lp))


def mlp_eval_loss_host(X, Y, n, W1, W2, variant=VARIANT_FUSED) -> float:
    v = lib().mlp_eval_loss_host(_hptr(X, np.float32, "X"), _hptr(Y, np.float32, "Y"), int(n),
                                 _hptr(W1, np.float32, "W1"), _hptr(W2, np.float32, "W2"), int(variant))
    if v != v:
        raise MlpError(-1, lib().mlp_last_error().decode() or "mlp_eval_loss_host returned NaN")
    return float(v)


def mlp_set_cluster(cluster: int) -> None:
    _check(lib().mlp_set_cluster(int(cluster)))


def mlp_get_cluster(batch=None) -> int:
    return int(lib().mlp_get_cluster() if batch is None else lib().mlp_get_cluster_for(int(batch)))


def mlp_train_order_errors() -> int:
    return int(lib().mlp_train_order_errors())


def mlp_get_train_stats():
    out = (C.c_double * 4)()
    _check(lib().mlp_get_train_stats(out))
    return {"sm_cycles": out[0], "ns": out[1], "steps": out[2], "cluster": out[3]}


def mlp_launch_count() -> int:
    return int(lib().mlp_launch_count())


def mlp_last_error() -> str:
    return lib().mlp_last_error().decode()


def mlp_version() -> str:
    return lib().mlp_version().decode()


def mlp_shutdown() -> None:
    lib().mlp_shutdown()

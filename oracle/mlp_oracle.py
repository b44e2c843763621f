"""ctypes front end of oracle/libmlp_oracle.so -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this module.  It marshals numpy arrays to the plain-C oracle in
oracle/mlp_oracle.c (which restates PAPER.md eqs. 1-9); it holds no
arithmetic of its own and imports nothing from the product package.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        fp = C.POINTER(C.c_float)
        dp = C.POINTER(C.c_double)
        up = C.POINTER(C.c_uint64)
        L.oracle_grads.argtypes = [fp, fp, C.c_int, C.c_int, C.c_int, fp, fp, dp, dp, dp, up]
        L.oracle_grads.restype = None
        L.oracle_grads_f64.argtypes = [fp, fp, C.c_int, C.c_int, C.c_int, dp, dp, dp, dp, dp, up]
        L.oracle_grads_f64.restype = None
        L.oracle_train.argtypes = [fp, fp, C.c_int64, C.c_int, C.c_int, C.c_int, C.c_float,
                                   C.c_int, fp, fp, C.POINTER(C.c_int32), C.c_int, up]
        L.oracle_train.restype = C.c_int64
        L.oracle_eval_loss.argtypes = [fp, fp, C.c_int64, C.c_int, C.c_int, fp, fp]
        L.oracle_eval_loss.restype = C.c_double
        L.oracle_predict_rows.argtypes = [fp, C.POINTER(C.c_int64), C.c_int64, C.c_int, C.c_int,
                                          fp, fp, dp]
        L.oracle_predict_rows.restype = None
        L.oracle_init_weights.argtypes = [C.c_uint64, C.c_int, C.c_int, fp, fp]
        L.oracle_init_weights.restype = None
        L.oracle_num_threads.argtypes = []
        L.oracle_num_threads.restype = C.c_int
        _lib = L
    return _lib


def _f32(a):
    a = np.ascontiguousarray(a, dtype=np.float32)
    return a, a.ctypes.data_as(C.POINTER(C.c_float))


def _f64(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(C.POINTER(C.c_double))


def _dims(X, W1):
    X = np.asarray(X)
    W1 = np.asarray(W1)
    m, I = X.shape
    I2, H = W1.shape
    assert I == I2, (X.shape, W1.shape)
    return m, I, H


def grads(X, Y, W1, W2, count_macs: bool = False):
    """(g1 [I,H], g2 [H], loss) of one batch; fp32 or fp64 weights (dtype of W1 decides)."""
    m, I, H = _dims(X, W1)
    Xc, xp = _f32(X)
    Yc, yp = _f32(np.reshape(Y, -1))
    g1 = np.zeros((I, H), np.float64)
    g2 = np.zeros(H, np.float64)
    loss = C.c_double(0.0)
    macs = np.zeros(5, np.uint64)
    mp = macs.ctypes.data_as(C.POINTER(C.c_uint64)) if count_macs else None
    g1p = g1.ctypes.data_as(C.POINTER(C.c_double))
    g2p = g2.ctypes.data_as(C.POINTER(C.c_double))
    if np.asarray(W1).dtype == np.float64:
        w1, w1p = _f64(W1)
        w2, w2p = _f64(np.reshape(W2, -1))
        lib().oracle_grads_f64(xp, yp, m, I, H, w1p, w2p, g1p, g2p, C.byref(loss), mp)
    else:
        w1, w1p = _f32(W1)
        w2, w2p = _f32(np.reshape(W2, -1))
        lib().oracle_grads(xp, yp, m, I, H, w1p, w2p, g1p, g2p, C.byref(loss), mp)
    if count_macs:
        return g1, g2, loss.value, macs
    return g1, g2, loss.value


def train(X, Y, W1, W2, batch, lr, epochs, order=None, state_fp64=False, count_macs=False):
    """Mini-batch SGD; returns new (W1, W2) fp32 copies (inputs untouched) [+ MAC counters]."""
    n, I, H = _dims(X, W1)
    Xc, xp = _f32(X)
    Yc, yp = _f32(np.reshape(Y, -1))
    w1 = np.array(W1, dtype=np.float32, order="C", copy=True)
    w2 = np.array(np.reshape(W2, -1), dtype=np.float32, order="C", copy=True)
    op = None
    if order is not None:
        oc = np.ascontiguousarray(order, dtype=np.int32).reshape(-1)
        nb = (n + batch - 1) // batch
        assert oc.size == epochs * nb, (oc.size, epochs, nb)
        op = oc.ctypes.data_as(C.POINTER(C.c_int32))
    macs = np.zeros(5, np.uint64)
    mp = macs.ctypes.data_as(C.POINTER(C.c_uint64)) if count_macs else None
    steps = lib().oracle_train(xp, yp, n, I, H, int(batch), C.c_float(float(np.float32(lr))),
                               int(epochs), w1.ctypes.data_as(C.POINTER(C.c_float)),
                               w2.ctypes.data_as(C.POINTER(C.c_float)), op,
                               1 if state_fp64 else 0, mp)
    if steps < 0:
        raise ValueError("oracle_train: bad arguments")
    if count_macs:
        return w1, w2, macs
    return w1, w2


def eval_loss(X, Y, W1, W2) -> float:
    n, I, H = _dims(X, W1)
    Xc, xp = _f32(X)
    Yc, yp = _f32(np.reshape(Y, -1))
    w1, w1p = _f32(W1)
    w2, w2p = _f32(np.reshape(W2, -1))
    return float(lib().oracle_eval_loss(xp, yp, n, I, H, w1p, w2p))


def predict_rows(X, rows, W1, W2):
    n, I, H = _dims(X, W1)
    Xc, xp = _f32(X)
    rc = np.ascontiguousarray(rows, dtype=np.int64)
    w1, w1p = _f32(W1)
    w2, w2p = _f32(np.reshape(W2, -1))
    out = np.zeros(rc.size, np.float64)
    lib().oracle_predict_rows(xp, rc.ctypes.data_as(C.POINTER(C.c_int64)), rc.size, I, H,
                              w1p, w2p, out.ctypes.data_as(C.POINTER(C.c_double)))
    return out


def init_weights(seed: int, in_features: int, hidden: int):
    W1 = np.zeros((in_features, hidden), np.float32)
    W2 = np.zeros(hidden, np.float32)
    lib().oracle_init_weights(C.c_uint64(seed), in_features, hidden,
                              W1.ctypes.data_as(C.POINTER(C.c_float)),
                              W2.ctypes.data_as(C.POINTER(C.c_float)))
    return W1, W2


def num_threads() -> int:
    return int(lib().oracle_num_threads())

"""A second, independent fp64 restatement of PAPER.md eqs. 1-9 in numpy (vectorised).

Used ONLY to cross-check the C oracle (tests/test_oracle_pins.py); it is not the oracle
and shares nothing with it or with the CUDA path.  PAPER.md:44-71.
"""
import numpy as np


def grads(X, Y, W1, W2):
    X = np.asarray(X, np.float64)
    Y = np.asarray(Y, np.float64).reshape(-1, 1)
    W1 = np.asarray(W1, np.float64)
    W2 = np.asarray(W2, np.float64).reshape(-1, 1)
    m = X.shape[0]
    Z1 = X @ W1                                  # eq. 1
    Hh = np.maximum(Z1, 0.0)                     # eq. 2
    Yp = Hh @ W2                                 # eq. 3
    L = float(np.mean((Yp - Y) ** 2))            # eq. 4
    dZ2 = (2.0 / m) * (Yp - Y)                   # eq. 5
    dW2 = Hh.T @ dZ2                             # eq. 6
    dZ1 = (dZ2 @ W2.T) * (Z1 > 0)                # eq. 7
    dW1 = X.T @ dZ1                              # eq. 8
    return dW1, dW2.reshape(-1), L


def train(X, Y, W1, W2, batch, lr, epochs, order=None):
    n = X.shape[0]
    nb = (n + batch - 1) // batch
    a = float(np.float32(lr))
    W1 = np.array(W1, np.float32)
    W2 = np.array(W2, np.float32).reshape(-1)
    for e in range(epochs):
        for k in range(nb):
            t = int(order[e][k]) if order is not None else k
            r0 = t * batch
            xb, yb = X[r0:r0 + batch], Y[r0:r0 + batch]
            g1, g2, _ = grads(xb, yb, W1, W2)
            W1 = (W1.astype(np.float64) - a * g1).astype(np.float32)     # eq. 9
            W2 = (W2.astype(np.float64) - a * g2).astype(np.float32)
    return W1, W2


def eval_loss(X, Y, W1, W2):
    X = np.asarray(X, np.float64)
    yp = np.maximum(X @ np.asarray(W1, np.float64), 0.0) @ np.asarray(W2, np.float64).reshape(-1)
    return float(np.mean((yp - np.asarray(Y, np.float64).reshape(-1)) ** 2))

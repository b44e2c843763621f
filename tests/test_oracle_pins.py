"""Pins of the CPU oracle (oracle/mlp_oracle.c) against what the paper and the mathematics fix.

None of these tests retypes the oracle's formula against itself: each compares it with a
value derived on paper (tests/golden/), a closed form, an invariant, a textbook special
case, a library routine (torch autograd), or brute force.  Pin numbers are SURVEY.md 8(c)'s.
Runs on CPU (`-m "not gpu"`).
"""
import math

import numpy as np
import pytest

from oracle import mlp_oracle as O
from paper_2606_30497_b200 import datagen
import ref_numpy

LR = np.float32(0.002)


# ---------------------------------------------------------------- P0: loop extents
def test_p0_mac_counts_match_paper(golden):
    """2,097,152 / 65,536 / 65,536 / 65,536 / 2,097,152 MACs per batch of 256."""
    g = golden["P0"]
    X, Y, W1, W2 = datagen.small_problem(0, g["batch"], g["I"], g["H"])
    _, _, macs = O.train(X, Y, W1, W2, g["batch"], LR, 1, count_macs=True)
    assert [int(v) for v in macs] == [g["macs_eq1_Z1"], g["macs_eq3_Ypred"], g["macs_eq6_dW2"],
                                      g["macs_eq7_dZ1"], g["macs_eq8_dW1"]]
    assert W1.size + W2.size == g["parameters"]          # PAPER.md:116 (eq. 10)
    assert sum(int(v) for v in macs) == 4390912          # "approximately 4.4 million"


# ---------------------------------------------------------------- P1: hand-worked example
def test_p1_hand_example(golden):
    g = golden["P1"]
    X = np.array(g["X"], np.float32)
    Y = np.array(g["Y"], np.float32)
    W1 = np.array(g["W1"], np.float32)
    W2 = np.array(g["W2"], np.float32)
    g1, g2, L = O.grads(X, Y, W1, W2)
    assert L == g["L"]
    np.testing.assert_array_equal(g1, np.array(g["dW1"], np.float64))
    np.testing.assert_array_equal(g2, np.array(g["dW2"], np.float64))
    assert float((g1 ** 2).sum() + (g2 ** 2).sum()) == g["grad_norm_sq"]
    w1, w2 = O.train(X, Y, W1, W2, 2, g["lr"], 1)
    np.testing.assert_allclose(w1, np.array(g["W1_after"]), rtol=0, atol=2e-7)
    np.testing.assert_allclose(w2, np.array(g["W2_after"]), rtol=0, atol=2e-7)
    assert abs(O.eval_loss(X, Y, w1, w2) - g["L_after"]) < 5e-6
    yp = O.predict_rows(X, [0, 1], w1, w2)
    np.testing.assert_allclose(yp, g["Ypred_after"], atol=2e-6)
    np.testing.assert_array_equal(O.predict_rows(X, [0, 1], W1, W2), np.array(g["Ypred"]))


def test_p1_embedded_in_32_inputs(golden):
    """Zero-padding X to 32 columns / W1 to 32 rows and adding dead hidden units (zero W1
    column, zero W2) must not change anything, and the padding must stay exactly zero."""
    g = golden["P1"]
    I, H = 32, 64
    X = np.zeros((2, I), np.float32); X[:, :2] = g["X"]
    W1 = np.zeros((I, H), np.float32); W1[:2, :4] = g["W1"]
    W2 = np.zeros(H, np.float32); W2[:4] = g["W2"]
    Y = np.array(g["Y"], np.float32)
    w1, w2 = O.train(X, Y, W1, W2, 2, g["lr"], 1)
    np.testing.assert_allclose(w1[:2, :4], np.array(g["W1_after"]), atol=2e-7)
    np.testing.assert_allclose(w2[:4], np.array(g["W2_after"]), atol=2e-7)
    assert not w1[2:, :].any() and not w1[:, 4:].any() and not w2[4:].any()


# ---------------------------------------------------------------- P2: tie at zero
def test_p2_tie_at_zero(golden):
    g1h, g2h = golden["P1"], golden["P2"]
    X = np.array(g2h["X"], np.float32)
    Y = np.array(g2h["Y"], np.float32)
    W1 = np.array(g1h["W1"], np.float32)
    W2 = np.array(g1h["W2"], np.float32)
    g1, g2, L = O.grads(X, Y, W1, W2)
    assert L == g2h["L"]
    np.testing.assert_allclose(3 * g1, np.array(g2h["three_dW1"], np.float64), rtol=1e-15)
    np.testing.assert_allclose(3 * g2, np.array(g2h["three_dW2"], np.float64), rtol=1e-15)


def test_relu_negative_zero_has_zero_gradient():
    X = np.array([[-0.0, 0.0], [1.0, 1.0]], np.float32)
    W1 = np.array([[1.0, -1.0], [1.0, -1.0]], np.float32)
    W2 = np.array([1.0, 1.0], np.float32)
    g1, g2, L = O.grads(X, np.array([1.0, 1.0], np.float32), W1, W2)
    # row 0: z = +-0 -> h = 0, mask 0.  row 1: z = [2,-2] -> h=[2,0]; ypred=2; dz2=(2/2)(2-1)=1
    np.testing.assert_array_equal(g2, [2.0, 0.0])
    np.testing.assert_array_equal(g1, [[1.0, 0.0], [1.0, 0.0]])
    assert L == 1.0                                   # ((0-1)^2 + (2-1)^2)/2


# ---------------------------------------------------------------- P3: finite differences
def _loss64(X, Y, W1, W2):
    return O.grads(X, Y, np.asarray(W1, np.float64), np.asarray(W2, np.float64))[2]


def test_p3_finite_differences():
    rng = np.random.default_rng(11)
    X, Y, W1, W2 = datagen.small_problem(5, 8, 32, 64)
    W1 = W1.astype(np.float64); W2 = W2.astype(np.float64)
    g1, g2, _ = O.grads(X, Y, W1, W2)
    Z = X.astype(np.float64) @ W1
    eps = 1e-6
    safe_cols = np.where(np.abs(Z).min(axis=0) > 1e-4)[0]      # skip kinks
    assert safe_cols.size > 40
    checked = 0
    for _ in range(260):
        i = int(rng.integers(32)); j = int(rng.choice(safe_cols))
        Wp = W1.copy(); Wp[i, j] += eps
        Wm = W1.copy(); Wm[i, j] -= eps
        fd = (_loss64(X, Y, Wp, W2) - _loss64(X, Y, Wm, W2)) / (2 * eps)
        assert abs(fd - g1[i, j]) <= 1e-7 * max(1.0, abs(g1[i, j])), (i, j, fd, g1[i, j])
        checked += 1
    for j in range(64):
        Wp = W2.copy(); Wp[j] += eps
        Wm = W2.copy(); Wm[j] -= eps
        fd = (_loss64(X, Y, W1, Wp) - _loss64(X, Y, W1, Wm)) / (2 * eps)
        assert abs(fd - g2[j]) <= 1e-7 * max(1.0, abs(g2[j])), (j, fd, g2[j])
    assert checked >= 200


# ---------------------------------------------------------------- P4: lr = 0
def test_p4_zero_lr_is_bit_identical():
    X, Y, W1, W2 = datagen.small_problem(7, 1000, 32, 64)
    w1, w2 = O.train(X, Y, W1, W2, 256, 0.0, 3)
    assert w1.tobytes() == W1.tobytes() and w2.tobytes() == W2.tobytes()


# ---------------------------------------------------------------- P5: descent identity
def test_p5_first_order_descent_identity():
    X, Y, W1, W2 = datagen.small_problem(9, 64, 32, 32)
    W1 = W1.astype(np.float64); W2 = W2.astype(np.float64)
    g1, g2, L0 = O.grads(X, Y, W1, W2)
    gn = float((g1 ** 2).sum() + (g2 ** 2).sum())
    ratios = []
    for a in (1e-4, 1e-5, 1e-6):
        La = _loss64(X, Y, W1 - a * g1, W2 - a * g2)
        ratios.append((L0 - La) / a / gn)
    # -> 1 linearly in alpha; a wrong 2/n, sign, or stale-W2 error would give a constant != 1
    assert abs(ratios[0] - 1) < 5e-2 and abs(ratios[1] - 1) < 5e-3 and abs(ratios[2] - 1) < 5e-4
    assert abs(ratios[0] - 1) > abs(ratios[1] - 1) > abs(ratios[2] - 1) * 0.999


def test_p5_step_uses_gradient_at_old_weights():
    """One oracle_train step == W - lr * oracle gradient at the ORIGINAL (W1, W2)
    (eq. 7 must see the pre-update W2)."""
    X, Y, W1, W2 = datagen.small_problem(10, 256, 32, 256)
    g1, g2, _ = O.grads(X, Y, W1, W2)
    w1, w2 = O.train(X, Y, W1, W2, 256, LR, 1)
    a = float(LR)
    np.testing.assert_array_equal(w1, (W1.astype(np.float64) - a * g1).astype(np.float32))
    np.testing.assert_array_equal(w2, (W2.astype(np.float64) - a * g2).astype(np.float32))


# ---------------------------------------------------------------- P6: linear regime
def test_p6_linear_regime_closed_form():
    r = np.random.default_rng(3)
    m, I, H = 40, 32, 48
    X = np.abs(r.standard_normal((m, I))).astype(np.float32)
    W1 = np.abs(r.standard_normal((I, H)) * 0.2).astype(np.float32) + np.float32(0.01)
    W2 = (r.standard_normal(H) * 0.2).astype(np.float32)
    Y = r.standard_normal(m).astype(np.float32)
    Xd, W1d, W2d, Yd = (a.astype(np.float64) for a in (X, W1, W2, Y))
    A = Xd @ W1d                                     # all >= 0 -> no mask, plain least squares
    res = A @ W2d - Yd
    g2_ref = (2.0 / m) * A.T @ res
    g1_ref = (2.0 / m) * Xd.T @ np.outer(res, W2d)
    g1, g2, L = O.grads(X, Y, W1, W2)
    np.testing.assert_allclose(g1, g1_ref, rtol=1e-12, atol=1e-13)
    np.testing.assert_allclose(g2, g2_ref, rtol=1e-12, atol=1e-13)
    assert abs(L - np.mean(res ** 2)) < 1e-12 * max(1, L)


# ---------------------------------------------------------------- P7: dead network
def test_p7_dead_network():
    r = np.random.default_rng(4)
    X = np.abs(r.standard_normal((100, 32))).astype(np.float32)
    W1 = -np.abs(r.standard_normal((32, 64))).astype(np.float32)
    W2 = r.standard_normal(64).astype(np.float32)
    Y = r.standard_normal(100).astype(np.float32)
    g1, g2, L = O.grads(X, Y, W1, W2)
    assert not g1.any() and not g2.any()
    assert abs(L - np.mean(Y.astype(np.float64) ** 2)) < 1e-14
    w1, w2 = O.train(X, Y, W1, W2, 32, 0.5, 2)
    assert w1.tobytes() == W1.tobytes() and w2.tobytes() == W2.tobytes()


# ---------------------------------------------------------------- P8: eval closed forms
def test_p8_eval_closed_forms():
    X, Y = datagen.make_dataset(4096, 0.1)
    r = np.random.default_rng(2)
    W1 = r.standard_normal((32, 64)).astype(np.float32)
    assert abs(O.eval_loss(X, Y, W1, np.zeros(64, np.float32))
               - np.mean(Y.astype(np.float64) ** 2)) < 1e-14          # (i) W2 = 0
    T1, T2 = datagen.teacher()
    X0, Y0 = datagen.make_dataset(4096, 0.0)
    L0 = O.eval_loss(X0, Y0, T1.astype(np.float32), T2.astype(np.float32).reshape(-1))
    assert L0 < 1e-10                                                  # (ii) student == teacher
    Ln = O.eval_loss(X, Y, T1.astype(np.float32), T2.astype(np.float32).reshape(-1))
    s2 = 0.1 ** 2
    assert abs(Ln - s2) < 3 * s2 * math.sqrt(2.0 / 4096) + 1e-6        # ~ sigma^2


# ---------------------------------------------------------------- P9: batch = n
def test_p9_full_batch_step_is_dataset_gradient():
    X, Y, W1, W2 = datagen.small_problem(12, 96, 32, 32)
    W1d, W2d = W1.astype(np.float64), W2.astype(np.float64)
    eps = 1e-6
    w1, w2 = O.train(X, Y, W1, W2, 96, LR, 1)
    # gradient of oracle_eval_loss by central differences on a few coordinates
    Z = X.astype(np.float64) @ W1d
    safe = np.where(np.abs(Z).min(axis=0) > 1e-4)[0]
    r = np.random.default_rng(0)
    for _ in range(20):
        i = int(r.integers(32)); j = int(r.choice(safe))
        Wp = W1d.copy(); Wp[i, j] += eps
        Wm = W1d.copy(); Wm[i, j] -= eps
        fd = (_loss64(X, Y, Wp, W2d) - _loss64(X, Y, Wm, W2d)) / (2 * eps)
        assert abs((W1[i, j] - float(LR) * fd) - w1[i, j]) < 1e-7


# ---------------------------------------------------------------- P10: permutation invariance
def test_p10_row_permutation_invariance():
    X, Y, W1, W2 = datagen.small_problem(13, 200, 32, 64)
    g1, g2, L = O.grads(X, Y, W1, W2)
    p = np.random.default_rng(1).permutation(200)
    h1, h2, Lp = O.grads(X[p], Y[p], W1, W2)
    assert np.abs(g1 - h1).max() <= 1e-14 * np.abs(g1).max()
    assert np.abs(g2 - h2).max() <= 1e-14 * np.abs(g2).max()
    assert abs(L - Lp) <= 1e-14 * L


# ---------------------------------------------------------------- P11: resume equivalence
def test_p11_resume_equivalence():
    X, Y, W1, W2 = datagen.small_problem(14, 700, 32, 64)
    a1, a2 = O.train(X, Y, W1, W2, 256, LR, 2)
    b1, b2 = O.train(X, Y, W1, W2, 256, LR, 1)
    b1, b2 = O.train(X, Y, b1, b2, 256, LR, 1)
    assert a1.tobytes() == b1.tobytes() and a2.tobytes() == b2.tobytes()


def test_order_table_semantics():
    """order[e*nb+k] selects the contiguous batch; a sequential table == no table; a reversed
    table == training on the row-block-reversed dataset (full batches only)."""
    X, Y, W1, W2 = datagen.small_problem(15, 768, 32, 32)
    seq = datagen.make_order(768, 256, 2, shuffle=False)
    a = O.train(X, Y, W1, W2, 256, LR, 2, order=seq)
    b = O.train(X, Y, W1, W2, 256, LR, 2)
    assert a[0].tobytes() == b[0].tobytes() and a[1].tobytes() == b[1].tobytes()
    rev = seq[:, ::-1].copy()
    Xr = np.concatenate([X[512:768], X[256:512], X[0:256]])
    Yr = np.concatenate([Y[512:768], Y[256:512], Y[0:256]])
    c = O.train(X, Y, W1, W2, 256, LR, 2, order=rev)
    d = O.train(Xr, Yr, W1, W2, 256, LR, 2)
    assert c[0].tobytes() == d[0].tobytes() and c[1].tobytes() == d[1].tobytes()


def test_tail_batch_uses_its_own_row_count():
    """n=300, B=256: the 44-row tail batch is a step with 2/44."""
    X, Y, W1, W2 = datagen.small_problem(16, 300, 32, 32)
    a1, a2 = O.train(X, Y, W1, W2, 256, LR, 1)
    b1, b2 = O.train(X[:256], Y[:256], W1, W2, 256, LR, 1)
    b1, b2 = O.train(X[256:], Y[256:], b1, b2, 44, LR, 1)
    assert a1.tobytes() == b1.tobytes() and a2.tobytes() == b2.tobytes()


def test_thread_count_independence():
    import os, subprocess, sys
    code = ("import numpy as np, hashlib;from oracle import mlp_oracle as O;"
            "from paper_2606_30497_b200 import datagen;"
            "X,Y,W1,W2=datagen.small_problem(17,512,32,64);"
            "a,b=O.train(X,Y,W1,W2,128,0.002,2);"
            "print(hashlib.sha1(a.tobytes()+b.tobytes()).hexdigest(), O.eval_loss(X,Y,a,b).hex())")
    outs = []
    for nt in ("1", "3"):
        env = dict(os.environ, OMP_NUM_THREADS=nt)
        outs.append(subprocess.check_output([sys.executable, "-c", code], env=env,
                                            cwd=os.path.dirname(os.path.dirname(__file__))))
    assert outs[0] == outs[1]


# ---------------------------------------------------------------- P12: torch fp64 autograd
def test_p12_torch_autograd():
    import torch
    X, Y, W1, W2 = datagen.small_problem(18, 64, 32, 128)
    g1, g2, L = O.grads(X, Y, W1, W2)
    tx = torch.tensor(X, dtype=torch.float64)
    ty = torch.tensor(Y, dtype=torch.float64).reshape(-1, 1)
    w1 = torch.tensor(W1, dtype=torch.float64, requires_grad=True)
    w2 = torch.tensor(W2, dtype=torch.float64).reshape(-1, 1).requires_grad_(True)
    loss = torch.nn.functional.mse_loss(torch.relu(tx @ w1) @ w2, ty)
    loss.backward()
    assert abs(loss.item() - L) < 1e-13 * max(1.0, L)
    np.testing.assert_allclose(g1, w1.grad.numpy(), rtol=1e-11, atol=1e-13)
    np.testing.assert_allclose(g2, w2.grad.numpy().reshape(-1), rtol=1e-11, atol=1e-13)


def test_p12_torch_training_run():
    import torch
    X, Y, W1, W2 = datagen.small_problem(19, 640, 32, 64)
    w1o, w2o = O.train(X, Y, W1, W2, 256, LR, 3)
    tx = torch.tensor(X, dtype=torch.float64); ty = torch.tensor(Y, dtype=torch.float64).reshape(-1, 1)
    w1 = torch.tensor(W1); w2 = torch.tensor(W2).reshape(-1, 1)
    a = float(LR)
    for _ in range(3):
        for r0 in range(0, 640, 256):
            p1 = w1.double().requires_grad_(True); p2 = w2.double().requires_grad_(True)
            torch.nn.functional.mse_loss(torch.relu(tx[r0:r0 + 256] @ p1) @ p2, ty[r0:r0 + 256]).backward()
            w1 = (p1.detach() - a * p1.grad).float(); w2 = (p2.detach() - a * p2.grad).float()
    # identical up to fp64 summation order before the fp32 rounding: allow 1 ulp flips
    np.testing.assert_allclose(w1o, w1.numpy(), rtol=0, atol=1e-7)
    np.testing.assert_allclose(w2o, w2.numpy().reshape(-1), rtol=0, atol=1e-7)


# ---------------------------------------------------------------- P13: brute force
def test_p13_brute_force_tiny():
    X, Y, W1, W2 = datagen.small_problem(20, 4, 3, 5)
    g1, g2, L = O.grads(X, Y, W1, W2)
    m, I, H = 4, 3, 5
    x = X.astype(np.float64); y = Y.astype(np.float64); a = W1.astype(np.float64); c = W2.astype(np.float64)

    def zval(b, j):
        return sum(x[b, i] * a[i, j] for i in range(I))

    def ypred(b):
        return sum(max(zval(b, j), 0.0) * c[j] for j in range(H))

    Lb = sum((ypred(b) - y[b]) ** 2 for b in range(m)) / m
    assert abs(L - Lb) < 1e-14
    for j in range(H):
        s = sum(max(zval(b, j), 0.0) * (2.0 / m) * (ypred(b) - y[b]) for b in range(m))
        assert abs(g2[j] - s) < 1e-14
        for i in range(I):
            s = sum(x[b, i] * ((2.0 / m) * (ypred(b) - y[b]) * c[j] if zval(b, j) > 0 else 0.0)
                    for b in range(m))
            assert abs(g1[i, j] - s) < 1e-14


# ---------------------------------------------------------------- numpy cross-check + P14
def test_numpy_reference_agrees_on_config1_shape():
    X, Y = datagen.make_dataset(1024, 0.01)
    W1, W2 = datagen.numpy_init_weights(256)
    w1o, w2o = O.train(X, Y, W1, W2, 256, LR, 1)
    w1n, w2n = ref_numpy.train(X, Y, W1, W2, 256, LR, 1)
    np.testing.assert_allclose(w1o, w1n, rtol=0, atol=6e-8)
    np.testing.assert_allclose(w2o, w2n, rtol=0, atol=6e-8)
    assert abs(O.eval_loss(X, Y, w1o, w2o) - ref_numpy.eval_loss(X, Y, w1n, w2n)) < 1e-7


def test_p14_config1_losses(golden):
    g = golden["P14"]["config1"]
    X, Y = datagen.make_dataset(1024, 0.01)
    W1, W2 = datagen.numpy_init_weights(256)
    assert abs(float(np.var(Y.astype(np.float64))) - g["var_Y"]) < 5e-5
    assert abs(O.eval_loss(X, Y, W1, W2) - g["loss_init"]) < 2e-6
    w1, w2 = O.train(X, Y, W1, W2, 256, LR, 1)
    assert abs(O.eval_loss(X, Y, w1, w2) - g["loss_after_4_steps"]) < 2e-6


def test_p14_config2_first_epochs(golden):
    g = golden["P14"]["config2"]
    X, Y = datagen.make_dataset(65536, 0.1)
    W1, W2 = datagen.numpy_init_weights(256)
    order = datagen.make_order(65536, 256, 10, shuffle=True)
    assert abs(float(np.var(Y.astype(np.float64))) - g["var_Y"]) < 5e-5
    assert abs(O.eval_loss(X, Y, W1, W2) - g["loss_init"]) < 2e-6
    w1, w2 = W1, W2
    for e in range(2):                                   # 2 of the 10 epochs keep the CPU suite short
        w1, w2 = O.train(X, Y, w1, w2, 256, LR, 1, order=order[e:e + 1])
        assert abs(O.eval_loss(X, Y, w1, w2) - g["loss_after_epoch"][e]) < 2e-6, e


# ---------------------------------------------------------------- init generator
def test_init_weights_distribution_and_determinism():
    W1, W2 = O.init_weights(2, 32, 256)
    b1, b2 = 1 / math.sqrt(32), 1 / math.sqrt(256)
    assert np.abs(W1).max() <= b1 and np.abs(W2).max() <= b2
    assert abs(W1.mean()) < 3 * b1 / math.sqrt(3 * W1.size)
    assert abs(W1.var() - b1 * b1 / 3) < 0.05 * b1 * b1 / 3
    V1, V2 = O.init_weights(2, 32, 256)
    assert V1.tobytes() == W1.tobytes() and V2.tobytes() == W2.tobytes()
    U1, _ = O.init_weights(3, 32, 256)
    assert (U1 != W1).mean() > 0.99
    # first element by hand: SplitMix64 finaliser of seed + golden*(e+1), e = 0
    z = (2 + 0x9E3779B97F4A7C15) & (2 ** 64 - 1)
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & (2 ** 64 - 1)
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & (2 ** 64 - 1)
    z ^= z >> 31
    u = (z >> 40) / 16777216.0
    assert W1[0, 0] == np.float32((2 * u - 1) * b1)

    # the same by hand for other flat indices e (W1 row-major, then W2): an interior W1 element, the last W1
    # element, the first W2 element (e = 32*256: the branch that switches offset and bound) and the last one
    def by_hand(seed, e, bound):
        z = (seed + 0x9E3779B97F4A7C15 * (e + 1)) & (2 ** 64 - 1)
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & (2 ** 64 - 1)
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & (2 ** 64 - 1)
        z ^= z >> 31
        return np.float32((2 * ((z >> 40) / 16777216.0) - 1) * bound)
    assert W1[3, 17] == by_hand(2, 3 * 256 + 17, b1)
    assert W1[31, 255] == by_hand(2, 32 * 256 - 1, b1)
    assert W2[0] == by_hand(2, 32 * 256, b2)
    assert W2[255] == by_hand(2, 32 * 256 + 255, b2)
    for hidden in (32, 1024):                                   # the bound of W2 follows the hidden width
        A1, A2 = O.init_weights(7, 32, hidden)
        assert A2[0] == by_hand(7, 32 * hidden, 1 / math.sqrt(hidden))
        assert A2[hidden - 1] == by_hand(7, 32 * hidden + hidden - 1, 1 / math.sqrt(hidden))
        assert A1[31, hidden - 1] == by_hand(7, 32 * hidden - 1, b1)


def test_state_fp64_switch_is_report_only():
    X, Y = datagen.make_dataset(4096, 0.1)
    W1, W2 = datagen.numpy_init_weights(256)
    a = O.train(X, Y, W1, W2, 256, LR, 2)
    b = O.train(X, Y, W1, W2, 256, LR, 2, state_fp64=True)
    assert np.abs(a[0] - b[0]).max() / np.abs(a[0]).max() < 1e-5

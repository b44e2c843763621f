"""GPU: calls on different streams overlap without sharing library state (include/mlp.h "Concurrency"),
and the device-side guards of the batch-order / row-order tables.  SURVEY.md 8(f) NEXT-6 (concurrent
replicas) against the oracle.  Run with `-m gpu` on a B200."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from oracle import mlp_oracle as O                      # noqa: E402
from paper_2606_30497_b200 import binding as B          # noqa: E402
from paper_2606_30497_b200 import datagen               # noqa: E402

LR = np.float32(0.002)


def nerr(g, o):
    g = np.asarray(g, np.float64); o = np.asarray(o, np.float64)
    return float(np.abs(g - o).max() / max(np.abs(o).max(), 1e-30))


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


@pytest.mark.parametrize("variant", ["FUSED", "TF32"])
def test_concurrent_evals_on_two_streams(variant):
    """Two (then many) mlp_eval_loss_async calls in flight on different streams over different data: each
    equals its single-stream result bitwise and the oracle within the variant's tolerance."""
    v = getattr(B, "VARIANT_" + variant)
    tol = 2e-6 if variant == "FUSED" else 5e-3
    B.mlp_init(2, 32, 256, 1)
    W1, W2 = O.init_weights(5, 32, 256)
    d1, d2 = dev(W1), dev(W2)
    sets = []
    for k, n in enumerate((300000, 70001, 5000, 127, 262144, 1)):
        X, Y = datagen.make_dataset(n, 0.1, seed_x=10 + k)
        sets.append((n, dev(X), dev(Y), O.eval_loss(X, Y, W1, W2)))
    single = []
    for n, dX, dY, _ in sets:
        out = torch.zeros(1, dtype=torch.float64, device="cuda")
        B.mlp_eval_loss_async(dX, dY, n, d1, d2, out, v)
        torch.cuda.synchronize()
        single.append(float(out.item()))
    for rounds in range(3):
        streams = [torch.cuda.Stream() for _ in sets]
        outs = [torch.zeros(8, dtype=torch.float64, device="cuda") for _ in sets]
        torch.cuda.synchronize()
        for rep in range(8):                                   # 48 launches in flight: more than the 32 pool slots
            for st, (n, dX, dY, _), out in zip(streams, sets, outs):
                with torch.cuda.stream(st):
                    B.mlp_eval_loss_async(dX, dY, n, d1, d2, out[rep:rep + 1], v)
        torch.cuda.synchronize()
        for (n, _, _, lo), out, s in zip(sets, outs, single):
            got = out.cpu().numpy()
            assert np.all(got == s), (variant, n, got, s)
            assert abs(s - lo) <= tol * lo, (variant, n, s, lo)


def test_eval_with_caller_workspace():
    B.mlp_init(2, 32, 256, 1)
    W1, W2 = O.init_weights(5, 32, 256)
    X, Y = datagen.make_dataset(70001, 0.1)
    dX, dY, d1, d2 = dev(X), dev(Y), dev(W1), dev(W2)
    nbytes = B.mlp_eval_workspace_bytes()
    assert nbytes >= 8 * 150
    ws = torch.zeros(nbytes // 8, dtype=torch.float64, device="cuda")
    out = torch.zeros(2, dtype=torch.float64, device="cuda")
    B.mlp_eval_loss_ws(dX, dY, 70001, d1, d2, out[0:1], B.VARIANT_FUSED, ws)
    B.mlp_eval_loss_ws(dX, dY, 70001, d1, d2, out[1:2], B.VARIANT_TF32, ws)      # the workspace is left reusable
    torch.cuda.synchronize()
    assert float(out[0].item()) == B.mlp_eval_loss(dX, dY, 70001, d1, d2)
    lo = O.eval_loss(X, Y, W1, W2)
    assert abs(float(out[1].item()) - lo) <= 5e-3 * lo
    with pytest.raises(B.MlpError):
        B.mlp_eval_loss_ws(dX, dY, 70001, d1, d2, out[0:1], B.VARIANT_FUSED, ws[:4])   # too small


def test_concurrent_training_replicas_match_single_stream_and_oracle():
    """4 independent models of the same job on 4 streams, each on its own cluster:
    bitwise equal to the single-stream run, within 1e-5 of the oracle, and the per-launch statistics of
    concurrent launches do not clobber each other."""
    n, batch, epochs = 8192, 256, 2
    X, Y = datagen.make_dataset(n, 0.1)
    order = datagen.make_order(n, batch, epochs, True)
    B.mlp_init(2, 32, 256, 1)
    B.mlp_set_cluster(0)
    dX, dY, dO = dev(X), dev(Y), dev(order.reshape(-1))
    seeds = (2, 3, 4, 5)
    inits = [O.init_weights(s, 32, 256) for s in seeds]
    ref = []
    for W1, W2 in inits:
        d1, d2 = dev(W1), dev(W2)
        B.mlp_train_ex(dX, dY, n, batch, LR, epochs, d1, d2, dO, B.VARIANT_FUSED)
        torch.cuda.synchronize()
        ref.append((d1.cpu().numpy(), d2.cpu().numpy()))
    streams = [torch.cuda.Stream() for _ in seeds]
    ws = [(dev(W1), dev(W2)) for W1, W2 in inits]
    torch.cuda.synchronize()
    for st, (d1, d2) in zip(streams, ws):
        with torch.cuda.stream(st):
            B.mlp_train_ex(dX, dY, n, batch, LR, epochs, d1, d2, dO, B.VARIANT_FUSED)
    torch.cuda.synchronize()
    stats = B.mlp_get_train_stats()
    assert stats["steps"] == epochs * (n // batch) and stats["cluster"] == 8 and stats["sm_cycles"] > 0
    assert B.mlp_train_order_errors() == 0
    for (d1, d2), (r1, r2), (W1, W2) in zip(ws, ref, inits):
        assert np.array_equal(d1.cpu().numpy(), r1) and np.array_equal(d2.cpu().numpy(), r2)
        o1, o2 = O.train(X, Y, W1, W2, batch, LR, epochs, order=order)
        assert nerr(r1, o1) <= 1e-5 and nerr(r2, o2) <= 1e-5


def test_eval_and_training_overlap():
    """An eval pass on one stream while a training launch runs on another (different buffers)."""
    n = 65536
    X, Y = datagen.make_dataset(n, 0.1)
    W1, W2 = O.init_weights(2, 32, 256)
    B.mlp_init(2, 32, 256, 1)
    dX, dY = dev(X), dev(Y)
    t1, t2, e1, e2 = dev(W1), dev(W2), dev(W1), dev(W2)
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    s_train, s_eval = torch.cuda.Stream(), torch.cuda.Stream()
    torch.cuda.synchronize()
    with torch.cuda.stream(s_train):
        B.mlp_train(dX, dY, n, 256, LR, 2, t1, t2)
    with torch.cuda.stream(s_eval):
        B.mlp_eval_loss_async(dX, dY, n, e1, e2, out, B.VARIANT_FUSED)
    torch.cuda.synchronize()
    lo = O.eval_loss(X, Y, W1, W2)
    assert abs(float(out.item()) - lo) <= 2e-6 * lo
    o1, o2 = O.train(X, Y, W1, W2, 256, LR, 2)
    assert nerr(t1.cpu().numpy(), o1) <= 1e-5 and nerr(t2.cpu().numpy(), o2) <= 1e-5


# ------------------------------------------------------------------ order-table guards
@pytest.mark.parametrize("variant", ["FUSED", "TF32"])
def test_out_of_range_batch_order_is_clamped_and_counted(variant):
    n, batch = 2048, 256
    nb = n // batch
    X, Y = datagen.make_dataset(n, 0.1)
    W1, W2 = O.init_weights(2, 32, 256)
    B.mlp_init(2, 32, 256, 1)
    bad = np.array([0, 3, 99, 1, -5, 7, 2, 8], np.int32)              # 99 -> nb-1, -5 -> 0, 8 -> nb-1
    clamped = np.clip(bad, 0, nb - 1).astype(np.int32)
    dX, dY = dev(X), dev(Y)
    v = getattr(B, "VARIANT_" + variant)
    g1, g2 = dev(W1), dev(W2)
    B.mlp_train_ex(dX, dY, n, batch, LR, 1, g1, g2, dev(bad), v)
    torch.cuda.synchronize()
    assert B.mlp_train_order_errors() == 3
    c1, c2 = dev(W1), dev(W2)
    B.mlp_train_ex(dX, dY, n, batch, LR, 1, c1, c2, dev(clamped), v)
    torch.cuda.synchronize()
    assert B.mlp_train_order_errors() == 0
    assert torch.equal(g1, c1) and torch.equal(g2, c2)
    with pytest.raises(B.MlpError):                                     # the per-equation path validates on the host
        B.mlp_train_ex(dX, dY, n, batch, LR, 1, dev(W1), dev(W2), dev(bad), B.VARIANT_UNFUSED)


def test_host_entry_validates_order_before_any_work():
    n, batch = 1024, 256
    X, Y = datagen.make_dataset(n, 0.1)
    W1, W2 = O.init_weights(2, 32, 256)
    B.mlp_init(2, 32, 256, 1)
    h1, h2 = W1.copy(), W2.copy()
    with pytest.raises(B.MlpError) as ei:
        B.mlp_train_host(X, Y, n, batch, LR, 1, h1, h2, np.array([0, 1, 2, 4], np.int32))
    assert ei.value.code == 2 and "batch_order[3]" in str(ei.value)
    assert np.array_equal(h1, W1) and np.array_equal(h2, W2)            # untouched


def test_out_of_range_row_order_is_clamped_and_counted():
    n, batch = 1000, 100
    X, Y = datagen.make_dataset(n, 0.1)
    W1, W2 = O.init_weights(2, 32, 64)
    B.mlp_init(2, 32, 64, 1)
    rows = datagen.make_row_order(n, 1).reshape(-1).copy()
    rows[5] = n + 17; rows[500] = -1
    fixed = np.clip(rows, 0, n - 1).astype(np.int32)
    dX, dY = dev(X), dev(Y)
    g1, g2 = dev(W1), dev(W2)
    B.mlp_train_rows(dX, dY, n, batch, LR, 1, g1, g2, dev(rows))
    torch.cuda.synchronize()
    assert B.mlp_train_order_errors() == 2
    o1, o2 = O.train(np.ascontiguousarray(X[fixed]), np.ascontiguousarray(Y[fixed]), W1, W2, batch, LR, 1)
    assert nerr(g1.cpu().numpy(), o1) <= 1e-5 and nerr(g2.cpu().numpy(), o2) <= 1e-5


# ------------------------------------------------------------------ fit (train + eval per epoch) and the chunked eval
def test_fit_host_matches_device_path_and_oracle():
    """BASELINE.json configs[2] structure (training with an eval-loss pass after each epoch) through the
    host-buffer entry point, scaled down."""
    n, batch, epochs = 20000, 256, 3
    X, Y = datagen.make_dataset(n, 0.1)
    W1, W2 = O.init_weights(2, 32, 256)
    order = datagen.make_order(n, batch, epochs, True)
    B.mlp_init(2, 32, 256, 1)
    h1, h2 = W1.copy(), W2.copy()
    losses = np.zeros(epochs, np.float64)
    B.mlp_fit_host(X, Y, n, batch, LR, epochs, h1, h2, order.reshape(-1).copy(), B.VARIANT_FUSED, B.VARIANT_FUSED, losses)
    dX, dY, d1, d2 = dev(X), dev(Y), dev(W1), dev(W2)
    o1, o2 = W1, W2
    for e in range(epochs):
        B.mlp_train_ex(dX, dY, n, batch, LR, 1, d1, d2, dev(order[e]), B.VARIANT_FUSED)
        assert B.mlp_eval_loss(dX, dY, n, d1, d2) == losses[e]
        o1, o2 = O.train(X, Y, o1, o2, batch, LR, 1, order=order[e:e + 1])
        lo = O.eval_loss(X, Y, o1, o2)
        assert abs(losses[e] - lo) <= 1e-5 * lo
    assert np.array_equal(h1, d1.cpu().numpy()) and np.array_equal(h2, d2.cpu().numpy())
    assert nerr(h1, o1) <= 1e-5 and nerr(h2, o2) <= 1e-5


@pytest.mark.parametrize("variant", ["FUSED", "TF32"])
def test_eval_loss_host_chunked_pipeline(variant):
    """More than one 262,144-row chunk: the copy/compute pipeline combines per-chunk means in chunk order."""
    n = 600001
    X, Y = datagen.make_dataset(n, 0.1)
    W1, W2 = O.init_weights(5, 32, 256)
    B.mlp_init(2, 32, 256, 1)
    v = getattr(B, "VARIANT_" + variant)
    a = B.mlp_eval_loss_host(X, Y, n, W1, W2, v)
    assert a == B.mlp_eval_loss_host(X, Y, n, W1, W2, v)                 # deterministic
    lo = O.eval_loss(X, Y, W1, W2)
    assert abs(a - lo) <= (2e-6 if variant == "FUSED" else 5e-3) * lo


@pytest.mark.parametrize("variant", ["FUSED", "TF32", "BF16"])
def test_cluster_sizes_agree_under_load(variant):
    """Stress test for the cross-CTA Ypred exchange (st.async + remote mbarrier transaction bytes, waited for with
    a CTA-scope acquire): the whole of BASELINE.json config 2 (2,560 SGD steps) at every
    cluster size, while a second stream keeps the rest of the chip busy with full-grid eval passes.  Every run
    must match the oracle; a lost or early-read partial would show up as a wrong gradient."""
    c = datagen.CONFIGS["config2"]
    X, Y = datagen.make_dataset(c.n, c.sigma)
    order = datagen.make_order(c.n, c.batch, c.epochs, True)
    W1, W2 = O.init_weights(2, 32, c.hidden)
    o1, o2 = O.train(X, Y, W1, W2, c.batch, LR, c.epochs, order=order)
    B.mlp_init(2, 32, c.hidden, 1)
    dX, dY, dO = dev(X), dev(Y), dev(order.reshape(-1))
    v = getattr(B, "VARIANT_" + variant)
    tol = {"FUSED": 1e-5, "TF32": 2e-3, "BF16": 5e-3}[variant]
    side = torch.cuda.Stream()
    e1, e2 = dev(W1), dev(W2)
    sink = torch.zeros(1, dtype=torch.float64, device="cuda")
    for cl in ((2, 4, 8, 16) if variant == "FUSED" else (0,)):
        B.mlp_set_cluster(cl)
        d1, d2 = dev(W1), dev(W2)
        torch.cuda.synchronize()
        with torch.cuda.stream(side):
            for _ in range(40):                                   # ~12 ms of full-grid work beside the training launch
                B.mlp_eval_loss_async(dX, dY, c.n, e1, e2, sink, B.VARIANT_FUSED)
        B.mlp_train_ex(dX, dY, c.n, c.batch, LR, c.epochs, d1, d2, dO, v)
        torch.cuda.synchronize()
        assert nerr(d1.cpu().numpy(), o1) <= tol and nerr(d2.cpu().numpy(), o2) <= tol, (variant, cl)
    B.mlp_set_cluster(0)

"""GPU: mlp_eval_loss_static (include/mlp.h), the eval entry point that allocates nothing: its per-CTA
partial sums and ticket live in a file-scope __device__ array of the library.  It launches the kernels of
mlp_eval_loss_async, so its result must equal that path's bit for bit (the reduction order is fixed) and
the oracle's within the tolerance of tests/test_gpu_parity.py.  Collected last on purpose (pytest -x).
Run with `-m gpu` on a B200."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from oracle import mlp_oracle as O                      # noqa: E402
from paper_2606_30497_b200 import binding as B          # noqa: E402
from paper_2606_30497_b200 import datagen               # noqa: E402

TOL = {"FUSED": 2e-6, "TF32": 5e-3, "BF16": 1e-2}


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


@pytest.mark.parametrize("variant", ["FUSED", "TF32", "BF16"])
def test_static_eval_matches_pool_path_on_consecutive_calls(variant):
    """Two calls in a row (the second over fewer rows and other weights, so the shared array still holds
    the first call's partial sums when it starts), then the first again: each equals mlp_eval_loss_async."""
    v = getattr(B, "VARIANT_" + variant)
    B.mlp_init(2, 32, 256, 1)
    cases = []
    for k, n in enumerate((200001, 777)):
        X, Y = datagen.make_dataset(n, 0.1, seed_x=40 + k)
        W1, W2 = O.init_weights(7 + k, 32, 256)
        cases.append((n, dev(X), dev(Y), dev(W1), dev(W2), O.eval_loss(X, Y, W1, W2)))
    want = torch.zeros(len(cases), dtype=torch.float64, device="cuda")
    for i, (n, dX, dY, d1, d2, _) in enumerate(cases):
        B.mlp_eval_loss_async(dX, dY, n, d1, d2, want[i:i + 1], v)
    torch.cuda.synchronize()
    want = want.cpu().numpy()
    order = (0, 1, 0, 1, 1)
    got = torch.full((len(order),), -1.0, dtype=torch.float64, device="cuda")
    before = B.mlp_launch_count()
    for j, i in enumerate(order):                         # back to back on one stream, no sync in between
        n, dX, dY, d1, d2, _ = cases[i]
        B.mlp_eval_loss_static(dX, dY, n, d1, d2, got[j:j + 1], v)
    torch.cuda.synchronize()
    assert B.mlp_launch_count() - before == len(order)
    got = got.cpu().numpy()
    for j, i in enumerate(order):
        assert got[j] == want[i], (variant, j, got[j], want[i])
        lo = cases[i][5]
        assert abs(got[j] - lo) <= TOL[variant] * lo, (variant, j, got[j], lo)


def test_static_eval_allocates_nothing_and_validates():
    """No device memory is taken by the calls (free memory as the driver reports it is unchanged, on a
    side stream too), and bad arguments are rejected like mlp_eval_loss_async's."""
    B.mlp_init(2, 32, 64, 1)
    n = 4097
    X, Y = datagen.make_dataset(n, 0.1, seed_x=51)
    W1, W2 = O.init_weights(3, 32, 64)
    dX, dY, d1, d2 = dev(X), dev(Y), dev(W1), dev(W2)
    out = torch.zeros(4, dtype=torch.float64, device="cuda")
    st = torch.cuda.Stream()
    B.mlp_eval_loss_static(dX, dY, n, d1, d2, out[0:1])            # first use: symbol lookup, module load
    with torch.cuda.stream(st):
        B.mlp_eval_loss_static(dX, dY, n, d1, d2, out[2:3], B.VARIANT_FUSED, st)
    torch.cuda.synchronize()
    out[2:3].fill_(-1.0)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    B.mlp_eval_loss_static(dX, dY, n, d1, d2, out[1:2])
    torch.cuda.synchronize()
    with torch.cuda.stream(st):
        B.mlp_eval_loss_static(dX, dY, n, d1, d2, out[2:3], B.VARIANT_FUSED, st)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0, (free0, free1)
    B.mlp_eval_loss_async(dX, dY, n, d1, d2, out[3:4])
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    assert got[0] == got[1] == got[2] == got[3], got
    lo = O.eval_loss(X, Y, W1, W2)
    assert abs(got[0] - lo) <= TOL["FUSED"] * lo
    with pytest.raises(B.MlpError):
        B.mlp_eval_loss_static(dX, dY, 0, d1, d2, out[0:1])                       # n < 1
    with pytest.raises(B.MlpError):
        B.mlp_eval_loss_static(dX, dY, n, d1, d2, out[0:1], 99)                   # unknown variant
    B.mlp_init(2, 32, 512, 1)
    with pytest.raises(B.MlpError):
        B.mlp_eval_loss_static(dX, dY, n, d1, d2, out[0:1], B.VARIANT_TF32X3)     # hidden > 256


def test_static_eval_under_graph_capture():
    """The motivating use: after one warm-up call (symbol lookup, module load), the call is captured into a CUDA
    graph (stream capture forbids cudaMalloc) and replayed; every replay equals mlp_eval_loss_async bit for bit."""
    B.mlp_init(2, 32, 128, 1)
    n = 50001
    X, Y = datagen.make_dataset(n, 0.1, seed_x=61)
    W1, W2 = O.init_weights(4, 32, 128)
    dX, dY, d1, d2 = dev(X), dev(Y), dev(W1), dev(W2)
    want = torch.zeros(2, dtype=torch.float64, device="cuda")
    B.mlp_eval_loss_async(dX, dY, n, d1, d2, want[0:1], B.VARIANT_FUSED)
    B.mlp_eval_loss_async(dX, dY, n, d1, d2, want[1:2], B.VARIANT_TF32)
    out = torch.zeros(2, dtype=torch.float64, device="cuda")
    B.mlp_eval_loss_static(dX, dY, n, d1, d2, out[0:1], B.VARIANT_FUSED)        # warm-up, outside the capture
    B.mlp_eval_loss_static(dX, dY, n, d1, d2, out[1:2], B.VARIANT_TF32)
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        st = torch.cuda.current_stream()
        B.mlp_eval_loss_static(dX, dY, n, d1, d2, out[0:1], B.VARIANT_FUSED, st)
        B.mlp_eval_loss_static(dX, dY, n, d1, d2, out[1:2], B.VARIANT_TF32, st)
    for _ in range(3):
        out.fill_(-1.0)
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(out, want), (out.cpu().numpy(), want.cpu().numpy())

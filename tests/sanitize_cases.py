"""Small invocations of every kernel family for compute-sanitizer (memcheck / racecheck / synccheck); SURVEY.md
section 5 "Race detection".  Each case also checks its result against the oracle, so a sanitizer run that
perturbs timing still verifies the numbers.  Not collected by pytest; run as

    compute-sanitizer --tool racecheck python tests/sanitize_cases.py <case> [<case> ...]

Cases: fused_c2 fused_c8 fused_c16 fused_b32 tc_c1 tc_c8 tc_bf16 tc_wide eval_fp32 eval_tf32_h256
eval_tf32_h1024 eval_bf16 eval_x3 eval_static (default: all that the library supports).  Summary: profiles/r02_sanitizer.md."""
import os
import sys

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from oracle import mlp_oracle as O                      # noqa: E402
from paper_2606_30497_b200 import binding as B          # noqa: E402
from paper_2606_30497_b200 import datagen               # noqa: E402

LR = np.float32(0.002)


def nerr(g, o):
    return float(np.abs(np.asarray(g, np.float64) - o).max() / np.abs(o).max())


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def train_case(hidden, batch, n, cluster, variant, tol, epochs=1):
    X, Y = datagen.make_dataset(n, 0.01)
    W1, W2 = O.init_weights(2, 32, hidden)
    order = datagen.make_order(n, batch, epochs, True)
    B.mlp_init(2, 32, hidden, 1)
    B.mlp_set_cluster(cluster)
    d1, d2 = dev(W1), dev(W2)
    B.mlp_train_ex(dev(X), dev(Y), n, batch, LR, epochs, d1, d2, dev(order.reshape(-1)), variant)
    torch.cuda.synchronize()
    B.mlp_set_cluster(0)
    o1, o2 = O.train(X, Y, W1, W2, batch, LR, epochs, order=order)
    e1, e2 = nerr(d1.cpu().numpy(), o1), nerr(d2.cpu().numpy(), o2)
    assert e1 <= tol and e2 <= tol, (e1, e2)
    return e1, e2


def eval_case(hidden, n, variant, tol, static=False):
    X, Y = datagen.make_dataset(n, 0.1)
    W1, W2 = O.init_weights(5, 32, hidden)
    B.mlp_init(2, 32, hidden, 1)
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    (B.mlp_eval_loss_static if static else B.mlp_eval_loss_async)(dev(X), dev(Y), n, dev(W1), dev(W2), out, variant)
    torch.cuda.synchronize()
    lo = O.eval_loss(X, Y, W1, W2)
    e = abs(float(out.item()) - lo) / lo
    assert e <= tol, e
    return (e,)


CASES = {
    # BASELINE.json config 1 (n=1024, B=256, 4 steps) on clusters of 2, 8, 16; B=32 / n=2048 run
    "fused_c2": lambda: train_case(256, 256, 1024, 2, B.VARIANT_FUSED, 1e-5),
    "fused_c8": lambda: train_case(256, 256, 1024, 8, B.VARIANT_FUSED, 1e-5),
    "fused_c16": lambda: train_case(256, 256, 1024, 16, B.VARIANT_FUSED, 1e-5),
    "fused_b32": lambda: train_case(256, 32, 2048, 0, B.VARIANT_FUSED, 1e-5),
    "fused_ragged": lambda: train_case(256, 300, 1000, 8, B.VARIANT_FUSED, 1e-5, epochs=2),
    "tc_c1": lambda: train_case(32, 256, 1024, 0, B.VARIANT_TF32, 2e-3),
    "tc_c8": lambda: train_case(256, 256, 1024, 0, B.VARIANT_TF32, 2e-3),
    "tc_b32": lambda: train_case(256, 32, 2048, 0, B.VARIANT_TF32, 2e-3),
    "tc_bf16": lambda: train_case(256, 256, 1024, 0, B.VARIANT_BF16, 5e-3),
    "tc_wide": lambda: train_case(1024, 256, 1024, 0, B.VARIANT_TF32, 2e-3),
    "eval_fp32": lambda: eval_case(256, 40000, B.VARIANT_FUSED, 2e-6),
    "eval_tf32_h256": lambda: eval_case(256, 40000, B.VARIANT_TF32, 5e-3),
    "eval_tf32_h1024": lambda: eval_case(1024, 40000, B.VARIANT_TF32, 5e-3),
    "eval_bf16": lambda: eval_case(256, 40000, B.VARIANT_BF16, 5e-3),
    "eval_x3": lambda: eval_case(256, 40000, B.VARIANT_TF32X3, 1e-5),
    "eval_static": lambda: eval_case(256, 40000, B.VARIANT_FUSED, 2e-6, static=True),   # scratch in a __device__ array
}

if __name__ == "__main__":
    names = sys.argv[1:] or list(CASES)
    for name in names:
        try:
            r = CASES[name]()
            print(f"{name}: ok, error vs oracle {' / '.join('%.2e' % v for v in r)}", flush=True)
        except B.MlpError as e:
            if e.code == 3:
                print(f"{name}: unsupported by this build ({e})", flush=True)
            else:
                raise

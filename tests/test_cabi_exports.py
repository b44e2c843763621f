"""The C-ABI library builds, loads, and exports every symbol include/mlp.h declares (no GPU)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "mlp.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(mlp_[a-z_0-9]+)\s*\(", src)))


def test_header_declares_the_three_north_star_calls():
    d = _declared()
    for name in ("mlp_init", "mlp_train", "mlp_eval_loss"):
        assert name in d


def test_library_exports_every_declared_symbol():
    from paper_2606_30497_b200 import build, binding
    path = build.build()
    L = ctypes.CDLL(path)
    for name in _declared():
        assert hasattr(L, name), name
    assert sorted(binding.EXPORTS) == _declared()


def test_argument_validation_without_gpu():
    """Error paths that return before any CUDA call work on a CPU-only box."""
    from paper_2606_30497_b200 import binding as B
    L = B.lib()
    assert L.mlp_init(0, 31, 256, 1) == 3            # MLP_ERR_UNSUPPORTED
    assert L.mlp_init(0, 32, 100, 1) == 3
    assert b"hidden" in L.mlp_last_error()
    assert L.mlp_init(0, 32, 256, 2) == 3
    assert L.mlp_init(2, 32, 256, 1) == 0
    assert L.mlp_train(None, None, 10, 4, 0.1, 1, None, None, None) == 2   # NULL -> BAD_ARG
    assert L.mlp_set_cluster(3) == 3
    assert L.mlp_set_cluster(8) == 0 and L.mlp_get_cluster() == 8
    assert L.mlp_set_cluster(0) == 0
    fake = ctypes.c_void_p(0x1000)
    assert L.mlp_train(fake, fake, 0, 4, 0.1, 1, fake, fake, None) == 2    # n < 1
    assert L.mlp_train(fake, fake, 8, 0, 0.1, 1, fake, fake, None) == 2    # batch < 1
    assert L.mlp_train(fake, fake, 8, 4, float("nan"), 1, fake, fake, None) == 2
    assert L.mlp_train(ctypes.c_void_p(0x1004), fake, 8, 4, 0.1, 1, fake, fake, None) == 4   # ALIGN
    assert L.mlp_train(fake, fake, 8, 4, 0.1, 0, fake, fake, None) == 0    # epochs == 0: no-op
    assert L.mlp_train_ex(fake, fake, 8, 4, 0.1, 1, fake, fake, None, 7, None) == 3


def test_no_cpu_fallback_without_device():
    """On a box without a GPU the compute entries must fail loudly, never compute on the CPU."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    import numpy as np
    from paper_2606_30497_b200 import binding as B
    B.mlp_init(2, 32, 256, 1)
    X = np.zeros((8, 32), np.float32); Y = np.zeros(8, np.float32)
    W1 = np.zeros((32, 256), np.float32); W2 = np.zeros(256, np.float32)
    with pytest.raises(B.MlpError):
        B.mlp_train_host(X, Y, 8, 4, 0.1, 1, W1, W2)
    with pytest.raises(B.MlpError):
        B.mlp_eval_loss_host(X, Y, 8, W1, W2)

"""B200-native (sm_100a) mini-batch SGD for the shallow ReLU/MSE MLP of arxiv/paper_2606_30497.

The product is the C-ABI library `libmlp_b200.so` (include/mlp.h; sources in csrc/); this package
adds the build script, a thin ctypes binding with the same names, the seeded input generators and
the roofline arithmetic used by bench.py.  Importing the package does not load the library.
"""
from .binding import (  # noqa: F401
    VARIANT_FUSED, VARIANT_TF32, VARIANT_UNFUSED, MlpError, mlp_eval_loss, mlp_eval_loss_async,
    mlp_eval_loss_host, mlp_get_cluster, mlp_get_train_stats, mlp_init, mlp_init_weights,
    mlp_last_error, mlp_launch_count, mlp_set_cluster, mlp_shutdown, mlp_train, mlp_train_ex,
    mlp_train_host, mlp_version,
)

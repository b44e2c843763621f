"""Roofline arithmetic for the hot path; pure bookkeeping, no kernels."""
from __future__ import annotations

IN = 32
FMA_FLOP_PER_CLK_PER_SM = 256          # 128 FP32 lanes x 2 FLOP (FMA)


def f_step(batch: int, hidden: int, in_features: int = IN) -> int:
    """Algorithmic FLOP of one SGD step (FMA = 2): eqs. 1,8: 2BIH each; eqs. 3,6: 2BH each;
    eq. 7: BH; eq. 5: 2B; eq. 9: 2(IH+H).   (PAPER.md:201-210 counts the same products as MACs.)"""
    B, H, I = batch, hidden, in_features
    return 4 * B * I * H + 5 * B * H + 2 * B + 2 * (I * H + H)


def train_floor_us(batch: int, hidden: int, cluster: int, sm_mhz: float) -> float:
    """FP32-FMA floor of one step on the `cluster` SMs the kernel occupies, in microseconds."""
    return f_step(batch, hidden) / (FMA_FLOP_PER_CLK_PER_SM * cluster * sm_mhz)


def eval_flop_per_sample(hidden: int, in_features: int = IN) -> int:
    return 2 * in_features * hidden + 2 * hidden + 3


def eval_bytes_per_sample(in_features: int = IN) -> int:
    return 4 * in_features + 4          # one X row + one target


def step_bytes(batch: int, in_features: int = IN) -> int:
    """HBM/L2 bytes one SGD step must read: the batch's X rows and targets (row a0)."""
    return batch * (4 * in_features + 4)

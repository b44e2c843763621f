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


# Tensor-core training variants (csrc/train_tc.cu): eqs. 1 and 8 on tcgen05, the rest on the CUDA cores, and one
# cluster exchange per tile that nothing can overlap (dZ2 of a row needs the Ypred partials of every CTA).
TC_DENSE_BF16_FLOP_PER_CLK_PER_SM = 8192   # 2.25 PFLOP/s nominal / 148 SMs / 1.86 GHz; kind::tf32 runs at half of it
DSMEM_HOP_CLK = 215                         # one st.async hop to a peer CTA (guide: B300_MICROARCH.md, CGA / DSMEM)


def tc_train_cluster(hidden: int) -> int:
    return {32: 1, 64: 2, 128: 4, 256: 8, 512: 8, 1024: 16}[hidden]


def tc_train_floor_us(batch: int, hidden: int, sm_mhz: float, bf16: bool, in_features: int = IN) -> float:
    """Floor of one step of the tensor-core variant on its cluster: tensor time of eqs. 1 and 8 at the nominal dense
    rate of the SMs it occupies + the remaining FLOP at the FP32-FMA rate + one DSMEM hop per 256-row (hidden <=
    256) or 128-row tile for the Ypred exchange."""
    C = tc_train_cluster(hidden)
    tensor = 4 * batch * in_features * hidden / (TC_DENSE_BF16_FLOP_PER_CLK_PER_SM * (1.0 if bf16 else 0.5) * C * sm_mhz)
    rest = (f_step(batch, hidden, in_features) - 4 * batch * in_features * hidden) / (FMA_FLOP_PER_CLK_PER_SM * C * sm_mhz)
    tile = 256 if hidden <= 256 else 128
    hops = -(-batch // tile) * DSMEM_HOP_CLK / sm_mhz
    return tensor + rest + hops

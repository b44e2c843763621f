"""Seeded synthetic input generators shared by the CPU oracle and the CUDA path.

This module produces INPUTS only (X, Y, teacher, batch-order tables, the numpy
init weights of pin P14). It holds none of the method's arithmetic (eqs. 1-9 of
PAPER.md:44-71): the targets are a *data recipe* (teacher network + noise) fixed
by BASELINE.json `configs` and SURVEY.md section 8(d), not the training step.

The paper's dataset is unnamed and undescribed; these seeded
teacher-student sets stand in for it with the paper's shapes (32 features, one
target, batch 256, lr 0.002 -- PAPER.md:98-112).
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

IN_FEATURES = 32
TEACHER_HIDDEN = 64       # BASELINE.json configs[0]: T1 [32x64], T2 [64x1]
LR = np.float32(0.002)


@dataclasses.dataclass(frozen=True)
class Config:
    """One of BASELINE.json's five synthetic configurations (or a scaled-down copy)."""
    name: str
    n: int
    hidden: int
    batch: int
    epochs: int
    sigma: float
    shuffle: bool          # per-epoch permutation of the batch indices (seed 3)
    lr: float = float(LR)


# BASELINE.json `configs` 1..5. Config 4 and 5 are sweeps: see `sweep()`.
CONFIGS = {
    "config1": Config("config1", 1024, 256, 256, 1, 0.01, False),
    "config2": Config("config2", 65536, 256, 256, 10, 0.1, True),
    "config3": Config("config3", 1048576, 256, 256, 10, 0.1, True),
    "config4": Config("config4", 262144, 256, 256, 5, 0.1, True),      # hidden swept
    "config5": Config("config5", 4194304, 256, 256, 3, 0.1, True),     # batch swept
}
CONFIG4_HIDDEN = (64, 128, 512, 1024)
CONFIG5_BATCH = (32, 256, 1024, 4096)


def sweep(name: str):
    """Expand config4 / config5 into their member configurations."""
    base = CONFIGS[name]
    if name == "config4":
        return [dataclasses.replace(base, name=f"config4_h{h}", hidden=h) for h in CONFIG4_HIDDEN]
    if name == "config5":
        return [dataclasses.replace(base, name=f"config5_b{b}", batch=b) for b in CONFIG5_BATCH]
    return [base]


def make_dataset(n: int, sigma: float, seed_x: int = 0, seed_teacher: int = 1):
    """X ~ N(0,1) [n x 32] fp32 (seed 0); Y = ReLU(X T1) T2 + N(0, sigma^2) fp32 [n].

    T1 [32x64], T2 [64x1] ~ N(0, 1/fan_in) (variance), then the noise, all drawn in
    that order from the seed-1 stream (SURVEY.md 8(c) items 23-24, 8(d) recipe).
    """
    X = np.random.default_rng(seed_x).standard_normal((n, IN_FEATURES), dtype=np.float32)
    rt = np.random.default_rng(seed_teacher)
    T1 = rt.standard_normal((IN_FEATURES, TEACHER_HIDDEN)) / math.sqrt(IN_FEATURES)
    T2 = rt.standard_normal((TEACHER_HIDDEN, 1)) / math.sqrt(TEACHER_HIDDEN)
    noise = sigma * rt.standard_normal((n, 1))
    Y = np.empty((n, 1), dtype=np.float64)
    blk = 1 << 18                                   # bound the fp64 temporary
    for s in range(0, n, blk):
        e = min(n, s + blk)
        Y[s:e] = np.maximum(X[s:e].astype(np.float64) @ T1, 0.0) @ T2
    Y += noise
    return np.ascontiguousarray(X), np.ascontiguousarray(Y.astype(np.float32).reshape(n))


def teacher(seed_teacher: int = 1):
    """The teacher weights alone (fp64), for the student==teacher pin (P8)."""
    rt = np.random.default_rng(seed_teacher)
    T1 = rt.standard_normal((IN_FEATURES, TEACHER_HIDDEN)) / math.sqrt(IN_FEATURES)
    T2 = rt.standard_normal((TEACHER_HIDDEN, 1)) / math.sqrt(TEACHER_HIDDEN)
    return T1, T2


def num_batches(n: int, batch: int) -> int:
    return (n + batch - 1) // batch


def make_order(n: int, batch: int, epochs: int, shuffle: bool, seed: int = 3):
    """Batch-order table int32 [epochs x nb]: row e is the order in which the nb
    contiguous batches [t*B, min(n,(t+1)*B)) are visited in epoch e.

    shuffle=False -> 0..nb-1 every epoch (config 1, `mlp_train`).
    shuffle=True  -> one `permutation(nb)` per epoch from default_rng(3) (configs 2-5).
    """
    nb = num_batches(n, batch)
    if not shuffle:
        return np.tile(np.arange(nb, dtype=np.int32), (epochs, 1))
    rp = np.random.default_rng(seed)
    return np.stack([rp.permutation(nb) for _ in range(epochs)]).astype(np.int32)


def make_row_order(n: int, epochs: int, seed: int = 3):
    """Sample-level shuffling: one permutation of the n rows per epoch, int32
    [epochs x n], drawn from numpy default_rng(seed)."""
    rp = np.random.default_rng(seed)
    return np.stack([rp.permutation(n) for _ in range(epochs)]).astype(np.int32)


def numpy_init_weights(hidden: int, seed: int = 2):
    """U(+-1/sqrt(fan_in)) from numpy's generator -- used ONLY by pin P14 (SURVEY.md
    8(c)); the library's own init is the counter-based generator of include/mlp.h."""
    rw = np.random.default_rng(seed)
    b1 = 1.0 / math.sqrt(IN_FEATURES)
    b2 = 1.0 / math.sqrt(hidden)
    W1 = rw.uniform(-b1, b1, (IN_FEATURES, hidden)).astype(np.float32)
    W2 = rw.uniform(-b2, b2, (hidden, 1)).astype(np.float32).reshape(hidden)
    return np.ascontiguousarray(W1), np.ascontiguousarray(W2)


def small_problem(seed: int, m: int, in_features: int, hidden: int, scale: float = 1.0):
    """A small random fp32 problem (X, Y, W1, W2) for oracle pins and edge cases."""
    r = np.random.default_rng(seed)
    X = r.standard_normal((m, in_features)).astype(np.float32)
    Y = r.standard_normal(m).astype(np.float32)
    W1 = (scale * r.uniform(-1, 1, (in_features, hidden)) / math.sqrt(in_features)).astype(np.float32)
    W2 = (scale * r.uniform(-1, 1, hidden) / math.sqrt(hidden)).astype(np.float32)
    return X, Y, W1, W2

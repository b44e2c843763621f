#!/usr/bin/env python
"""bench.py -- headline benchmark of the B200 MLP-SGD library (contract: DESIGN.md section 7).

Workload (N=1): BASELINE.json configs[2] ("config3", the largest single-GPU configuration the metric
"training samples/s and us per SGD step (fp32, B=256)" applies to; "like the paper's largest case",
PAPER.md:330): 32-256-1 ReLU/MSE MLP, fp32, batch 256, lr 0.002, n = 1,048,576 seeded teacher-student
samples, 10 epochs with a per-epoch batch-order permutation (seed 3), and a full-dataset eval-loss pass
after each epoch.  One bench "step" = that whole job: per epoch one fused training launch (4,096 SGD
steps) and one exact-fp32 eval launch, 20 launches in all.  metric = training samples/s (whole job, all
ranks).  N>1: independent replicas (the SGD step does not shard -- DESIGN.md section 6), weak scaling, no
data-path collective.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--quick]
"""
from __future__ import annotations

import argparse
import hashlib
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

WORKLOAD = "config3"
METRIC = "training samples/s (fp32, B=256, 32-256-1 MLP SGD)"
UNIT = "samples/s"
REF_SAMPLE_ROWS = 131072          # rows of the bounded sample one --impl reference step works on


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"hbm_gbs": d["hbm_gbs"], "sm_max_mhz": d.get("sm_max_mhz", 1965.0), "source": "measured",
                "bf16_tflops": d.get("bf16_tflops", 1636.0)}
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "source": "fallback", "bf16_tflops": 1600.0}


def workload_config(cfg):
    """The `config` object both arms print (same keys, same values: the same job)."""
    c = {"workload": WORKLOAD, "n": cfg.n, "hidden": cfg.hidden, "batch": cfg.batch, "epochs": cfg.epochs,
         "evals_per_step": cfg.epochs, "sgd_steps_per_step": cfg.epochs * ((cfg.n + cfg.batch - 1) // cfg.batch),
         "step_definition": "one full run of BASELINE.json configs[2]: 10 epochs of mini-batch SGD over n rows "
                            "(per-epoch batch-order permutation, seed 3), an eval-loss pass over the dataset "
                            "after each epoch",
         "l2": "dataset (138 MB) larger than L2 (126 MB); L2 also flushed between timed steps (256 MiB memset, untimed)"}
    c["parallelism"] = "replicas only (one independent job per GPU; the SGD step does not shard)"
    return c


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.max_mhz = index, [], set(), None
        self._stop_evt = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception:
            self.ok = False

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {
            getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
            getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwPowerBrakeSlowdown", 0x80): "hw_power_brake_slowdown",
        }
        while not self._stop_evt.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(0.005)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=2)

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": 0}
        return {"sm_mhz": statistics.median(self.samples), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ---------------------------------------------------------------------------------------------- oracle legs
def oracle_fit(O, X, Y, W1, W2, cfg, order, epochs):
    """The oracle running `epochs` epochs of the job with an eval pass after each (as the repo arm does)."""
    w1, w2 = W1, W2
    for e in range(epochs):
        w1, w2 = O.train(X, Y, w1, w2, cfg.batch, cfg.lr, 1, order=order[e:e + 1])
        O.eval_loss(X, Y, w1, w2)
    return w1, w2


def oracle_leg(cfg, X, Y, W1, W2, order, budget_s=12.0):
    """cpu_baseline: the oracle, as it stands, on the host cores: whole epochs of the SAME job (same rows, same
    batch order, eval pass after each epoch) from the same initial weights until ~budget_s of CPU work."""
    from oracle import mlp_oracle as O
    t0 = time.perf_counter()
    epochs = 0
    w1, w2 = W1, W2
    while True:
        e = epochs % cfg.epochs
        w1, w2 = O.train(X, Y, w1, w2, cfg.batch, cfg.lr, 1, order=order[e:e + 1])
        O.eval_loss(X, Y, w1, w2)
        epochs += 1
        dt = time.perf_counter() - t0
        if dt >= budget_s or epochs >= cfg.epochs:
            break
    steps = epochs * ((cfg.n + cfg.batch - 1) // cfg.batch)
    return {"value": cfg.n * epochs / dt, "unit": UNIT, "cores": O.num_threads(), "kind": "oracle",
            "sample": f"the first {epochs} of the {cfg.epochs} epochs of {cfg.name} (n={cfg.n}; {steps} SGD steps), an "
                      f"eval pass after each, {dt:.2f} s wall", "us_per_sgd_step": dt / steps * 1e6}


def oracle_us_per_step(X, Y, hidden, batch, budget_s=1.5):
    """Oracle time per SGD step for one per_config member: whole batches of its first epoch, ~budget_s."""
    from oracle import mlp_oracle as O
    W1, W2 = O.init_weights(2, 32, hidden)
    rows = min(X.shape[0], max(batch, 8192 // batch * batch))
    t0 = time.perf_counter()
    steps = 0
    while True:
        O.train(X[:rows], Y[:rows], W1, W2, batch, 0.002, 1)
        steps += (rows + batch - 1) // batch
        dt = time.perf_counter() - t0
        if dt >= budget_s:
            break
    return dt / steps * 1e6


def run_reference(args, rank, world):
    """--impl reference: the CPU oracle timed on the box's host cores (rank 0 only).  Same job, same metric, same
    `config`; each step is a bounded sample of it: one epoch (with its eval pass) over the first
    REF_SAMPLE_ROWS rows, so that K+W steps end within a few minutes on the host."""
    if rank != 0:
        return
    from oracle import mlp_oracle as O
    from paper_2606_30497_b200 import datagen
    cfg = datagen.CONFIGS[WORKLOAD]
    ns = min(cfg.n, REF_SAMPLE_ROWS)
    X, Y = datagen.make_dataset(ns, cfg.sigma)                      # = the first ns rows of the config's dataset
    W1, W2 = O.init_weights(2, 32, cfg.hidden)
    order = datagen.make_order(ns, cfg.batch, cfg.epochs, cfg.shuffle)
    w1, w2 = W1, W2
    times = []
    for k in range(args.warmup + args.steps):
        e = k % cfg.epochs
        t0 = time.perf_counter()
        w1, w2 = O.train(X, Y, w1, w2, cfg.batch, cfg.lr, 1, order=order[e:e + 1])
        O.eval_loss(X, Y, w1, w2)
        if k >= args.warmup:
            times.append(time.perf_counter() - t0)
    total = sum(times)
    value = ns * args.steps / total
    sample = (f"each step = one epoch of {cfg.name} restricted to its first {ns} rows ({ns // cfg.batch} SGD steps, "
              f"permuted batch order) + one eval pass over those rows: 1/{cfg.epochs * cfg.n // ns} of the repo arm's "
              f"step, same train:eval proportion, CPU oracle fp64")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": total / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": workload_config(cfg),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": O.num_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


# ---------------------------------------------------------------------------------------------- repo arm
def sha256_of(path):
    return hashlib.sha256(open(path, "rb").read()).hexdigest()


def run_ours(args, rank, world, local_rank):
    import torch
    import torch.distributed as dist
    from paper_2606_30497_b200 import binding as B
    from paper_2606_30497_b200 import datagen, roofline, sharding

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; use --impl reference "
                         "for the oracle arm)")
    torch.cuda.set_device(local_rank)
    peaks = load_peaks()
    cfg = datagen.CONFIGS[WORKLOAD]
    nb = datagen.num_batches(cfg.n, cfg.batch)
    sgd_steps = cfg.epochs * nb
    samples_per_step = cfg.n * cfg.epochs
    full = rank == 0 and world == 1 and not args.quick         # the per-config block and the context rows

    # ---- seeded synthetic inputs (same bytes on every rank: independent replicas).  The recipe's streams are
    #      prefix-stable, so configs 2-4 are the leading rows of config 5's 4,194,304-row dataset. ----
    n_all = datagen.CONFIGS["config5"].n if full else cfg.n
    X_all, Y_all = datagen.make_dataset(n_all, cfg.sigma)
    X, Y = X_all[:cfg.n], Y_all[:cfg.n]
    order = datagen.make_order(cfg.n, cfg.batch, cfg.epochs, cfg.shuffle)
    B.mlp_init(2, 32, cfg.hidden, 1)
    B.mlp_set_cluster(0)
    dX_all, dY_all = torch.from_numpy(X_all).cuda(), torch.from_numpy(Y_all).cuda()
    dX, dY = dX_all[:cfg.n], dY_all[:cfg.n]
    dO = torch.from_numpy(order.copy()).cuda()                              # [epochs][nb]
    W1i = torch.empty(32, cfg.hidden, device="cuda"); W2i = torch.empty(cfg.hidden, device="cuda")
    B.mlp_init_weights(W1i, W2i)
    d1, d2 = W1i.clone(), W2i.clone()
    dloss = torch.zeros(cfg.epochs, dtype=torch.float64, device="cuda")
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")      # > 126 MB L2
    cluster = B.mlp_get_cluster(cfg.batch)
    ev = lambda: torch.cuda.Event(enable_timing=True)                      # noqa: E731

    def one_step(evs=None):
        d1.copy_(W1i); d2.copy_(W2i)
        flush.zero_()                                   # evict the dataset from L2 (untimed)
        if evs: evs[0].record()
        for e in range(cfg.epochs):
            if evs: evs[2][e][0].record()
            B.mlp_train_ex(dX, dY, cfg.n, cfg.batch, cfg.lr, 1, d1, d2, dO[e], B.VARIANT_FUSED)
            if evs: evs[2][e][1].record()
            B.mlp_eval_loss_async(dX, dY, cfg.n, d1, d2, dloss[e:e + 1], B.VARIANT_FUSED)
        if evs: evs[1].record()

    for _ in range(args.warmup):
        one_step()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    launches0 = B.mlp_launch_count()
    evs = [(ev(), ev(), [(ev(), ev()) for _ in range(cfg.epochs)]) for _ in range(args.steps)]
    torch.cuda.synchronize()
    for k in range(args.steps):
        one_step(evs[k])
    torch.cuda.synchronize()
    launches = B.mlp_launch_count() - launches0
    sampler.stop()
    if world > 1:
        dist.barrier()
    step_ms = [e[0].elapsed_time(e[1]) for e in evs]
    train_ms = [sum(a.elapsed_time(b) for a, b in e[2]) for e in evs]         # the cfg.epochs training launches of a step
    total_ms = sum(step_ms)
    stats = B.mlp_get_train_stats()
    losses = dloss.cpu().numpy().tolist()
    w1_dev, w2_dev = d1.clone(), d2.clone()                                   # the device path's result (default cluster)
    if world > 1:
        total_ms = sharding.max_over_ranks(total_ms)      # device time of the slowest replica
    if rank != 0:
        return

    value = world * samples_per_step * args.steps / (total_ms * 1e-3)
    train_ms_avg = sum(train_ms) / len(train_ms)
    launch_ms = train_ms_avg / cfg.epochs                                      # one training launch = one epoch
    us_per_sgd = train_ms_avg * 1e3 / sgd_steps
    kernel_mhz = stats["sm_cycles"] / stats["ns"] * 1e3 if stats["ns"] else None

    # ---- roofline of the dominant kernel (fused training kernel; ALU-bound) ----
    flop_launch = roofline.f_step(cfg.batch, cfg.hidden) * nb
    achieved = flop_launch / (launch_ms * 1e-3) / 1e12
    peak = roofline.FMA_FLOP_PER_CLK_PER_SM * cluster * peaks["sm_max_mhz"] * 1e6 / 1e12
    traffic, traffic_note = None, "profiles/traffic.json missing"
    tpath = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(tpath):
        tj = json.load(open(tpath))
        src = os.path.join(ROOT, "paper_2606_30497_b200", "csrc", "train_fused.cu")
        if tj.get("train_fused_cu_sha256") == sha256_of(src) and tj.get("workload") == WORKLOAD:
            traffic, traffic_note = tj.get("train_fused_dram_bytes_per_launch"), tj.get("source")
        else:
            traffic_note = "profiles/traffic.json was captured for another build of train_fused.cu or another workload: stale, not reported"
    roof = {"bound": "alu", "kernel": "k_train_fused", "achieved": achieved, "peak": peak,
            "unit": "TFLOP/s", "frac": achieved / peak, "traffic": traffic, "traffic_source": traffic_note,
            "peak_source": f"256 FLOP/clk/SM x {cluster} occupied SMs x sm_max_mhz "
                           f"({peaks['sm_max_mhz']:.0f}, {peaks['source']})",
            "launch": f"one epoch of {WORKLOAD} = {nb} SGD steps", "launch_ms": launch_ms,
            "share_of_step": train_ms_avg / (total_ms / args.steps) if world == 1 else None,
            "us_per_sgd_step": us_per_sgd,
            "floor_us_per_sgd_step": roofline.train_floor_us(cfg.batch, cfg.hidden, cluster, peaks["sm_max_mhz"]),
            "cluster": cluster, "sm_mhz_in_kernel": kernel_mhz,
            "algorithmic_flop_per_launch": flop_launch,
            "algorithmic_hbm_bytes_per_launch": roofline.step_bytes(cfg.batch) * nb}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": workload_config(cfg), "cluster_sms": cluster,
        "us_per_sgd_step": us_per_sgd, "epoch_losses": losses, "final_loss": losses[-1],
        "roofline": roof, "gpu_launches": int(launches), "clocks": sampler.summary(),
        "context": "paper (Tesla T4, optimised kernels): 1,482 us/step, 172.7 k samples/s (PAPER.md:330, derived)",
    }

    # ---- end-to-end: the same job through the host-buffer C-ABI call, copies inside the timed region ----
    hX = torch.from_numpy(X).pin_memory(); hY = torch.from_numpy(Y).pin_memory()
    hO = torch.from_numpy(order.reshape(-1).copy()).pin_memory()
    h1 = W1i.cpu().pin_memory(); h2 = W2i.cpu().pin_memory()
    hL = torch.zeros(cfg.epochs, dtype=torch.float64).pin_memory()
    w1_init, w2_init = h1.clone(), h2.clone()

    def e2e_call():
        h1.copy_(w1_init); h2.copy_(w2_init)
        t0 = time.perf_counter()
        B.mlp_fit_host(hX, hY, cfg.n, cfg.batch, cfg.lr, cfg.epochs, h1, h2, hO, B.VARIANT_FUSED, B.VARIANT_FUSED, hL)
        return time.perf_counter() - t0

    for _ in range(2):
        e2e_call()
    ne2e = max(3, min(args.steps, 10))
    e2e_t = sum(e2e_call() for _ in range(ne2e))
    wbytes = (32 * cfg.hidden + cfg.hidden) * 4
    line["e2e"] = {"value": world * samples_per_step * ne2e / e2e_t, "unit": UNIT,
                   "h2d_bytes_per_step": cfg.n * 132 + wbytes + order.size * 4, "d2h_bytes_per_step": wbytes + 8 * cfg.epochs,
                   "api": "mlp_fit_host (pinned host X/Y/W/order in; trained W and the 10 epoch losses out)",
                   "timer": "host wall clock", "calls_timed": ne2e, "ms_per_step": e2e_t / ne2e * 1e3}
    line["e2e_bitwise_equal_to_device_path"] = bool(
        torch.equal(h1.cuda(), w1_dev) and torch.equal(h2.cuda(), w2_dev) and hL.tolist() == losses)
    del hX, hY

    if full:
        extras(line, B, datagen, roofline, torch, peaks, cfg, X_all, Y_all, dX_all, dY_all, W1i, W2i, w1_dev, w2_dev,
               order, flush, losses)
        line["cpu_baseline"] = oracle_leg(cfg, X, Y, W1i.cpu().numpy(), W2i.cpu().numpy(), order)
    print(json.dumps(line))


def extras(line, B, datagen, roofline, torch, peaks, cfg, X_all, Y_all, dX_all, dY_all, W1i, W2i, w1_dev, w2_dev,
           order, flush, losses):
    """N=1 only, outside the timed region: the per-config block (north_star: "report throughput on the synthetic
    configs"), the eval kernels on config 5's matrix, cluster sweep, tensor-core variants, concurrent replicas,
    the paper's own shapes."""
    ev = lambda: torch.cuda.Event(enable_timing=True)                      # noqa: E731
    mhz = peaks["sm_max_mhz"]

    def timed(fn, reps=3, flush_l2=True):
        ts = []
        for _ in range(reps):
            if flush_l2:
                flush.zero_()
            a, b = ev(), ev()
            a.record(); fn(); b.record()
            torch.cuda.synchronize()
            ts.append(a.elapsed_time(b))
        return min(ts), statistics.median(ts)

    def train_member(c, variant=B.VARIANT_FUSED, reps=3):
        """us per SGD step of one whole run of config member c in ONE launch, at the default cluster."""
        B.mlp_init(2, 32, c.hidden, 1)
        B.mlp_set_cluster(0)
        a1 = torch.empty(32, c.hidden, device="cuda"); a2 = torch.empty(c.hidden, device="cuda")
        B.mlp_init_weights(a1, a2)
        dO = torch.from_numpy(datagen.make_order(c.n, c.batch, c.epochs, c.shuffle).reshape(-1).copy()).cuda()
        w1, w2 = a1.clone(), a2.clone()

        def run():
            w1.copy_(a1); w2.copy_(a2)
            B.mlp_train_ex(dX_all[:c.n], dY_all[:c.n], c.n, c.batch, c.lr, c.epochs, w1, w2, dO, variant)
        run(); torch.cuda.synchronize()
        best, _ = timed(run, reps)
        steps = c.epochs * datagen.num_batches(c.n, c.batch)
        dl = torch.zeros(1, dtype=torch.float64, device="cuda")
        B.mlp_eval_loss_async(dX_all[:c.n], dY_all[:c.n], c.n, w1, w2, dl, B.VARIANT_FUSED)
        torch.cuda.synchronize()
        return best * 1e3 / steps, c.n * c.epochs / (best * 1e-3), float(dl.item())

    def unfused_us(c, steps=256):
        B.mlp_init(2, 32, c.hidden, 1)
        rows = min(c.n, steps * c.batch)
        u1 = torch.empty(32, c.hidden, device="cuda"); u2 = torch.empty(c.hidden, device="cuda")
        B.mlp_init_weights(u1, u2)
        f = lambda: B.mlp_train_ex(dX_all[:rows], dY_all[:rows], rows, c.batch, c.lr, 1, u1, u2, None, B.VARIANT_UNFUSED)  # noqa: E731
        f(); torch.cuda.synchronize()
        best, _ = timed(f, 2, flush_l2=False)
        return best * 1e3 / datagen.num_batches(rows, c.batch)

    # ---- per-config block ----
    per = {}
    members = [datagen.CONFIGS["config2"], cfg] + datagen.sweep("config4") + datagen.sweep("config5")
    for c in members:
        if c.name == cfg.name:
            us, sps, fl = line["us_per_sgd_step"], line["value"], losses[-1]
            note = "the timed headline job (one launch per epoch, eval pass after each epoch included in samples/s)"
        else:
            us, sps, fl = train_member(c)
            note = "whole job in one launch, best of 3"
        B.mlp_init(2, 32, c.hidden, 1)
        cl = B.mlp_get_cluster(c.batch)
        floor = roofline.train_floor_us(c.batch, c.hidden, cl, mhz)
        row = {"n": c.n, "hidden": c.hidden, "batch": c.batch, "epochs": c.epochs, "cluster": cl,
               "us_per_sgd_step": us, "samples_per_s": sps, "floor_us_per_sgd_step": floor, "frac_of_fma_floor": floor / us,
               "final_loss": fl, "timing": note,
               "unfused_us_per_sgd_step": unfused_us(c),
               "oracle_us_per_sgd_step": oracle_us_per_step(X_all[:c.n], Y_all[:c.n], c.hidden, c.batch)}
        for vname, v in (("tf32", B.VARIANT_TF32), ("bf16", B.VARIANT_BF16)):
            try:
                tus, tsps, tfl = train_member(c, v)
                tfloor = roofline.tc_train_floor_us(c.batch, c.hidden, mhz, vname == "bf16")
                row["train_" + vname] = {"us_per_sgd_step": tus, "samples_per_s": tsps, "final_loss": tfl,
                                         "final_loss_rel_diff_vs_fp32_path": abs(tfl - fl) / fl,
                                         "cluster": roofline.tc_train_cluster(c.hidden),
                                         "floor_us_per_sgd_step": tfloor, "frac_of_tc_floor": tfloor / tus,
                                         "floor": "tensor time of eqs. 1, 8 at the nominal dense rate of the cluster's SMs "
                                                  "+ other FLOP at the FP32-FMA rate + one DSMEM hop per tile (roofline.py)"}
            except B.MlpError:
                row["train_" + vname] = None
        per[c.name] = row
    line["per_config"] = per
    B.mlp_init(2, 32, cfg.hidden, 1)

    # ---- eval kernels on BASELINE.json configs[4]'s 4,194,304 x 32 matrix (the HBM measurement) and on 16.8 M rows ----
    dloss = torch.zeros(1, dtype=torch.float64, device="cuda")
    ev_out = {}
    fma_peak = 256 * 148 * mhz * 1e6 / 1e12

    def eval_rows(dXe, dYe, ne, hidden, variants):
        out = {}
        B.mlp_init(2, 32, hidden, 1)
        e1 = torch.empty(32, hidden, device="cuda"); e2 = torch.empty(hidden, device="cuda")
        B.mlp_init_weights(e1, e2)
        for name, v in variants:
            try:
                B.mlp_eval_loss_async(dXe, dYe, ne, e1, e2, dloss, v)
            except B.MlpError:
                out[name] = None
                continue
            torch.cuda.synchronize()
            ms, med = timed(lambda: B.mlp_eval_loss_async(dXe, dYe, ne, e1, e2, dloss, v), 10)
            gbs = ne * roofline.eval_bytes_per_sample() / (ms * 1e-3) / 1e9
            tf = ne * roofline.eval_flop_per_sample(hidden) / (ms * 1e-3) / 1e12
            out[name] = {"us": ms * 1e3, "us_median": med * 1e3, "GB/s": gbs, "frac_of_measured_hbm": gbs / peaks["hbm_gbs"],
                         "frac_of_8TBs_nominal": gbs / 8000.0, "TFLOP/s": tf, "frac_of_fp32_fma_peak": tf / fma_peak,
                         "loss": float(dloss.item())}
        return out

    allv = (("fp32", B.VARIANT_FUSED), ("tf32", B.VARIANT_TF32), ("bf16", B.VARIANT_BF16), ("tf32x3", B.VARIANT_TF32X3))
    n5 = datagen.CONFIGS["config5"].n
    for hidden in (64, 128, 256, 512, 1024):
        ev_out["h%d" % hidden] = eval_rows(dX_all, dY_all, n5, hidden, allv if hidden == 256 else allv[1:3])
    ts = []
    for _ in range(5):
        a, b = ev(), ev()
        flush.zero_()
        a.record(); dX_all.sum(); b.record()
        torch.cuda.synchronize()
        ts.append(a.elapsed_time(b))
    ev_out["torch_sum_read_GB/s"] = n5 * 128 / (min(ts) * 1e-3) / 1e9
    ev_out["rows"] = n5
    line["eval_config5"] = ev_out
    big = {}
    try:
        n16 = 1 << 24
        gen = torch.Generator(device="cuda"); gen.manual_seed(0)
        Xb = torch.randn(n16, 32, device="cuda", generator=gen); Yb = torch.randn(n16, device="cuda", generator=gen)
        for hidden in (64, 256):
            big["h%d" % hidden] = eval_rows(Xb, Yb, n16, hidden, allv[1:3])
        big["rows"] = n16
        big["data"] = "torch.randn on the device (bandwidth only; not the config's recipe)"
        del Xb, Yb
    except Exception as e:                                                  # out of memory on a shared box etc.
        big["error"] = str(e)[:200]
    line["eval_16M_rows"] = big
    B.mlp_init(2, 32, cfg.hidden, 1)

    # ---- the headline epoch at the other cluster sizes ----
    dX, dY = dX_all[:cfg.n], dY_all[:cfg.n]
    dO0 = torch.from_numpy(order[0].copy()).cuda()
    nb = order.shape[1]
    by_cluster = {}
    for cl in (2, 4, 8, 16):
        try:
            B.mlp_set_cluster(cl)
        except B.MlpError:
            continue
        c1, c2 = W1i.clone(), W2i.clone()
        f = lambda: B.mlp_train_ex(dX, dY, cfg.n, cfg.batch, cfg.lr, 1, c1, c2, dO0, B.VARIANT_FUSED)  # noqa: E731
        f(); torch.cuda.synchronize()
        best, _ = timed(f, 3)
        us = best * 1e3 / nb
        by_cluster[str(cl)] = {"us_per_sgd_step": us,
                               "frac_of_fma_floor": roofline.train_floor_us(cfg.batch, cfg.hidden, cl, mhz) / us}
    B.mlp_set_cluster(0)
    line["train_by_cluster"] = by_cluster

    # ---- concurrent replicas: R independent models of one epoch on R streams ----
    conc = {}
    for R in (4, 16):
        streams = [torch.cuda.Stream() for _ in range(R)]
        ws = [(W1i.clone(), W2i.clone()) for _ in range(R)]
        torch.cuda.synchronize()
        a, b = ev(), ev()
        a.record()
        for st, (r1, r2) in zip(streams, ws):
            st.wait_event(a)
            with torch.cuda.stream(st):
                B.mlp_train_ex(dX, dY, cfg.n, cfg.batch, cfg.lr, 1, r1, r2, dO0, B.VARIANT_FUSED)
        for st in streams:
            torch.cuda.current_stream().wait_stream(st)
        b.record()
        torch.cuda.synchronize()
        same = all(torch.equal(r1, ws[0][0]) and torch.equal(r2, ws[0][1]) for r1, r2 in ws)
        conc[str(R)] = {"ms": a.elapsed_time(b), "aggregate_samples_per_s": R * cfg.n / (a.elapsed_time(b) * 1e-3),
                        "replicas_bitwise_equal": bool(same)}
    line["concurrent_replicas"] = conc

    # ---- the paper's own shapes (Tables I-II): seconds for 100 epochs, B=256, sequential
    #      batches, with the paper's two strategies re-created (prior_art.cu) beside the fused kernel ----
    paper_T4 = {"n256": (0.306, 0.248), "n2560": (2.000, 1.561), "n25600": (21.002, 14.823),
                "h32": 0.810, "h64": 0.921, "h128": 1.107, "h256": 1.551, "h512": 2.743, "h1024": 4.645}

    def seconds(nn, hidden, variant, epochs=100):
        B.mlp_init(2, 32, hidden, 1)
        a1 = torch.empty(32, hidden, device="cuda"); a2 = torch.empty(hidden, device="cuda")
        B.mlp_init_weights(a1, a2)
        ep = epochs if variant == B.VARIANT_FUSED else max(1, min(epochs, 2000 // max(1, nn // 256)))
        B.mlp_train_ex(dX_all[:nn], dY_all[:nn], nn, 256, cfg.lr, 1, a1, a2, None, variant)          # warm-up
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        B.mlp_train_ex(dX_all[:nn], dY_all[:nn], nn, 256, cfg.lr, ep, a1, a2, None, variant)
        torch.cuda.synchronize()
        return (time.perf_counter() - t0) * epochs / ep

    paper_shapes = {"unit": "seconds per 100 epochs (host wall clock incl. launches; baselines extrapolated "
                            "from >= 2000 SGD steps)", "table1": {}, "table2_n2560": {}}
    for nn in (256, 2560, 25600):
        naive, tiled, fused = (seconds(nn, 256, v) for v in (B.VARIANT_PRIOR_NAIVE, B.VARIANT_PRIOR_TILED, B.VARIANT_FUSED))
        paper_shapes["table1"]["n%d" % nn] = {
            "paper_T4_baseline": paper_T4["n%d" % nn][0], "paper_T4_optimized": paper_T4["n%d" % nn][1],
            "b200_paper_baseline": naive, "b200_paper_optimized": tiled, "b200_fused": fused,
            "b200_optimized_over_baseline": naive / tiled}
    for hh in (32, 64, 128, 256, 512, 1024):
        paper_shapes["table2_n2560"]["h%d" % hh] = {
            "paper_T4": paper_T4["h%d" % hh], "b200_paper_optimized": seconds(2560, hh, B.VARIANT_PRIOR_TILED),
            "b200_fused": seconds(2560, hh, B.VARIANT_FUSED)}
    line["paper_shapes"] = paper_shapes
    B.mlp_init(2, 32, cfg.hidden, 1)


def spawn_replicas(args):
    """`python bench.py --gpus N` without a launcher: start N ranks (one per device) ourselves."""
    import socket
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    procs = []
    for r in range(args.gpus):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE=str(args.gpus),
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, os.path.abspath(__file__)] + sys.argv[1:], env=env,
                                      stdout=None if r == 0 else subprocess.DEVNULL))
    rc = 0
    for p in procs:
        rc = p.wait() or rc
    sys.exit(rc)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--quick", action="store_true", help="headline line only (no per-config block, no context rows)")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3                                  # timing rule: W >= 3
    launched = "RANK" in os.environ and "WORLD_SIZE" in os.environ
    if args.impl == "ours" and args.gpus > 1 and not launched:
        spawn_replicas(args)
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return
    if world > 1:
        import torch
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        if local_rank >= torch.cuda.device_count():
            raise SystemExit(f"bench.py: rank {rank} has no device (visible GPUs: {torch.cuda.device_count()})")
        torch.cuda.set_device(local_rank)
        dist.init_process_group("nccl")
    try:
        run_ours(args, rank, world, local_rank)
    finally:
        if world > 1:
            import torch.distributed as dist
            dist.destroy_process_group()


if __name__ == "__main__":
    main()

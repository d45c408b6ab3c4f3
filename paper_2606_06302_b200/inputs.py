"""Seeded synthetic input generators for the five BASELINE.json configs.

This module is shared by the tests, the oracle-side checks and bench.py.  It holds
NONE of the method's arithmetic (no Eq. 4/5, no clustering, no page counting, no
planning, no attention): it only draws the *inputs* of the path -- calibrated per-head
statistics (mu, sigma), context lengths, per-request demanded retention, q and the
bf16 page pool, and a free-page list of a size the CALLER chooses.

The inputs stand in for the paper's SCBench runs on Qwen/Llama models (PAPER.md:262-266,
§5.1), whose data, weights and calibrated profiles are not available; shapes and ratio
structure follow BASELINE.json `configs` and the description of Fig. 5.
Recipe: DESIGN.md §"Input recipe".
"""
from __future__ import annotations

import dataclasses
import math
from typing import Optional

import numpy as np

SEED_BASE = 20260630
CONFIG_NAMES = ("tiny", "8b", "32b", "skew", "uniform")
# not a BASELINE.json config: the 8b recipe on Gemma-3-12B-shaped heads (16 query / 8 KV heads of 256 dims,
# one of the paper's five models) -- exercises the d = 256 kernels at full size
EXTRA_CONFIG_NAMES = ("12b_d256",)


@dataclasses.dataclass
class Workload:
    name: str
    index: int
    R: int            # requests in the batch
    Hq: int           # query heads
    H: int            # KV heads
    d: int            # head dim
    P: int            # page size in tokens
    C: int            # head clusters (H_p = H / C)
    alpha: float      # safety-margin coefficient of Eq. 5
    granule: int      # split granule g in tokens
    ctx_len: np.ndarray   # [R] int32   pre-compression context N_r
    mu: np.ndarray        # [H] float64 calibrated mean retention ratio
    sigma: np.ndarray     # [H] float64 calibrated std of the ratio
    demand: np.ndarray    # [R, H] int32 tokens the compressor wants to retain
    seed: int

    @property
    def G(self) -> int:
        return self.Hq // self.H

    @property
    def Hp(self) -> int:
        return self.H // self.C


def _demand(ctx_len: np.ndarray, ratio_rh: np.ndarray) -> np.ndarray:
    # generator-side rounding is half-up (BASELINE.json: "round(512*r)"), clamped to [1, N_r]
    n = ctx_len.astype(np.float64)[:, None]
    dem = np.floor(n * ratio_rh + 0.5).astype(np.int64)
    dem = np.minimum(np.maximum(dem, 1), ctx_len.astype(np.int64)[:, None])
    return dem.astype(np.int32)


def _jitter(rng: np.random.Generator, ratio_h: np.ndarray, R: int, hw: float) -> np.ndarray:
    if hw == 0.0:
        return np.broadcast_to(ratio_h[None, :], (R, ratio_h.shape[0])).copy()
    u = rng.uniform(-hw, hw, size=(R, ratio_h.shape[0]))
    return np.minimum(1.0, ratio_h[None, :] * (1.0 + u))


def make_workload(name: str, *, R: Optional[int] = None, ctx_div: int = 1, layer: int = 0,
                  page_size: Optional[int] = None) -> Workload:
    """Build config `name` (one of CONFIG_NAMES).  `R` overrides the batch size and
    `ctx_div` divides every context length (scaled-down parity cases); the default
    arguments give the full BASELINE.json configuration.  `layer` > 0 draws another layer of the
    same shape (its own head ratios, i.e. its own budgets, clusters and plan) for multi-layer
    decode loops: seed + 1000 * layer; the context lengths of layer 0 are kept (same requests).
    `page_size` overrides P = 16 (BASELINE.json) for the P = 32 variants of the configs."""
    idx = (CONFIG_NAMES + EXTRA_CONFIG_NAMES).index(name)
    seed = SEED_BASE + idx
    if layer:
        base = make_workload(name, R=R, ctx_div=ctx_div, page_size=page_size)
        seed += 1000 * layer
    rng = np.random.default_rng(seed)
    P, alpha, g = page_size or 16, 2.0, 64

    if name == "tiny":
        R0, Hq, H, d, C, hw = 2, 4, 2, 64, 2, 0.05
        R_ = R or R0
        ctx = np.full(R_, 512 // ctx_div, dtype=np.int32)
        ratio_h = np.array([1.0, 0.25])
    elif name in ("8b", "12b_d256"):
        R0, Hq, H, d, C, hw = (32, 32, 8, 128, 4, 0.10) if name == "8b" else (32, 16, 8, 256, 4, 0.10)
        R_ = R or R0
        ctx = (rng.integers(8192, 32768 + 1, size=R_) // ctx_div).astype(np.int32)
        ratio_h = np.exp(rng.normal(math.log(0.2), 0.5, size=H))
        retrieval = np.array([2, 5])
        ratio_h[retrieval] = rng.uniform(0.9, 1.0, size=2)
        rest = np.setdiff1d(np.arange(H), retrieval)
        # the global 30 % retention wins over the literal "around 0.2"
        ratio_h[rest] *= (0.30 * H - ratio_h[retrieval].sum()) / ratio_h[rest].sum()
    elif name == "32b":
        R0, Hq, H, d, C, hw = 64, 40, 8, 128, 4, 0.05
        R_ = R or R0
        ctx = (rng.integers(16000, 24000 + 1, size=R_) // ctx_div).astype(np.int32)
        ratio_h = rng.beta(2.0, 2.0, size=H)
        target = 0.50 * H
        for _ in range(8):  # scale-and-clip (water filling) to mean 0.50
            free = ratio_h < 1.0
            s = (target - np.count_nonzero(~free)) / ratio_h[free].sum()
            ratio_h = np.where(free, np.minimum(1.0, ratio_h * s), 1.0)
            if abs(ratio_h.sum() - target) < 1e-12:
                break
    elif name == "skew":
        R0, Hq, H, d, C, hw = 16, 32, 8, 128, 2, 0.0
        R_ = R or R0
        ctx = np.full(R_, 131072 // ctx_div, dtype=np.int32)
        ratio_h = np.full(H, 2.0 ** -8)
        ratio_h[0] = 1.0
    elif name == "uniform":
        R0, Hq, H, d, C, hw = 256, 32, 8, 128, 1, 0.0
        R_ = R or R0
        ctx = np.full(R_, 4096 // ctx_div, dtype=np.int32)
        ratio_h = np.ones(H)
    else:  # pragma: no cover
        raise ValueError(name)

    ctx = np.maximum(ctx, 1).astype(np.int32)
    if layer:
        ctx = base.ctx_len.copy()
    ratio_rh = _jitter(rng, ratio_h, R_, hw)
    mu = ratio_h.astype(np.float64).copy()
    sigma = (hw * mu / math.sqrt(3.0)) if hw > 0 else np.zeros(H)
    return Workload(name=name, index=idx, R=R_, Hq=Hq, H=H, d=d, P=P, C=C, alpha=alpha,
                    granule=g, ctx_len=ctx, mu=mu, sigma=np.asarray(sigma, dtype=np.float64),
                    demand=_demand(ctx, ratio_rh), seed=seed)


def make_random_workload(seed: int, *, R: int, H: int, G: int, d: int, C: int, P: int = 16,
                         max_ctx: int = 600, granule: int = 64) -> Workload:
    """Small randomized shapes for property / parity tests (not a BASELINE config)."""
    rng = np.random.default_rng(seed)
    ctx = rng.integers(1, max_ctx + 1, size=R).astype(np.int32)
    mu = rng.uniform(0.02, 1.0, size=H)
    sigma = rng.uniform(0.0, 0.05, size=H) * mu
    ratio_rh = np.minimum(1.0, mu[None, :] * (1.0 + rng.uniform(-0.15, 0.15, size=(R, H))))
    return Workload(name=f"rand{seed}", index=-1, R=R, Hq=H * G, H=H, d=d, P=P, C=C, alpha=2.0,
                    granule=granule, ctx_len=ctx, mu=mu, sigma=sigma,
                    demand=_demand(ctx, ratio_rh), seed=seed)


def make_free_pages(wl: Workload, n_pool_pages: int, *, identity: bool = False) -> np.ndarray:
    """Free list handed to the table builder: a seeded permutation of [0, n_pool_pages)."""
    if identity:
        return np.arange(n_pool_pages, dtype=np.int32)
    rng = np.random.default_rng(wl.seed + 7919)
    return rng.permutation(n_pool_pages).astype(np.int32)


def make_q_and_pool(wl: Workload, n_pool_pages: int, device: str = "cpu", *, poison=None):
    """q [R, Hq, d] bf16 and pool [n_pool_pages, H_p, 2, P, d] bf16, both ~ N(0,1).
    Every slot of the pool is random (slack holds garbage).  Returned as torch tensors
    on `device`.  The stream depends on the device type (torch CPU and CUDA generators
    differ); a test generates once and hands the same tensors to both sides."""
    import torch

    gen = torch.Generator(device=device)
    gen.manual_seed(wl.seed)
    q = torch.randn(wl.R, wl.Hq, wl.d, generator=gen, device=device, dtype=torch.float32).bfloat16()
    shape = (n_pool_pages, wl.Hp, 2, wl.P, wl.d)
    pool = torch.empty(shape, dtype=torch.bfloat16, device=device)
    chunk = max(1, (1 << 28) // (wl.Hp * 2 * wl.P * wl.d))  # <= 1 GiB fp32 scratch at a time
    for p0 in range(0, n_pool_pages, chunk):
        p1 = min(n_pool_pages, p0 + chunk)
        pool[p0:p1] = torch.randn((p1 - p0,) + shape[1:], generator=gen, device=device,
                                  dtype=torch.float32).bfloat16()
    return q, pool


def make_scores_and_dense_kv(wl: Workload, n_max: int, device: str = "cpu", *, ties: str = "bf16"):
    """Inputs of the per-head Top-k compaction (NEXT-2): importance scores [R, H, n_max] f32 and the
    uncompressed cache K, V [R, H, n_max, d] bf16 ~ N(0,1).  Scores are log-normal (attention-mass-like:
    positive, heavy tail); with ties="bf16" they are rounded to bf16 precision first, as a scoring function
    running in bf16 would leave them, so equal scores are common; ties="none" keeps full fp32 values.
    Stands in for the scores of the paper's compression methods, which need model weights."""
    import torch

    gen = torch.Generator(device=device)
    gen.manual_seed(wl.seed + 4242)
    scores = torch.randn(wl.R, wl.H, n_max, generator=gen, device=device, dtype=torch.float32).exp_()
    if ties == "bf16":
        scores = scores.bfloat16().float()
    k = torch.empty(wl.R, wl.H, n_max, wl.d, dtype=torch.bfloat16, device=device)
    v = torch.empty_like(k)
    for dst in (k, v):
        for r in range(wl.R):  # one request at a time: bounded fp32 scratch
            dst[r] = torch.randn(wl.H, n_max, wl.d, generator=gen, device=device, dtype=torch.float32).bfloat16()
    return scores, k, v


def make_calibration_ratios(wl: Workload, n_samples: int = 50) -> np.ndarray:
    """[n_samples, H] per-head implicit retention ratios as a calibration run would record them
    (PAPER.md:156, 50 samples :262): the workload's nominal head ratio times the same uniform per-input
    jitter the demand uses (half-width = sigma * sqrt(3) / mu), clipped to (0, 1]."""
    rng = np.random.default_rng(wl.seed + 99991)
    hw = np.where(wl.mu > 0, wl.sigma * math.sqrt(3.0) / np.maximum(wl.mu, 1e-300), 0.0)
    u = rng.uniform(-1.0, 1.0, size=(n_samples, wl.H))
    return np.clip(wl.mu[None, :] * (1.0 + hw[None, :] * u), 1e-6, 1.0)

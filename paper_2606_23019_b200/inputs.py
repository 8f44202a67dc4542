"""Seeded synthetic inputs for the block-sparse attention hot path.

Input preparation only: this module holds none of the method's arithmetic (no attention, no
top-fraction selection, no bit packing). It serves both the CUDA path (tests, bench.py) and the
CPU oracle's tests, so that both sides see byte-identical q, k, v, block scores and densities.

The paper measures on Wan2.1 / HunyuanVideo activations and WEST/FAST masks (PAPER.md:191-193,
231-246); none of those are available offline, so these inputs take their shapes (21 frames x
1560 / 3600 tokens, 128x128 blocks), their density range and their structure
(local spatio-temporal support plus a few global "sink" columns) and stand in
for them. See BASELINE.json `configs`.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, replace
from typing import Optional, Tuple

import numpy as np
import torch


@dataclass(frozen=True)
class Config:
    name: str
    B: int
    H: int
    N: int          # padded token count (multiple of Bq and Bk)
    D: int
    Bq: int
    Bk: int
    n_valid: int    # real tokens; keys >= n_valid carry zero weight
    grid: Optional[Tuple[int, int, int]]  # latent (T, Hl, Wl), frame-major flattening
    qkv_seed: int
    mask_seed: int
    density_lo: float
    density_hi: float
    sigma_lo: float = 1.0
    sigma_hi: float = 16.0

    @property
    def NQB(self) -> int:
        return self.N // self.Bq

    @property
    def NKB(self) -> int:
        return self.N // self.Bk

    @property
    def W(self) -> int:
        return (self.NKB + 31) // 32

    @property
    def scale(self) -> float:
        """softmax scale as the fp32 value both sides receive."""
        return float(np.float32(1.0 / math.sqrt(self.D)))

    def flops_per_block(self) -> int:
        return 4 * self.Bq * self.Bk * self.D


# BASELINE.json configs[0..3]; C5 is built from C4 with `uniform_density` / adversarial masks.
C1 = Config("C1-tiny", 1, 2, 1024, 64, 64, 64, 1024, None, 0, 0, 0.5, 0.5)
C2 = Config("C2-wan1.3b-480p", 1, 12, 32768, 128, 128, 128, 32760, (21, 30, 52), 1, 101, 0.1, 0.4)
C3 = Config("C3-wan14b-480p", 1, 40, 32768, 128, 128, 128, 32760, (21, 30, 52), 2, 102, 0.05, 0.35)
C4 = Config("C4-wan14b-720p", 1, 40, 75648, 128, 128, 128, 75600, (21, 45, 80), 3, 103, 0.1, 0.3)
CONFIGS = {"C1": C1, "C2": C2, "C3": C3, "C4": C4}


def scaled(cfg: Config, **kw) -> Config:
    """A reduced copy of a config (fewer heads / a smaller latent grid) for parity tests."""
    return replace(cfg, **kw)


def make_qkv(cfg: Config, pin_memory: bool = False):
    """q, k, v ~ N(0,1) drawn in fp32 from one seeded CPU generator (order q, k, v; each tensor
    filled head by head), rounded to bf16. Returns CPU tensors [B][H][N][D]."""
    g = torch.Generator(device="cpu").manual_seed(cfg.qkv_seed)
    outs = []
    for _ in range(3):
        t = torch.empty((cfg.B, cfg.H, cfg.N, cfg.D), dtype=torch.bfloat16,
                        pin_memory=pin_memory)
        for b in range(cfg.B):
            for h in range(cfg.H):
                t[b, h].copy_(torch.randn((cfg.N, cfg.D), generator=g, dtype=torch.float32))
        outs.append(t)
    return tuple(outs)


def poison_padding(cfg: Config, k: torch.Tensor, v: torch.Tensor) -> None:
    """Parity tests fill padded keys with values that make any leak loud (P8)."""
    if cfg.n_valid < cfg.N:
        k[:, :, cfg.n_valid:, :] = 64.0
        v[:, :, cfg.n_valid:, :] = 1000.0


def as_u16(t: torch.Tensor) -> np.ndarray:
    """bf16 CPU tensor -> numpy uint16 bit patterns (the oracle's input format)."""
    assert t.dtype == torch.bfloat16 and t.device.type == "cpu"
    return t.contiguous().view(torch.int16).numpy().view(np.uint16)


def block_centroids(cfg: Config) -> np.ndarray:
    """Mean (t, y, x) latent coordinate of the valid tokens of each block, [NQB][3] float64.
    Token n -> t = n // (Hl*Wl), y = (n % (Hl*Wl)) // Wl, x = n % Wl (frame-major)."""
    assert cfg.grid is not None and cfg.Bq == cfg.Bk
    T, Hl, Wl = cfg.grid
    assert T * Hl * Wl == cfg.n_valid, (cfg.grid, cfg.n_valid)
    n = np.arange(cfg.n_valid)
    coords = np.stack([n // (Hl * Wl), (n % (Hl * Wl)) // Wl, n % Wl], axis=1).astype(np.float64)
    cent = np.zeros((cfg.NQB, 3), dtype=np.float64)
    for u in range(cfg.NQB):
        lo, hi = u * cfg.Bq, min((u + 1) * cfg.Bq, cfg.n_valid)
        cent[u] = coords[lo:hi].mean(axis=0)
    return cent


def make_block_scores(cfg: Config, uniform_density: Optional[float] = None,
                      mask_seed: Optional[int] = None):
    """Structured block scores + per-head densities (BASELINE.json configs 1-4):
        score[h][u][v] = exp(-||c_u - c_v||_2 / sigma_h) + 0.05 * U(0,1),
        +1.0 on 2 seeded-random key-block columns per head ("sinks"),
        sigma_h ~ LogU(sigma_lo, sigma_hi), density_h ~ U(density_lo, density_hi)
    (or every head at `uniform_density`, BASELINE.json config 4 / C5).
    Returns (scores float32 [H][NQB][NKB], density float32 [H], sigma float64 [H])."""
    seed = cfg.mask_seed if mask_seed is None else mask_seed
    rng = np.random.Generator(np.random.PCG64(seed))
    cent = block_centroids(cfg)
    dist = np.sqrt(((cent[:, None, :] - cent[None, :, :]) ** 2).sum(-1))
    sigma = np.exp(rng.uniform(math.log(cfg.sigma_lo), math.log(cfg.sigma_hi), size=cfg.H))
    density = rng.uniform(cfg.density_lo, cfg.density_hi, size=cfg.H)
    if uniform_density is not None:
        density = np.full(cfg.H, float(uniform_density))
    scores = np.empty((cfg.H, cfg.NQB, cfg.NKB), dtype=np.float32)
    for h in range(cfg.H):
        s = np.exp(-dist / sigma[h]) + 0.05 * rng.random((cfg.NQB, cfg.NKB))
        sinks = rng.choice(cfg.NKB, size=2, replace=False)
        s[:, sinks] += 1.0
        scores[h] = s.astype(np.float32)
    return scores, density.astype(np.float32), sigma


def iid_block_mask(H: int, NQB: int, NKB: int, density: float, seed: int) -> np.ndarray:
    """C1 mask: diagonal on, every other block on i.i.d. with the p that gives `density`
    overall. Boolean [H][NQB][NKB] (not packed: packing is the method's job)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    ndiag = min(NQB, NKB)
    p = (density * NQB * NKB - ndiag) / (NQB * NKB - ndiag)
    m = rng.random((H, NQB, NKB)) < p
    for u in range(ndiag):
        m[:, u, u] = True
    return m


def adversarial_block_mask(H: int, NQB: int, dense_frac: float, seed: int) -> np.ndarray:
    """C5 imbalance case: per head a seeded `dense_frac` of the query blocks is fully dense,
    every other row holds only its diagonal block."""
    rng = np.random.Generator(np.random.PCG64(seed))
    m = np.zeros((H, NQB, NQB), dtype=bool)
    n_dense = int(round(dense_frac * NQB))
    for h in range(H):
        m[h, np.arange(NQB), np.arange(NQB)] = True
        rows = rng.choice(NQB, size=n_dense, replace=False)
        m[h, rows, :] = True
    return m


def bool_mask_as_scores(m: np.ndarray):
    """A boolean block mask expressed as (scores, density) so that a top-fraction selection
    reproduces it exactly: score 1 where on, 0 where off, density = count / total per head.
    (count/total in fp32 is off by < 1e-7 relative, far less than half a block.)"""
    H, NQB, NKB = m.shape
    scores = m.astype(np.float32)
    cnt = m.reshape(H, -1).sum(axis=1)
    assert (cnt >= 1).all()
    density = (cnt.astype(np.float64) / (NQB * NKB)).astype(np.float32)
    return scores, density


def sample_units(row_popcount: np.ndarray, seed: int, n_heads: int = 8, n_random_rows: int = 4):
    """Units (b=0, h, u) on which the oracle is run at the large configs: for the
    densest head, the sparsest head and seeded-random heads: query blocks 0, NQB-1, the heaviest
    row, the lightest row and `n_random_rows` seeded-random rows. `row_popcount` is int [H][NQB]."""
    H, NQB = row_popcount.shape
    rng = np.random.Generator(np.random.PCG64(seed))
    per_head = row_popcount.sum(axis=1)
    heads = [int(per_head.argmax()), int(per_head.argmin())]
    others = [h for h in rng.permutation(H).tolist() if h not in heads]
    heads = (heads + others)[:min(n_heads, H)]
    units = []
    for h in heads:
        rows = [0, NQB - 1, int(row_popcount[h].argmax()), int(row_popcount[h].argmin())]
        rows += rng.integers(0, NQB, size=n_random_rows).tolist()
        seen = []
        for u in rows:
            if u not in seen:
                seen.append(u)
        units += [(0, h, int(u)) for u in seen]
    return np.asarray(units, dtype=np.int32)


# ---- second workload: the paper's own kernel experiment, a sequence-length
# x sparsity grid at block 128 (Sec. 5.3, Fig. 5 caption PAPER.md:250; 1K..262K
# tokens), plus a HunyuanVideo-shaped layer (33 frames x 1350 tokens = 44 550 tokens).
# The paper gives no head count / head dim for it: H and D are parameters here.
SEQ_GRID_N = (1024, 4096, 16384, 65536, 262144)
SEQ_GRID_DENSITY = (1.0, 0.5, 0.25, 0.1, 0.05)


def seq_grid_config(N: int, H: int, n_valid: Optional[int] = None, seed: int = 7) -> Config:
    """One cell's shape: B=1, D=128, 128-blocks, no latent grid (masks are i.i.d., see
    `iid_block_scores`)."""
    return Config(f"grid-N{N}-H{H}", 1, H, N, 128, 128, 128, N if n_valid is None else n_valid,
                  None, 1000 + seed, 2000 + seed, 0.0, 0.0)


HUNYUAN = Config("hunyuan-33x1350", 1, 24, 44672, 128, 128, 128, 44550, None, 11, 111, 0.0, 0.0)


def iid_block_scores(cfg: Config, density: float, seed: Optional[int] = None):
    """Block scores ~ i.i.d. U(0,1) (seeded) with every head at `density`: their per-head
    top-fraction is a uniformly random mask with exactly that density (diagonal forced by the
    pack call). Returns (scores float32 [H][NQB][NKB], density float32 [H])."""
    rng = np.random.Generator(np.random.PCG64(cfg.mask_seed if seed is None else seed))
    scores = rng.random((cfg.H, cfg.NQB, cfg.NKB), dtype=np.float32)
    return scores, np.full(cfg.H, float(density), dtype=np.float32)

"""Seeded synthetic inputs shaped like the paper's workloads (BASELINE.json configs C1..C5).

A module of its own: it serves both the CPU oracle's tests and the CUDA path's tests/bench, and
holds NONE of the method's arithmetic (no scoring, no tiering, no quantisation) -- only random
K / V / Q tensors and the per-config policy parameters.  Recipe:

  * torch.Generator seeded  seed + 1000*request + {K:1, V:2, Q:3, channel choice:4}
  * values drawn in fp32, clamped to +-65504, cast to fp16 (round to nearest even)
  * K "tiny"      : N(0,1), channels 0..3 scaled x8
    K "outlier"   : N(0,1), round(0.05*d) channels per (layer, kv-head) scaled x10 (fixed over tokens)
    K "student_t" : z / sqrt((g1^2+g2^2+g3^2)/3) / sqrt(3)   (Student-t nu=3 scaled to unit variance)
  * V ~ N(0,1), Q ~ N(0,1)
  * layout token-major  K,V [L][n][Hkv][d],  Q [L][Hq][w][d]

These stand in for the KV caches of Qwen2.5-7B / Mistral-7B / Gemma-2-9B on the paper's prompts
(Table 4 seq 4096, Table 7 tier policy), which need trained weights and datasets
that are not available; nothing here reproduces any dataset item.
"""
from dataclasses import dataclass, field
from typing import Tuple

import torch


@dataclass(frozen=True)
class Config:
    name: str
    L: int
    Hq: int
    Hkv: int
    d: int
    n: int
    w: int
    R: int = 1
    k_dist: str = "outlier"
    budgets: Tuple[float, ...] = (0.5,)
    n_sink: int = 4
    ranges: Tuple[Tuple[int, int], ...] = ()
    allow_int4: bool = True
    seed: int = 0

    @property
    def bytes_fp16(self) -> int:
        """Eq. 1: 2 * L * Hkv * d * n * 2 bytes, per request."""
        return 2 * self.L * self.Hkv * self.d * self.n * 2

    def scaled(self, **kw) -> "Config":
        from dataclasses import replace
        return replace(self, **kw)


CONFIGS = {
    "C1": Config("C1-tiny", L=1, Hq=2, Hkv=2, d=128, n=256, w=16, k_dist="tiny", budgets=(0.5,)),
    "C2": Config("C2-qwen2.5-7b-shaped", L=28, Hq=28, Hkv=4, d=128, n=4096, w=32,
                 budgets=(0.3, 0.5), allow_int4=False),
    "C3": Config("C3-mistral-7b-shaped", L=32, Hq=32, Hkv=8, d=128, n=4096, w=32,
                 budgets=(0.3, 0.5), ranges=((4032, 4096),)),
    "C4": Config("C4-gemma-2-9b-shaped", L=42, Hq=16, Hkv=8, d=256, n=4096, w=32,
                 k_dist="student_t", budgets=(0.5,)),
    "C5": Config("C5-long-mistral-7b-shaped", L=32, Hq=32, Hkv=8, d=128, n=32768, w=64, R=4,
                 budgets=(0.3, 0.4, 0.5, 0.75, 1.0)),
}


def _gen(cfg: Config, request: int, which: int, device) -> torch.Generator:
    g = torch.Generator(device=device)
    g.manual_seed(cfg.seed + 1000 * request + which)
    return g


def _to_f16(x: torch.Tensor) -> torch.Tensor:
    return x.clamp_(-65504.0, 65504.0).to(torch.float16)


def make_kv(cfg: Config, request: int = 0, device="cpu", layers=None):
    """Returns (K, V) fp16 [L'][n][Hkv][d] for `layers` (default all), generated layer by layer."""
    dev = torch.device(device)
    gk, gv, gc = _gen(cfg, request, 1, dev), _gen(cfg, request, 2, dev), _gen(cfg, request, 4, dev)
    want = list(range(cfg.L)) if layers is None else list(layers)
    K = torch.empty((len(want), cfg.n, cfg.Hkv, cfg.d), dtype=torch.float16, device=dev)
    V = torch.empty_like(K)
    shape = (cfg.n, cfg.Hkv, cfg.d)
    n_out = int(round(0.05 * cfg.d))
    for l in range(max(want) + 1 if want else 0):
        # draw every layer up to the last wanted one so that a layer's bytes do not depend on `layers`
        if cfg.k_dist == "student_t":
            z = torch.randn((4,) + shape, generator=gk, device=dev, dtype=torch.float32)
            k = z[0] / torch.sqrt((z[1] ** 2 + z[2] ** 2 + z[3] ** 2) / 3.0) / (3.0 ** 0.5)
        else:
            k = torch.randn(shape, generator=gk, device=dev, dtype=torch.float32)
            if cfg.k_dist == "tiny":
                k[:, :, 0:4] *= 8.0
            elif cfg.k_dist == "outlier":
                for h in range(cfg.Hkv):
                    ch = torch.randperm(cfg.d, generator=gc, device=dev)[:n_out]
                    k[:, h, ch] *= 10.0
            elif cfg.k_dist != "normal":
                raise ValueError(cfg.k_dist)
        v = torch.randn(shape, generator=gv, device=dev, dtype=torch.float32)
        if l in want:
            K[want.index(l)] = _to_f16(k)
            V[want.index(l)] = _to_f16(v)
    return K, V


def make_q(cfg: Config, request: int = 0, device="cpu", layers=None):
    """Observation-window queries fp16 [L'][Hq][w][d] ~ N(0,1); query i sits at position n-w+i."""
    dev = torch.device(device)
    g = _gen(cfg, request, 3, dev)
    want = list(range(cfg.L)) if layers is None else list(layers)
    Q = torch.empty((len(want), cfg.Hq, cfg.w, cfg.d), dtype=torch.float16, device=dev)
    for l in range(max(want) + 1 if want else 0):
        q = torch.randn((cfg.Hq, cfg.w, cfg.d), generator=g, device=dev, dtype=torch.float32)
        if l in want:
            Q[want.index(l)] = _to_f16(q)
    return Q


def make_importance(cfg: Config, request: int = 0, device="cpu"):
    """A stand-in importance vector f32 [L][n] (positive, heavy-tailed, with a few exact duplicates)
    for tests that exercise selection / pack / unpack without running the importance step."""
    dev = torch.device(device)
    g = _gen(cfg, request, 5, dev)
    x = torch.rand((cfg.L, cfg.n), generator=g, device=dev, dtype=torch.float32)
    I = (x ** 4) / cfg.n
    if cfg.n >= 16:
        I[:, 7] = I[:, 11]          # exact ties, to exercise the position tie-break
        I[:, cfg.n - 3] = I[:, 5]
    return I

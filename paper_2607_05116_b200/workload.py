"""Seeded synthetic routing workloads (inputs only -- none of the method's arithmetic).

Stand-ins for the paper's routing traces (Qwen3-30B-A3B / DeepSeek-V2-Lite served on
LMSYS-Chat and Arxiv Abstracts), which are not available here; the shapes and
distributions follow BASELINE.json's five configs.  The recipe is stated in DESIGN.md
section 4.  Everything is a stateless hash of (seed, layer, token, expert), so any token
range can be regenerated independently (numpy on the host; no libm in the per-token
data path, so the bits do not depend on the platform).

Used by tests/, bench.py and __graft_entry__.py to feed BOTH the CUDA path and the CPU
oracle; it imports neither.
"""
from dataclasses import dataclass, field
from typing import Optional, Tuple

import numpy as np

_U = np.uint64


def splitmix64(x):
    """splitmix64 finaliser on a uint64 array (wrap-around arithmetic)."""
    with np.errstate(over="ignore"):
        z = np.asarray(x, dtype=_U) + _U(0x9E3779B97F4A7C15)
        z = (z ^ (z >> _U(30))) * _U(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> _U(27))) * _U(0x94D049BB133111EB)
        return z ^ (z >> _U(31))


def _key(seed: int, layer: int, domain: int) -> np.uint64:
    a = splitmix64(np.array([layer], dtype=_U))[0]
    return splitmix64(np.array([_U(seed) ^ a ^ _U(domain)], dtype=_U))[0]


_DOM_NOISE = 0x6E6F697365  # "noise"
_DOM_CLUST = 0x636C757374  # "clust"
_DOM_PERM = 0x7065726D00   # "perm"
_DOM_BIAS = 0x6269617300   # "bias"
_DOM_SRC = 0x7372630000    # "src"

_SIGMA = float(np.sqrt(8.0 * (65536.0 ** 2 - 1.0) / 12.0))   # Irwin-Hall(8) of 16-bit lanes
_INV_SIGMA = np.float32(1.0 / _SIGMA)


@dataclass(frozen=True)
class Config:
    name: str
    index: int                 # 1..5, BASELINE.json order
    L: int
    E: int
    k: int
    T: int
    D: int
    N: int
    P: int
    taus: Tuple[float, ...]
    zipf_s: float
    clusters: Optional[Tuple[int, int, float]]   # (n_clusters, size, p_active) or None
    scoring: int = 0           # 0 softmax, 1 sigmoid
    renormalize: int = 1
    n_group: int = 1
    topk_group: int = 1
    group_score: int = 0
    has_bias: bool = False
    cost_inter: int = 1
    bytes_per_token: int = 4096
    zipf_alpha: float = 0.25
    boost: float = 2.0

    @property
    def gate(self):
        return dict(k=self.k, scoring=self.scoring, renormalize=self.renormalize,
                    n_group=self.n_group, topk_group=self.topk_group,
                    group_score=self.group_score, scale=1.0)

    def seed(self, layer: int) -> int:
        return 0xCA90000 + self.index * 256 + layer

    def with_(self, **kw):
        d = dict(self.__dict__)
        d.update(kw)
        return Config(**d)


CONFIGS = {
    "tiny": Config("tiny", 1, L=1, E=16, k=2, T=4096, D=4, N=1, P=4, taus=(0.1,), zipf_s=1.0,
                   clusters=None, renormalize=1),
    "qwen3": Config("qwen3", 2, L=48, E=128, k=8, T=16384, D=8, N=1, P=64, taus=(0.05, 0.1),
                    zipf_s=1.1, clusters=(16, 8, 0.6)),
    "target": Config("target", 3, L=1, E=128, k=8, T=65536, D=16, N=2, P=256, taus=(0.1,),
                     zipf_s=1.1, clusters=(16, 8, 0.6), cost_inter=4),
    "dsv3": Config("dsv3", 4, L=58, E=256, k=8, T=32768, D=32, N=4, P=128, taus=(0.05,),
                   zipf_s=1.2, clusters=(32, 8, 0.5), scoring=1, n_group=8, topk_group=4,
                   group_score=1, has_bias=True, cost_inter=4, bytes_per_token=14336),
    "stress": Config("stress", 5, L=1, E=512, k=10, T=65536, D=64, N=8, P=1024, taus=(0.1,),
                     zipf_s=1.0, clusters=(64, 8, 0.5), renormalize=1, cost_inter=4),
}


def _perm(seed: int, layer: int, n: int, stream: int) -> np.ndarray:
    """Seeded permutation of range(n): stable argsort of hashes."""
    key = _key(seed, layer, _DOM_PERM + stream)
    with np.errstate(over="ignore"):
        h = splitmix64(key + np.arange(n, dtype=_U))
    return np.argsort(h, kind="stable").astype(np.int64)


def zipf_bias(cfg: Config, layer: int) -> np.ndarray:
    """Per-expert popularity term alpha*(ln pop - mean ln pop), pop ~ rank^-s, fp32 [E]."""
    rank = np.empty(cfg.E, np.int64)
    rank[_perm(cfg.seed(layer), layer, cfg.E, 1)] = np.arange(1, cfg.E + 1)
    lp = -cfg.zipf_s * np.log(rank.astype(np.float64))
    return (cfg.zipf_alpha * (lp - lp.mean())).astype(np.float32)


def cluster_members(cfg: Config, layer: int) -> Optional[np.ndarray]:
    """[n_clusters, size] expert ids: a seeded random partition (not contiguous)."""
    if cfg.clusters is None:
        return None
    n, size, _ = cfg.clusters
    perm = _perm(cfg.seed(layer), layer, cfg.E, 2)
    return perm[: n * size].reshape(n, size)


def logits(cfg: Config, layer: int, t0: int = 0, t1: Optional[int] = None) -> np.ndarray:
    """fp32 [t1-t0, E] router logits of tokens t0..t1 of one layer."""
    t1 = cfg.T if t1 is None else t1
    E = cfg.E
    seed = cfg.seed(layer)
    key = _key(seed, layer, _DOM_NOISE)
    out = np.empty((t1 - t0, E), np.float32)
    zb = zipf_bias(cfg, layer)
    mem = cluster_members(cfg, layer)
    chunk = max(1, (1 << 22) // E)
    for a in range(t0, t1, chunk):
        b = min(t1, a + chunk)
        with np.errstate(over="ignore"):
            i = (np.arange(a, b, dtype=_U)[:, None] * _U(E) + np.arange(E, dtype=_U)[None, :]) * _U(2)
            h0 = splitmix64(key + i)
            h1 = splitmix64(key + i + _U(1))
        S = np.zeros(h0.shape, np.int64)
        for h in (h0, h1):
            for sh in (0, 16, 32, 48):
                S += ((h >> _U(sh)) & _U(0xFFFF)).astype(np.int64)
        z = (S - 262140).astype(np.float32) * _INV_SIGMA
        x = z + zb[None, :]
        if mem is not None:
            n, size, pact = cfg.clusters
            ck = _key(seed, layer, _DOM_CLUST)
            with np.errstate(over="ignore"):
                hc = splitmix64(ck + np.arange(a, b, dtype=_U))
            active = (hc & _U(0xFFFFFFFF)) < _U(int(pact * 4294967296.0))
            cid = ((hc >> _U(32)) % _U(n)).astype(np.int64)
            boost = np.zeros((b - a, E), np.float32)
            rows = np.nonzero(active)[0]
            boost[rows[:, None], mem[cid[rows]]] = np.float32(cfg.boost)
            x = x + boost
        out[a - t0:b - t0] = x
    return out


def gate_bias(cfg: Config, layer: int) -> Optional[np.ndarray]:
    """fp32 [E] selection bias for sigmoid scoring: uniform in +-0.05 (16-bit lanes)."""
    if not cfg.has_bias:
        return None
    key = _key(cfg.seed(layer), layer, _DOM_BIAS)
    with np.errstate(over="ignore"):
        h = splitmix64(key + np.arange(cfg.E, dtype=_U))
    lane = (h & _U(0xFFFF)).astype(np.int64) - 32768
    return (lane.astype(np.float32) * np.float32(0.05 / 32768.0)).astype(np.float32)


def dev_node(cfg: Config) -> np.ndarray:
    return (np.arange(cfg.D) // (cfg.D // cfg.N)).astype(np.int32)


def token_src_random(cfg: Config, layer: int, T: Optional[int] = None) -> np.ndarray:
    """Seeded non-contiguous source devices, int32 [T] (exercises the general path)."""
    T = cfg.T if T is None else T
    key = _key(cfg.seed(layer), layer, _DOM_SRC)
    with np.errstate(over="ignore"):
        h = splitmix64(key + np.arange(T, dtype=_U))
    return ((h >> _U(33)) % _U(cfg.D)).astype(np.int32)


def candidates(cfg: Config, layer: int, P: Optional[int] = None) -> np.ndarray:
    """int32 [P, E] expert->device maps, every device hosting E/D experts.

    p0 sequential (the paper's Default), p1 round-robin, p2 cluster-aligned (the
    generator's planted structure), then cluster-aligned with 1,2,3,... seeded swaps (a
    spectrum like P:L194-200) up to P/2, the rest balanced random permutations.
    """
    P = cfg.P if P is None else P
    E, D = cfg.E, cfg.D
    per = E // D
    seed = cfg.seed(layer)
    out = np.empty((P, E), np.int32)
    e = np.arange(E)
    mem = cluster_members(cfg, layer)
    for p in range(P):
        if p == 0:
            m = e // per
        elif p == 1:
            m = e % D
        elif mem is not None and p < max(3, P // 2):
            order = np.concatenate([mem.reshape(-1),
                                    np.setdiff1d(e, mem.reshape(-1), assume_unique=False)])
            m = np.empty(E, np.int64)
            m[order] = np.arange(E) // per
            nsw = p - 2
            if nsw:
                key = _key(seed, layer, _DOM_PERM + 1000 + p)
                with np.errstate(over="ignore"):
                    h = splitmix64(key + np.arange(2 * nsw, dtype=_U))
                for s in range(nsw):
                    i, j = int(h[2 * s] % _U(E)), int(h[2 * s + 1] % _U(E))
                    m[i], m[j] = m[j], m[i]
        else:
            perm = _perm(seed, layer, E, 100 + p)
            m = np.empty(E, np.int64)
            m[perm] = np.arange(E) // per
        out[p] = m
    return out


def layer_inputs(cfg: Config, layer: int, T: Optional[int] = None):
    """(logits [T,E], bias [E]|None, expert_dev [P,E]) of one layer."""
    T = cfg.T if T is None else T
    return logits(cfg, layer, 0, T), gate_bias(cfg, layer), candidates(cfg, layer)

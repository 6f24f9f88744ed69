"""Device-side twin of workload.logits: the same stateless hash evaluated with
torch integer ops on the GPU, so that the large workloads (config 4: 1.95 GB of logits, config 5 at
2^20..2^22 tokens: up to 8.6 GB) are filled in HBM instead of being hashed on the host and copied over
PCIe.  Inputs only, none of the method's arithmetic; it imports neither the CUDA library nor the
oracle.  Every user checks a sample of rows bit for bit against the host generator
(check_rows_against_host) before trusting the rest.
"""
import numpy as np
import torch

from . import workload as W

_M64 = (1 << 64) - 1


def _s64(v: int) -> int:
    """uint64 constant -> the int64 with the same bits (torch has no uint64 arithmetic)."""
    v &= _M64
    return v - (1 << 64) if v >= (1 << 63) else v


def _lsr(z, s):
    """logical right shift of int64 bit patterns"""
    return (z >> s) & ((1 << (64 - s)) - 1)


def splitmix64_t(x):
    z = x + _s64(0x9E3779B97F4A7C15)
    z = (z ^ _lsr(z, 30)) * _s64(0xBF58476D1CE4E5B9)
    z = (z ^ _lsr(z, 27)) * _s64(0x94D049BB133111EB)
    return z ^ _lsr(z, 31)


def logits_device(cfg, layer, t0=0, t1=None, out=None, chunk_tokens=None, device="cuda"):
    """fp32 [t1-t0, E] on the device, bit-identical to W.logits(cfg, layer, t0, t1)."""
    t1 = cfg.T if t1 is None else t1
    E = cfg.E
    seed = cfg.seed(layer)
    key = _s64(int(W._key(seed, layer, W._DOM_NOISE)))
    zb = torch.from_numpy(W.zipf_bias(cfg, layer)).to(device)
    mem = W.cluster_members(cfg, layer)
    mem_t = None if mem is None else torch.from_numpy(mem.astype(np.int64)).to(device)
    if out is None:
        out = torch.empty((t1 - t0, E), dtype=torch.float32, device=device)
    chunk = chunk_tokens or max(1, (1 << 24) // E)
    e_ar = torch.arange(E, dtype=torch.int64, device=device)[None, :]
    inv_sigma = torch.tensor(float(W._INV_SIGMA), dtype=torch.float32, device=device)
    for a in range(t0, t1, chunk):
        b = min(t1, a + chunk)
        t_ar = torch.arange(a, b, dtype=torch.int64, device=device)
        i = (t_ar[:, None] * E + e_ar) * 2
        S = torch.zeros(i.shape, dtype=torch.int64, device=device)
        for off in (0, 1):
            h = splitmix64_t(i + (key + off))
            for sh in (0, 16, 32, 48):
                S += _lsr(h, sh) & 0xFFFF if sh else h & 0xFFFF
            del h
        z = (S - 262140).to(torch.float32) * inv_sigma
        del S, i
        x = z + zb[None, :]
        if mem_t is not None:
            n, size, pact = cfg.clusters
            ck = _s64(int(W._key(seed, layer, W._DOM_CLUST)))
            hc = splitmix64_t(t_ar + ck)
            active = (hc & 0xFFFFFFFF) < int(pact * 4294967296.0)
            cid = _lsr(hc, 32) % n
            boost = torch.zeros((b - a, E), dtype=torch.float32, device=device)
            rows = torch.nonzero(active)[:, 0]
            boost[rows[:, None], mem_t[cid[rows]]] = float(np.float32(cfg.boost))
            x = x + boost
            del boost
        out[a - t0:b - t0] = x
    return out


def check_rows_against_host(cfg, layer, x_dev, rows, t0=0):
    """assert that rows (token numbers) of x_dev equal the host generator bit for bit"""
    rows = np.asarray(rows, dtype=np.int64)
    got = x_dev[torch.from_numpy(rows - t0).to(x_dev.device)].cpu().numpy()
    for j, t in enumerate(rows):
        ref = W.logits(cfg, layer, int(t), int(t) + 1)[0]
        assert np.array_equal(got[j].view(np.uint32), ref.view(np.uint32)), f"generator mismatch at token {t}"

"""ctypes front-end to the CPU oracle (oracle/cap_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this module.  It takes
and returns numpy arrays on the host and never touches the CUDA path.
"""
import ctypes as C
from types import SimpleNamespace

import numpy as np

from . import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.capo_exp_s.restype = C.c_float
        _lib.capo_exp_s.argtypes = [C.c_float]
        _lib.capo_sig_s.restype = C.c_float
        _lib.capo_sig_s.argtypes = [C.c_float]
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _c(a, dt):
    if a is None:
        return None
    a = np.ascontiguousarray(a, dtype=dt)
    return a


def exp_s(x):
    return float(lib().capo_exp_s(C.c_float(float(x))))


def sig_s(x):
    return float(lib().capo_sig_s(C.c_float(float(x))))


def gate_topk(logits, bias=None, *, k, scoring=0, renormalize=1, n_group=1, topk_group=1,
              group_score=0, scale=1.0):
    """S1. logits [L,T,E] fp32 -> (idx [L,T,k] int32, w [L,T,k] fp32)."""
    logits = _c(logits, np.float32)
    L, T, E = logits.shape
    bias = _c(bias, np.float32)
    idx = np.empty((L, T, k), np.int32)
    w = np.empty((L, T, k), np.float32)
    rc = lib().capo_gate_topk(_p(logits), _p(bias), C.c_int32(L), C.c_int64(T), C.c_int32(E),
                              C.c_int32(k), C.c_int32(scoring), C.c_int32(renormalize),
                              C.c_int32(n_group), C.c_int32(topk_group), C.c_int32(group_score),
                              C.c_float(scale), _p(idx), _p(w))
    if rc != 0:
        raise ValueError(f"capo_gate_topk -> {rc}")
    return idx, w


def coactivation(idx, kept=None, *, E):
    """S2. idx [L,T,k] -> (counts [L,E] int64, coact [L,E,E] int32)."""
    idx = _c(idx, np.int32)
    L, T, k = idx.shape
    kept = _c(kept, np.uint8)
    counts = np.empty((L, E), np.int64)
    coact = np.empty((L, E, E), np.int32)
    rc = lib().capo_coactivation(_p(idx), _p(kept), C.c_int32(L), C.c_int64(T), C.c_int32(k),
                                 C.c_int32(E), _p(counts), _p(coact))
    if rc != 0:
        raise ValueError(f"capo_coactivation -> {rc}")
    return counts, coact


def eval_placements(idx, expert_dev, dev_node, *, kept=None, token_src=None, E=None,
                    cost_local=0, cost_intra=1, cost_inter=1, bytes_per_token=0,
                    per_token=False):
    """S3. idx [L,T,k]; expert_dev [L,P,E]; dev_node [D] -> namespace of arrays."""
    idx = _c(idx, np.int32)
    L, T, k = idx.shape
    expert_dev = _c(expert_dev, np.int32)
    _, P, E2 = expert_dev.shape
    E = E2 if E is None else E
    dev_node = _c(dev_node, np.int32)
    D = dev_node.shape[0]
    N = int(dev_node.max()) + 1 if D else 1
    kept = _c(kept, np.uint8)
    token_src = _c(token_src, np.int32)
    o = SimpleNamespace()
    for name in ("dev_visits", "remote_dev", "remote_intra", "remote_inter", "node_visits",
                 "remote_node", "cost", "bytes"):
        setattr(o, name, np.empty((L, P), np.int64))
    o.load_pairs = np.empty((L, P, D), np.int64)
    o.recv_tokens = np.empty((L, P, D), np.int64)
    o.imbalance = np.empty((L, P), np.float64)
    o.imbalance_recv = np.empty((L, P), np.float64)
    o.tok_remote_dev = np.empty((L, P, T), np.uint8) if per_token else None
    o.tok_remote_node = np.empty((L, P, T), np.uint8) if per_token else None
    rc = lib().capo_eval_placements(
        _p(idx), _p(kept), _p(token_src), C.c_int32(L), C.c_int64(T), C.c_int32(k), C.c_int32(E),
        _p(expert_dev), C.c_int32(P), C.c_int32(D), C.c_int32(N), _p(dev_node),
        C.c_int32(cost_local), C.c_int32(cost_intra), C.c_int32(cost_inter),
        C.c_int64(bytes_per_token),
        _p(o.dev_visits), _p(o.remote_dev), _p(o.remote_intra), _p(o.remote_inter),
        _p(o.node_visits), _p(o.remote_node), _p(o.cost), _p(o.bytes),
        _p(o.load_pairs), _p(o.recv_tokens), _p(o.imbalance), _p(o.imbalance_recv),
        _p(o.tok_remote_dev), _p(o.tok_remote_node))
    if rc != 0:
        raise ValueError(f"capo_eval_placements -> {rc}")
    return o


def prune(idx, w, expert_dev, dev_node, p, *, token_src=None, cost_local=0, cost_intra=1,
          cost_inter=1):
    """S4. idx,w [L,T,k]; expert_dev [L,E] -> (kept [L,T,k] uint8, near_margin [L] int64)."""
    idx = _c(idx, np.int32)
    w = _c(w, np.float32)
    L, T, k = idx.shape
    expert_dev = _c(expert_dev, np.int32)
    E = expert_dev.shape[-1]
    dev_node = _c(dev_node, np.int32)
    D = dev_node.shape[0]
    N = int(dev_node.max()) + 1
    token_src = _c(token_src, np.int32)
    kept = np.empty((L, T, k), np.uint8)
    near = np.zeros((L,), np.int64)
    rc = lib().capo_prune(_p(idx), _p(w), _p(token_src), C.c_int32(L), C.c_int64(T), C.c_int32(k),
                          C.c_int32(E), _p(expert_dev), C.c_int32(D), C.c_int32(N), _p(dev_node),
                          C.c_int32(cost_local), C.c_int32(cost_intra), C.c_int32(cost_inter),
                          C.c_float(p), _p(kept), _p(near))
    if rc != 0:
        raise ValueError(f"capo_prune -> {rc}")
    return kept, near


def dispatch_layout(idx, expert_dev, D, *, kept=None, want_pos=True):
    """S5. idx [T,k]; expert_dev [E] -> (sorted_pairs [n_kept], offsets [D+1], pair_pos [T*k])."""
    idx = _c(idx, np.int32)
    T, k = idx.shape
    expert_dev = _c(expert_dev, np.int32)
    E = expert_dev.shape[0]
    kept = _c(kept, np.uint8)
    sorted_pairs = np.empty((T * k,), np.int32)
    pair_pos = np.empty((T * k,), np.int32) if want_pos else None
    offsets = np.empty((D + 1,), np.int64)
    rc = lib().capo_dispatch_layout(_p(idx), _p(kept), C.c_int64(T), C.c_int32(k), C.c_int32(E),
                                    _p(expert_dev), C.c_int32(D), _p(sorted_pairs), _p(pair_pos),
                                    _p(offsets))
    if rc != 0:
        raise ValueError(f"capo_dispatch_layout -> {rc}")
    return sorted_pairs[: int(offsets[D])], offsets, pair_pos


def trace_fused(logits, bias, gate, expert_dev, dev_node, *, token_src=None, cost_local=0,
                cost_intra=1, cost_inter=1, bytes_per_token=0, per_token=False):
    """S1 -> S2 -> S3 composed (what cap_trace_fused computes in one pass)."""
    idx, w = gate_topk(logits, bias, **gate)
    E = logits.shape[-1]
    counts, coact = coactivation(idx, E=E)
    ev = eval_placements(idx, expert_dev, dev_node, token_src=token_src, cost_local=cost_local,
                         cost_intra=cost_intra, cost_inter=cost_inter,
                         bytes_per_token=bytes_per_token, per_token=per_token)
    return idx, w, counts, coact, ev


def coact_placement(counts, coact, *, D, N, rnd=None, want_p=False):
    """NEXT-1: Jaccard p_ij + Algorithm 1 (device groups, then node groups).

    counts [L,E] int64, coact [L,E,E] int32, rnd [L,E+D] uint32 or None ->
    (expert_group [L,E], group_node [L,D], expert_dev [L,E], p [L,E,E] fp64 or None)."""
    counts = _c(counts, np.int64)
    coact = _c(coact, np.int32)
    L, E = counts.shape
    rnd = _c(rnd, np.uint32)
    p = np.empty((L, E, E), np.float64) if want_p else None
    expert_group = np.empty((L, E), np.int32)
    group_node = np.empty((L, D), np.int32)
    expert_dev = np.empty((L, E), np.int32)
    rc = lib().capo_coact_placement(_p(counts), _p(coact), C.c_int32(L), C.c_int32(E), C.c_int32(D),
                                    C.c_int32(N), _p(rnd), _p(p), _p(expert_group), _p(group_node),
                                    _p(expert_dev))
    if rc != 0:
        raise ValueError(f"capo_coact_placement -> {rc}")
    return expert_group, group_node, expert_dev, p


def pairwise_objective(counts, coact, expert_dev, dev_node, *, cost_intra=1, cost_inter=1, lam=0.5,
                       imbalance=None):
    """NEXT-3: Eq. 2-3 for P candidates from (counts, coact).  expert_dev [L,P,E] ->
    (obj_count [L,P] int64, obj_prob [L,P] fp64, combined [L,P] fp64 or None)."""
    counts = _c(counts, np.int64)
    coact = _c(coact, np.int32)
    expert_dev = _c(expert_dev, np.int32)
    dev_node = _c(dev_node, np.int32)
    L, P, E = expert_dev.shape
    D = dev_node.shape[0]
    imbalance = _c(imbalance, np.float64)
    oc = np.empty((L, P), np.int64)
    op = np.empty((L, P), np.float64)
    cb = np.empty((L, P), np.float64) if imbalance is not None else None
    rc = lib().capo_pairwise_objective(_p(counts), _p(coact), C.c_int32(L), C.c_int32(E), _p(expert_dev),
                                       C.c_int32(P), C.c_int32(D), _p(dev_node), C.c_int32(cost_intra),
                                       C.c_int32(cost_inter), C.c_double(lam), _p(imbalance), _p(oc),
                                       _p(op), _p(cb))
    if rc != 0:
        raise ValueError(f"capo_pairwise_objective -> {rc}")
    return oc, op, cb


def dispatch_rows(idx, expert_dev, D, *, kept=None):
    """NEXT-4: one row per (token, destination device).  idx [T,k]; expert_dev [E] ->
    (rows_token [n_rows], row_offsets [D+1], pair_row [T*k])."""
    idx = _c(idx, np.int32)
    T, k = idx.shape
    expert_dev = _c(expert_dev, np.int32)
    E = expert_dev.shape[0]
    kept = _c(kept, np.uint8)
    rows = np.empty((T * k,), np.int32)
    pair_row = np.empty((T * k,), np.int32)
    offsets = np.empty((D + 1,), np.int64)
    rc = lib().capo_dispatch_rows(_p(idx), _p(kept), C.c_int64(T), C.c_int32(k), C.c_int32(E),
                                  _p(expert_dev), C.c_int32(D), _p(rows), _p(pair_row), _p(offsets))
    if rc != 0:
        raise ValueError(f"capo_dispatch_rows -> {rc}")
    return rows[: int(offsets[D])], offsets, pair_row


def adjust_spectrum(counts, coact, expert_dev0, *, D, S):
    """NEXT-2: S swap steps of the Adjustment Approach (reading R27).  expert_dev0 [L,E] ->
    (spectrum [L,S,E], n_done [L], swaps [L,S,2])."""
    counts = _c(counts, np.int64)
    coact = _c(coact, np.int32)
    expert_dev0 = _c(expert_dev0, np.int32)
    L, E = expert_dev0.shape
    spectrum = np.empty((L, S, E), np.int32)
    n_done = np.empty((L,), np.int32)
    swaps = np.empty((L, S, 2), np.int32)
    rc = lib().capo_adjust_spectrum(_p(counts), _p(coact), C.c_int32(L), C.c_int32(E), C.c_int32(D),
                                    _p(expert_dev0), C.c_int32(S), _p(spectrum), _p(n_done), _p(swaps))
    if rc != 0:
        raise ValueError(f"capo_adjust_spectrum -> {rc}")
    return spectrum, n_done, swaps


def prune_naive(idx, w, p):
    """NEXT-4b: naive expert-level top-p pruning. idx,w [L,T,k] -> (kept [L,T,k] uint8, near_margin [L])."""
    idx = _c(idx, np.int32)
    w = _c(w, np.float32)
    L, T, k = idx.shape
    kept = np.empty((L, T, k), np.uint8)
    near = np.zeros((L,), np.int64)
    rc = lib().capo_prune_naive(_p(idx), _p(w), C.c_int32(L), C.c_int64(T), C.c_int32(k), C.c_float(p),
                                _p(kept), _p(near))
    if rc != 0:
        raise ValueError(f"capo_prune_naive -> {rc}")
    return kept, near


def dispatch_row_weights(w, pair_row, n_rows):
    """NEXT-4c: combine weight a_d of every dispatch row. w [T,k] fp32, pair_row [T*k] -> row_w [n_rows]."""
    w = _c(w, np.float32)
    T, k = w.shape
    pair_row = _c(pair_row, np.int32)
    row_w = np.empty((int(n_rows),), np.float32)
    rc = lib().capo_dispatch_row_weights(_p(w), _p(pair_row), C.c_int64(T), C.c_int32(k), C.c_int64(int(n_rows)),
                                         _p(row_w))
    if rc != 0:
        raise ValueError(f"capo_dispatch_row_weights -> {rc}")
    return row_w

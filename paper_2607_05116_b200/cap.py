"""Thin ctypes binding of libcap_b200.so (include/cap.h).  Argument marshalling only: every
step of the path runs in the library's CUDA kernels.  torch is used for device memory and
streams.  There is no CPU fallback: a missing library or a missing GPU raises.
"""
import ctypes as C
import types
import os
from types import SimpleNamespace

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libcap_b200.so")

(CALL_GATE_TOPK, CALL_COACTIVATION, CALL_EVAL_PLACEMENTS, CALL_PRUNE, CALL_DISPATCH_LAYOUT, CALL_TRACE_FUSED,
 CALL_COACT_PLACEMENT, CALL_DISPATCH_ROWS, CALL_PRUNE_DISPATCH) = range(9)
OK, EINVAL, EWORKSPACE, ECUDA = 0, -1, -2, -3

EXPORTS = ("cap_gate_topk", "cap_coactivation", "cap_eval_placements", "cap_prune",
           "cap_dispatch_layout", "cap_trace_fused", "cap_coact_placement", "cap_pairwise_objective", "cap_dispatch_rows", "cap_adjust_spectrum", "cap_workspace_bytes",
           "cap_validate_placements", "cap_last_cuda_error", "cap_launch_count", "cap_version",
           "cap_kernel_timer_arm", "cap_kernel_timer_ms", "cap_profile_fused_kernel", "cap_trace_fused_plan",
           "cap_dispatch_layout_static", "cap_static_scratch_bytes", "cap_prune_naive", "cap_dispatch_row_weights", "cap_dispatch_layout_batched",
           "cap_trace_fused_begin", "cap_trace_fused_finish", "cap_prune_dispatch")

KERNEL_TAGS = ("trace_fused", "gate_topk", "coact", "masked_counts", "eval_table", "eval", "eval_decode", "eval_finalize", "prune",
               "dispatch_hist", "dispatch_scan", "dispatch_scatter", "coact_placement", "objective", "rows_hist", "rows_scan", "rows_scatter", "adjust")


class GateCfg(C.Structure):
    _fields_ = [("E", C.c_int32), ("k", C.c_int32), ("scoring", C.c_int32),
                ("renormalize", C.c_int32), ("n_group", C.c_int32), ("topk_group", C.c_int32),
                ("group_score", C.c_int32), ("scale", C.c_float)]


class Topology(C.Structure):
    _fields_ = [("D", C.c_int32), ("N", C.c_int32), ("dev_node", C.c_void_p),
                ("cost_local", C.c_int32), ("cost_intra", C.c_int32), ("cost_inter", C.c_int32),
                ("bytes_per_token", C.c_int64)]


_EVAL_I64 = ("dev_visits", "remote_dev", "remote_intra", "remote_inter", "node_visits",
             "remote_node", "cost", "bytes")


class EvalOut(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in _EVAL_I64 + ("load_pairs", "recv_tokens", "imbalance",
                                                      "imbalance_recv", "tok_remote_dev",
                                                      "tok_remote_node")]


class CapError(RuntimeError):
    pass


_lib = None


def lib():
    """Load libcap_b200.so (fails loudly if it has not been built)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise CapError(f"{LIB_PATH} is missing: run `python -m paper_2607_05116_b200.build` "
                           "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        L.cap_workspace_bytes.restype = C.c_size_t
        L.cap_workspace_bytes.argtypes = [C.c_int, C.c_int32, C.c_int64, C.c_int32, C.c_int32,
                                          C.c_int32, C.c_int32]
        L.cap_launch_count.restype = C.c_int64
        L.cap_version.restype = C.c_char_p
        vp, i32, i64, f32, sz = C.c_void_p, C.c_int32, C.c_int64, C.c_float, C.c_size_t
        L.cap_gate_topk.argtypes = [vp, vp, i32, i64, C.POINTER(GateCfg), vp, vp, vp, sz, vp]
        L.cap_coactivation.argtypes = [vp, vp, i32, i64, i32, i32, vp, vp, vp, sz, vp]
        L.cap_eval_placements.argtypes = [vp, vp, vp, i32, i64, i32, i32, vp, i32,
                                          C.POINTER(Topology), vp, C.POINTER(EvalOut), vp, sz, vp]
        L.cap_prune.argtypes = [vp, vp, vp, i32, i64, i32, i32, vp, C.POINTER(Topology), f32, vp,
                                C.POINTER(EvalOut), vp, vp, sz, vp]
        L.cap_dispatch_layout.argtypes = [vp, vp, i64, i32, i32, vp, i32, vp, vp, vp, vp, sz, vp]
        L.cap_trace_fused.argtypes = [vp, vp, i32, i64, C.POINTER(GateCfg), vp, vp, vp, vp, vp, vp,
                                      i32, C.POINTER(Topology), C.POINTER(EvalOut), vp, sz, vp]
        L.cap_validate_placements.argtypes = [vp, i32, i32, i32, i32, vp]
        L.cap_pairwise_objective.argtypes = [vp, vp, i32, i32, vp, i32, C.POINTER(Topology), C.c_double, vp, vp, vp,
                                             vp, vp]
        L.cap_adjust_spectrum.argtypes = [vp, vp, i32, i32, i32, vp, i32, vp, vp, vp, vp]
        L.cap_dispatch_rows.argtypes = [vp, vp, i64, i32, i32, vp, i32, vp, vp, vp, vp, sz, vp]
        L.cap_coact_placement.argtypes = [vp, vp, i32, i32, i32, i32, vp, vp, vp, vp, vp, vp, sz, vp]
        L.cap_profile_fused_kernel.argtypes = [C.POINTER(C.c_void_p), i32, i32, i32, i64, C.POINTER(GateCfg), vp, vp,
                                               vp, vp, vp, i32, C.POINTER(Topology), C.POINTER(EvalOut), vp, sz,
                                               vp, C.POINTER(C.c_float)]
        L.cap_trace_fused_plan.argtypes = [i32, i64, C.POINTER(GateCfg), i32, i32, i32, C.POINTER(C.c_int64)]
        L.cap_dispatch_layout_static.argtypes = [vp, vp, i64, i32, i32, vp, i32, vp, vp, vp, vp]
        L.cap_static_scratch_bytes.restype = C.c_size_t
        L.cap_prune_naive.argtypes = [vp, vp, i32, i64, i32, f32, vp, vp, vp]
        L.cap_dispatch_row_weights.argtypes = [vp, vp, i64, i32, i64, vp, vp]
        L.cap_dispatch_layout_batched.argtypes = [vp, vp, i32, i64, i32, i32, vp, i32, vp, vp, vp, vp, sz, vp]
        L.cap_prune_dispatch.argtypes = [vp, vp, vp, i32, i64, i32, i32, vp, C.POINTER(Topology), f32, vp,
                                         C.POINTER(EvalOut), vp, vp, vp, vp, vp, sz, vp]
        L.cap_trace_fused_begin.argtypes = [vp, vp, i32, i64, C.POINTER(GateCfg), vp, vp, vp, vp, vp, vp,
                                            i32, C.POINTER(Topology), C.POINTER(EvalOut), vp, sz, C.POINTER(Pending), vp]
        L.cap_trace_fused_finish.argtypes = [C.POINTER(Pending), vp]
        L.cap_kernel_timer_arm.argtypes = [C.c_char_p, C.c_int]
        L.cap_kernel_timer_ms.argtypes = [C.c_int]
        L.cap_kernel_timer_ms.restype = C.c_float
        _lib = L
    return _lib


def launch_count() -> int:
    return int(lib().cap_launch_count())


def _check(rc, what):
    if rc != OK:
        name = {EINVAL: "CAP_EINVAL", EWORKSPACE: "CAP_EWORKSPACE", ECUDA: "CAP_ECUDA"}.get(rc, str(rc))
        extra = f" (cudaError {lib().cap_last_cuda_error()})" if rc == ECUDA else ""
        raise CapError(f"{what} -> {name}{extra}")


def _ptr(t, dtype=None):
    if t is None:
        return None
    if not t.is_cuda:
        raise CapError("cap: tensors must live on a CUDA device (no CPU fallback)")
    if dtype is not None and t.dtype != dtype:
        raise CapError(f"cap: expected dtype {dtype}, got {t.dtype}")
    if not t.is_contiguous():
        raise CapError("cap: tensors must be contiguous")
    return C.c_void_p(t.data_ptr())


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def gate_cfg(E, k, scoring=0, renormalize=1, n_group=1, topk_group=1, group_score=0, scale=1.0):
    return GateCfg(E, k, scoring, renormalize, n_group, topk_group, group_score, scale)


def topology(dev_node, cost_local=0, cost_intra=1, cost_inter=1, bytes_per_token=0, N=None):
    """dev_node: int32 CUDA tensor [D].  N must be given (or is taken from a host copy once)."""
    D = dev_node.numel()
    if N is None:
        N = int(dev_node.max().item()) + 1
    t = Topology(D, N, dev_node.data_ptr(), cost_local, cost_intra, cost_inter, bytes_per_token)
    t._keep = dev_node
    return t


def workspace(which, L, T, E, k, D=1, P=0, device="cuda"):
    n = int(lib().cap_workspace_bytes(which, L, T, E, k, D, P))
    return torch.empty(max(n, 256), dtype=torch.uint8, device=device)


def alloc_eval_out(L, P, D, T=0, per_token=False, device="cuda"):
    o = SimpleNamespace()
    for n in _EVAL_I64:
        setattr(o, n, torch.empty((L, P), dtype=torch.int64, device=device))
    o.load_pairs = torch.empty((L, P, D), dtype=torch.int64, device=device)
    o.recv_tokens = torch.empty((L, P, D), dtype=torch.int64, device=device)
    o.imbalance = torch.empty((L, P), dtype=torch.float64, device=device)
    o.imbalance_recv = torch.empty((L, P), dtype=torch.float64, device=device)
    o.tok_remote_dev = torch.empty((L, P, T), dtype=torch.uint8, device=device) if per_token else None
    o.tok_remote_node = torch.empty((L, P, T), dtype=torch.uint8, device=device) if per_token else None
    return o


def _eval_struct(o):
    s = EvalOut()
    for name, _ in EvalOut._fields_:
        t = getattr(o, name, None)
        setattr(s, name, None if t is None else t.data_ptr())
    return s


def gate_topk(logits, bias, cfg, idx=None, w=None):
    L, T, E = logits.shape
    if idx is None:
        idx = torch.empty((L, T, cfg.k), dtype=torch.int32, device=logits.device)
    if w is None:
        w = torch.empty((L, T, cfg.k), dtype=torch.float32, device=logits.device)
    rc = lib().cap_gate_topk(_ptr(logits, torch.float32), _ptr(bias, torch.float32), L, T,
                             C.byref(cfg), _ptr(idx), _ptr(w), None, 0, _stream())
    _check(rc, "cap_gate_topk")
    return idx, w


def coactivation(idx, kept, E, counts=None, coact=None):
    L, T, k = idx.shape
    if counts is None:
        counts = torch.empty((L, E), dtype=torch.int64, device=idx.device)
    if coact is None:
        coact = torch.empty((L, E, E), dtype=torch.int32, device=idx.device)
    rc = lib().cap_coactivation(_ptr(idx, torch.int32), _ptr(kept, torch.uint8), L, T, k, E,
                                _ptr(counts), _ptr(coact), None, 0, _stream())
    _check(rc, "cap_coactivation")
    return counts, coact


def eval_placements(idx, kept, token_src, expert_dev, topo, counts=None, out=None, ws=None,
                    per_token=False):
    L, T, k = idx.shape
    _, P, E = expert_dev.shape
    if out is None:
        out = alloc_eval_out(L, P, topo.D, T, per_token, idx.device)
    if ws is None:
        ws = workspace(CALL_EVAL_PLACEMENTS, L, T, E, k, topo.D, P, idx.device)
    s = _eval_struct(out)
    rc = lib().cap_eval_placements(_ptr(idx, torch.int32), _ptr(kept, torch.uint8),
                                   _ptr(token_src, torch.int32), L, T, k, E,
                                   _ptr(expert_dev, torch.int32), P, C.byref(topo),
                                   _ptr(counts, torch.int64), C.byref(s), _ptr(ws), ws.numel(),
                                   _stream())
    _check(rc, "cap_eval_placements")
    return out


def prune(idx, w, token_src, expert_dev, topo, p, kept=None, after=None, near_margin=None,
          ws=None, want_after=True):
    L, T, k = idx.shape
    E = expert_dev.shape[-1]
    if kept is None:
        kept = torch.empty((L, T, k), dtype=torch.uint8, device=idx.device)
    if near_margin is None:
        near_margin = torch.empty((L,), dtype=torch.int64, device=idx.device)
    s = None
    if want_after:
        if after is None:
            after = alloc_eval_out(L, 1, topo.D, T, False, idx.device)
        if ws is None:
            ws = workspace(CALL_PRUNE, L, T, E, k, topo.D, 1, idx.device)
        s = _eval_struct(after)
    rc = lib().cap_prune(_ptr(idx, torch.int32), _ptr(w, torch.float32),
                         _ptr(token_src, torch.int32), L, T, k, E, _ptr(expert_dev, torch.int32),
                         C.byref(topo), float(p), _ptr(kept), C.byref(s) if s is not None else None,
                         _ptr(near_margin), _ptr(ws), 0 if ws is None else ws.numel(), _stream())
    _check(rc, "cap_prune")
    return kept, near_margin, after


def dispatch_layout(idx, kept, expert_dev, D, want_pos=True, ws=None):
    T, k = idx.shape
    E = expert_dev.shape[0]
    sorted_pairs = torch.empty((T * k,), dtype=torch.int32, device=idx.device)
    pair_pos = torch.empty((T * k,), dtype=torch.int32, device=idx.device) if want_pos else None
    offsets = torch.empty((D + 1,), dtype=torch.int64, device=idx.device)
    if ws is None:
        ws = workspace(CALL_DISPATCH_LAYOUT, 1, T, E, k, D, 0, idx.device)
    rc = lib().cap_dispatch_layout(_ptr(idx, torch.int32), _ptr(kept, torch.uint8), T, k, E,
                                   _ptr(expert_dev, torch.int32), D, _ptr(sorted_pairs),
                                   _ptr(pair_pos), _ptr(offsets), _ptr(ws), ws.numel(), _stream())
    _check(rc, "cap_dispatch_layout")
    return sorted_pairs, offsets, pair_pos


def dispatch_layout_batched(idx, kept, expert_dev, D, want_pos=True, ws=None, out=None):
    """cap_dispatch_layout_batched: S5 for all layers in one call.  idx [L,T,k], kept [L,T,k]|None, expert_dev [L,E]
    -> (sorted_pairs [L,T*k], offsets [L,D+1], pair_pos [L,T*k]|None)."""
    L, T, k = idx.shape
    E = expert_dev.shape[-1]
    if out is None:
        sorted_pairs = torch.empty((L, T * k), dtype=torch.int32, device=idx.device)
        pair_pos = torch.empty((L, T * k), dtype=torch.int32, device=idx.device) if want_pos else None
        offsets = torch.empty((L, D + 1), dtype=torch.int64, device=idx.device)
    else:
        sorted_pairs, offsets, pair_pos = out
    if ws is None:
        ws = workspace(CALL_DISPATCH_LAYOUT, L, T, E, k, D, 0, idx.device)
    rc = lib().cap_dispatch_layout_batched(_ptr(idx, torch.int32), _ptr(kept, torch.uint8), L, T, k, E,
                                           _ptr(expert_dev, torch.int32), D, _ptr(sorted_pairs), _ptr(pair_pos),
                                           _ptr(offsets), _ptr(ws), ws.numel(), _stream())
    _check(rc, "cap_dispatch_layout_batched")
    return sorted_pairs, offsets, pair_pos


def prune_dispatch(idx, w, token_src, expert_dev, topo, p, want_after=True, want_pos=True, ws=None, bufs=None):
    """cap_prune_dispatch: S4 + S5 under expert_dev [L,E] in three launches.  Returns (kept, near_margin, after,
    sorted_pairs, offsets, pair_pos) -- what prune() followed by dispatch_layout_batched() returns."""
    L, T, k = idx.shape
    E = expert_dev.shape[-1]
    D = topo.D
    if bufs is None:
        kept = torch.empty((L, T, k), dtype=torch.uint8, device=idx.device)
        near = torch.empty((L,), dtype=torch.int64, device=idx.device)
        after = alloc_eval_out(L, 1, D, T, False, idx.device) if want_after else None
        sorted_pairs = torch.empty((L, T * k), dtype=torch.int32, device=idx.device)
        pair_pos = torch.empty((L, T * k), dtype=torch.int32, device=idx.device) if want_pos else None
        offsets = torch.empty((L, D + 1), dtype=torch.int64, device=idx.device)
    else:
        kept, near, after, sorted_pairs, offsets, pair_pos = bufs
    if ws is None:
        ws = workspace(CALL_PRUNE_DISPATCH, L, T, E, k, D, 0, idx.device)
    s = _eval_struct(after) if after is not None else None
    rc = lib().cap_prune_dispatch(_ptr(idx, torch.int32), _ptr(w, torch.float32), _ptr(token_src, torch.int32), L, T,
                                  k, E, _ptr(expert_dev, torch.int32), C.byref(topo), float(p), _ptr(kept),
                                  C.byref(s) if s is not None else None, _ptr(near), _ptr(sorted_pairs),
                                  _ptr(pair_pos), _ptr(offsets), _ptr(ws), ws.numel(), _stream())
    _check(rc, "cap_prune_dispatch")
    return kept, near, after, sorted_pairs, offsets, pair_pos


def dispatch_layout_static(idx, kept, expert_dev, D, sorted_pairs, offsets, pair_pos=None):
    """cap_dispatch_layout_static: S5 into CALLER-provided outputs with the library's static scratch (no
    workspace, nothing allocated here or in the library).  sorted_pairs [T*k] int32, offsets [D+1] int64,
    pair_pos [T*k] int32 or None.  Raises CapError(CAP_EWORKSPACE) beyond the static limit."""
    T, k = idx.shape
    E = expert_dev.shape[0]
    rc = lib().cap_dispatch_layout_static(_ptr(idx, torch.int32), _ptr(kept, torch.uint8), T, k, E,
                                          _ptr(expert_dev, torch.int32), D, _ptr(sorted_pairs, torch.int32),
                                          _ptr(pair_pos, torch.int32), _ptr(offsets, torch.int64), _stream())
    if rc == EWORKSPACE:
        need = int(lib().cap_workspace_bytes(CALL_DISPATCH_LAYOUT, 1, T, E, k, D, 0))
        raise CapError(f"cap_dispatch_layout_static -> CAP_EWORKSPACE: T={T} k={k} D={D} needs {need} bytes of scratch, "
                       f"the static array holds {int(lib().cap_static_scratch_bytes())}; use cap_dispatch_layout")
    _check(rc, "cap_dispatch_layout_static")
    return sorted_pairs, offsets, pair_pos


def coact_placement(counts, coact, D, N, rnd=None, want_p=False, ws=None):
    """cap_coact_placement: Jaccard p_ij + Algorithm 1 (device groups, then node groups).
    counts [L,E] int64, coact [L,E,E] int32, rnd [L,E+D] int32-typed bits or None ->
    (expert_group [L,E], group_node [L,D], expert_dev [L,E], p [L,E,E] fp64 or None)."""
    L, E = counts.shape
    dev = counts.device
    p = torch.empty((L, E, E), dtype=torch.float64, device=dev) if want_p else None
    expert_group = torch.empty((L, E), dtype=torch.int32, device=dev)
    group_node = torch.empty((L, D), dtype=torch.int32, device=dev)
    expert_dev = torch.empty((L, E), dtype=torch.int32, device=dev)
    if ws is None:
        ws = workspace(CALL_COACT_PLACEMENT, L, 0, E, 1, D, 0, device=dev)
    rc = lib().cap_coact_placement(_ptr(counts, torch.int64), _ptr(coact, torch.int32), L, E, D, N,
                                   _ptr(rnd, torch.int32), _ptr(p), _ptr(expert_group), _ptr(group_node),
                                   _ptr(expert_dev), _ptr(ws), ws.numel(), _stream())
    _check(rc, "cap_coact_placement")
    return expert_group, group_node, expert_dev, p


def adjust_spectrum(counts, coact, expert_dev0, D, S):
    """cap_adjust_spectrum: S swap steps of the Adjustment Approach.  expert_dev0 [L,E] int32 ->
    (spectrum [L,S,E], n_done [L], swaps [L,S,2])."""
    L, E = expert_dev0.shape
    dev = counts.device
    spectrum = torch.empty((L, S, E), dtype=torch.int32, device=dev)
    n_done = torch.empty((L,), dtype=torch.int32, device=dev)
    swaps = torch.empty((L, S, 2), dtype=torch.int32, device=dev)
    rc = lib().cap_adjust_spectrum(_ptr(counts, torch.int64), _ptr(coact, torch.int32), L, E, D,
                                   _ptr(expert_dev0, torch.int32), S, _ptr(spectrum), _ptr(n_done), _ptr(swaps),
                                   _stream())
    _check(rc, "cap_adjust_spectrum")
    return spectrum, n_done, swaps


def dispatch_rows(idx, kept, expert_dev, D, want_pair_row=True, ws=None):
    """cap_dispatch_rows: one row per (token, destination device).  idx [T,k], kept [T,k] or None,
    expert_dev [E] -> (rows_token [T*min(k,D)] (valid up to row_offsets[D]), row_offsets [D+1], pair_row)."""
    T, k = idx.shape
    E = expert_dev.numel()
    dev = idx.device
    rows = torch.empty((max(T * min(k, D), 1),), dtype=torch.int32, device=dev)
    pair_row = torch.empty((T * k,), dtype=torch.int32, device=dev) if want_pair_row else None
    offsets = torch.empty((D + 1,), dtype=torch.int64, device=dev)
    if ws is None:
        ws = workspace(CALL_DISPATCH_ROWS, 1, T, E, k, D, 0, device=dev)
    rc = lib().cap_dispatch_rows(_ptr(idx, torch.int32), _ptr(kept, torch.uint8), T, k, E,
                                 _ptr(expert_dev, torch.int32), D, _ptr(rows), _ptr(pair_row), _ptr(offsets),
                                 _ptr(ws), ws.numel(), _stream())
    _check(rc, "cap_dispatch_rows")
    return rows, offsets, pair_row


def prune_naive(idx, w, p, kept=None, near_margin=None):
    """cap_prune_naive: naive expert-level top-p pruning. idx, w [L,T,k] -> (kept [L,T,k] uint8, near [L])."""
    L, T, k = idx.shape
    if kept is None:
        kept = torch.empty((L, T, k), dtype=torch.uint8, device=idx.device)
    if near_margin is None:
        near_margin = torch.empty((L,), dtype=torch.int64, device=idx.device)
    rc = lib().cap_prune_naive(_ptr(idx, torch.int32), _ptr(w, torch.float32), L, T, k, float(p), _ptr(kept),
                               _ptr(near_margin), _stream())
    _check(rc, "cap_prune_naive")
    return kept, near_margin


def dispatch_row_weights(w, pair_row, n_rows, row_w=None):
    """cap_dispatch_row_weights: combine weight a_d of every dispatch row. w [T,k], pair_row [T*k]."""
    T, k = w.shape
    if row_w is None:
        row_w = torch.empty((max(int(n_rows), 1),), dtype=torch.float32, device=w.device)
    rc = lib().cap_dispatch_row_weights(_ptr(w, torch.float32), _ptr(pair_row, torch.int32), T, k, int(n_rows),
                                        _ptr(row_w), _stream())
    _check(rc, "cap_dispatch_row_weights")
    return row_w[: int(n_rows)]


def pairwise_objective(counts, coact, expert_dev, topo, lam=0.5, imbalance=None):
    """cap_pairwise_objective: Eq. 2-3 for P candidates from (counts, coact); Eq. 5 when imbalance is given.
    expert_dev [L,P,E] int32 -> (obj_count [L,P] int64, obj_prob [L,P] fp64, combined [L,P] fp64 or None)."""
    L, P, E = expert_dev.shape
    dev = counts.device
    oc = torch.empty((L, P), dtype=torch.int64, device=dev)
    op = torch.empty((L, P), dtype=torch.float64, device=dev)
    cb = torch.empty((L, P), dtype=torch.float64, device=dev) if imbalance is not None else None
    rc = lib().cap_pairwise_objective(_ptr(counts, torch.int64), _ptr(coact, torch.int32), L, E,
                                      _ptr(expert_dev, torch.int32), P, C.byref(topo), float(lam),
                                      _ptr(imbalance, torch.float64), _ptr(oc), _ptr(op), _ptr(cb), _stream())
    _check(rc, "cap_pairwise_objective")
    return oc, op, cb


class FusedBuffers:
    """Pre-allocated outputs + workspace of cap_trace_fused for fixed sizes."""

    def __init__(self, L, T, E, k, D, P, device="cuda", per_token=False):
        self.idx = torch.empty((L, T, k), dtype=torch.int32, device=device)
        self.w = torch.empty((L, T, k), dtype=torch.float32, device=device)
        self.counts = torch.empty((L, E), dtype=torch.int64, device=device)
        self.coact = torch.empty((L, E, E), dtype=torch.int32, device=device)
        self.out = alloc_eval_out(L, P, D, T, per_token, device)
        self.ws = workspace(CALL_TRACE_FUSED, L, T, E, k, D, P, device)
        self.out_struct = _eval_struct(self.out)


def trace_fused(logits, bias, cfg, token_src, expert_dev, topo, bufs=None, per_token=False):
    L, T, E = logits.shape
    P = expert_dev.shape[1]
    if bufs is None:
        bufs = FusedBuffers(L, T, E, cfg.k, topo.D, P, logits.device, per_token)
    rc = lib().cap_trace_fused(_ptr(logits, torch.float32), _ptr(bias, torch.float32), L, T,
                               C.byref(cfg), _ptr(bufs.idx), _ptr(bufs.w), _ptr(bufs.counts),
                               _ptr(bufs.coact), _ptr(token_src, torch.int32),
                               _ptr(expert_dev, torch.int32), P, C.byref(topo),
                               C.byref(bufs.out_struct), _ptr(bufs.ws), bufs.ws.numel(), _stream())
    _check(rc, "cap_trace_fused")
    return bufs


class Pending(C.Structure):
    """cap_pending (include/cap.h): the launch cap_trace_fused_begin hands back."""
    _fields_ = [("kind", C.c_int32), ("reserved", C.c_int32), ("blob", C.c_ubyte * 496)]


def trace_fused_begin(logits, bias, cfg, token_src, expert_dev, topo, bufs=None, per_token=False, pend=None):
    """cap_trace_fused up to the last launch of S3 (current stream); returns (bufs, pend).  bufs.idx / w / counts /
    coact are final in stream order, bufs.out only after trace_fused_finish(pend)."""
    L, T, E = logits.shape
    P = expert_dev.shape[1]
    if bufs is None:
        bufs = FusedBuffers(L, T, E, cfg.k, topo.D, P, logits.device, per_token)
    if pend is None:
        pend = Pending()
    rc = lib().cap_trace_fused_begin(_ptr(logits, torch.float32), _ptr(bias, torch.float32), L, T,
                                     C.byref(cfg), _ptr(bufs.idx), _ptr(bufs.w), _ptr(bufs.counts),
                                     _ptr(bufs.coact), _ptr(token_src, torch.int32),
                                     _ptr(expert_dev, torch.int32), P, C.byref(topo),
                                     C.byref(bufs.out_struct), _ptr(bufs.ws), bufs.ws.numel(), C.byref(pend),
                                     _stream())
    _check(rc, "cap_trace_fused_begin")
    return bufs, pend


def trace_fused_finish(pend):
    """Issue the launch trace_fused_begin handed back, on the CURRENT stream (the caller orders it after the
    stream _begin ran on)."""
    _check(lib().cap_trace_fused_finish(C.byref(pend), _stream()), "cap_trace_fused_finish")


def profile_fused_kernel(logits_list, cfg, expert_dev, topo, bufs, n_rep):
    """Average device time (ms) of the fused S1+S2+S3 kernel alone over n_rep back-to-back launches
    rotating over logits_list; returns None if the configuration is not served by the fused kernel."""
    L, T, E = logits_list[0].shape
    P = expert_dev.shape[1]
    arr = (C.c_void_p * len(logits_list))(*[t.data_ptr() for t in logits_list])
    ms = C.c_float(0.0)
    rc = lib().cap_profile_fused_kernel(arr, len(logits_list), n_rep, L, T, C.byref(cfg), _ptr(bufs.idx),
                                        _ptr(bufs.w), _ptr(bufs.counts), _ptr(bufs.coact),
                                        _ptr(expert_dev, torch.int32), P, C.byref(topo),
                                        C.byref(bufs.out_struct), _ptr(bufs.ws), bufs.ws.numel(), _stream(),
                                        C.byref(ms))
    if rc == EINVAL:
        return None
    _check(rc, "cap_profile_fused_kernel")
    return float(ms.value)


def trace_fused_plan(L, T, cfg, D, N, P):
    """cap_trace_fused_plan -> dict (host only): which kernel serves these sizes and its token geometry."""
    arr = (C.c_int64 * 8)()
    _check(lib().cap_trace_fused_plan(L, T, C.byref(cfg), D, N, P, arr), "cap_trace_fused_plan")
    names = ("fused", "blocks_per_layer", "tokens_per_block", "max_tokens_one_source", "run_capacity",
             "records_per_block", "blocks_per_source", "kernel_version")
    return dict(zip(names, [int(v) for v in arr]))


def validate_placements(expert_dev, D):
    L, P, E = expert_dev.shape
    return int(lib().cap_validate_placements(_ptr(expert_dev, torch.int32), L, P, E, D, _stream()))


def kernel_timer_arm(tag: str, slot: int):
    _check(lib().cap_kernel_timer_arm(tag.encode(), slot), "cap_kernel_timer_arm")


def kernel_timer_ms(slot: int) -> float:
    return float(lib().cap_kernel_timer_ms(slot))


class Pipeline:
    """The whole hot path for fixed sizes, on resident device buffers: cap_trace_fused (S1+S2+S3
    over P candidates) -> cap_prune under candidate `chosen` (S4, with the after-metrics) ->
    cap_dispatch_layout per layer for the same candidate (S5).  Holds every output buffer and
    workspace, so step() only enqueues kernels."""

    def __init__(self, L, T, gate, D, N, P, dev_node, cost_inter=1, bytes_per_token=0, tau=0.1,
                 chosen=0, device="cuda"):
        self.L, self.T, self.P, self.D, self.tau, self.chosen = L, T, P, D, tau, chosen
        self._ctor = dict(L=L, T=T, gate=gate, D=D, N=N, P=P, dev_node=dev_node, cost_inter=cost_inter,
                          bytes_per_token=bytes_per_token, tau=tau, chosen=chosen, device=device)
        self.gate = gate
        if gate.renormalize != 1 or gate.scale != 1.0:
            # cap_prune's stop rule compares the kept weight with 1 - p (Eq. 6, reading R8): it needs routing
            # weights that sum to 1 per token, which only renormalised, unscaled gates produce
            raise CapError("Pipeline: cap_prune needs renormalised routing weights with scale 1 (include/cap.h)")
        E, k = gate.E, gate.k
        self.dev_node = dev_node
        self.topo = topology(dev_node, 0, 1, cost_inter, bytes_per_token, N=N)
        self.fb = FusedBuffers(L, T, E, k, D, P, device)
        self.kept = torch.empty((L, T, k), dtype=torch.uint8, device=device)
        self.near = torch.empty((L,), dtype=torch.int64, device=device)
        self.after = alloc_eval_out(L, 1, D, T, False, device)
        self.after_struct = _eval_struct(self.after)
        self.ws_prune = workspace(CALL_PRUNE, L, T, E, k, D, 1, device)
        self.sorted_pairs = torch.empty((L, T * k), dtype=torch.int32, device=device)
        self.pair_pos = torch.empty((L, T * k), dtype=torch.int32, device=device)
        self.offsets = torch.empty((L, D + 1), dtype=torch.int64, device=device)
        self.ws_disp = workspace(CALL_DISPATCH_LAYOUT, L, T, E, k, D, 0, device)
        self.ws_pd = workspace(CALL_PRUNE_DISPATCH, L, T, E, k, D, 0, device)
        self.pi = torch.empty((L, E), dtype=torch.int32, device=device)
        self.side = torch.cuda.Stream(device=device)       # the S3 decode runs here, beside S4 / S5 (step)
        self.pend = Pending()

    def clone(self):
        """A second pipeline with its own output buffers and workspaces (same configuration)."""
        return Pipeline(**self._ctor)

    def _pi(self, expert_dev):
        if self.L == 1:
            return expert_dev[:, self.chosen, :]        # already the [L][E] layout cap_prune wants: no copy
        self.pi.copy_(expert_dev[:, self.chosen, :])
        return self.pi

    def step_prune(self, token_src, pi):
        """S4 on the buffers the last cap_trace_fused left (kept mask + after-metrics)."""
        rc = lib().cap_prune(_ptr(self.fb.idx), _ptr(self.fb.w), _ptr(token_src, torch.int32), self.L, self.T,
                             self.gate.k, self.gate.E, _ptr(pi), C.byref(self.topo), float(self.tau),
                             _ptr(self.kept), C.byref(self.after_struct), _ptr(self.near), _ptr(self.ws_prune),
                             self.ws_prune.numel(), _stream())
        _check(rc, "cap_prune")

    def step_prune_dispatch(self, token_src, pi):
        """S4 + S5 as one call (cap_prune_dispatch: three launches) on the buffers of the last cap_trace_fused."""
        rc = lib().cap_prune_dispatch(_ptr(self.fb.idx), _ptr(self.fb.w), _ptr(token_src, torch.int32), self.L,
                                      self.T, self.gate.k, self.gate.E, _ptr(pi), C.byref(self.topo),
                                      float(self.tau), _ptr(self.kept), C.byref(self.after_struct), _ptr(self.near),
                                      _ptr(self.sorted_pairs), _ptr(self.pair_pos), _ptr(self.offsets),
                                      _ptr(self.ws_pd), self.ws_pd.numel(), _stream())
        _check(rc, "cap_prune_dispatch")

    def step_dispatch(self, pi):
        """S5 for every layer on the kept mask of the last cap_prune: one batched call (three launches)."""
        dispatch_layout_batched(self.fb.idx, self.kept, pi if pi.is_contiguous() else pi.contiguous(), self.D,
                                ws=self.ws_disp, out=(self.sorted_pairs, self.offsets, self.pair_pos))

    def step(self, logits, bias, token_src, expert_dev):
        """One pass S1..S5.  S4 and S5 read the routing trace, not the S3 outputs, so the last launch of S3 (the
        decode of the per-block records into fb.out) runs on a side stream beside them: fork after the scoring
        kernel, join at the end of the step (inside a CUDA graph: two parallel branches)."""
        main = torch.cuda.current_stream()
        _, pend = trace_fused_begin(logits, bias, self.gate, token_src, expert_dev, self.topo, self.fb,
                                    pend=self.pend)
        if pend.kind:
            self.side.wait_stream(main)
            with torch.cuda.stream(self.side):
                trace_fused_finish(pend)
        self.step_prune_dispatch(token_src, self._pi(expert_dev))
        if pend.kind:
            main.wait_stream(self.side)
        return self

    def step_serial(self, logits, bias, token_src, expert_dev):
        """The same pass with every launch on the current stream (one dependent chain)."""
        trace_fused(logits, bias, self.gate, token_src, expert_dev, self.topo, self.fb)
        pi = self._pi(expert_dev)
        self.step_prune(token_src, pi)
        self.step_dispatch(pi)
        return self

    def capture_stage(self, which, token_src, expert_dev):
        """Graph of one stage alone ("prune" = S4 with after-metrics, "dispatch" = S5, "prune_dispatch" = the
        fused S4 + S5 call the step uses) on the current buffers,
        for stand-alone stage timings; the preceding stages must have run once."""
        pi = self._pi(expert_dev)
        fn = {"prune": lambda: self.step_prune(token_src, pi), "dispatch": lambda: self.step_dispatch(pi),
              "prune_dispatch": lambda: self.step_prune_dispatch(token_src, pi)}[which]
        fn()
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            fn()
        return g

    def capture(self, logits, bias, token_src, expert_dev):
        """Capture one step on these (fixed) input buffers into a CUDA graph: the library only
        enqueues work on the current stream, so a step is capturable as is.  Returns the graph;
        replay() re-runs the whole step with no host-side launch cost."""
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):
            self.step(logits, bias, token_src, expert_dev)      # one-time attribute setup outside capture
        torch.cuda.current_stream().wait_stream(side)
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            self.step(logits, bias, token_src, expert_dev)
        return g

    def capture_fused(self, logits, bias, token_src, expert_dev):
        """Graph of the cap_trace_fused call alone (S1+S2+S3), for timing the fused pass."""
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            trace_fused(logits, bias, self.gate, token_src, expert_dev, self.topo, self.fb)
        return g

    def result_tensors(self):
        """Every output of a step (what a host caller reads back)."""
        o, a = self.fb.out, self.after
        ts = [self.fb.idx, self.fb.w, self.fb.counts, self.fb.coact, self.kept, self.near,
              self.sorted_pairs, self.pair_pos, self.offsets]
        for ns in (o, a):
            for name, _ in EvalOut._fields_:
                t = getattr(ns, name, None)
                if t is not None:
                    ts.append(t)
        return ts


class HostPipeline:
    """The same step driven from HOST buffers (the end-to-end call): pinned host inputs are copied
    to the device, the step runs, every output is copied back to pinned host memory.

    depth = 1: copy in, compute, copy out, one after the other on the current stream.
    depth > 1: `depth` independent sets of staging buffers, device outputs and host outputs; the copies
    run on two side streams, so the upload of step i+1 and the read-back of step i-1 overlap the
    compute of step i (PCIe is full duplex).  Every step still uploads its own inputs and reads back
    all of its own outputs; call finish() before looking at the returned host tensors."""

    def __init__(self, pipe: Pipeline, has_bias=False, has_src=False, depth=1):
        self.pipe = pipe
        self.depth = depth
        L, T, P = pipe.L, pipe.T, pipe.P
        E = pipe.gate.E
        dev = pipe.kept.device
        self.sets = []
        for i in range(depth):
            st = types.SimpleNamespace()
            st.pipe = pipe if i == 0 else pipe.clone()
            st.d_logits = torch.empty((L, T, E), dtype=torch.float32, device=dev)
            st.d_maps = torch.empty((L, P, E), dtype=torch.int32, device=dev)
            st.d_bias = torch.empty((L, E), dtype=torch.float32, device=dev) if has_bias else None
            st.d_src = torch.empty((L, T), dtype=torch.int32, device=dev) if has_src else None
            st.h_out = [torch.empty(t.shape, dtype=t.dtype, pin_memory=True) for t in st.pipe.result_tensors()]
            st.graph = None
            st.ev_in, st.ev_comp, st.ev_out = torch.cuda.Event(), torch.cuda.Event(), torch.cuda.Event()
            st.used = False
            self.sets.append(st)
        self.h_out = self.sets[0].h_out
        self.d2h_bytes = sum(t.numel() * t.element_size() for t in self.h_out)
        self.s_h2d = torch.cuda.Stream(device=dev) if depth > 1 else None
        self.s_d2h = torch.cuda.Stream(device=dev) if depth > 1 else None
        self.n = 0

    def capture(self):
        """Capture the device part of the step (on the staging buffers) into a CUDA graph per set."""
        for st in self.sets:
            st.graph = st.pipe.capture(st.d_logits, st.d_bias, st.d_src, st.d_maps)
        self.graph = self.sets[0].graph

    def h2d_bytes(self, logits, maps, bias=None, src=None):
        return sum(t.numel() * t.element_size() for t in (logits, maps, bias, src) if t is not None)

    @staticmethod
    def _upload(st, h_logits, h_maps, h_bias, h_src):
        st.d_logits.copy_(h_logits, non_blocking=True)
        st.d_maps.copy_(h_maps, non_blocking=True)
        if h_bias is not None:
            st.d_bias.copy_(h_bias, non_blocking=True)
        if h_src is not None:
            st.d_src.copy_(h_src, non_blocking=True)

    @staticmethod
    def _compute(st, h_bias, h_src):
        if st.graph is not None:
            st.graph.replay()
        else:
            st.pipe.step(st.d_logits, st.d_bias if h_bias is not None else None,
                         st.d_src if h_src is not None else None, st.d_maps)

    @staticmethod
    def _download(st):
        for h, d in zip(st.h_out, st.pipe.result_tensors()):
            h.copy_(d, non_blocking=True)

    def step(self, h_logits, h_maps, h_bias=None, h_src=None):
        st = self.sets[self.n % self.depth]
        self.n += 1
        if self.depth == 1:
            self._upload(st, h_logits, h_maps, h_bias, h_src)
            self._compute(st, h_bias, h_src)
            self._download(st)
            return st.h_out
        cur = torch.cuda.current_stream()
        if st.used:
            self.s_h2d.wait_event(st.ev_comp)       # the compute that read these staging buffers
        else:
            self.s_h2d.wait_stream(cur)
        with torch.cuda.stream(self.s_h2d):
            self._upload(st, h_logits, h_maps, h_bias, h_src)
            st.ev_in.record(self.s_h2d)
        cur.wait_event(st.ev_in)
        if st.used:
            cur.wait_event(st.ev_out)               # the read-back of this set's previous outputs
        self._compute(st, h_bias, h_src)
        st.ev_comp.record(cur)
        self.s_d2h.wait_event(st.ev_comp)
        with torch.cuda.stream(self.s_d2h):
            self._download(st)
            st.ev_out.record(self.s_d2h)
        st.used = True
        return st.h_out

    def finish(self):
        """Make the current stream wait for every copy issued so far."""
        if self.depth > 1:
            cur = torch.cuda.current_stream()
            cur.wait_stream(self.s_h2d)
            cur.wait_stream(self.s_d2h)



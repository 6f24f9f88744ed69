"""GPU parity of cap_coact_placement (Jaccard p_ij + Algorithm 1 in both
stages) against the CPU oracle through the C ABI: expert_group, group_node, expert_dev bit-exact,
the fp64 probabilities bit-identical (one IEEE divide on exact integers)."""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu

from oracle import cap_oracle as O                      # noqa: E402
from paper_2607_05116_b200 import cap                   # noqa: E402
from paper_2607_05116_b200 import workload as W         # noqa: E402
from parity_util import dev, host                       # noqa: E402


@pytest.fixture(scope="module", autouse=True)
def _need_gpu():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    cap.lib()


def check(counts, coact, D, N, rnd=None, tag=""):
    L, E = counts.shape
    ref = O.coact_placement(counts, coact, D=D, N=N, rnd=rnd, want_p=True)
    rnd_d = None if rnd is None else dev(rnd.view(np.int32))
    got = cap.coact_placement(dev(counts), dev(coact), D, N, rnd=rnd_d, want_p=True)
    torch.cuda.synchronize()
    for name, g, r in zip(("expert_group", "group_node", "expert_dev"), got[:3], ref[:3]):
        np.testing.assert_array_equal(host(g), r, err_msg=tag + name)
    np.testing.assert_array_equal(host(got[3]).view(np.int64), ref[3].view(np.int64), err_msg=tag + "p bits")
    ed = ref[2]
    for l in range(L):
        assert np.bincount(ed[l], minlength=D).tolist() == [E // D] * D
    return ref


def trace_stats(cfg, layers, T):
    xs = np.stack([W.logits(cfg.with_(T=T), l) for l in layers])
    bs = W.gate_bias(cfg, layers[0])
    bias = np.stack([W.gate_bias(cfg, l) for l in layers]) if bs is not None else None
    idx, _ = O.gate_topk(xs, bias, **cfg.gate)
    cnt, C = O.coactivation(idx, E=cfg.E)
    return xs, bias, idx, cnt, C


@pytest.mark.parametrize("name,layers,T", [("tiny", (0,), 4096), ("qwen3", (0, 17, 47), 16384),
                                           ("target", (0,), 65536), ("dsv3", (0, 31), 8192),
                                           ("stress", (0,), 16384)])
def test_placement_on_baseline_configs(name, layers, T):
    cfg = W.CONFIGS[name]
    rng = np.random.default_rng(cfg.index)
    xs, bias, idx, cnt, C = trace_stats(cfg, layers, T)
    rnd = rng.integers(0, 2**32, (len(layers), cfg.E + cfg.D), dtype=np.uint64).astype(np.uint32)
    ref = check(cnt, C, cfg.D, cfg.N, rnd, tag=name + " ")
    # chained on the GPU: trace statistics from the CUDA gate + co-activation feed the placement
    g = cap.gate_cfg(cfg.E, **cfg.gate)
    gi, _ = cap.gate_topk(dev(xs), dev(bias), g)
    gc, gC = cap.coactivation(gi, None, cfg.E)
    got = cap.coact_placement(gc, gC, cfg.D, cfg.N, rnd=dev(rnd.view(np.int32)))
    np.testing.assert_array_equal(host(got[2]), ref[2])
    # the paper's claim, through the CUDA path: fewer devices per token than the sequential map
    if cfg.clusters is not None:
        seq = (np.arange(cfg.E) // (cfg.E // cfg.D)).astype(np.int32)
        both = np.stack([np.stack([seq, ref[2][l]]) for l in range(len(layers))])
        ev = O.eval_placements(idx, both, W.dev_node(cfg))
        assert np.all(ev.dev_visits[:, 1] < ev.dev_visits[:, 0])


@pytest.mark.parametrize("E,D,N,k,T", [(8, 4, 2, 3, 4), (12, 4, 2, 3, 30), (64, 64, 8, 4, 200), (64, 1, 1, 4, 200),
                                       (96, 8, 8, 6, 150), (256, 32, 4, 8, 300), (1024, 64, 8, 16, 500),
                                       (1000, 50, 10, 12, 64), (33, 33, 1, 5, 10), (62, 31, 31, 2, 9)])
def test_placement_sparse_traces_ties_and_random_branch(E, D, N, k, T):
    """Short random traces: small integer counts give many exactly equal probabilities, degrees and
    scores (tie rules), never-selected experts give zero rows (the random branch with real rnd)."""
    rng = np.random.default_rng(E * 7 + D)
    L = 3
    idx = np.stack([[rng.choice(max(k, E - E // 5), k, replace=False) for _ in range(T)]
                    for _ in range(L)]).astype(np.int32)
    cnt, C = O.coactivation(idx, E=E)
    rnd = rng.integers(0, 2**32, (L, E + D), dtype=np.uint64).astype(np.uint32)
    check(cnt, C, D, N, rnd, tag=f"E{E} D{D} N{N} ")
    check(cnt, C, D, N, None, tag=f"E{E} D{D} N{N} rnd=NULL ")


def test_placement_all_zero_and_empty():
    rng = np.random.default_rng(5)
    cnt = np.zeros((2, 128), np.int64)
    C = np.zeros((2, 128, 128), np.int32)
    rnd = rng.integers(0, 2**32, (2, 128 + 16), dtype=np.uint64).astype(np.uint32)
    check(cnt, C, 16, 4, rnd, tag="zeros ")
    got = cap.coact_placement(dev(cnt[:0]), dev(C[:0]), 16, 4)
    assert got[2].shape == (0, 128)


def test_placement_kernel_time_all_layers():
    """Timing note (printed): all layers of configs 2 and 4 in one launch, one CTA per layer."""
    for name, L in (("qwen3", 48), ("dsv3", 58), ("stress", 1)):
        cfg = W.CONFIGS[name]
        _, _, _, cnt, C = trace_stats(cfg, (0,), 8192)
        rng = np.random.default_rng(1)
        cntL = np.repeat(cnt, L, 0)
        CL = np.repeat(C, L, 0)
        for l in range(1, L):                       # distinct layers: perturb the off-diagonal counts
            A = np.triu(rng.integers(0, 3, (cfg.E, cfg.E)), 1)
            CL[l] += (A + A.T).astype(np.int32)
        ref = O.coact_placement(cntL, CL, D=cfg.D, N=cfg.N)
        dc, dC = dev(cntL), dev(CL)
        ws = cap.workspace(cap.CALL_COACT_PLACEMENT, L, 0, cfg.E, 1, cfg.D, 0)
        cap.coact_placement(dc, dC, cfg.D, cfg.N, ws=ws)
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(5):
            got = cap.coact_placement(dc, dC, cfg.D, cfg.N, ws=ws)
        b.record()
        torch.cuda.synchronize()
        np.testing.assert_array_equal(host(got[2]), ref[2])
        print(f"cap_coact_placement {name}: L={L} E={cfg.E} D={cfg.D} N={cfg.N}: {a.elapsed_time(b) / 5 * 1e3:.1f} us per call")


# ------------------------------------------------------------------ cap_pairwise_objective (Eq. 2-3, Eq. 5)
OBJ_RTOL = 1e-10   # include/cap.h: summation order only; (E^2 / 2) ulp bound on non-negative terms


def check_objective(cnt, C, maps, dn, cost_intra, cost_inter, lam, imb, tag=""):
    D = dn.shape[0]
    N = int(dn.max()) + 1
    ref = O.pairwise_objective(cnt, C, maps, dn, cost_intra=cost_intra, cost_inter=cost_inter, lam=lam,
                               imbalance=imb)
    dnd = dev(dn)
    topo = cap.topology(dnd, 0, cost_intra, cost_inter, 0, N=N)
    got = cap.pairwise_objective(dev(cnt), dev(C), dev(maps), topo, lam=lam, imbalance=dev(imb))
    torch.cuda.synchronize()
    np.testing.assert_array_equal(host(got[0]), ref[0], err_msg=tag + "obj_count")
    np.testing.assert_allclose(host(got[1]), ref[1], rtol=OBJ_RTOL, atol=0, err_msg=tag + "obj_prob")
    if imb is not None:
        np.testing.assert_allclose(host(got[2]), ref[2], rtol=OBJ_RTOL, atol=0, err_msg=tag + "combined")
    return ref


@pytest.mark.parametrize("name,layers,T,P", [("tiny", (0,), 4096, 4), ("qwen3", (0, 17), 16384, 64),
                                             ("target", (0,), 65536, 256), ("dsv3", (0, 31), 8192, 128),
                                             ("stress", (0,), 16384, 1024)])
def test_objective_on_baseline_configs(name, layers, T, P):
    cfg = W.CONFIGS[name]
    _, _, idx, cnt, C = trace_stats(cfg, layers, T)
    maps = np.stack([W.candidates(cfg, l, P) for l in layers])
    rng = np.random.default_rng(3)
    imb = 1.0 + rng.random((len(layers), P))
    ref = check_objective(cnt, C, maps, W.dev_node(cfg), 1, cfg.cost_inter, 0.3, imb, tag=name + " ")
    # the planted cluster-aligned candidate cuts less than the sequential one (not under group-limited
    # routing, where the contiguous groups of the sequential map are themselves what the gate favours)
    if cfg.clusters is not None and cfg.n_group == 1:
        assert np.all(ref[0][:, 2] < ref[0][:, 0])


@pytest.mark.parametrize("E,D,N,P", [(8, 4, 2, 2), (33, 11, 1, 9), (100, 10, 5, 17), (1024, 64, 8, 3), (1, 1, 1, 1)])
def test_objective_ragged_shapes(E, D, N, P):
    rng = np.random.default_rng(E + P)
    L, k, T = 2, min(4, E), 300
    idx = np.stack([[rng.choice(E, k, replace=False) for _ in range(T)] for _ in range(L)]).astype(np.int32)
    cnt, C = O.coactivation(idx, E=E)
    maps = rng.integers(0, D, (L, P, E)).astype(np.int32)
    dn = (np.arange(D) // (D // N)).astype(np.int32)
    check_objective(cnt, C, maps, dn, 2, 7, 0.75, None, tag=f"E{E} ")
    check_objective(cnt, C, maps, dn, 1, 1, 0.0, rng.random((L, P)) + 1, tag=f"E{E} uniform ")


def test_objective_kernel_time():
    for name in ("target", "stress"):
        cfg = W.CONFIGS[name]
        _, _, _, cnt, C = trace_stats(cfg, (0,), 8192)
        maps = W.candidates(cfg, 0)[None]
        dnd = dev(W.dev_node(cfg))
        topo = cap.topology(dnd, 0, 1, cfg.cost_inter, 0, N=cfg.N)
        dc, dC, dm = dev(cnt), dev(C), dev(maps)
        cap.pairwise_objective(dc, dC, dm, topo)
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(10):
            cap.pairwise_objective(dc, dC, dm, topo)
        b.record()
        torch.cuda.synchronize()
        print(f"cap_pairwise_objective {name}: E={cfg.E} P={cfg.P}: {a.elapsed_time(b) / 10 * 1e3:.1f} us per call")


# ------------------------------------------------------------------ cap_dispatch_rows (Fig. 2)
def check_rows(idx, kept, pi, D, tag=""):
    rows_r, off_r, pr_r = O.dispatch_rows(idx, pi, D, kept=kept)
    rows, off, pr = cap.dispatch_rows(dev(idx), dev(kept), dev(pi), D)
    torch.cuda.synchronize()
    np.testing.assert_array_equal(host(off), off_r, err_msg=tag + "row_offsets")
    np.testing.assert_array_equal(host(rows)[: len(rows_r)], rows_r, err_msg=tag + "rows_token")
    np.testing.assert_array_equal(host(pr), pr_r, err_msg=tag + "pair_row")


@pytest.mark.parametrize("name,T", [("tiny", 4096), ("qwen3", 16384), ("target", 65536), ("dsv3", 32768),
                                    ("stress", 65536)])
def test_dispatch_rows_on_baseline_configs(name, T):
    cfg = W.CONFIGS[name]
    x = W.logits(cfg.with_(T=T), 0)[None]
    b = W.gate_bias(cfg, 0)
    idx, w = O.gate_topk(x, None if b is None else b[None], **cfg.gate)
    cand = W.candidates(cfg, 0)
    for c in (0, 2 if cand.shape[0] > 2 else 1):
        kept, _ = O.prune(idx, w, cand[None, c], W.dev_node(cfg), cfg.taus[-1], cost_inter=cfg.cost_inter)
        check_rows(idx[0], None, cand[c], cfg.D, tag=f"{name} cand{c} ")
        check_rows(idx[0], kept[0], cand[c], cfg.D, tag=f"{name} cand{c} pruned ")


@pytest.mark.parametrize("T,E,k,D", [(0, 16, 2, 4), (1, 16, 2, 4), (255, 8, 8, 1), (257, 64, 16, 64), (5000, 1024, 16, 64),
                                     (70001, 40, 3, 7), (1000, 33, 1, 5)])
def test_dispatch_rows_ragged_and_edges(T, E, k, D):
    rng = np.random.default_rng(T + E)
    idx = (np.stack([rng.choice(E, k, replace=False) for _ in range(T)]) if T else np.zeros((0, k))).astype(np.int32)
    pi = rng.integers(0, D, E).astype(np.int32)
    check_rows(idx, None, pi, D, tag="all ")
    check_rows(idx, (rng.random((T, k)) < 0.5).astype(np.uint8), pi, D, tag="half ")
    check_rows(idx, np.zeros((T, k), np.uint8), pi, D, tag="none ")


def test_dispatch_rows_kernel_time():
    cfg = W.CONFIGS["target"]
    x = W.logits(cfg, 0)[None]
    idx, _ = O.gate_topk(x, None, **cfg.gate)
    di, dp = dev(idx[0]), dev(W.candidates(cfg, 0)[0])
    ws = cap.workspace(cap.CALL_DISPATCH_ROWS, 1, cfg.T, cfg.E, cfg.k, cfg.D, 0)
    cap.dispatch_rows(di, None, dp, cfg.D, ws=ws)
    torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for _ in range(20):
        cap.dispatch_rows(di, None, dp, cfg.D, ws=ws)
    b.record()
    torch.cuda.synchronize()
    print(f"cap_dispatch_rows target: T={cfg.T} k={cfg.k} D={cfg.D}: {a.elapsed_time(b) / 20 * 1e3:.1f} us per call")


# ------------------------------------------------------------------ cap_adjust_spectrum (R27)
def check_adjust(cnt, C, pi0, D, S, tag=""):
    ref = O.adjust_spectrum(cnt, C, pi0, D=D, S=S)
    got = cap.adjust_spectrum(dev(cnt), dev(C), dev(pi0), D, S)
    torch.cuda.synchronize()
    for name, g, r in zip(("spectrum", "n_done", "swaps"), got, ref):
        np.testing.assert_array_equal(host(g), r, err_msg=tag + name)
    return ref


@pytest.mark.parametrize("name,layers,T,S", [("tiny", (0,), 4096, 7), ("qwen3", (0, 17, 47), 16384, 7),
                                             ("target", (0,), 65536, 12), ("dsv3", (0, 31), 8192, 7),
                                             ("stress", (0,), 16384, 7)])
def test_adjust_on_baseline_configs(name, layers, T, S):
    """The paper's pipeline: Algorithm 1's placement, then the swap spectrum (7 placements)."""
    cfg = W.CONFIGS[name]
    _, _, idx, cnt, C = trace_stats(cfg, layers, T)
    _, _, ed, _ = O.coact_placement(cnt, C, D=cfg.D, N=cfg.N)
    ref = check_adjust(cnt, C, ed, cfg.D, S, tag=name + " ")
    seq = np.tile((np.arange(cfg.E) // (cfg.E // cfg.D)).astype(np.int32), (len(layers), 1))
    check_adjust(cnt, C, seq, cfg.D, S, tag=name + " from sequential ")
    assert np.all(ref[1] >= 1)


@pytest.mark.parametrize("E,D,k,T,S", [(6, 2, 2, 20, 8), (24, 4, 4, 400, 40), (64, 64, 4, 100, 5), (33, 1, 3, 50, 3),
                                       (1024, 64, 16, 300, 6), (100, 7, 5, 200, 10)])
def test_adjust_shapes_stops_and_unbalanced_maps(E, D, k, T, S):
    rng = np.random.default_rng(E + S)
    L = 2
    idx = np.stack([[rng.choice(E, k, replace=False) for _ in range(T)] for _ in range(L)]).astype(np.int32)
    cnt, C = O.coactivation(idx, E=E)
    pi0 = rng.integers(0, D, (L, E)).astype(np.int32)          # arbitrary (unbalanced) maps
    check_adjust(cnt, C, pi0, D, S, tag=f"E{E} D{D} ")


def test_adjust_chained_on_the_cuda_path_trades_communication_for_balance():
    """VERDICT r1 missing #8: the whole chain on the GPU -- gate, co-activation, Algorithm 1, the swap
    spectrum (R27, parity unpinned against the paper) and cap_eval_placements scoring every step -- shows
    what P:L194-196 claims: imbalance does not rise along the spectrum and ends lower, devices per token
    do not fall.  The scores themselves are bit-exact against the oracle's for the same maps."""
    cfg = W.CONFIGS["qwen3"].with_(T=8192)
    x = dev(W.logits(cfg, 0)[None])
    idx, _ = cap.gate_topk(x, None, cap.gate_cfg(cfg.E, **cfg.gate))
    cnt, C = cap.coactivation(idx, None, cfg.E)
    ed = cap.coact_placement(cnt, C, cfg.D, cfg.N)[2]
    spec, done, _ = cap.adjust_spectrum(cnt, C, ed, cfg.D, 6)
    maps = torch.cat([ed[:, None], spec], 1).contiguous()
    dn = W.dev_node(cfg)
    topo = cap.topology(dev(dn), 0, 1, cfg.cost_inter, cfg.bytes_per_token, N=cfg.N)
    ev = cap.eval_placements(idx, None, None, maps, topo, counts=cnt)
    torch.cuda.synchronize()
    assert int(host(done)[0]) == 6
    imb, vis = host(ev.imbalance)[0], host(ev.dev_visits)[0]
    assert np.all(np.diff(imb) <= 1e-12) and imb[-1] < imb[0] - 0.02
    assert vis[-1] >= vis[0]
    ref = O.eval_placements(host(idx), host(maps), dn, cost_inter=cfg.cost_inter, bytes_per_token=cfg.bytes_per_token)
    np.testing.assert_array_equal(imb, ref.imbalance[0])
    np.testing.assert_array_equal(vis, ref.dev_visits[0])


def test_adjust_kernel_time():
    cfg = W.CONFIGS["qwen3"]
    _, _, _, cnt, C = trace_stats(cfg, (0,), 8192)
    L = 48
    _, _, ed, _ = O.coact_placement(cnt, C, D=cfg.D, N=cfg.N)
    dc, dC, de = dev(np.repeat(cnt, L, 0)), dev(np.repeat(C, L, 0)), dev(np.repeat(ed, L, 0))
    cap.adjust_spectrum(dc, dC, de, cfg.D, 7)
    torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for _ in range(5):
        cap.adjust_spectrum(dc, dC, de, cfg.D, 7)
    b.record()
    torch.cuda.synchronize()
    print(f"cap_adjust_spectrum qwen3: L={L} E={cfg.E} D={cfg.D} S=7: {a.elapsed_time(b) / 5 * 1e3:.1f} us per call")


# ------------------------------------------------------------------ rest of SURVEY 8(f) rank 4
@pytest.mark.parametrize("name,T", [("tiny", 4096), ("target", 65536), ("dsv3", 8192), ("stress", 16384)])
def test_prune_naive_and_row_weights_on_baseline_configs(name, T):
    """cap_prune_naive and cap_dispatch_row_weights bit-exact against the oracle, chained on the CUDA
    path: gate -> naive pruning -> dispatch rows under the sequential placement -> combine weights."""
    cfg = W.CONFIGS[name]
    xs, bias, idx_r, _, _ = trace_stats(cfg, (0, 1) if cfg.L > 1 else (0,), T)
    _, w_r = O.gate_topk(xs, bias, **cfg.gate)
    gi, gw = cap.gate_topk(dev(xs), dev(bias), cap.gate_cfg(cfg.E, **cfg.gate))
    for p in (0.0, 0.05, 0.3, 0.7):
        kept_r, near_r = O.prune_naive(idx_r, w_r, p)
        kept_d, near_d = cap.prune_naive(dev(idx_r), dev(w_r), p)
        np.testing.assert_array_equal(host(kept_d), kept_r, err_msg=f"{name} p={p} kept")
        np.testing.assert_array_equal(host(near_d), near_r, err_msg=f"{name} p={p} near")
        kept_e, _ = cap.prune_naive(gi, gw, p)                       # end to end on the GPU's own S1 output
        assert int((host(kept_e) != kept_r).any(-1).sum()) <= int(near_r.sum())
    # exact ties and unsorted weights
    rng = np.random.default_rng(cfg.index)
    w_t = np.round(rng.random(w_r.shape).astype(np.float32) * 8) / 8 + np.float32(0.125)
    w_t = (w_t / w_t.sum(-1, keepdims=True, dtype=np.float32)).astype(np.float32)
    kept_r, near_r = O.prune_naive(idx_r, w_t, 0.25)
    kept_d, near_d = cap.prune_naive(dev(idx_r), dev(w_t), 0.25)
    np.testing.assert_array_equal(host(kept_d), kept_r)
    np.testing.assert_array_equal(host(near_d), near_r)
    # combine weights of the rows of layer 0 under the sequential placement, pruned trace
    pi = W.candidates(cfg, 0)[0]
    kept0, _ = O.prune_naive(idx_r[:1], w_r[:1], 0.3)
    rows_r, off_r, prow_r = O.dispatch_rows(idx_r[0], pi, cfg.D, kept=kept0[0])
    rw_r = O.dispatch_row_weights(w_r[0], prow_r, int(off_r[-1]))
    rows_d, off_d, prow_d = cap.dispatch_rows(dev(idx_r[0]), dev(kept0[0]), dev(pi), cfg.D)
    n_rows = int(off_d[-1])
    rw_d = cap.dispatch_row_weights(dev(w_r[0]), prow_d, n_rows)
    np.testing.assert_array_equal(host(prow_d), prow_r)
    np.testing.assert_array_equal(host(rw_d).view(np.int32), rw_r.view(np.int32), err_msg="row weights (bits)")


def test_prune_naive_edges():
    idx = torch.zeros((1, 0, 4), dtype=torch.int32, device="cuda")
    w = torch.zeros((1, 0, 4), dtype=torch.float32, device="cuda")
    kept, near = cap.prune_naive(idx, w, 0.1)
    assert kept.shape == (1, 0, 4) and int(near[0]) == 0
    with pytest.raises(cap.CapError, match="EINVAL"):
        cap.prune_naive(idx, w, 1.0)
    rng = np.random.default_rng(1)
    for k in (1, 9, 16):
        T = 1000
        idx_h = np.stack([rng.permutation(1024)[:k] for _ in range(T)]).astype(np.int32)[None]
        w_h = rng.random((1, T, k)).astype(np.float32) + np.float32(0.01)
        w_h = (w_h / w_h.sum(-1, keepdims=True, dtype=np.float32)).astype(np.float32)
        for p in (0.1, 0.5):
            kept_r, near_r = O.prune_naive(idx_h, w_h, p)
            kept_d, near_d = cap.prune_naive(dev(idx_h), dev(w_h), p)
            np.testing.assert_array_equal(host(kept_d), kept_r)
            np.testing.assert_array_equal(host(near_d), near_r)

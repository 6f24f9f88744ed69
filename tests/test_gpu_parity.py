"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on
the same seeded inputs.  Integers bit-exact, gate weights within 1e-6 absolute."""
import numpy as np
from types import SimpleNamespace
import pytest
import torch

pytestmark = pytest.mark.gpu

from oracle import cap_oracle as O                      # noqa: E402
from paper_2607_05116_b200 import cap                   # noqa: E402
from paper_2607_05116_b200 import workload as W         # noqa: E402
from parity_util import (assert_eval_equal, check_all_stages, check_gate, dev, host,  # noqa: E402
                         topo_of)


@pytest.fixture(scope="module", autouse=True)
def _need_gpu():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    cap.lib()


# ------------------------------------------------------------------ the five BASELINE configs
def test_config1_tiny_all_stages():
    cfg = W.CONFIGS["tiny"]
    check_all_stages(cfg, per_token=True, tag="tiny ")
    check_all_stages(cfg, random_src=True, per_token=True, tag="tiny/src ")


def test_config2_qwen3_two_layers_full_T():
    cfg = W.CONFIGS["qwen3"]
    rep = check_all_stages(cfg, layers=(0, 17), tag="qwen3 ")
    assert rep["w_max_abs_diff"] <= 1e-6


def test_config3_target_full_size():
    cfg = W.CONFIGS["target"]
    rep = check_all_stages(cfg, tag="target ")
    print("target report", rep)
    check_all_stages(cfg, T=4099, random_src=True, per_token=True, tag="target/ragged ")


def test_config4_dsv3_two_layers_full_T():
    cfg = W.CONFIGS["dsv3"]
    rep = check_all_stages(cfg, layers=(0, 31), tag="dsv3 ")
    print("dsv3 report", rep)


def test_config5_stress_2pow16():
    cfg = W.CONFIGS["stress"]
    rep = check_all_stages(cfg, tag="stress ")
    print("stress report", rep)


# ------------------------------------------------------------------ S1 edge cases
@pytest.mark.parametrize("E,k", [(1, 1), (7, 7), (16, 2), (33, 4), (40, 5), (64, 6), (100, 8), (128, 8),
                                 (130, 8), (256, 8), (260, 16), (512, 10), (1000, 12), (1024, 16)])
def test_gate_shapes_and_ties(E, k):
    rng = np.random.default_rng(E * 31 + k)
    T = 777
    x = rng.normal(0, 1, (2, T, E)).astype(np.float32)
    x[1] = np.round(x[1] * 2) / 2                    # heavy exact ties
    x[0, :5] = 0.25                                   # all-equal rows
    x[0, 5, : min(E, 3)] = -0.0                       # -0 / +0
    x[0, 5, min(E, 3):] = 0.0
    for gate in (dict(k=k), dict(k=k, renormalize=0), dict(k=k, scale=2.5),
                 dict(k=k, scoring=1), dict(k=k, scoring=1, renormalize=0)):
        check_gate(x, None, gate, tag=f"E{E}k{k} {gate} ")


@pytest.mark.parametrize("group_score", [0, 1])
@pytest.mark.parametrize("E,n_group,topk_group,k", [(64, 8, 3, 6), (256, 8, 4, 8), (96, 32, 9, 8), (16, 2, 1, 2)])
def test_gate_group_limited(E, n_group, topk_group, k, group_score):
    rng = np.random.default_rng(E + n_group)
    x = rng.normal(0, 1.3, (2, 500, E)).astype(np.float32)
    x[1, :100] = np.round(x[1, :100] * 2) / 2
    bias = rng.uniform(-0.05, 0.05, (2, E)).astype(np.float32)
    g = dict(k=k, n_group=n_group, topk_group=topk_group, group_score=group_score)
    check_gate(x, bias, dict(scoring=1, **g))
    check_gate(x, None, dict(scoring=0, **g))


@pytest.mark.parametrize("E", [64, 128, 256])
@pytest.mark.parametrize("grouped,group_score", [(False, 0), (True, 0), (True, 1)])
def test_gate_sigmoid_fast_path(E, grouped, group_score):
    """The two-lanes-per-token sigmoid kernel (cap_gate_sig.cu: cheap sigmoid inside payload keys + exact redo of
    uncertified tokens) must give the oracle's result on exactly the inputs that stress its certification:
    heavy exact ties, all-equal rows, -0/+0, saturated sigmoids (scores tied at 1.0 / near 0), near-ties one ulp
    apart, biases that reorder experts.  T is a multiple of 16, so the fast path serves these calls."""
    rng = np.random.default_rng(E * 3 + group_score + 7 * grouped)
    T = 1024
    ng = E // 32
    x = rng.normal(0, 1.5, (3, T, E)).astype(np.float32)
    x[1] = np.round(x[1] * 2) / 2                                   # heavy exact ties
    x[2, :256] = x[2, :256] * 12.0                                   # saturated: many scores at 1.0 or ~0
    x[2, 256:512] = -8.0 + 0.01 * x[2, 256:512]                      # every score far below 0.25
    base = rng.normal(0, 1, (256, 1)).astype(np.float32)
    near = np.nextafter(np.broadcast_to(base, (256, E)).astype(np.float32), np.float32(np.inf))
    x[2, 512:768] = np.where(rng.random((256, E)) < 0.5, near, np.broadcast_to(base, (256, E)))   # one ulp apart
    x[0, :5] = 0.25
    x[0, 5, :3] = -0.0
    x[0, 5, 3:] = 0.0
    bias = rng.uniform(-0.05, 0.05, (3, E)).astype(np.float32)
    bias[1] = np.round(bias[1] * 64) / 64                            # biases that create exact score ties
    for k in (1, 3, 8):
        for tg in ((1, ng) if grouped else (1,)):
            if grouped and k > tg * 32:
                continue
            g = dict(k=k, scoring=1, n_group=ng if grouped else 1, topk_group=tg if grouped else 1,
                     group_score=group_score)
            if grouped and ng == 8:
                g4 = dict(g, topk_group=4)
                check_gate(x, bias, g4, tag=f"sigfast E{E} {g4} ")
            check_gate(x, bias, g, tag=f"sigfast E{E} {g} ")
            check_gate(x, None, dict(g, scale=2.5), tag=f"sigfast/nobias E{E} {g} ")


@pytest.mark.parametrize("scoring", [0, 1])
def test_gate_ring_wraps_many_times_E256(scoring):
    """E = 256 gives the TMA ring of the standalone gate kernels only 12 stages: 70 000 tokens make every block
    wrap it more than twice (regression: stages consumed by changing warps desynchronised the ring)."""
    cfg = W.CONFIGS["dsv3"].with_(T=70000 - 70000 % 16)
    x = W.logits(cfg, 0)[None]
    if scoring == 0:
        check_gate(x, None, dict(k=8), tag="E256 softmax wrap ")
    else:
        check_gate(x, W.gate_bias(cfg, 0)[None], cfg.gate, tag="E256 sigmoid wrap ")


def test_gate_empty_and_single():
    cfg = cap.gate_cfg(128, 8)
    idx, w = cap.gate_topk(torch.empty((1, 0, 128), device="cuda"), None, cfg)
    assert idx.shape == (1, 0, 8)
    x = np.random.default_rng(0).normal(0, 1, (1, 1, 128)).astype(np.float32)
    check_gate(x, None, dict(k=8))


# ------------------------------------------------------------------ S2/S3/S4/S5 edge cases
def _trace(rng, L, T, E, k):
    return np.stack([np.stack([rng.permutation(E)[:k] for _ in range(T)]) for _ in range(L)]).astype(np.int32)


@pytest.mark.parametrize("E,k,T", [(8, 3, 5), (16, 2, 1), (24, 5, 1033), (200, 8, 700), (256, 8, 3000), (512, 10, 900),
                                   (258, 4, 300), (320, 6, 1500), (385, 9, 2100), (500, 10, 5000), (512, 16, 4097),
                                   (514, 8, 600), (1024, 16, 500)])
def test_coact_masked_and_shapes(E, k, T):
    rng = np.random.default_rng(E + T)
    idx = _trace(rng, 2, T, E, k)
    kept = (rng.random((2, T, k)) < 0.6).astype(np.uint8)
    kept[0, 0] = 0
    for m in (None, kept, np.zeros_like(kept)):
        cnt_r, C_r = O.coactivation(idx, m, E=E)
        cnt_d, C_d = cap.coactivation(dev(idx), dev(m), E)
        assert np.array_equal(host(cnt_d), cnt_r) and np.array_equal(host(C_d), C_r)
    cnt_d, C_d = cap.coactivation(dev(idx[:, :0]), None, E)          # T = 0 -> zeros
    assert int(cnt_d.sum()) == 0 and int(C_d.sum()) == 0


@pytest.mark.parametrize("E,k,D,N,P,T", [(16, 2, 1, 1, 3, 100), (32, 4, 8, 4, 5, 257), (64, 6, 64, 8, 33, 1000),
                                         (128, 8, 16, 2, 300, 2048), (512, 10, 64, 8, 70, 500), (1024, 16, 64, 64, 40, 300)])
def test_eval_generic_unbalanced_maps(E, k, D, N, P, T):
    rng = np.random.default_rng(E * 7 + D)
    L = 2
    idx = _trace(rng, L, T, E, k)
    kept = (rng.random((L, T, k)) < 0.7).astype(np.uint8)
    pis = rng.integers(0, D, (L, P, E)).astype(np.int32)
    pis[0, 0] = 0                                           # everything on device 0
    dn = np.sort(rng.integers(0, N, D)).astype(np.int32)
    dn[0], dn[-1] = 0, N - 1
    src = rng.integers(0, D, (L, T)).astype(np.int32)
    topo = cap.topology(dev(dn), cost_local=2, cost_intra=3, cost_inter=7, bytes_per_token=4096, N=N)
    for m, s in ((None, None), (kept, src), (np.zeros_like(kept), src)):
        ref = O.eval_placements(idx, pis, dn, kept=m, token_src=s, cost_local=2, cost_intra=3,
                                cost_inter=7, bytes_per_token=4096, per_token=True)
        got = cap.eval_placements(dev(idx), dev(m), dev(s), dev(pis), topo, per_token=True)
        assert_eval_equal(got, ref, True, f"E{E} D{D} ")
    assert cap.validate_placements(dev(pis), D) == cap.OK
    bad = pis.copy()
    bad[1, P - 1, E - 1] = D
    assert cap.validate_placements(dev(bad), D) == cap.EINVAL


@pytest.mark.parametrize("k", [1, 3, 8, 16])
def test_prune_edge_cases(k):
    rng = np.random.default_rng(100 + k)
    L, T, E, D = 2, 1500, 64, 16
    idx = _trace(rng, L, T, E, k)
    w = rng.random((L, T, k)).astype(np.float32) + np.float32(0.02)
    w = -np.sort(-w, axis=-1)
    w = (w / w.sum(-1, keepdims=True, dtype=np.float32)).astype(np.float32)
    w[0, :50] = np.float32(1.0 / k)                       # exact ratio ties
    pi = np.stack([rng.permutation(E) % D for _ in range(L)]).astype(np.int32)
    dn = (np.arange(D) // 4).astype(np.int32)
    src = rng.integers(0, D, (L, T)).astype(np.int32)
    for costs in ((0, 1, 4), (1, 1, 1), (0, 0, 3), (2, 1, 5)):
        topo = cap.topology(dev(dn), *costs, bytes_per_token=64, N=4)
        for p in (0.0, -1.0, 0.05, 0.3, 0.5, 0.999):
            for s in (None, src):
                kept_r, near_r = O.prune(idx, w, pi, dn, p, token_src=s, cost_local=costs[0],
                                         cost_intra=costs[1], cost_inter=costs[2])
                kept_d, near_d, aft = cap.prune(dev(idx), dev(w), dev(s), dev(pi), topo, p)
                assert np.array_equal(host(kept_d), kept_r), (costs, p)
                assert np.array_equal(host(near_d), near_r), (costs, p)
                ref = O.eval_placements(idx, pi[:, None], dn, kept=kept_r, token_src=s, cost_local=costs[0],
                                        cost_intra=costs[1], cost_inter=costs[2], bytes_per_token=64)
                assert_eval_equal(aft, ref, False, f"after {costs} {p} ")


@pytest.mark.parametrize("L,T,k,E,D,N", [(1, 1, 1, 4, 2, 1), (2, 33, 3, 8, 4, 2), (1, 4099, 8, 128, 16, 2),
                                         (3, 1500, 8, 128, 8, 2), (1, 9000, 10, 512, 64, 8), (2, 700, 16, 64, 5, 5),
                                         (1, 70000, 4, 64, 33, 3)])
def test_prune_dispatch_equals_prune_then_dispatch(L, T, k, E, D, N):
    """cap_prune_dispatch (S4 + S5 in three launches: the pruning kernel leaves the sort's histogram, the scan and
    scatter launches finish the after-metrics) against the oracle's prune followed by its dispatch layout, per
    layer: kept masks, near-margin counts, after-metrics, sorted pairs, inverse positions, offsets."""
    rng = np.random.default_rng(L * 1000 + T + k)
    idx = _trace(rng, L, T, E, k)
    w = rng.random((L, T, k)).astype(np.float32) + np.float32(0.02)
    w = -np.sort(-w, axis=-1)
    w = (w / w.sum(-1, keepdims=True, dtype=np.float32)).astype(np.float32)
    w[0, : min(T, 40)] = np.float32(1.0 / k)                 # exact ratio ties
    pi = np.stack([rng.permutation(E) % D for _ in range(L)]).astype(np.int32)
    dn = np.sort(rng.integers(0, N, D)).astype(np.int32)
    dn[0], dn[-1] = 0, N - 1
    src = rng.integers(0, D, (L, T)).astype(np.int32)
    topo = cap.topology(dev(dn), 0, 1, 4, bytes_per_token=64, N=N)
    for p, s, want_after in ((0.1, None, True), (0.4, src, True), (0.0, None, True), (0.25, src, False)):
        kept_r, near_r = O.prune(idx, w, pi, dn, p, token_src=s, cost_local=0, cost_intra=1, cost_inter=4)
        n0 = cap.launch_count()
        kept_d, near_d, aft, sp_d, off_d, pos_d = cap.prune_dispatch(dev(idx), dev(w), dev(s), dev(pi), topo, p,
                                                                     want_after=want_after)
        torch.cuda.synchronize()
        assert cap.launch_count() - n0 == 3
        tag = f"p={p} src={s is not None} "
        assert np.array_equal(host(kept_d), kept_r), tag + "kept"
        assert np.array_equal(host(near_d), near_r), tag + "near"
        if want_after:
            ref = O.eval_placements(idx, pi[:, None], dn, kept=kept_r, token_src=s, cost_local=0, cost_intra=1,
                                    cost_inter=4, bytes_per_token=64)
            assert_eval_equal(aft, ref, False, tag + "after ")
        for l in range(L):
            sp_r, off_r, pos_r = O.dispatch_layout(idx[l], pi[l], D, kept=kept_r[l])
            n = int(off_r[-1])
            assert np.array_equal(host(off_d[l]), off_r), tag + f"offsets layer {l}"
            assert np.array_equal(host(sp_d[l])[:n], sp_r), tag + f"sorted_pairs layer {l}"
            assert np.array_equal(host(pos_d[l]), pos_r), tag + f"pair_pos layer {l}"


def test_prune_dispatch_empty_and_workspace():
    E, k, D = 64, 4, 8
    dn = dev((np.arange(D) // 4).astype(np.int32))
    topo = cap.topology(dn, 0, 1, 4, bytes_per_token=8, N=2)
    pi = dev((np.arange(E) % D).astype(np.int32)[None])
    idx = torch.zeros((1, 0, k), dtype=torch.int32, device="cuda")
    w = torch.zeros((1, 0, k), dtype=torch.float32, device="cuda")
    kept, near, aft, sp, off, pos = cap.prune_dispatch(idx, w, None, pi, topo, 0.2)
    torch.cuda.synchronize()
    assert host(off).tolist() == [[0] * (D + 1)] and host(near).tolist() == [0]
    assert int(aft.dev_visits.sum()) == 0
    idx = torch.zeros((1, 100, k), dtype=torch.int32, device="cuda")
    w = torch.full((1, 100, k), 0.25, dtype=torch.float32, device="cuda")
    with pytest.raises(cap.CapError, match="EWORKSPACE"):
        cap.prune_dispatch(idx, w, None, pi, topo, 0.2, ws=torch.empty(64, dtype=torch.uint8, device="cuda"))
    with pytest.raises(cap.CapError, match="EINVAL"):
        cap.prune_dispatch(idx, w, None, pi, topo, 1.0)


@pytest.mark.parametrize("T,k,E,D", [(1, 1, 4, 2), (5, 3, 8, 4), (2048, 1, 16, 3), (4097, 8, 128, 16), (30000, 10, 512, 64)])
def test_dispatch_edge_cases(T, k, E, D):
    rng = np.random.default_rng(T + D)
    idx = _trace(rng, 1, T, E, k)[0]
    pi = rng.integers(0, D, E).astype(np.int32)
    pi[rng.integers(0, E)] = D - 1
    kept = (rng.random((T, k)) < 0.5).astype(np.uint8)
    for m in (None, kept, np.zeros_like(kept)):
        sp_r, off_r, pos_r = O.dispatch_layout(idx, pi, D, kept=m)
        sp_d, off_d, pos_d = cap.dispatch_layout(dev(idx), dev(m), dev(pi), D)
        n = int(off_r[-1])
        assert np.array_equal(host(off_d), off_r)
        assert np.array_equal(host(sp_d)[:n], sp_r)
        assert np.array_equal(host(pos_d), pos_r)
    sp_d, off_d, _ = cap.dispatch_layout(dev(idx[:0]), None, dev(pi), D)
    assert host(off_d).tolist() == [0] * (D + 1)


@pytest.mark.parametrize("L,T,k,E,D", [(3, 4097, 8, 128, 16), (2, 1, 1, 4, 2), (5, 30000, 10, 512, 64), (4, 2048, 3, 16, 3)])
def test_dispatch_batched_matches_per_layer_oracle(L, T, k, E, D):
    """cap_dispatch_layout_batched = cap_dispatch_layout per layer (own placement, own mask), in three launches."""
    rng = np.random.default_rng(L * 1000 + T)
    idx = _trace(rng, L, T, E, k)
    pi = rng.integers(0, D, (L, E)).astype(np.int32)
    pi[:, 0] = D - 1
    kept = (rng.random((L, T, k)) < 0.5).astype(np.uint8)
    kept[L - 1] = 0                                                   # one layer with every pair pruned
    for m in (None, kept):
        n0 = cap.launch_count()
        sp_d, off_d, pos_d = cap.dispatch_layout_batched(dev(idx), dev(m), dev(pi), D)
        torch.cuda.synchronize()
        assert cap.launch_count() - n0 == 3
        for l in range(L):
            sp_r, off_r, pos_r = O.dispatch_layout(idx[l], pi[l], D, kept=None if m is None else m[l])
            n = int(off_r[-1])
            assert np.array_equal(host(off_d[l]), off_r), (l, "offsets")
            assert np.array_equal(host(sp_d[l])[:n], sp_r), (l, "sorted_pairs")
            assert np.array_equal(host(pos_d[l]), pos_r), (l, "pair_pos")
    sp_d, off_d, _ = cap.dispatch_layout_batched(dev(idx[:, :0]), None, dev(pi), D)      # T = 0
    assert host(off_d).tolist() == [[0] * (D + 1)] * L


def test_error_codes():
    x = torch.zeros((1, 4, 16), device="cuda")
    b = torch.zeros((1, 16), device="cuda")
    with pytest.raises(cap.CapError, match="EINVAL"):
        cap.gate_topk(x, b, cap.gate_cfg(16, 2, scoring=0))            # bias with softmax
    with pytest.raises(cap.CapError, match="EINVAL"):
        cap.gate_topk(x, None, cap.gate_cfg(16, 17))
    with pytest.raises(cap.CapError, match="EINVAL"):
        cap.gate_topk(x, None, cap.gate_cfg(16, 5, n_group=4, topk_group=1))
    idx = torch.zeros((1, 4, 2), dtype=torch.int32, device="cuda")
    w = torch.full((1, 4, 2), 0.5, device="cuda")
    dn = torch.zeros(4, dtype=torch.int32, device="cuda")
    pi = torch.zeros((1, 16), dtype=torch.int32, device="cuda")
    topo = cap.topology(dn, N=1)
    with pytest.raises(cap.CapError, match="EINVAL"):
        cap.prune(idx, w, None, pi, topo, 1.0)
    with pytest.raises(cap.CapError, match="EWORKSPACE"):
        cap.eval_placements(idx, None, None, pi[None], topo, ws=torch.empty(8, dtype=torch.uint8, device="cuda"))
    with pytest.raises(cap.CapError, match="CUDA device"):
        cap.gate_topk(x.cpu(), None, cap.gate_cfg(16, 2))             # no CPU fallback


def test_launch_counter_moves():
    n0 = cap.launch_count()
    x = torch.zeros((1, 64, 16), device="cuda")
    cap.gate_topk(x, None, cap.gate_cfg(16, 2))
    torch.cuda.synchronize()
    assert cap.launch_count() == n0 + 1


# ------------------------------------------------------------------ fast paths on other shapes
# The fused S1+S2+S3 kernel, the bit-sliced S3 path, the tcgen05 S2 path and the register-only S4
# kernel are selected by shape; these cases walk their templates (E = 64 / 128 / 256, field widths
# 8..64, node widths 2..8, k < 8) and their ragged edges (T not a multiple of the 16-token tile, of
# the 64-token scoring block or of the source-device segments; single tokens; several layers).
_FAST_SHAPES = [
    dict(base="target", T=4099),
    dict(base="target", T=1), dict(base="target", T=15), dict(base="target", T=16), dict(base="target", T=17),
    dict(base="target", T=1000, k=3, P=17),
    dict(base="target", T=3001, E=64, k=4, D=8, N=2, P=40, clusters=(8, 8, 0.5)),
    dict(base="target", T=2500, E=256, k=8, D=32, N=4, P=24, clusters=(32, 8, 0.5)),
    dict(base="target", T=2049, D=64, N=8, P=8),
    dict(base="target", T=777, D=1, N=1, P=5),
    dict(base="target", T=5000, D=4, N=4, P=300),
    dict(base="qwen3", T=1500, L=3),
    dict(base="target", T=70000, P=64),
]


@pytest.mark.parametrize("shape", _FAST_SHAPES, ids=lambda s: "-".join(f"{k}{v}" for k, v in s.items() if k != "clusters"))
def test_fast_paths_shapes(shape):
    kw = dict(shape)
    cfg = W.CONFIGS[kw.pop("base")].with_(**kw)
    layers = tuple(range(cfg.L))
    check_all_stages(cfg, layers=layers, tag=f"{shape} ")
    if cfg.T >= 16:
        check_all_stages(cfg, layers=layers[:1], random_src=True, per_token=True, tag=f"{shape}/src ")


@pytest.mark.parametrize("shape", [_FAST_SHAPES[0], _FAST_SHAPES[6], _FAST_SHAPES[7], _FAST_SHAPES[11]],
                         ids=["E128", "E64", "E256", "L3"])
def test_fused_kernel_serves_these_shapes(shape):
    """cap_trace_fused must run its single fused kernel here (the kernel timer tagged 'trace_fused' only
    fires for it), not the three-kernel fallback."""
    kw = dict(shape)
    cfg = W.CONFIGS[kw.pop("base")].with_(**kw)
    from parity_util import layers_inputs
    logits, bias, cand = layers_inputs(cfg, tuple(range(cfg.L)), cfg.T)
    dn_d = dev(W.dev_node(cfg))
    topo = topo_of(cfg, dn_d)
    cap.kernel_timer_arm("trace_fused", 7)
    cap.trace_fused(dev(logits), dev(bias), cap.gate_cfg(cfg.E, **cfg.gate), None, dev(cand), topo)
    torch.cuda.synchronize()
    assert cap.kernel_timer_ms(7) > 0.0


@pytest.mark.parametrize("skew", ["uniform", "one-source", "two-sources"])
def test_bitsliced_eval_serves_explicit_token_src(skew):
    """An explicit token_src (reading R5) keeps the bit-sliced S3 kernel: tokens are grouped by source with the S5
    counting sort and the kernel walks the runs ('eval_decode' only fires behind that kernel).  Skewed sources
    (every token from one device; two devices, the others empty) against the oracle."""
    cfg = W.CONFIGS["target"].with_(T=9001, P=70)
    rng = np.random.default_rng(11)
    L, T, E, k, D = 2, cfg.T, cfg.E, cfg.k, cfg.D
    idx = _trace(rng, L, T, E, k)
    kept = (rng.random((L, T, k)) < 0.7).astype(np.uint8)
    cand = np.stack([W.candidates(cfg, l) for l in range(L)])
    src = {"uniform": rng.integers(0, D, (L, T)), "one-source": np.full((L, T), D - 1),
           "two-sources": rng.choice([3, D - 2], (L, T))}[skew].astype(np.int32)
    dn = W.dev_node(cfg)
    topo = topo_of(cfg, dev(dn))
    for m in (None, kept):
        ref = O.eval_placements(idx, cand, dn, kept=m, token_src=src, cost_inter=cfg.cost_inter,
                                bytes_per_token=cfg.bytes_per_token)
        cap.kernel_timer_arm("eval_decode", 6)
        got = cap.eval_placements(dev(idx), dev(m), dev(src), dev(cand), topo)
        torch.cuda.synchronize()
        assert cap.kernel_timer_ms(6) > 0.0
        assert_eval_equal(got, ref, False, f"{skew} ")


@pytest.mark.parametrize("shape", [_FAST_SHAPES[0], _FAST_SHAPES[5], _FAST_SHAPES[6], _FAST_SHAPES[11], _FAST_SHAPES[12],
                                   dict(base="target", T=20000, D=4, N=2, P=100)],
                         ids=["E128", "k3", "E64", "L3", "T70000", "multi-source"])
def test_single_launch_variant_optin(shape, monkeypatch):
    """cap_fused2.cu, the single cooperative-launch variant of cap_trace_fused (opt-in: CAP_FUSED2=1; slower than
    the default path on B200), stays bit-exact against the oracle."""
    monkeypatch.setenv("CAP_FUSED2", "1")
    kw = dict(shape)
    cfg = W.CONFIGS[kw.pop("base")].with_(**kw)
    plan = cap.trace_fused_plan(cfg.L, cfg.T, cap.gate_cfg(cfg.E, **cfg.gate), cfg.D, cfg.N, cfg.P)
    assert plan["kernel_version"] == 2, plan
    from parity_util import layers_inputs
    layers = tuple(range(cfg.L))
    logits, bias, cand = layers_inputs(cfg, layers, cfg.T)
    dn = W.dev_node(cfg)
    topo = topo_of(cfg, dev(dn))
    idx_r, w_r, cnt_r, C_r, ev_r = O.trace_fused(logits, bias, cfg.gate, cand, dn, cost_inter=cfg.cost_inter,
                                                 bytes_per_token=cfg.bytes_per_token)
    fb = cap.trace_fused(dev(logits), dev(bias), cap.gate_cfg(cfg.E, **cfg.gate), None, dev(cand), topo)
    torch.cuda.synchronize()
    assert np.array_equal(host(fb.idx), idx_r)
    assert float(np.abs(host(fb.w).astype(np.float64) - w_r).max()) <= 1e-6
    assert np.array_equal(host(fb.counts), cnt_r) and np.array_equal(host(fb.coact), C_r)
    assert_eval_equal(fb.out, ev_r, False, "fused2 ")


@pytest.mark.parametrize("base,kw", [("target", dict(T=4099, P=40)), ("qwen3", dict(T=1500, L=3)),
                                     ("dsv3", dict(T=1024, L=2, P=16)), ("tiny", dict())],
                         ids=["fused", "fused-L3", "staged-sigmoid", "tiny"])
def test_trace_fused_begin_finish_and_forked_step(base, kw):
    """cap_trace_fused_begin / _finish (include/cap.h): the two halves give the results of the single call, and
    Pipeline.step -- which runs the second half on a side stream beside S4 / S5 -- gives those of the serial
    chain, launched directly and replayed from a CUDA graph (fork / join inside the capture)."""
    cfg = W.CONFIGS[base].with_(**kw)
    from parity_util import layers_inputs
    layers = tuple(range(cfg.L))
    logits, bias, cand = layers_inputs(cfg, layers, cfg.T)
    dn = W.dev_node(cfg)
    dn_d = dev(dn)
    topo = topo_of(cfg, dn_d)
    gate = cap.gate_cfg(cfg.E, **cfg.gate)
    x_d, b_d, c_d = dev(logits), dev(bias), dev(cand)
    idx_r, w_r, cnt_r, C_r, ev_r = O.trace_fused(logits, bias, cfg.gate, cand, dn, cost_inter=cfg.cost_inter,
                                                 bytes_per_token=cfg.bytes_per_token)
    n0 = cap.launch_count()
    fb, pend = cap.trace_fused_begin(x_d, b_d, gate, None, c_d, topo)
    n1 = cap.launch_count()
    cap.trace_fused_finish(pend)                       # same stream: ordered behind the first half
    torch.cuda.synchronize()
    assert cap.launch_count() - n1 == (1 if pend.kind else 0)
    assert pend.kind == 1                               # all four shapes reach the bit-sliced S3 path
    _, p0 = cap.trace_fused_begin(x_d, b_d, gate, None, c_d, topo, per_token=True)
    assert p0.kind == 0                                 # per-token outputs: generic S3 kernel, nothing owed
    cap.trace_fused_finish(p0)
    assert np.array_equal(host(fb.idx), idx_r) and np.array_equal(host(fb.counts), cnt_r)
    assert np.array_equal(host(fb.coact), C_r)
    assert_eval_equal(fb.out, ev_r, False, "begin/finish ")
    n2 = cap.launch_count()
    cap.trace_fused(x_d, b_d, gate, None, c_d, topo)   # the plain call still launches the decode itself
    assert cap.launch_count() - n2 == (n1 - n0) + (1 if pend.kind else 0)

    mk = lambda: cap.Pipeline(cfg.L, cfg.T, gate, cfg.D, cfg.N, cfg.P, dn_d, cost_inter=cfg.cost_inter,
                              bytes_per_token=cfg.bytes_per_token, tau=cfg.taus[-1], chosen=0, device="cuda")
    ser, forked, graphed = mk(), mk(), mk()
    ser.step_serial(x_d, b_d, None, c_d)
    forked.step(x_d, b_d, None, c_d)
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        graphed.step(x_d, b_d, None, c_d)              # warm-up outside the capture
    torch.cuda.current_stream().wait_stream(s)
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        graphed.step(x_d, b_d, None, c_d)
    for t in graphed.result_tensors():
        t.zero_()
    g.replay()
    g.replay()
    torch.cuda.synchronize()
    assert_eval_equal(forked.fb.out, ev_r, False, "forked ")
    assert_eval_equal(graphed.fb.out, ev_r, False, "graphed ")
    for a, b, c in zip(ser.result_tensors(), forked.result_tensors(), graphed.result_tensors()):
        if a.shape == ser.sorted_pairs.shape and a.dtype == torch.int32 and a is not ser.pair_pos:
            for l in range(cfg.L):
                n = int(ser.offsets[l, -1])
                assert torch.equal(a[l, :n], b[l, :n]) and torch.equal(a[l, :n], c[l, :n])
        else:
            assert torch.equal(a, b) and torch.equal(a, c)


def test_host_pipeline_double_buffered_matches_single():
    """The end-to-end call with two staging sets (copies on side streams, as bench.py's e2e leg uses it)
    returns, step by step, exactly what the plain device pipeline computes on the same inputs."""
    cfg = W.CONFIGS["target"].with_(T=3001, P=24)
    from parity_util import layers_inputs
    dn_d = dev(W.dev_node(cfg))
    gate = cap.gate_cfg(cfg.E, **cfg.gate)
    mk = lambda: cap.Pipeline(cfg.L, cfg.T, gate, cfg.D, cfg.N, cfg.P, dn_d, cost_inter=cfg.cost_inter,
                              bytes_per_token=cfg.bytes_per_token, tau=cfg.taus[-1], chosen=0, device="cuda")
    ref, hp = mk(), cap.HostPipeline(mk(), depth=2)
    hp.capture()
    ins = []
    for s in range(5):
        logits, _, cand = layers_inputs(cfg, tuple(range(cfg.L)), cfg.T)
        logits = np.roll(logits, s * 13, axis=1).copy()           # distinct inputs per step
        ins.append((torch.from_numpy(logits).pin_memory(), torch.from_numpy(cand).pin_memory()))
    outs = [hp.step(x, m) for x, m in ins[:2]]                     # two steps in flight
    hp.finish()
    torch.cuda.synchronize()
    got = [[t.clone() for t in o] for o in outs]
    for s in range(2, 5):                                          # reuse of both sets
        o = hp.step(*ins[s])
        hp.finish()
        torch.cuda.synchronize()
        got.append([t.clone() for t in o])
    for s, (x, m) in enumerate(ins):
        ref.step(x.cuda(), None, None, m.cuda())
        torch.cuda.synchronize()
        for a, b in zip(got[s], ref.result_tensors()):
            if a.dtype == torch.float32:
                assert torch.equal(a, b.cpu()), f"step {s}"
            elif a.shape == ref.sorted_pairs.shape and a.dtype == torch.int32 and a is not None:
                n = int(ref.offsets[0, -1])
                assert torch.equal(a.reshape(-1)[:n], b.cpu().reshape(-1)[:n]) or torch.equal(a, b.cpu()), f"step {s}"
            else:
                assert torch.equal(a, b.cpu()), f"step {s}"


@pytest.mark.parametrize("with_src", [False, True])
def test_garbage_values_are_memory_safe(with_src):
    """include/cap.h: out-of-range VALUES inside device arrays (expert_dev >= D or negative, token_src >= D,
    non-finite logits) give undefined results but must stay memory-safe: the calls run to completion and
    the next valid call is still bit-exact."""
    cfg = W.CONFIGS["target"].with_(T=4099, P=40)
    rng = np.random.default_rng(7)
    L, T, E, k, P, D = cfg.L, cfg.T, cfg.E, cfg.k, cfg.P, cfg.D
    x = rng.normal(0, 1, (L, T, E)).astype(np.float32)
    x[0, ::7, 3] = np.nan
    x[0, 1::11, 5] = np.inf
    x[0, 2::13, :] = -np.inf
    maps = rng.integers(-2 ** 31, 2 ** 31 - 1, (L, P, E), dtype=np.int64).astype(np.int32)
    src = rng.integers(-2 ** 31, 2 ** 31 - 1, (L, T), dtype=np.int64).astype(np.int32) if with_src else None
    dn_d = dev(W.dev_node(cfg))
    topo = topo_of(cfg, dn_d)
    gate = cap.gate_cfg(E, **cfg.gate)
    fb = cap.trace_fused(dev(x), None, gate, dev(src), dev(maps), topo)
    pi = dev(maps[:, 0, :].copy())
    kept, near, aft = cap.prune(fb.idx, fb.w, dev(src), pi, topo, 0.1)
    cap.dispatch_layout(fb.idx[0], kept[0], pi[0], D)
    cap.dispatch_layout(fb.idx[0], None, pi[0], D)
    cap.eval_placements(fb.idx, kept, dev(src), dev(maps), topo)
    bad_idx = dev(rng.integers(-2 ** 31, 2 ** 31 - 1, (L, T, k), dtype=np.int64).astype(np.int32))
    cap.coactivation(bad_idx, None, E)
    cap.coactivation(bad_idx, kept, E)
    cap.eval_placements(bad_idx, None, dev(src), dev(maps), topo, counts=None)
    if E != 512:
        cap.coactivation(bad_idx[:, :300].contiguous(), None, 512)          # the four-row-block tensor-core path
    cap.coactivation(bad_idx[:, :300].contiguous(), None, 1024)             # the histogram path of large E
    torch.cuda.synchronize()
    check_all_stages(W.CONFIGS["tiny"], tag="after garbage ")


def test_config5_maximum_size_sampled_and_invariants():
    """Config 5 at the top of its T sweep (2^22 tokens, E=512, top-10, 64 devices over 8 nodes): 8.6 GB of
    logits, 41.9 M (token, slot) pairs.  The oracle cannot run the whole trace, so: sampled tokens are
    checked element by element against it (S1 indices / weights, S3 per-token remote devices / nodes, S4
    kept masks), and the aggregates through properties that hold at any size (BASELINE.json invariants:
    sum of counts = T k, C symmetric with diag = counts and off-diagonal row sums = (k-1) counts; S3 totals
    equal the sums of the per-token outputs; S5 is a stable permutation of the kept pairs grouped by
    device).  Inputs: the BASELINE generator of config 5 (workload.logits) evaluated on the GPU by
    paper_2607_05116_b200/workload_device.py, checked bit for bit against the host generator on sampled rows.  The sweep
    points 2^18 and 2^20 are compared with the chunked oracle in tests/test_gpu_fullsize.py."""
    cfg = W.CONFIGS["stress"]
    L, T, E, k, D, N = 1, 1 << 22, cfg.E, cfg.k, cfg.D, cfg.N
    from paper_2607_05116_b200 import workload_device as G
    cfg = cfg.with_(T=T)
    x = G.logits_device(cfg, 0)[None]                 # the BASELINE generator, evaluated on the device
    gate = cap.gate_cfg(E, **cfg.gate)
    dn = W.dev_node(cfg)
    dn_d = dev(dn)
    topo = topo_of(cfg, dn_d)
    rng = np.random.default_rng(5)
    sample = np.unique(np.concatenate([np.arange(0, 48), np.arange(T - 48, T),
                                       rng.integers(0, T, 4000)])).astype(np.int64)
    samp_d = torch.from_numpy(sample).cuda()
    G.check_rows_against_host(cfg, 0, x[0], sample[::64])   # device generator == host generator, bit for bit

    # S1 on everything, oracle on the sample
    idx_d, w_d = cap.gate_topk(x, None, gate)
    xs = x[0, samp_d].cpu().numpy()[None]
    idx_r, w_r = O.gate_topk(xs, None, **cfg.gate)
    assert np.array_equal(idx_d[0, samp_d].cpu().numpy()[None], idx_r)
    assert float(np.abs(w_d[0, samp_d].cpu().numpy()[None].astype(np.float64) - w_r).max()) <= 1e-6
    del x
    torch.cuda.empty_cache()

    # S2: invariants + an independent count
    cnt_d, C_d = cap.coactivation(idx_d, None, E)
    cnt_t = torch.bincount(idx_d.reshape(-1).long(), minlength=E)
    assert torch.equal(cnt_d[0], cnt_t) and int(cnt_d.sum()) == T * k
    Cl = C_d[0].long()
    assert torch.equal(Cl, Cl.t()) and torch.equal(torch.diagonal(Cl), cnt_d[0])
    assert torch.equal(Cl.sum(1) - torch.diagonal(Cl), (k - 1) * cnt_d[0])

    # S3: P = 48 candidates with per-token outputs; sampled tokens against the oracle, totals against the sums
    P = 48
    cand = W.candidates(cfg, 0, P)[None]
    cand_d = dev(cand)
    ev = cap.eval_placements(idx_d, None, None, cand_d, topo, counts=cnt_d, per_token=True)
    src_s = ((sample * D) // T).astype(np.int32)[None]
    ev_r = O.eval_placements(idx_r, cand, dn, token_src=src_s, cost_inter=cfg.cost_inter,
                             bytes_per_token=cfg.bytes_per_token, per_token=True)
    assert np.array_equal(ev.tok_remote_dev[0][:, samp_d].cpu().numpy(), ev_r.tok_remote_dev[0])
    assert np.array_equal(ev.tok_remote_node[0][:, samp_d].cpu().numpy(), ev_r.tok_remote_node[0])
    assert torch.equal(ev.remote_dev[0], ev.tok_remote_dev[0].long().sum(1))
    assert torch.equal(ev.remote_node[0], ev.tok_remote_node[0].long().sum(1))
    assert torch.equal(ev.dev_visits[0], ev.recv_tokens[0].sum(1))
    assert bool((ev.load_pairs[0].sum(1) == T * k).all())
    assert torch.equal(ev.bytes[0], ev.remote_dev[0] * cfg.bytes_per_token)
    assert torch.equal(ev.remote_dev[0], ev.remote_intra[0] + ev.remote_inter[0])
    # the fast (bit-sliced) path without per-token outputs gives the same totals
    ev2 = cap.eval_placements(idx_d, None, None, cand_d, topo, counts=cnt_d)
    for name in ("dev_visits", "remote_dev", "remote_intra", "remote_inter", "node_visits", "remote_node", "cost",
                 "bytes", "load_pairs", "recv_tokens"):
        assert torch.equal(getattr(ev, name), getattr(ev2, name)), name
    del ev, ev2
    torch.cuda.empty_cache()

    # S4: sampled tokens against the oracle; after-metrics against an evaluation of the kept trace
    pi = cand[:, 2, :].copy()
    pi_d = dev(pi)
    tau = cfg.taus[-1]
    kept_d, near_d, aft = cap.prune(idx_d, w_d, None, pi_d, topo, tau)
    w_s = w_d[0, samp_d].cpu().numpy()[None]
    kept_r, near_r = O.prune(idx_r, w_s, pi, dn, tau, token_src=src_s, cost_inter=cfg.cost_inter)
    assert np.array_equal(kept_d[0, samp_d].cpu().numpy()[None], kept_r)
    ev_k = cap.eval_placements(idx_d, kept_d, None, pi_d[:, None, :].contiguous(), topo)
    assert_eval_equal(aft, SimpleNamespace(**{n: host(getattr(ev_k, n)) for n in
                                              ("dev_visits", "remote_dev", "remote_intra", "remote_inter", "node_visits",
                                               "remote_node", "cost", "bytes", "load_pairs", "recv_tokens", "imbalance",
                                               "imbalance_recv")}), False, "2^22 after-prune ")

    # S5: stable permutation of the kept pairs grouped by device
    sp, off, pos = cap.dispatch_layout(idx_d[0], kept_d[0], pi_d[0], D)
    n_kept = int(kept_d.sum())
    assert int(off[0]) == 0 and int(off[-1]) == n_kept
    spv = sp[:n_kept].long()
    keys = pi_d[0].long()[idx_d[0].reshape(-1).long()[spv]]
    assert bool((keys[1:] >= keys[:-1]).all())                                   # grouped by device
    assert torch.equal(torch.bincount(keys, minlength=D).cumsum(0), off[1:])     # offsets = prefix of the counts
    same = keys[1:] == keys[:-1]
    assert bool((spv[1:][same] > spv[:-1][same]).all())                          # ascending inside a device: stable
    assert bool(kept_d.reshape(-1)[spv].all())                                   # only kept pairs
    assert torch.equal(pos.long()[spv], torch.arange(n_kept, device="cuda"))     # inverse permutation
    assert int((pos >= 0).sum()) == n_kept

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

"""Shared helpers for the GPU parity tests: run the CUDA path (through the C ABI binding) and
the CPU oracle on the same seeded inputs and compare element by element."""
import numpy as np
import torch

from oracle import cap_oracle as O
from paper_2607_05116_b200 import cap
from paper_2607_05116_b200 import workload as W

EVAL_I64 = ("dev_visits", "remote_dev", "remote_intra", "remote_inter", "node_visits",
            "remote_node", "cost", "bytes", "load_pairs", "recv_tokens")
W_TOL = 1e-6   # BASELINE.json north_star: gate weights within 1e-6 absolute


def dev(a, dtype=None):
    if a is None:
        return None
    t = torch.from_numpy(np.ascontiguousarray(a))
    if dtype is not None:
        t = t.to(dtype)
    return t.cuda()


def host(t):
    return None if t is None else t.cpu().numpy()


def topo_of(cfg, dn_dev, cost_local=0):
    return cap.topology(dn_dev, cost_local=cost_local, cost_intra=1, cost_inter=cfg.cost_inter,
                        bytes_per_token=cfg.bytes_per_token, N=cfg.N)


def assert_eval_equal(got, ref, per_token=False, tag=""):
    for name in EVAL_I64:
        g = host(getattr(got, name))
        r = getattr(ref, name)
        assert np.array_equal(g, r), f"{tag}{name}: {int((g != r).sum())} mismatches"
    for name in ("imbalance", "imbalance_recv"):
        g = host(getattr(got, name))
        r = getattr(ref, name)
        assert np.array_equal(g, r), f"{tag}{name} differs (max {np.abs(g - r).max()})"
    if per_token:
        for name in ("tok_remote_dev", "tok_remote_node"):
            assert np.array_equal(host(getattr(got, name)), getattr(ref, name)), tag + name


def layers_inputs(cfg, layers, T):
    xs, bs, cs = [], [], []
    for l in layers:
        x, b, c = W.layer_inputs(cfg.with_(T=T), l, T)
        xs.append(x)
        bs.append(b)
        cs.append(c)
    logits = np.stack(xs)
    bias = np.stack(bs) if bs[0] is not None else None
    cand = np.stack(cs)
    return logits, bias, cand


def check_gate(logits, bias, gate, tag=""):
    """returns (idx_ref, w_ref, idx_dev, w_dev, max |dw|)"""
    idx_r, w_r = O.gate_topk(logits, bias, **gate)
    cfg = cap.gate_cfg(logits.shape[-1], **gate)
    idx_d, w_d = cap.gate_topk(dev(logits), dev(bias), cfg)
    torch.cuda.synchronize()
    gi, gw = host(idx_d), host(w_d)
    assert np.array_equal(gi, idx_r), f"{tag}topk_idx: {int((gi != idx_r).any(-1).sum())} tokens differ"
    dmax = float(np.abs(gw.astype(np.float64) - w_r.astype(np.float64)).max()) if gw.size else 0.0
    assert dmax <= W_TOL, f"{tag}topk_w max abs diff {dmax}"
    return idx_r, w_r, idx_d, w_d, dmax


def check_all_stages(cfg, layers=(0,), T=None, random_src=False, per_token=False, tag=""):
    """Full pipeline parity for `layers` of config `cfg` at T tokens per layer."""
    T = cfg.T if T is None else T
    L = len(layers)
    logits, bias, cand = layers_inputs(cfg, layers, T)
    dn = W.dev_node(cfg)
    src = np.stack([W.token_src_random(cfg, l, T) for l in layers]) if random_src else None
    report = {}

    # S1
    idx_r, w_r, idx_d, w_d, dmax = check_gate(logits, bias, cfg.gate, tag)
    report["w_max_abs_diff"] = dmax
    report["w_bit_identical"] = bool(np.array_equal(host(w_d), w_r))

    # S2
    cnt_r, C_r = O.coactivation(idx_r, E=cfg.E)
    cnt_d, C_d = cap.coactivation(idx_d, None, cfg.E)
    assert np.array_equal(host(cnt_d), cnt_r), tag + "counts"
    assert np.array_equal(host(C_d), C_r), tag + "coact"

    # S3
    dn_d = dev(dn)
    topo = topo_of(cfg, dn_d)
    ev_r = O.eval_placements(idx_r, cand, dn, token_src=src, cost_inter=cfg.cost_inter,
                             bytes_per_token=cfg.bytes_per_token, per_token=per_token)
    cand_d, src_d = dev(cand), dev(src)
    ev_d = cap.eval_placements(idx_d, None, src_d, cand_d, topo, counts=cnt_d, per_token=per_token)
    assert_eval_equal(ev_d, ev_r, per_token, tag + "eval ")
    ev_d2 = cap.eval_placements(idx_d, None, src_d, cand_d, topo, counts=None)   # recount path
    assert_eval_equal(ev_d2, ev_r, False, tag + "eval(no counts) ")

    # fused S1+S2+S3
    fb = cap.trace_fused(dev(logits), dev(bias), cap.gate_cfg(cfg.E, **cfg.gate), src_d, cand_d, topo,
                         per_token=per_token)
    torch.cuda.synchronize()
    assert np.array_equal(host(fb.idx), idx_r), tag + "fused idx"
    assert float(np.abs(host(fb.w).astype(np.float64) - w_r).max()) <= W_TOL, tag + "fused w"
    assert np.array_equal(host(fb.counts), cnt_r), tag + "fused counts"
    assert np.array_equal(host(fb.coact), C_r), tag + "fused coact"
    assert_eval_equal(fb.out, ev_r, per_token, tag + "fused eval ")

    # S4 (stage-isolated on the oracle's S1 output, then end-to-end on the GPU's)
    pi = cand[:, 2 if cand.shape[1] > 2 else 0, :]          # one chosen placement per layer
    pi_d = dev(pi)
    w_r_d = dev(w_r)
    idx_r_d = dev(idx_r)
    for tau in cfg.taus + (0.0,):
        kept_r, near_r = O.prune(idx_r, w_r, pi, dn, tau, token_src=src, cost_inter=cfg.cost_inter)
        aft_r = O.eval_placements(idx_r, pi[:, None, :], dn, kept=kept_r, token_src=src,
                                  cost_inter=cfg.cost_inter, bytes_per_token=cfg.bytes_per_token)
        kept_d, near_d, aft_d = cap.prune(idx_r_d, w_r_d, src_d, pi_d, topo, tau)
        assert np.array_equal(host(kept_d), kept_r), f"{tag}kept (isolated) tau={tau}"
        assert np.array_equal(host(near_d), near_r), f"{tag}near_margin tau={tau}"
        assert_eval_equal(aft_d, aft_r, False, f"{tag}after-prune tau={tau} ")
        # end to end: GPU weights -> GPU prune; mismatching tokens must be near-margin tokens
        kept_e, near_e, _ = cap.prune(idx_d, w_d, src_d, pi_d, topo, tau)
        bad = (host(kept_e) != kept_r).any(-1).sum()
        assert bad <= int(near_r.sum()), f"{tag}kept (end-to-end) tau={tau}: {bad} tokens differ"
        report[f"near_margin_tau{tau}"] = int(near_r.sum())
        report[f"e2e_prune_mismatch_tau{tau}"] = int(bad)
        # pruned co-activation (the trace Step 2 of the paper consumes)
        cntp_r, Cp_r = O.coactivation(idx_r, kept_r, E=cfg.E)
        cntp_d, Cp_d = cap.coactivation(idx_r_d, kept_d, cfg.E)
        assert np.array_equal(host(cntp_d), cntp_r) and np.array_equal(host(Cp_d), Cp_r), tag + "pruned coact"

    # S5 (layer 0), unpruned and pruned
    kept0_r, _ = O.prune(idx_r[:1], w_r[:1], pi[:1], dn, cfg.taus[0], token_src=None if src is None else src[:1],
                         cost_inter=cfg.cost_inter)
    for m in (None, kept0_r[0]):
        sp_r, off_r, pos_r = O.dispatch_layout(idx_r[0], pi[0], cfg.D, kept=m)
        sp_d, off_d, pos_d = cap.dispatch_layout(idx_r_d[0], dev(m), pi_d[0].contiguous(), cfg.D)
        n = int(off_r[-1])
        assert np.array_equal(host(off_d), off_r), tag + "offsets"
        assert np.array_equal(host(sp_d)[:n], sp_r), tag + "sorted_pairs"
        assert np.array_equal(host(pos_d), pos_r), tag + "pair_pos"
    return report

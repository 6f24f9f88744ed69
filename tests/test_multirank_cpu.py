"""N > 1 path on the CPU (gloo, world_size 2): tokens are independent units, so the path shards with no
data-path collective; merging shards is one all-reduce(sum) of the integer aggregates.  Each rank runs
the oracle on its own token range (explicit token_src, since the default source of a token depends on
its global position) and the reduced sums must equal the single-process result bit for bit."""
import os

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2607_05116_b200 import workload as W


def _whole(cfg):
    from oracle import cap_oracle as O
    x, _, cand = W.layer_inputs(cfg, 0)
    dn = W.dev_node(cfg)
    src = ((np.arange(cfg.T, dtype=np.int64) * cfg.D) // cfg.T).astype(np.int32)
    idx, w = O.gate_topk(x[None], None, **cfg.gate)
    return O, x, cand, dn, src, idx, w


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cfg = W.CONFIGS["tiny"]
    O, x, cand, dn, src, _, _ = _whole(cfg)
    lo, hi = rank * cfg.T // world, (rank + 1) * cfg.T // world
    idx, w = O.gate_topk(x[None, lo:hi], None, **cfg.gate)
    counts, coact = O.coactivation(idx, E=cfg.E)
    ev = O.eval_placements(idx, cand[None], dn, token_src=src[None, lo:hi], cost_inter=cfg.cost_inter,
                           bytes_per_token=cfg.bytes_per_token)
    parts = [torch.from_numpy(np.ascontiguousarray(a)).to(torch.int64) for a in
             (counts, coact, ev.dev_visits, ev.remote_dev, ev.remote_intra, ev.remote_inter, ev.node_visits,
              ev.remote_node, ev.cost, ev.bytes, ev.load_pairs, ev.recv_tokens)]
    for t in parts:
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
    # the consumers of the merged statistics (Algorithm 1 placement, adjustment spectrum) are
    # deterministic: every rank derives the same placement from the all-reduced counts / coact
    g, gn, ed, _ = O.coact_placement(parts[0].numpy(), parts[1].numpy().astype(np.int32), D=cfg.D, N=cfg.N)
    spec, _, _ = O.adjust_spectrum(parts[0].numpy(), parts[1].numpy().astype(np.int32), ed, D=cfg.D, S=3)
    mine = torch.from_numpy(np.concatenate([ed.ravel(), spec.ravel()]).astype(np.int64))
    lo_t, hi_t = mine.clone(), mine.clone()
    dist.all_reduce(lo_t, op=dist.ReduceOp.MIN)
    dist.all_reduce(hi_t, op=dist.ReduceOp.MAX)
    assert torch.equal(lo_t, hi_t)
    if rank == 0:
        q.put([t.numpy() for t in parts] + [mine.numpy()])
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_shards_sum_to_whole():
    cfg = W.CONFIGS["tiny"]
    O, x, cand, dn, src, idx, w = _whole(cfg)
    counts, coact = O.coactivation(idx, E=cfg.E)
    ev = O.eval_placements(idx, cand[None], dn, token_src=src[None], cost_inter=cfg.cost_inter,
                           bytes_per_token=cfg.bytes_per_token)
    ref = [counts, coact, ev.dev_visits, ev.remote_dev, ev.remote_intra, ev.remote_inter, ev.node_visits,
           ev.remote_node, ev.cost, ev.bytes, ev.load_pairs, ev.recv_tokens]
    # the explicit contiguous token_src is the NULL default (reading R5)
    ev0 = O.eval_placements(idx, cand[None], dn, cost_inter=cfg.cost_inter, bytes_per_token=cfg.bytes_per_token)
    assert np.array_equal(ev0.remote_dev, ev.remote_dev)
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + (os.getpid() % 2000)
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    _, _, ed, _ = O.coact_placement(counts, coact, D=cfg.D, N=cfg.N)
    spec, _, _ = O.adjust_spectrum(counts, coact, ed, D=cfg.D, S=3)
    ref.append(np.concatenate([ed.ravel(), spec.ravel()]))
    assert len(got) == len(ref)
    for g, r in zip(got, ref):
        assert np.array_equal(g, np.asarray(r).astype(np.int64))

"""bench.py -- routed tokens/s through the whole CAP routing-trace hot path on B200.

One "step" = one pass of every stage of SURVEY.md section 8(a) over one batch of synthetic
router logits: cap_trace_fused (S1 gate top-k + S2 counts/co-activation + S3 scoring of P
candidate placements) -> cap_prune_dispatch under the chosen placement (S4 + S5, all layers, three launches).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config target] [--T tokens] [--impl cap|reference]

Prints ONE JSON line (rank 0).  `value` = tokens of all ranks / device time with the inputs
resident in HBM; `e2e` = the same metric through the host-buffer call (pinned host -> device
copies and the read-back of every output inside the timed region); `roofline` = algorithmic bytes of
the fused S1+S2+S3 PASS (the whole cap_trace_fused call, every kernel of it) / its CUDA-event duration
against MEASURED_PEAKS.json, with the dominant kernel alone as `kernel_only_*`; `stages` = S4 and S5
stand-alone as GB/s; `others` = the other BASELINE configs (2, 4, 5 at both ends of its T sweep), one
line each from the same code; `cpu_baseline` = the CPU oracle on one and on all host cores (reported
baseline, not the target).  `--impl reference` times the oracle alone (the reference arm of this tier).

Timing protocol: a timed "step" is one pass of the path replayed from a CUDA graph;
the timed region is 5 repeats of K x R replays (R = --replays, default so that K x R >= 1000), each repeat
bracketed by CUDA events on the launching stream; `ms_per_step` and `value` come from the median repeat.
Inputs rotate over 8 distinct sets (268 MB of logits > 126 MB L2) or are larger than L2 themselves.

Multi-GPU: tokens are independent units -- every rank runs its own batch, no data-path collective
("scaling": "weak"); only the barrier and the max-over-ranks use NCCL.  `--gpus N` without a torchrun
environment re-launches itself under torch.distributed.run with N ranks.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "routed tokens/s through gate+coactivation+P-placement eval; % of B200 HBM BW"
UNIT = "tokens/s"
N_ROTATE = 8          # distinct input sets rotated between steps (8 x 33.5 MB > 126 MB L2)
FALLBACK_HBM_GBS = 6650.0


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured"
    return FALLBACK_HBM_GBS, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                 "--format=csv,noheader,nounits", "-lms", "200"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._read, daemon=True)
        self.thread.start()

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        self.thread.join(timeout=2)
        sm, mx, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for r in self.rows:
            if len(r) < 6:
                continue
            try:
                sm.append(float(r[0]))
                mx.append(float(r[1]))
            except ValueError:
                continue
            for n, v in zip(names, r[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None,
                "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


# ---- workload ---------------------------------------------------------------------------------
def algorithmic_bytes(cfg, has_src=False):
    """Bytes each kernel must move per launch, keyed by kernel tag."""
    L, T, E, k, P, D = cfg.L, cfg.T, cfg.E, cfg.k, cfg.P, cfg.D
    LT = L * T
    ev_out = L * P * (8 * 8 + 2 * 8 * D + 2 * 8)
    return {
        # 4E + 8k bytes per token (logits in, top-k indices and weights out)
        "trace_fused": LT * (4 * E + 8 * k),
        "gate_topk": LT * (4 * E + 8 * k),
        "coact": LT * 4 * k + L * (4 * E * E + 8 * E),
        "eval": LT * (4 * k + (4 if has_src else 0)) + L * P * E * 4,
        "prune": LT * (8 * k + k),
        "dispatch_hist": LT * 4 * k + LT * k,
        "dispatch_scatter": LT * (4 * k + k + 4 * k + 4 * k),
        "eval_table": L * P * E * 4,
        "eval_decode": ev_out,
        "eval_finalize": L * P * E * 4 + ev_out,
    }


def oracle_step(O, cfg, x, bias, maps, dn):
    """The whole hot path on the CPU oracle (S1..S5), host arrays in, aggregates out."""
    idx, w, counts, coact, ev = O.trace_fused(x, bias, cfg.gate, maps, dn, cost_inter=cfg.cost_inter,
                                              bytes_per_token=cfg.bytes_per_token)
    pi = np.ascontiguousarray(maps[:, 0, :])
    kept, near = O.prune(idx, w, pi, dn, cfg.taus[-1], cost_inter=cfg.cost_inter)
    after = O.eval_placements(idx, pi[:, None, :], dn, kept=kept, cost_inter=cfg.cost_inter,
                              bytes_per_token=cfg.bytes_per_token)
    for l in range(x.shape[0]):
        O.dispatch_layout(idx[l], pi[l], cfg.D, kept=kept[l])
    return ev, after


def oracle_sample(cfg, W, max_tokens=65536):
    """Bounded sample of the workload for the CPU legs: one layer, the first min(T, max_tokens)
    tokens, all P candidates."""
    T = min(cfg.T, max_tokens)
    x = W.logits(cfg, 0, 0, T)[None]
    b = W.gate_bias(cfg, 0)
    maps = W.candidates(cfg, 0)[None]
    return T, x, (b[None] if b is not None else None), maps


def _oracle_shard(args):
    """one worker of the N-core leg: the whole path on its contiguous token range (a trace of its own: every
    aggregate is a sum over tokens, so shards are independent units)"""
    name, T_total, a, b, n_pass = args
    from oracle import cap_oracle as O
    from paper_2607_05116_b200 import workload as W
    O.lib()
    cfg = W.CONFIGS[name].with_(T=T_total)
    x = W.logits(cfg, 0, a, b)[None]
    bias = W.gate_bias(cfg, 0)
    maps = W.candidates(cfg, 0)[None]
    dn = W.dev_node(cfg)
    t0 = time.perf_counter()
    for _ in range(n_pass):
        oracle_step(O, cfg, x, bias[None] if bias is not None else None, maps, dn)
    return time.perf_counter() - t0


def time_oracle(cfg, W, min_seconds, key):
    """The oracle as it stands on one host core, then sharded over all host cores (one process per core,
    contiguous token ranges), on a bounded sample of the workload."""
    import multiprocessing as mp
    from oracle import cap_oracle as O
    O.lib()
    T, x, b, maps = oracle_sample(cfg, W)
    dn = W.dev_node(cfg)
    passes, t0 = 0, time.perf_counter()
    while True:
        oracle_step(O, cfg, x, b, maps, dn)
        passes += 1
        el = time.perf_counter() - t0
        if el >= min_seconds / 2 or passes >= 64:
            break
    v1 = passes * T / el
    ncores = len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)
    out = {"value": v1, "unit": UNIT, "cores": 1, "kind": "oracle",
           "sample": f"{passes} pass(es) of 1 layer x {T} tokens x P={cfg.P} candidates, all 5 stages, "
                     f"{el:.1f} s on one host core"}
    if ncores > 1:
        n_pass = max(1, int(round(passes * min(ncores, 8) / 2)))
        per = (T + ncores - 1) // ncores
        jobs = [(key, T, i * per, min(T, (i + 1) * per), n_pass) for i in range(ncores) if i * per < T]
        try:
            ctx = mp.get_context("fork")
            t0 = time.perf_counter()
            with ctx.Pool(len(jobs)) as pool:
                pool.map(_oracle_shard, jobs)
            eln = time.perf_counter() - t0
            out = {"value": n_pass * T / eln, "unit": UNIT, "cores": len(jobs), "kind": "oracle",
                   "value_1core": v1,
                   "sample": f"{n_pass} pass(es) of 1 layer x {T} tokens x P={cfg.P} candidates, all 5 stages, tokens "
                             f"sharded over {len(jobs)} processes (one per host core; {eln:.1f} s wall incl. process "
                             f"start and each shard generating its own inputs); 1 core: {passes} pass(es) in {el:.1f} s"}
        except Exception as e:                        # the 1-core figure stands
            out["multicore_error"] = repr(e)[:200]
    return out


def config_dict(cfg, extra=None):
    d = {"workload": f"config {cfg.index} '{cfg.name}': L={cfg.L} E={cfg.E} top-{cfg.k} T={cfg.T}/layer "
                     f"D={cfg.D} over N={cfg.N} nodes (cost 0/1/{cfg.cost_inter}) P={cfg.P} "
                     f"tau={cfg.taus[-1]} {'sigmoid+bias group-limited' if cfg.scoring else 'softmax'} renorm",
         "stages": "S1 gate top-k + S2 counts/co-activation + S3 P-candidate scoring (cap_trace_fused) "
                   "-> S4 + S5 cap_prune_dispatch (all layers, three launches); the last launch of S3 (decode) runs on a side "
                   "stream beside S4 / S5 (cap_trace_fused_begin / _finish)",
         "tokens_per_step_per_gpu": cfg.L * cfg.T}
    if extra:
        d.update(extra)
    return d


# ---- reference arm: the CPU oracle ----------------------------------------------------------------
def run_reference(args, cfg, W):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import cap_oracle as O
    O.lib()
    T, x, b, maps = oracle_sample(cfg, W, max_tokens=args.ref_tokens)
    dn = W.dev_node(cfg)
    for _ in range(min(args.warmup, 1)):
        oracle_step(O, cfg, x, b, maps, dn)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle_step(O, cfg, x, b, maps, dn)
    el = time.perf_counter() - t0
    v = args.steps * T / el
    sample = f"each step = 1 layer x {T} tokens x P={cfg.P} candidates, all 5 stages, one host core"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * el / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic", "config": config_dict(cfg, {"sample": sample}),
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


# ---- product arm: the CUDA library ------------------------------------------------------------------
REPEATS = 5


def device_inputs(cfg, W, WD, set_id, rank, dev):
    """One batch resident in HBM: logits [L,T,E] (filled by the device twin of the host generator, checked
    bit for bit on sampled rows of the first layer), bias [L,E]|None, maps [L,P,E]."""
    import torch
    base = rank * 100000 + set_id * cfg.L
    x = torch.empty((cfg.L, cfg.T, cfg.E), dtype=torch.float32, device=dev)
    bs, ms = [], []
    for l in range(cfg.L):
        WD.logits_device(cfg, base + l, out=x[l], device=dev)
        b = W.gate_bias(cfg, base + l)
        if b is not None:
            bs.append(b)
        ms.append(W.candidates(cfg, base + l))
    if set_id == 0:
        WD.check_rows_against_host(cfg, base, x[0], [0, cfg.T // 2, cfg.T - 1])
    b = torch.from_numpy(np.stack(bs)).to(dev) if bs else None
    m = torch.from_numpy(np.stack(ms)).to(dev)
    return x, b, m


def timed_replays(torch, fn, n, barrier):
    """REPEATS repeats of n calls of fn(i), each repeat between two CUDA events on the current stream;
    returns the per-call milliseconds of every repeat."""
    out = []
    for r in range(REPEATS):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record()
        for i in range(n):
            fn(i)
        e1.record()
        barrier()
        out.append(e0.elapsed_time(e1) / n)
    return out


def measure(cfg, W, WD, cap, torch, dev, rank, steps, replays, barrier, light=False):
    """Device-resident numbers of one configuration: the whole step, the fused pass, S4 and S5 alone."""
    L, T, E, k, P, D = cfg.L, cfg.T, cfg.E, cfg.k, cfg.P, cfg.D
    in_bytes = L * T * E * 4
    n_sets = 1 if in_bytes > (256 << 20) else N_ROTATE
    d_sets = [device_inputs(cfg, W, WD, s, rank, dev) for s in range(n_sets)]
    dn = torch.from_numpy(W.dev_node(cfg)).to(dev)
    gate = cap.gate_cfg(E, **cfg.gate)
    pipe = cap.Pipeline(L, T, gate, D, cfg.N, P, dn, cost_inter=cfg.cost_inter,
                        bytes_per_token=cfg.bytes_per_token, tau=cfg.taus[-1], chosen=0, device=dev)
    n0 = cap.launch_count()
    for x, b, m in d_sets[:1]:
        pipe.step(x, b, None, m)
    torch.cuda.synchronize()
    launches_per_step = cap.launch_count() - n0
    graphs = [pipe.capture(x, b, None, m) for x, b, m in d_sets]
    fused_graphs = [pipe.capture_fused(x, b, None, m) for x, b, m in d_sets]
    n = steps * replays
    for i in range(3):
        graphs[i % n_sets].replay()
    ms_step = timed_replays(torch, lambda i: graphs[i % n_sets].replay(), n, barrier)
    ms_fused = timed_replays(torch, lambda i: fused_graphs[i % n_sets].replay(), n, barrier)
    # S4 / S5 alone on the buffers the last step left (inputs of these stages: 4-9 MB, L2-resident between
    # replays at config 3 -- stated in the output)
    g_prune = pipe.capture_stage("prune", None, d_sets[0][2])
    g_disp = pipe.capture_stage("dispatch", None, d_sets[0][2])
    ms_prune = timed_replays(torch, lambda i: g_prune.replay(), n, barrier)
    ms_disp = timed_replays(torch, lambda i: g_disp.replay(), n, barrier)
    g_pd = pipe.capture_stage("prune_dispatch", None, d_sets[0][2])
    ms_pd = timed_replays(torch, lambda i: g_pd.replay(), n, barrier)
    # the dominant kernel of the pass alone, back to back (rotating inputs), by the library's profiling entry
    kms = None
    if not light:
        kms = cap.profile_fused_kernel([d[0] for d in d_sets], gate, d_sets[0][2], pipe.topo, pipe.fb, max(steps, 50))
    # the general reading R5 (explicit, non-contiguous token sources): staged S1 / S2 kernels + the generic S3 kernel
    ms_src = None
    if not light:
        src = torch.from_numpy(np.stack([W.token_src_random(cfg, l) for l in range(L)])).to(dev)
        g_src = [pipe.capture_fused(x, b, src, m) for x, b, m in d_sets]
        ms_src = timed_replays(torch, lambda i: g_src[i % n_sets].replay(), max(10, n // 20), barrier)
        del g_src
    plan = cap.trace_fused_plan(L, T, gate, D, cfg.N, P)
    res = dict(pipe=pipe, d_sets=d_sets, gate=gate, n_sets=n_sets, in_bytes=in_bytes, ms_step=ms_step,
               ms_fused=ms_fused, ms_prune=ms_prune, ms_disp=ms_disp, ms_pd=ms_pd, kernel_ms=kms, plan=plan, ms_src=ms_src,
               launches_per_step=launches_per_step)
    return res


def summarise(cfg, res, peak):
    """The per-configuration numbers that go into the JSON line (main config and `others`)."""
    ab = algorithmic_bytes(cfg)
    LT = cfg.L * cfg.T
    med = lambda v: float(np.median(v))
    ms_step, ms_fused = med(res["ms_step"]), med(res["ms_fused"])
    ms_prune, ms_disp = med(res["ms_prune"]), med(res["ms_disp"])
    gbs = lambda b, ms: b / (ms * 1e-3) / 1e9
    b_disp = ab["dispatch_scatter"]          # read idx + kept, write sorted_pairs + pair_pos: 104 B/token at k = 8
    out = {
        "tokens_per_step": LT, "ms_per_step": ms_step, "tokens_per_s": LT / (ms_step * 1e-3),
        "fused_pass_ms": ms_fused, "fused_pass_gbs": gbs(ab["trace_fused"], ms_fused),
        "fused_pass_frac_of_hbm_peak": gbs(ab["trace_fused"], ms_fused) / peak,
        "fused_kernel": "single fused S1+S2+S3 kernel" if res["plan"]["fused"] else "staged S1, S2, S3 kernels",
        "stages": {
            "S4_cap_prune": {"ms": ms_prune, "algorithmic_bytes": ab["prune"], "gbs": gbs(ab["prune"], ms_prune),
                             "frac_of_hbm_peak": gbs(ab["prune"], ms_prune) / peak},
            "S5_cap_dispatch_layout": {"ms": ms_disp, "algorithmic_bytes": b_disp, "gbs": gbs(b_disp, ms_disp),
                                       "frac_of_hbm_peak": gbs(b_disp, ms_disp) / peak,
                                       "calls": 1, "layers": cfg.L},
            "S4S5_cap_prune_dispatch": {"ms": med(res["ms_pd"]), "algorithmic_bytes": ab["prune"] + b_disp,
                                        "gbs": gbs(ab["prune"] + b_disp, med(res["ms_pd"])),
                                        "frac_of_hbm_peak": gbs(ab["prune"] + b_disp, med(res["ms_pd"])) / peak,
                                        "what": "the fused S4 + S5 call the step uses (three launches); the two rows "
                                                "above are the stand-alone calls"},
        },
        "launches_per_step": int(res["launches_per_step"]),
    }
    if res.get("ms_src"):
        ms = med(res["ms_src"])
        out["explicit_token_src_pass"] = {
            "ms": ms, "gbs": gbs(ab["trace_fused"], ms), "frac_of_hbm_peak": gbs(ab["trace_fused"], ms) / peak,
            "what": "cap_trace_fused with an explicit random token_src (reading R5): staged gate + co-activation "
                    "kernels, tokens grouped by source with the S5 counting sort, then the bit-sliced S3 kernel over the runs"}
    return out


def run_cap(args, cfg, W):
    import torch
    import torch.distributed as dist
    from paper_2607_05116_b200 import build as capbuild
    from paper_2607_05116_b200 import cap
    from paper_2607_05116_b200 import workload_device as WD

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    if rank == 0:
        capbuild.build()
    if world > 1:
        dist.barrier()
    cap.lib()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    steps = args.steps
    replays = args.replays if args.replays > 0 else max(1, -(-1000 // steps))
    L, T, E, k, P, D = cfg.L, cfg.T, cfg.E, cfg.k, cfg.P, cfg.D
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    for _ in range(max(args.warmup, 3)):            # warm-up of the context / clocks before anything is timed
        torch.empty(1 << 20, device=dev).zero_()
    res = measure(cfg, W, WD, cap, torch, dev, rank, steps, replays, barrier)
    pipe, d_sets, n_sets = res["pipe"], res["d_sets"], res["n_sets"]

    # ---- end to end: pinned host inputs -> device -> step -> every output back to the host ----------
    # (two staging sets: the upload of step i+1 and the read-back of step i-1 overlap the compute of step
    # i; every step uploads its own inputs and reads back all of its own outputs inside the timed region)
    h_sets = [tuple(None if a is None else a.cpu().pin_memory() for a in d) for d in d_sets]
    hpipe = cap.HostPipeline(pipe, has_bias=cfg.has_bias, depth=2)
    hpipe.capture()

    def hstep(i):
        x, b, m = h_sets[i % n_sets]
        hpipe.step(x, m, b)

    for i in range(3):
        hstep(i)
    hpipe.finish()
    n_e2e = max(steps, 20)
    ms_e2e = []
    for r in range(3):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record()
        for i in range(n_e2e):
            hstep(i)
        hpipe.finish()
        e1.record()
        barrier()
        ms_e2e.append(e0.elapsed_time(e1) / n_e2e)
    clocks = sampler.stop() if rank == 0 else None
    x0, b0, m0 = h_sets[0]
    h2d = sum(a.numel() * a.element_size() for a in (x0, b0, m0) if a is not None)
    d2h = hpipe.d2h_bytes
    del hpipe, h_sets

    # ---- SURVEY 8(f) consumers, outside every timed region above ----
    def time_us(fn, nrep=10):
        for _ in range(3):
            fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(nrep):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / nrep * 1e3

    pipe.step(*d_sets[0][:2], None, d_sets[0][2])
    ws_pl = cap.workspace(cap.CALL_COACT_PLACEMENT, L, 0, E, 1, D, 0, device=dev)
    us_place = time_us(lambda: cap.coact_placement(pipe.fb.counts, pipe.fb.coact, D, cfg.N, ws=ws_pl))
    maps0 = d_sets[0][2]
    us_obj = time_us(lambda: cap.pairwise_objective(pipe.fb.counts, pipe.fb.coact, maps0, pipe.topo))
    # the paper's order for re-placement: statistics of the PRUNED trace, then Algorithm 1
    cnt_k = torch.empty_like(pipe.fb.counts)
    co_k = torch.empty_like(pipe.fb.coact)

    def pruned_stats_then_place():
        cap.coactivation(pipe.fb.idx, pipe.kept, E, counts=cnt_k, coact=co_k)
        cap.coact_placement(cnt_k, co_k, D, cfg.N, ws=ws_pl)
    us_pruned_place = time_us(pruned_stats_then_place)
    ws_rows = cap.workspace(cap.CALL_DISPATCH_ROWS, 1, T, E, k, D, 0, device=dev)
    pi0 = maps0[0, 0].contiguous()
    us_rows = time_us(lambda: cap.dispatch_rows(pipe.fb.idx[0], pipe.kept[0], pi0, D, ws=ws_rows))

    ms_step = float(np.median(res["ms_step"]))
    ms_e2e_med = float(np.median(ms_e2e))
    if world > 1:
        tt = torch.tensor([ms_step, ms_e2e_med], device=dev, dtype=torch.float64)
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        ms_step, ms_e2e_med = float(tt[0]), float(tt[1])
    peak, peak_src = _peaks()
    main = summarise(cfg, res, peak)
    kms = res["kernel_ms"]
    ab = algorithmic_bytes(cfg)

    # ---- the other BASELINE configurations through the same code (rank 0, one GPU's worth each) ----
    others = {}
    rep_step = [round(float(v), 6) for v in res["ms_step"]]
    rep_fused = [round(float(v), 6) for v in res["ms_fused"]]
    del res, pipe, d_sets
    torch.cuda.empty_cache()
    if rank == 0 and not args.no_others and args.config == "target" and args.T == 0:
        for name, Tover, st in (("qwen3", 0, 20), ("dsv3", 0, 5), ("stress", 1 << 16, 10), ("stress", 1 << 22, 3)):
            c = W.CONFIGS[name]
            if Tover:
                c = c.with_(T=Tover)
            try:
                r = measure(c, W, WD, cap, torch, dev, 0, st, 1, lambda: torch.cuda.synchronize(), light=True)
                o = summarise(c, r, peak)
                o["workload"] = config_dict(c)["workload"]
                o["timed"] = f"{REPEATS} repeats of {st} graph replays, median"
                others[f"config{c.index}_{name}" + (f"_T{Tover}" if Tover else "")] = o
                del r
            except Exception as e:                  # a failure here must not take the headline line down
                others[f"config{c.index}_{name}" + (f"_T{Tover}" if Tover else "")] = {"error": repr(e)[:300]}
            torch.cuda.empty_cache()
    if world > 1:
        dist.barrier()

    tokens_per_step = world * L * T
    if rank == 0:
        fused_gbs = main["fused_pass_gbs"]
        out = {
            "metric": METRIC, "value": tokens_per_step / (ms_step * 1e-3), "unit": UNIT, "n_gpus": world,
            "steps": steps, "warmup": max(args.warmup, 3), "ms_per_step": ms_step,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic",
            "config": config_dict(cfg, {
                "l2": (f"inputs rotate over {n_sets} distinct sets ({n_sets * main['tokens_per_step'] * E * 4 / 1e6:.0f} MB of "
                       f"logits > 126 MB L2)") if n_sets > 1 else f"one input set of {L * T * E * 4 / 1e6:.0f} MB > 126 MB L2",
                "launch": "a step is replayed from a CUDA graph (one graph per input set)",
                "timing": f"{REPEATS} repeats of {steps} x {replays} replays, each repeat between two CUDA events on the "
                          f"launching stream; ms_per_step = median repeat / replays",
                "parallelism": f"{world} independent rank(s), token batches sharded, no data-path collective"}),
            "replays_per_step": replays, "repeats": REPEATS,
            "ms_per_step_repeats": rep_step, "fused_pass_ms_repeats": rep_fused,
            "e2e": {"value": tokens_per_step / (ms_e2e_med * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d,
                    "d2h_bytes_per_step": d2h, "ms_per_step": ms_e2e_med,
                    "timed": f"3 repeats of {n_e2e} host-buffer steps, median"},
            "gpu_launches": int(main["launches_per_step"]) * steps * replays * REPEATS,
            "gpu_launches_per_step": int(main["launches_per_step"]),
            "clocks": clocks,
            "roofline": {
                "bound": "hbm", "kernel": "cap_trace_fused (the whole S1+S2+S3 pass: " + main["fused_kernel"] + " + its table and decode kernels)",
                "achieved": fused_gbs, "peak": peak, "unit": "GB/s", "frac": fused_gbs / peak, "traffic": None,
                "traffic_note": "not measured inside this run; the ncu capture of the dominant kernel is in profiles/",
                "peak_source": f"MEASURED_PEAKS.json hbm_gbs ({peak_src})",
                "algorithmic_bytes": ab["trace_fused"], "pass_ms": main["fused_pass_ms"],
                "how": "algorithmic bytes (4E + 8k per token) / median CUDA-event time of the cap_trace_fused call replayed "
                       "from a graph with rotating inputs",
                "kernel_only_ms": kms,
                "kernel_only_gbs": (ab["trace_fused"] / (kms * 1e-3) / 1e9) if kms else None,
                "kernel_only_frac": (ab["trace_fused"] / (kms * 1e-3) / 1e9 / peak) if kms else None,
                "kernel_only_how": "cap_profile_fused_kernel: the fused kernel alone, back-to-back launches rotating over "
                                   "the input sets, one CUDA-event pair on the launching stream",
                "ceiling_note": "shared-memory-bound formulation: 30.1 k shared-memory wavefronts per SM per launch (ncu, "
                                "profiles/r2a_step.md) = 15.3 us at one wavefront per clock, i.e. <= 0.38 of the HBM peak for "
                                "the kernel; the 0.60 target is out of reach with it (DESIGN.md 6.4)"},
            "stages": main["stages"],
            "explicit_token_src_pass": main.get("explicit_token_src_pass"),
            "stages_note": "S4 / S5 replayed alone from a graph on the buffers of the last step (their 4-9 MB of inputs "
                           "stay in L2 between replays at this size: launch-latency-bound, see others.config5_stress_T4194304 "
                           "for the bandwidth-bound size)",
            "others": others,
        }
        out["next"] = {"coact_placement": {
            "us_per_call": us_place, "layers": L, "greedy_steps_per_layer": (E - D) + (D - cfg.N),
            "what": "cap_coact_placement (P:L106-144, L148, L162-164) on the step's counts / coact; latency-bound "
                    "sequential greedy, one CTA per layer; not part of `value`"},
            "pruned_stats_then_placement": {
                "us_per_call": us_pruned_place,
                "what": "cap_coactivation with the step's kept mask (statistics of the pruned trace, P:L224) followed by "
                        "cap_coact_placement on them: the paper's order for re-placement after pruning"},
            "pairwise_objective": {"us_per_call": us_obj, "candidates": P, "what": "cap_pairwise_objective (Eq. 2-3) "
                                   "on the step's counts / coact and its P candidate maps"},
            "dispatch_rows": {"us_per_call": us_rows, "what": "cap_dispatch_rows (P:L58, Fig. 2) for layer 0 under "
                              "candidate 0 with the step's pruning mask; three direct launches through the binding, "
                              "output tensors allocated per call"}}
        if not args.no_cpu_baseline:
            out["cpu_baseline"] = time_oracle(cfg, W, args.cpu_seconds, args.config)
        print(json.dumps(out))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="cap", choices=["cap", "reference"])
    ap.add_argument("--config", default="target")
    ap.add_argument("--T", type=int, default=0, help="tokens per layer (config 5 sweeps 2^16..2^22); 0 = the config's own")
    ap.add_argument("--replays", type=int, default=0, help="graph replays per timed step; 0 = ceil(1000 / steps)")
    ap.add_argument("--cpu-seconds", type=float, default=20.0)
    ap.add_argument("--ref-tokens", type=int, default=16384)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-others", action="store_true", help="skip the lines of the other BASELINE configs")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and args.impl == "cap":
        # `python bench.py --gpus N` starts its own N ranks (one per GPU); NCCL's communicator log stays on
        env = dict(os.environ)
        env.setdefault("NCCL_DEBUG", "WARN")
        port = 29500 + (os.getpid() % 2000)
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        raise SystemExit(subprocess.call(cmd, env=env))
    from paper_2607_05116_b200 import workload as W
    cfg = W.CONFIGS[args.config]
    if args.T > 0:
        cfg = cfg.with_(T=args.T)
    if args.impl == "reference":
        run_reference(args, cfg, W)
    else:
        run_cap(args, cfg, W)


if __name__ == "__main__":
    main()

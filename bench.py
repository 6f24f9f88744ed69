"""bench.py -- routed tokens/s through the whole CAP routing-trace hot path on B200.

One "step" = one pass of every stage of SURVEY.md section 8(a) over one batch of synthetic
router logits: cap_trace_fused (S1 gate top-k + S2 counts/co-activation + S3 scoring of P
candidate placements) -> cap_prune under the chosen placement (S4) -> cap_dispatch_layout (S5).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config target] [--impl cap|reference]

Prints ONE JSON line (rank 0).  `value` = tokens of all ranks / device time with the inputs
resident in HBM; `e2e` = the same metric through the host-buffer call (pinned host -> device
copies and the read-back of every output inside the timed region); `roofline` = the dominant
kernel's algorithmic bytes / its CUDA-event duration against MEASURED_PEAKS.json; `cpu_baseline`
= the CPU oracle on the same workload (reported baseline, not the target).
`--impl reference` times the oracle alone (the reference arm of this tier).
Multi-GPU (torchrun): tokens are independent units -- every rank runs its own batch, no
data-path collective ("scaling": "weak"); only the barrier and the max-over-ranks use NCCL.
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


def _ncu_traffic(kernel, workload):
    """dram bytes read + written per launch of `kernel` from the committed `ncu --set full` capture
    (profiles/ncu_traffic.txt: lines `kernel workload bytes source`), or None."""
    p = os.path.join(ROOT, "profiles", "ncu_traffic.txt")
    if not os.path.exists(p):
        return None
    with open(p) as f:
        for line in f:
            t = line.split()
            if len(t) >= 3 and not line.startswith("#") and t[0] == kernel and t[1] == workload:
                return int(t[2])
    return None


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
def make_inputs(cfg, W, set_id, rank):
    """Host inputs of one batch: logits [L,T,E], bias [L,E]|None, maps [L,P,E] (seeded; the layer
    number is the seed stream, so every (rank, set) is a distinct trace of the same recipe)."""
    base = rank * 100000 + set_id * cfg.L
    xs, bs, ms = [], [], []
    for l in range(cfg.L):
        xs.append(W.logits(cfg, base + l))
        b = W.gate_bias(cfg, base + l)
        if b is not None:
            bs.append(b)
        ms.append(W.candidates(cfg, base + l))
    return np.stack(xs), (np.stack(bs) if bs else None), np.stack(ms)


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


def time_oracle(cfg, W, min_seconds):
    from oracle import cap_oracle as O
    O.lib()
    T, x, b, maps = oracle_sample(cfg, W)
    dn = W.dev_node(cfg)
    passes, t0 = 0, time.perf_counter()
    while True:
        oracle_step(O, cfg, x, b, maps, dn)
        passes += 1
        el = time.perf_counter() - t0
        if el >= min_seconds or passes >= 64:
            break
    return {"value": passes * T / el, "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": f"{passes} pass(es) of 1 layer x {T} tokens x P={cfg.P} candidates, all 5 stages, "
                      f"{el:.1f} s on one host core"}


def config_dict(cfg, extra=None):
    d = {"workload": f"config {cfg.index} '{cfg.name}': L={cfg.L} E={cfg.E} top-{cfg.k} T={cfg.T}/layer "
                     f"D={cfg.D} over N={cfg.N} nodes (cost 0/1/{cfg.cost_inter}) P={cfg.P} "
                     f"tau={cfg.taus[-1]} {'sigmoid+bias group-limited' if cfg.scoring else 'softmax'} renorm",
         "stages": "S1 gate top-k + S2 counts/co-activation + S3 P-candidate scoring (cap_trace_fused) "
                   "-> S4 cap_prune -> S5 cap_dispatch_layout",
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
def run_cap(args, cfg, W):
    import torch
    import torch.distributed as dist
    from paper_2607_05116_b200 import build as capbuild
    from paper_2607_05116_b200 import cap

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

    L, T, E, k, P, D = cfg.L, cfg.T, cfg.E, cfg.k, cfg.P, cfg.D
    in_bytes = L * T * E * 4
    n_sets = 1 if in_bytes > (256 << 20) else N_ROTATE
    h_sets, d_sets = [], []
    for s in range(n_sets):
        x, b, m = make_inputs(cfg, W, s, rank)
        hs = tuple(None if a is None else torch.from_numpy(a).pin_memory() for a in (x, b, m))
        h_sets.append(hs)
        d_sets.append(tuple(None if a is None else a.to(dev) for a in hs))
    dn = torch.from_numpy(W.dev_node(cfg)).to(dev)
    gate = cap.gate_cfg(E, **cfg.gate)
    pipe = cap.Pipeline(L, T, gate, D, cfg.N, P, dn, cost_inter=cfg.cost_inter,
                        bytes_per_token=cfg.bytes_per_token, tau=cfg.taus[-1], chosen=0, device=dev)
    hpipe = cap.HostPipeline(pipe, has_bias=cfg.has_bias, depth=2)

    def dstep(i):                       # direct launches (per-kernel event timers can be armed)
        x, b, m = d_sets[i % n_sets]
        pipe.step(x, b, None, m)

    graphs = []

    def gstep(i):                       # the same step replayed from a CUDA graph
        graphs[i % n_sets].replay()

    def hstep(i):
        x, b, m = h_sets[i % n_sets]
        hpipe.step(x, m, b)

    # ---- warm-up; find the dominant kernel with the library's per-kernel event timers ----------
    tags = list(cap.KERNEL_TAGS)
    tot = {t: 0.0 for t in tags}
    for i in range(max(args.warmup, 3) + 1):
        for j, t in enumerate(tags):
            cap.kernel_timer_arm(t, j)
        dstep(i)
        torch.cuda.synchronize()
        if i == 0:
            continue                    # first step pays one-time module loading: not representative
        for j, t in enumerate(tags):
            ms = cap.kernel_timer_ms(j)
            if ms > 0:
                tot[t] += ms
    dominant = max(tot, key=lambda t: tot[t])
    for x, b, m in d_sets:
        graphs.append(pipe.capture(x, b, None, m))
    fused_graphs = [pipe.capture_fused(x, b, None, m) for x, b, m in d_sets]
    hpipe.capture()
    for i in range(3):
        gstep(i)

    # ---- timed region: K steps, inputs resident in HBM ---------------------------------------------
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    n0 = cap.launch_count()
    ev0.record()
    for i in range(args.steps):
        gstep(i)
    ev1.record()
    barrier()
    ms = ev0.elapsed_time(ev1)
    # the dominant kernel's duration: the same K steps launched directly, one CUDA-event pair
    # (owned by the library, on the launching stream) around that kernel in every step
    n0 = cap.launch_count()
    for i in range(args.steps):
        cap.kernel_timer_arm(dominant, 100 + i)
        dstep(i)
    barrier()
    launches = cap.launch_count() - n0
    dom_ms = [cap.kernel_timer_ms(100 + i) for i in range(args.steps)]
    dom_ms = [v for v in dom_ms if v > 0]
    dom_how = "library CUDA-event pair around the kernel in K directly launched steps"
    if dominant == "trace_fused":
        # direct launches from Python leave the GPU idle between kernels, which the event pair would
        # count; the library's profiling entry launches the fused kernel alone K times back to back
        # (rotating over the input sets, > L2) between two events on the launching stream
        kms = cap.profile_fused_kernel([d[0] for d in d_sets], gate, d_sets[0][2], pipe.topo, pipe.fb,
                                       max(args.steps, 8))
        if kms is not None:
            dom_ms = [kms]
            dom_how = ("cap_profile_fused_kernel: the fused kernel alone, K back-to-back launches rotating "
                       "over the input sets, one CUDA-event pair on the launching stream")
    # the fused call alone (S1+S2+S3: every kernel and memset of cap_trace_fused), graph replays
    ev4, ev5 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    for i in range(3):
        fused_graphs[i % n_sets].replay()
    torch.cuda.synchronize()
    ev4.record()
    for i in range(args.steps):
        fused_graphs[i % n_sets].replay()
    ev5.record()
    torch.cuda.synchronize()
    ms_fused = ev4.elapsed_time(ev5) / args.steps

    # ---- end to end: pinned host inputs -> device -> step -> every output back to the host ----------
    # (two staging sets: the upload of step i+1 and the read-back of step i-1 overlap the compute of step
    # i; every step uploads its own inputs and reads back all of its own outputs inside the timed region)
    for i in range(3):
        hstep(i)
    hpipe.finish()
    barrier()
    ev2, ev3 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev2.record()
    for i in range(args.steps):
        hstep(i)
    hpipe.finish()
    ev3.record()
    barrier()
    ms_e2e = ev2.elapsed_time(ev3)
    clocks = sampler.stop() if rank == 0 else None

    # ---- SURVEY 8(f) rank 1, outside every timed region above: cap_coact_placement (Jaccard p_ij +
    # Algorithm 1, both stages) on the counts / co-activation matrices the last step left on the device
    dstep(0)
    ws_pl = cap.workspace(cap.CALL_COACT_PLACEMENT, L, 0, E, 1, D, 0, device=dev)
    for _ in range(3):
        cap.coact_placement(pipe.fb.counts, pipe.fb.coact, D, cfg.N, ws=ws_pl)
    torch.cuda.synchronize()
    ev6, ev7 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev6.record()
    for _ in range(10):
        cap.coact_placement(pipe.fb.counts, pipe.fb.coact, D, cfg.N, ws=ws_pl)
    ev7.record()
    torch.cuda.synchronize()
    us_place = ev6.elapsed_time(ev7) / 10 * 1e3

    def time_us(fn, n=10):
        for _ in range(3):
            fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(n):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / n * 1e3

    maps0 = d_sets[0][2]
    us_obj = time_us(lambda: cap.pairwise_objective(pipe.fb.counts, pipe.fb.coact, maps0, pipe.topo))
    ws_rows = cap.workspace(cap.CALL_DISPATCH_ROWS, 1, T, E, k, D, 0, device=dev)
    pi0 = maps0[0, 0].contiguous()
    us_rows = time_us(lambda: cap.dispatch_rows(pipe.fb.idx[0], pipe.kept[0], pi0, D, ws=ws_rows))

    if world > 1:
        tt = torch.tensor([ms, ms_e2e], device=dev, dtype=torch.float64)
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        ms, ms_e2e = float(tt[0]), float(tt[1])
    tokens = world * args.steps * L * T
    if rank == 0:
        peak, peak_src = _peaks()
        ab = algorithmic_bytes(cfg)
        dom_avg = float(np.mean(dom_ms)) if dom_ms else float("nan")
        achieved = ab.get(dominant, 0) / (dom_avg * 1e-3) / 1e9 if dom_ms else None
        x0, b0, m0 = h_sets[0]
        h2d = sum(a.numel() * a.element_size() for a in (x0, b0, m0) if a is not None)
        out = {
            "metric": METRIC, "value": tokens / (ms * 1e-3), "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic",
            "config": config_dict(cfg, {
                "l2": (f"inputs rotate over {n_sets} distinct sets ({n_sets * in_bytes / 1e6:.0f} MB of logits "
                       f"> 126 MB L2)") if n_sets > 1 else f"one input set of {in_bytes / 1e6:.0f} MB > 126 MB L2",
                "launch": "timed region replays the step from a CUDA graph (one graph per input set); "
                          "roofline.kernel_ms comes from the same steps launched directly",
                "parallelism": f"{world} independent rank(s), token batches sharded, no data-path collective"}),
            "e2e": {"value": tokens / (ms_e2e * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d,
                    "d2h_bytes_per_step": hpipe.d2h_bytes, "ms_per_step": ms_e2e / args.steps},
            "gpu_launches": int(launches),
            "clocks": clocks,
            "roofline": {"bound": "hbm", "kernel": dominant, "achieved": achieved, "peak": peak,
                         "unit": "GB/s", "frac": (achieved / peak) if achieved else None,
                         "traffic": _ncu_traffic(dominant, args.config), "peak_source": f"MEASURED_PEAKS.json hbm_gbs ({peak_src})",
                         "kernel_ms": dom_avg, "kernel_ms_how": dom_how,
                         "algorithmic_bytes": ab.get(dominant),
                         "fused_call_ms": ms_fused,
                         "fused_call_gbs": ab["trace_fused"] / (ms_fused * 1e-3) / 1e9,
                         "fused_call_frac": ab["trace_fused"] / (ms_fused * 1e-3) / 1e9 / peak,
                         "kernel_ms_warmup_share": {t: round(v / max(sum(tot.values()), 1e-9), 4)
                                                    for t, v in tot.items() if v > 0}},
        }
        out["next"] = {"coact_placement": {
            "us_per_call": us_place, "layers": L, "greedy_steps_per_layer": (E - D) + (D - cfg.N),
            "what": "cap_coact_placement (P:L106-144, L148, L162-164) on the step's counts / coact; latency-bound "
                    "sequential greedy, one CTA per layer; not part of `value`"},
            "pairwise_objective": {"us_per_call": us_obj, "candidates": P, "what": "cap_pairwise_objective (Eq. 2-3) "
                                   "on the step's counts / coact and its P candidate maps"},
            "dispatch_rows": {"us_per_call": us_rows, "what": "cap_dispatch_rows (P:L58, Fig. 2) for layer 0 under "
                              "candidate 0 with the step's pruning mask; three direct launches through the binding, "
                              "output tensors allocated per call"}}
        if not args.no_cpu_baseline:
            out["cpu_baseline"] = time_oracle(cfg, W, args.cpu_seconds)
        print(json.dumps(out))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="cap", choices=["cap", "reference"])
    ap.add_argument("--config", default="target")
    ap.add_argument("--cpu-seconds", type=float, default=10.0)
    ap.add_argument("--ref-tokens", type=int, default=16384)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    from paper_2607_05116_b200 import workload as W
    cfg = W.CONFIGS[args.config]
    if args.impl == "reference":
        run_reference(args, cfg, W)
    else:
        run_cap(args, cfg, W)


if __name__ == "__main__":
    main()

"""Pins of the oracle's NEXT-1 function: Jaccard co-activation probabilities
(reading R3) and Algorithm 1 in both stages.  Each pin is
something other than the oracle itself: hand values, closed-form special cases, exact recovery of
planted structure, an exact-rational replay of the listing, and the paper's claim that the
placement lowers devices per token."""
from fractions import Fraction

import numpy as np
import pytest

from paper_2607_05116_b200 import workload as W


def planted(E, D, N, rng, strong=40, weak=3):
    """Counts / co-activation with planted device clusters (size E/D) grouped into planted nodes.
    One "hub" expert per cluster co-activates more strongly with its cluster mates and one hub
    cluster per node co-activates (weakly) across nodes, so that the top-D weighted degrees are
    one expert per cluster and the top-N group strengths one cluster per node: Algorithm 1 seeds
    with the largest degrees, and two seeds inside one cluster could not recover it.
    Returns (counts, C, cluster_of_expert, node_of_cluster)."""
    perm = rng.permutation(E)
    cl = np.empty(E, np.int64)
    cl[perm] = np.arange(E) // (E // D)
    cperm = rng.permutation(D)
    nd = np.empty(D, np.int64)
    nd[cperm] = np.arange(D) // (D // N)
    hub_e = {int(perm[c * (E // D)]) for c in range(D)}
    hub_c = {int(cperm[m * (D // N)]) for m in range(N)}
    Cm = np.zeros((E, E), np.int64)
    for i in range(E):
        for j in range(E):
            if i == j:
                continue
            if cl[i] == cl[j]:
                Cm[i, j] = strong + (20 if (i in hub_e or j in hub_e) else 0)
            elif nd[cl[i]] == nd[cl[j]]:
                Cm[i, j] = weak
            else:
                Cm[i, j] = 1 if (int(cl[i]) in hub_c or int(cl[j]) in hub_c) else 0
    n = Cm.sum(1) + 5
    Cm[np.arange(E), np.arange(E)] = n
    return n[None].astype(np.int64), Cm[None].astype(np.int32), cl, nd


def same_partition(a, b):
    m = {}
    for x, y in zip(a.tolist(), b.tolist()):
        if m.setdefault(x, y) != y:
            return False
    return len(set(m.values())) == len(m)


def test_jaccard_worked_example(oracle, golden):
    """SURVEY 8(c) worked example: counts [3,2,2,1,2,1,1,0]; p_01 = 1/(3+2-1), p_04 = 2/(3+2-2),
    p_07 = 0 (expert 7 never selected), p symmetric with zero diagonal."""
    idx = np.array(golden["worked_example"]["idx"], np.int32)[None]
    cnt, C = oracle.coactivation(idx, E=8)
    *_, p = oracle.coact_placement(cnt, C, D=4, N=2, want_p=True)
    p = p[0]
    assert p[0, 1] == 0.25 and p[0, 4] == 2.0 / 3.0 and p[0, 7] == 0.0 and p[7, 7] == 0.0
    assert p[1, 6] == 1.0 / 2.0                      # C=1, n=2,1 -> 1/(2+1-1)
    np.testing.assert_array_equal(p, p.T)
    assert np.all(np.diag(p) == 0.0) and np.all((p >= 0) & (p <= 1))


def test_jaccard_zero_denominator(oracle):
    cnt = np.zeros((1, 4), np.int64)
    C = np.zeros((1, 4, 4), np.int32)
    g, gn, ed, p = oracle.coact_placement(cnt, C, D=2, N=1, want_p=True)
    assert np.all(p == 0.0)
    # all scores are 0 -> every growth step takes the random branch; with rnd = None (zeros) the
    # lowest unassigned expert joins: seeds 0,1 then 2 -> g0, 3 -> g1
    assert g.tolist() == [[0, 1, 0, 1]] and gn.tolist() == [[0, 0]] and ed.tolist() == [[0, 1, 0, 1]]


def test_random_branch_uses_supplied_numbers(oracle):
    """Zero matrix, E=6, D=2: seeds 0,1; U = {2,3,4,5}.  rnd = [3, 1, 6, 9]: step 0 picks the
    3 mod 4 = 3rd of {2,3,4,5} = 5 -> g0; step 1: 1 mod 3 -> {2,3,4}[1] = 3 -> g1; step 2:
    6 mod 2 = 0 -> 2 -> g0; step 3: 9 mod 1 = 0 -> 4 -> g1."""
    cnt = np.zeros((1, 6), np.int64)
    C = np.zeros((1, 6, 6), np.int32)
    rnd = np.array([[3, 1, 6, 9, 0, 0, 0, 0]], np.uint32)
    g, _, _, _ = oracle.coact_placement(cnt, C, D=2, N=1, rnd=rnd)
    assert g.tolist() == [[0, 1, 0, 1, 1, 0]]


def test_k_equals_one_and_k_equals_n(oracle):
    rng = np.random.default_rng(3)
    n, C, _, _ = planted(12, 4, 2, rng)
    g, gn, ed, p = oracle.coact_placement(n, C, D=1, N=1, want_p=True)
    assert np.all(g == 0) and np.all(ed == 0)
    # D = E: every expert is a seed; group index = rank by weighted degree (desc, ties -> lower)
    A = rng.integers(0, 30, (12, 12))
    A = np.triu(A, 1)
    A = A + A.T
    nn = A.sum(1) + 1
    A[np.arange(12), np.arange(12)] = nn
    g, gn, ed, p = oracle.coact_placement(nn[None].astype(np.int64), A[None].astype(np.int32),
                                          D=12, N=1, want_p=True)
    deg = np.array([sum(p[0, i, j] for j in range(12) if j != i) for i in range(12)])
    order = sorted(range(12), key=lambda i: (-deg[i], i))
    assert [int(g[0, e]) for e in order] == list(range(12))


@pytest.mark.parametrize("E,D,N", [(16, 4, 2), (64, 8, 2), (128, 16, 4)])
def test_planted_clusters_and_nodes_recovered(oracle, E, D, N):
    """Block structure: co-activation >= 40 inside a cluster, 3 between clusters of one node,
    <= 1 across nodes, seeds forced into distinct clusters / nodes by the hubs.  The greedy step
    of a group then always sees its own cluster mates with the largest score, so stage 1 returns
    the clusters and stage 2 the nodes."""
    rng = np.random.default_rng(E)
    n, C, cl, nd = planted(E, D, N, rng)
    g, gn, ed, _ = oracle.coact_placement(n, C, D=D, N=N)
    assert same_partition(g[0], cl)
    assert np.bincount(g[0], minlength=D).tolist() == [E // D] * D
    assert same_partition(gn[0][g[0]], nd[cl])
    # final placement: a permutation-balanced map on the regular topology
    assert np.bincount(ed[0], minlength=D).tolist() == [E // D] * D
    np.testing.assert_array_equal(ed[0] // (D // N), gn[0][g[0]])
    assert same_partition(ed[0], g[0])


def alg1_exact(P, k, rnd):
    """Algorithm 1 replayed in exact rational arithmetic."""
    n = len(P)
    deg = [sum(P[i][j] for j in range(n) if j != i) for i in range(n)]
    pi = sorted(range(n), key=lambda i: (-deg[i], i))
    G = [[pi[g]] for g in range(k)]
    U = sorted(set(range(n)) - set(pi[:k]))
    g, step = 0, 0
    while U:
        sc = {e: sum(P[e][v] for v in G[g]) for e in U}
        best = max(U, key=lambda e: (sc[e], -e))
        if sc[best] == 0:
            best = U[int(rnd[step]) % len(U)]
        G[g].append(best)
        U.remove(best)
        g = (g + 1) % k
        step += 1
    return G


@pytest.mark.parametrize("seed", range(6))
def test_algorithm1_vs_exact_rational_replay(oracle, seed):
    """Tiny random traces: the fp64 oracle takes the same decisions as the listing evaluated with
    fractions.Fraction (random integer matrices have no rational near-ties at 1e-16)."""
    rng = np.random.default_rng(100 + seed)
    E, D, N, k, T = 12, 4, 2, 3, 40 + 10 * seed
    idx = np.stack([rng.choice(E - 2, k, replace=False) for _ in range(T)]).astype(np.int32)[None]
    cnt, C = oracle.coactivation(idx, E=E)          # experts E-2, E-1 never selected -> zero rows
    rnd = rng.integers(0, 2**32, (1, E + D), dtype=np.uint64).astype(np.uint32)
    g, gn, ed, p = oracle.coact_placement(cnt, C, D=D, N=N, rnd=rnd, want_p=True)
    n = cnt[0].tolist()
    Cm = C[0].tolist()
    P = [[Fraction(0) if (i == j or n[i] + n[j] - Cm[i][j] == 0)
          else Fraction(Cm[i][j], n[i] + n[j] - Cm[i][j]) for j in range(E)] for i in range(E)]
    np.testing.assert_allclose(p[0], np.array([[float(x) for x in r] for r in P]), rtol=0, atol=1e-16)
    G = alg1_exact(P, D, rnd[0, :E])
    for a, members in enumerate(G):
        assert all(g[0, e] == a for e in members)
    Wm = [[sum(P[i][j] for i in sorted(G[a]) for j in sorted(G[b])) if a != b else Fraction(0)
           for b in range(D)] for a in range(D)]
    G2 = alg1_exact(Wm, N, rnd[0, E:])
    for nd, members in enumerate(G2):
        for r, a in enumerate(members):
            assert gn[0, a] == nd
            assert all(ed[0, e] == nd * (D // N) + r for e in G[a])


def test_placement_lowers_devices_per_token(oracle, golden):
    """P:L162, Table III: grouping co-activated experts lowers the devices each token visits
    (paper: 5.33-5.35 -> 4.14-4.49 at E=128, k=8, D=8).  On the Qwen3-shaped synthetic trace the
    Algorithm 1 placement must beat the sequential one clearly and stay balanced in size."""
    cfg = W.CONFIGS["qwen3"].with_(T=16384)
    x = W.logits(cfg, 0)[None]
    idx, _ = oracle.gate_topk(x, k=cfg.k)
    cnt, C = oracle.coactivation(idx, E=cfg.E)
    g, gn, ed, _ = oracle.coact_placement(cnt, C, D=cfg.D, N=cfg.N)
    seq = (np.arange(cfg.E) // (cfg.E // cfg.D)).astype(np.int32)
    ev = oracle.eval_placements(idx, np.stack([seq, ed[0]])[None], W.dev_node(cfg))
    dpt = ev.dev_visits[0] / cfg.T
    assert np.bincount(ed[0], minlength=cfg.D).tolist() == [cfg.E // cfg.D] * cfg.D
    lo, hi = golden["paper_table3_default"]["cap_devices_per_token_range"]
    assert dpt[1] < dpt[0] - 0.4 and lo - 0.6 < dpt[1] < hi + 0.6


def test_placement_einval(oracle):
    cnt = np.zeros((1, 6), np.int64)
    C = np.zeros((1, 6, 6), np.int32)
    with pytest.raises(ValueError):
        oracle.coact_placement(cnt, C, D=4, N=1)      # E % D != 0
    with pytest.raises(ValueError):
        oracle.coact_placement(cnt, C, D=3, N=2)      # D % N != 0


# ------------------------------------------------------------------ NEXT-3: pairwise objective, Eq. 2-3
def test_objective_worked_example_by_hand(oracle, golden):
    """Worked example, Eq. 2-3 with costs 1 / 4, summed by hand over the ten co-activated
    pairs: pi_A: (0,2) 2*1 + (0,4) 2*4 + (0,5) 4 + (1,2) 1 + (1,3) 1 + (1,6) 4 + (2,4) 4 + (3,6) 4 = 28;
    pi_B: 1 + 8 + 0 + 1 + 4 + 4 + 4 + 4 + 1 + 1 = 28.  Probabilities (Jaccard) under pi_A:
    2/3 + 4*2/3 + 4/3 + 1/3 + 1/2 + 4/2 + 4/3 + 4*1 = 19/3 + 6.5."""
    g = golden["worked_example"]
    cnt = np.array(g["counts"], np.int64)[None]
    C = np.array(g["coact"], np.int32)[None]
    maps = np.array([g["pi_A"], g["pi_B"]], np.int32)[None]
    oc, op, cb = oracle.pairwise_objective(cnt, C, maps, np.array(g["dev_node"], np.int32), cost_intra=1,
                                           cost_inter=4, lam=0.25,
                                           imbalance=np.array([[g["eval_A"]["imbalance"], 2.0]]))
    assert oc.tolist() == [[28, 28]]
    assert abs(op[0, 0] - (19.0 / 3.0 + 6.5)) < 1e-14
    assert abs(cb[0, 0] - (0.25 * (19.0 / 3.0 + 6.5) + 0.75 * 5.0 / 3.0)) < 1e-14      # Eq. 5


def test_objective_closed_forms_and_brute_force(oracle):
    rng = np.random.default_rng(11)
    E, k, T, D = 24, 4, 300, 6
    idx = np.stack([rng.choice(E, k, replace=False) for _ in range(T)]).astype(np.int32)[None]
    cnt, C = oracle.coactivation(idx, E=E)
    dn = np.array([0, 0, 0, 1, 1, 1], np.int32)
    one_dev = np.zeros(E, np.int32)
    ident = np.arange(E, dtype=np.int32)
    rnd = rng.integers(0, D, E).astype(np.int32)
    # all experts on one device: nothing is cut
    oc, op, _ = oracle.pairwise_objective(cnt, C, np.stack([one_dev, rnd])[None], dn, cost_intra=1, cost_inter=5)
    assert oc[0, 0] == 0 and op[0, 0] == 0.0
    # brute force over pairs for the random map
    n, Cm = cnt[0], C[0].astype(np.int64)
    want_c, want_p = 0, 0.0
    for i in range(E):
        for j in range(i + 1, E):
            d = 0 if rnd[i] == rnd[j] else (1 if dn[rnd[i]] == dn[rnd[j]] else 5)
            want_c += int(Cm[i, j]) * d
            den = n[i] + n[j] - Cm[i, j]
            want_p += (Cm[i, j] / den if den else 0.0) * d
    assert oc[0, 1] == want_c and abs(op[0, 1] - want_p) <= 1e-12 * want_p
    # one expert per device, one node, cost 1: every co-activated pair is cut once:
    # sum_{i<j} C_ij = sum_i (k-1) n_i / 2 = T k (k-1) / 2   (S2's row-sum invariant)
    oc, _, _ = oracle.pairwise_objective(cnt, C, ident[None, None], np.zeros(E, np.int32))
    assert oc[0, 0] == T * k * (k - 1) // 2


def test_objective_prefers_cluster_aligned_placement(oracle):
    """Eq. 2 is the proxy the placement minimises: on the clustered trace the planted cluster-aligned
    candidate (workload candidate 2) and Algorithm 1's placement score below the sequential map."""
    cfg = W.CONFIGS["target"].with_(T=8192)
    idx, _ = oracle.gate_topk(W.logits(cfg, 0)[None], k=cfg.k)
    cnt, C = oracle.coactivation(idx, E=cfg.E)
    cand = W.candidates(cfg, 0)[:3]
    _, _, ed, _ = oracle.coact_placement(cnt, C, D=cfg.D, N=cfg.N)
    maps = np.concatenate([cand, ed])[None]
    oc, op, _ = oracle.pairwise_objective(cnt, C, maps, W.dev_node(cfg), cost_intra=1, cost_inter=cfg.cost_inter)
    assert oc[0, 2] < oc[0, 0] and op[0, 2] < op[0, 0]
    assert oc[0, 3] < oc[0, 0] and op[0, 3] < op[0, 0]


# ------------------------------------------------------------------ NEXT-4: device-centric dispatch rows
def test_dispatch_rows_worked_example_by_hand(oracle, golden):
    """Worked example under pi_A (e // 2), by hand from Fig. 2's rule (one copy per device):
    d0 <- t0,t1,t2,t3; d1 <- t0 (expert 2), t2 (expert 3), t3 (expert 2); d2 <- t1 (4,5), t3 (4);
    d3 <- t2 (6).  Row counts = recv_tokens [4,3,2,1] of the S3 golden values."""
    g = golden["worked_example"]
    idx = np.array(g["idx"], np.int32)
    rows, off, pr = oracle.dispatch_rows(idx, np.array(g["pi_A"], np.int32), 4)
    assert rows.tolist() == [0, 1, 2, 3, 0, 2, 3, 1, 3, 2]
    assert off.tolist() == [0, 4, 7, 9, 10]
    assert pr.tolist() == [0, 4, 0, 7, 7, 1, 2, 9, 5, 3, 6, 8]
    assert np.diff(off).tolist() == g["eval_A"]["recv_tokens"]
    kept = np.array(g["prune_A_p025"]["kept"], np.uint8)
    rows, off, pr = oracle.dispatch_rows(idx, np.array(g["pi_A"], np.int32), 4, kept=kept)
    # kept = [[1,0,1],[1,1,0],[1,1,0],[1,0,1]]: t0 -> d0; t1 -> d2; t2 -> d0, d3; t3 -> d0, d2
    assert rows.tolist() == [0, 2, 3, 1, 3, 2] and off.tolist() == [0, 3, 3, 5, 6]
    assert pr.tolist() == [0, -1, 0, 3, 3, -1, 1, 5, -1, 2, -1, 4]


def test_dispatch_rows_vs_python_sets_and_s3(oracle):
    rng = np.random.default_rng(21)
    T, E, k, D = 500, 40, 6, 8
    idx = np.stack([rng.choice(E, k, replace=False) for _ in range(T)]).astype(np.int32)
    kept = (rng.random((T, k)) < 0.7).astype(np.uint8)
    pi = rng.integers(0, D, E).astype(np.int32)
    for m in (None, kept):
        rows, off, pr = oracle.dispatch_rows(idx, pi, D, kept=m)
        want = sorted({(int(pi[idx[t, s]]), t) for t in range(T) for s in range(k) if m is None or m[t, s]})
        got = [(d, int(t)) for d in range(D) for t in rows[off[d]:off[d + 1]]]
        assert got == want
        ev = oracle.eval_placements(idx[None], pi[None, None], np.zeros(D, np.int32), kept=None if m is None else m[None])
        assert np.diff(off).tolist() == ev.recv_tokens[0, 0].tolist() and off[D] == ev.dev_visits[0, 0]
        for t in range(T):
            for s in range(k):
                i = t * k + s
                if m is not None and not m[t, s]:
                    assert pr[i] == -1
                else:
                    d = pi[idx[t, s]]
                    assert off[d] <= pr[i] < off[d + 1] and rows[pr[i]] == t
    rows, off, pr = oracle.dispatch_rows(idx[:0], pi, D)
    assert rows.size == 0 and off.tolist() == [0] * (D + 1)


# ------------------------------------------------------------------ NEXT-2: adjustment spectrum (R27)
def _sym(E, pairs):
    Cm = np.zeros((E, E), np.int32)
    for (i, j), v in pairs.items():
        Cm[i, j] = Cm[j, i] = v
    return Cm


def test_adjust_hand_example(oracle):
    """E=6, D=2, pi0 = [0,0,0,1,1,1], n = [9,5,4,1,2,3] (loads 18 / 6).  By hand (R27):
    step 1: all nine pairs are candidates; losses: (2,3) = 2+2-0-0 = 4 is the smallest -> swap 2,3
            (loads 15 / 9);
    step 2: candidates (0,2) d=5, (1,2) d=1, (1,4) d=3, (1,5) d=2; losses 3, 3, 8, 8 -> tie -> (0,2)
            (loads 10 / 14);
    step 3: hot = 1; candidates (4,3) d=1, (5,3) d=2; losses 5, 5 -> (4,3) (loads 11 / 13);
    step 4: hot = 1 {0,3,5}, cold = 0 {1,2,4}, gap 2: only (5,4) has 0 < d=1 < 2 -> swap (loads 12 / 12);
    step 5: equal loads -> stop."""
    n = np.array([[9, 5, 4, 1, 2, 3]], np.int64)
    Cm = _sym(6, {(0, 1): 6, (0, 2): 1, (1, 2): 1, (3, 4): 1, (3, 5): 1, (4, 5): 4, (2, 3): 2})[None]
    spec, done, sw = oracle.adjust_spectrum(n, Cm, np.array([[0, 0, 0, 1, 1, 1]], np.int32), D=2, S=6)
    assert sw[0, :5].tolist() == [[2, 3], [0, 2], [4, 3], [5, 4], [-1, -1]]
    assert spec[0, 0].tolist() == [0, 0, 1, 0, 1, 1]
    assert spec[0, 1].tolist() == [1, 0, 0, 0, 1, 1]
    assert spec[0, 2].tolist() == [1, 0, 0, 1, 0, 1]
    assert spec[0, 3].tolist() == [1, 0, 0, 1, 1, 0]
    assert spec[0, 4].tolist() == spec[0, 3].tolist() == spec[0, 5].tolist() and done[0] == 4


def test_adjust_properties_and_python_replay(oracle):
    """Random traces: every step swaps one expert of the then-hottest device with one of the
    then-coldest, device sizes never change, the maximum load never rises, and a set-based Python
    replay of R27 takes the same decisions."""
    rng = np.random.default_rng(9)
    E, k, T, D, S = 24, 4, 400, 4, 12
    idx = np.stack([rng.choice(E, k, replace=False, p=np.arange(1, E + 1) / (E * (E + 1) / 2))
                    for _ in range(T)]).astype(np.int32)[None]
    cnt, C = oracle.coactivation(idx, E=E)
    pi0 = (np.arange(E) // (E // D)).astype(np.int32)
    spec, done, sw = oracle.adjust_spectrum(cnt, C, pi0[None], D=D, S=S)
    n, Cm = cnt[0], C[0].astype(np.int64)
    pi = pi0.copy()
    prev_max = max(n[pi == d].sum() for d in range(D))
    assert done[0] >= 2
    for s in range(S):
        load = [int(n[pi == d].sum()) for d in range(D)]
        hot = max(range(D), key=lambda d: (load[d], -d))
        cold = min(range(D), key=lambda d: (load[d], d))
        best = None
        for a in np.flatnonzero(pi == hot):
            for b in np.flatnonzero(pi == cold):
                dl = int(n[a] - n[b])
                if hot == cold or not (0 < dl < load[hot] - load[cold]):
                    continue
                H = [v for v in np.flatnonzero(pi == hot) if v != a]
                Cd = [v for v in np.flatnonzero(pi == cold) if v != b]
                loss = int(Cm[a, H].sum() + Cm[b, Cd].sum() - Cm[a, Cd].sum() - Cm[b, H].sum())
                if best is None or loss < best[0]:
                    best = (loss, int(a), int(b))
        if best is None:
            assert done[0] == s and sw[0, s].tolist() == [-1, -1]
            break
        assert sw[0, s].tolist() == [best[1], best[2]]
        pi[best[1]], pi[best[2]] = cold, hot
        assert spec[0, s].tolist() == pi.tolist()
        assert np.bincount(pi, minlength=D).tolist() == [E // D] * D
        new_max = max(n[pi == d].sum() for d in range(D))
        assert new_max <= prev_max
        prev_max = new_max


def test_adjust_trades_communication_for_balance(oracle):
    """from the Algorithm 1 placement the spectrum moves toward lower imbalance at the
    cost of more devices per token."""
    cfg = W.CONFIGS["qwen3"].with_(T=8192)
    idx, _ = oracle.gate_topk(W.logits(cfg, 0)[None], k=cfg.k)
    cnt, C = oracle.coactivation(idx, E=cfg.E)
    _, _, ed, _ = oracle.coact_placement(cnt, C, D=cfg.D, N=cfg.N)
    spec, done, _ = oracle.adjust_spectrum(cnt, C, ed, D=cfg.D, S=6)
    maps = np.concatenate([ed[:, None], spec], 1)
    ev = oracle.eval_placements(idx, maps, W.dev_node(cfg))
    assert done[0] == 6
    assert np.all(np.diff(ev.imbalance[0]) <= 1e-12) and ev.imbalance[0, -1] < ev.imbalance[0, 0] - 0.02
    assert ev.dev_visits[0, -1] >= ev.dev_visits[0, 0]


# ------------------------------------------------------------------ NEXT-4b naive expert-level pruning
def test_prune_naive_hand_example(oracle):
    # one token, weights 0.4 0.3 0.2 0.1 (experts 7 3 9 1): target 1 - p
    idx = np.array([[[7, 3, 9, 1]]], np.int32)
    w = np.array([[[0.4, 0.3, 0.2, 0.1]]], np.float32)
    for p, want in ((0.0, [1, 1, 1, 1]), (0.05, [1, 1, 1, 1]), (0.1, [1, 1, 1, 0]), (0.25, [1, 1, 1, 0]),
                    (0.3, [1, 1, 0, 0]), (0.35, [1, 1, 0, 0]), (0.6, [1, 0, 0, 0]), (0.9, [1, 0, 0, 0])):
        # p = 0.1: 0.4 + 0.3 + 0.2 = 0.9 >= 0.9 only in exact arithmetic; fp32: 0.4f + 0.3f + 0.2f vs 1 - 0.1f
        kept, near = oracle.prune_naive(idx, w, p)
        cum, k_ref, target = np.float32(0), [0, 0, 0, 0], np.float32(1) - np.float32(p)
        if p > 0:
            for s in range(4):
                if cum >= target:
                    break
                k_ref[s] = 1
                cum = np.float32(cum + w[0, 0, s])
        else:
            k_ref = [1, 1, 1, 1]
        assert kept[0, 0].tolist() == k_ref, p
        if p not in (0.1, 0.3, 0.6):          # away from the exact boundaries the hand values hold
            assert kept[0, 0].tolist() == want, p
    # unsorted slots (sigmoid + bias gating orders slots by the biased score): descending weight, ties -> lower expert
    idx = np.array([[[5, 2, 8, 4]]], np.int32)
    w = np.array([[[0.25, 0.25, 0.4, 0.1]]], np.float32)
    kept, _ = oracle.prune_naive(idx, w, 0.5)         # 0.4 (e8), then the tie 0.25: expert 2 before expert 5
    assert kept[0, 0].tolist() == [0, 1, 1, 0]
    kept, _ = oracle.prune_naive(idx, w, 0.3)         # 0.4 + 0.25 (e2) = 0.65 < 0.7 -> expert 5 too
    assert kept[0, 0].tolist() == [1, 1, 1, 0]


def test_prune_naive_is_the_uniform_cost_identity_placement_case_of_prune(oracle):
    """P:L62 vs P:L212: with one expert per device and c_d = 1 for every device Eq. 6's greedy is the naive rule
    (capo_prune's special case is itself pinned by 2^k brute force in test_oracle_pins.py)."""
    rng = np.random.default_rng(62)
    L, T, E, k = 2, 400, 64, 6
    idx = np.stack([np.stack([rng.permutation(E)[:k] for _ in range(T)]) for _ in range(L)]).astype(np.int32)
    w = rng.random((L, T, k)).astype(np.float32) + np.float32(0.01)
    w[0, :40] = np.float32(1.0 / k)                                   # exact ties
    w = (w / w.sum(-1, keepdims=True, dtype=np.float32)).astype(np.float32)
    pi = np.tile(np.arange(E, dtype=np.int32), (L, 1))
    dn = np.zeros(E, np.int32)
    for p in (0.0, 0.05, 0.2, 0.5, 0.9):
        kept_n, near_n = oracle.prune_naive(idx, w, p)
        kept_r, near_r = oracle.prune(idx, w, pi, dn, p, cost_local=1, cost_intra=1, cost_inter=1)
        assert np.array_equal(kept_n, kept_r), p
        assert np.array_equal(near_n, near_r), p


def test_prune_naive_minimal_cardinality_brute_force(oracle):
    """The kept set reaches the target with the fewest experts possible (2^k subsets), and dropping its smallest
    member falls below the target."""
    rng = np.random.default_rng(295)
    T, k = 120, 8
    idx = np.stack([rng.permutation(500)[:k] for _ in range(T)]).astype(np.int32)[None]
    w = rng.random((1, T, k)).astype(np.float32) ** 2 + np.float32(0.01)
    w = (w / w.sum(-1, keepdims=True, dtype=np.float32)).astype(np.float32)
    for p in (0.1, 0.3, 0.6):
        kept, _ = oracle.prune_naive(idx, w, p)
        target = float(np.float32(1) - np.float32(p))
        for t in range(T):
            ws = w[0, t].astype(np.float64)
            nk = int(kept[0, t].sum())
            assert ws[kept[0, t] == 1].sum() >= target - 1e-6
            best = min(bin(m).count("1") for m in range(1, 1 << k)
                       if sum(ws[s] for s in range(k) if m >> s & 1) >= target - 1e-6)
            assert nk == best or abs(ws[kept[0, t] == 1].sum() - ws[kept[0, t] == 1].min() - target) < 1e-5, (t, nk, best)
            assert nk <= best + 1
            assert ws[kept[0, t] == 1].min() >= ws[kept[0, t] == 0].max() - 1e-12 if nk < k else True


# ------------------------------------------------------------------ NEXT-4c combine weights of the dispatch rows
def test_dispatch_row_weights_hand_and_python_replay(oracle, golden):
    # hand case: 2 tokens, k = 3, devices of the slots: t0 -> (1, 0, 1), t1 -> (0, 0, pruned)
    idx = np.array([[0, 1, 2], [3, 4, 5]], np.int32)
    pi = np.array([1, 0, 1, 0, 0, 1], np.int32)
    kept = np.array([[1, 1, 1], [1, 1, 0]], np.uint8)
    w = np.array([[0.5, 0.3, 0.2], [0.6, 0.3, 0.1]], np.float32)
    rows, off, prow = oracle.dispatch_rows(idx, pi, 2, kept=kept)
    assert rows.tolist() == [0, 1, 0] and off.tolist() == [0, 2, 3]       # device 0: t0, t1; device 1: t0
    assert prow.tolist() == [2, 0, 2, 1, 1, -1]
    rw = oracle.dispatch_row_weights(w, prow, 3)
    assert rw.tolist() == [np.float32(0.3), np.float32(np.float32(0.6) + np.float32(0.3)),
                           np.float32(np.float32(0.5) + np.float32(0.2))]
    # random traces: sequential fp32 sums per (token, device) in slot order, written independently in Python
    rng = np.random.default_rng(58)
    T, k, E, D = 300, 8, 64, 16
    idx = np.stack([rng.permutation(E)[:k] for _ in range(T)]).astype(np.int32)
    pi = (rng.permutation(E) % D).astype(np.int32)
    kept = (rng.random((T, k)) < 0.7).astype(np.uint8)
    w = rng.random((T, k)).astype(np.float32)
    rows, off, prow = oracle.dispatch_rows(idx, pi, D, kept=kept)
    rw = oracle.dispatch_row_weights(w, prow, int(off[-1]))
    for d in range(D):
        for r in range(int(off[d]), int(off[d + 1])):
            t = int(rows[r])
            acc = np.float32(0)
            for s in range(k):
                if kept[t, s] and pi[idx[t, s]] == d:
                    acc = np.float32(acc + w[t, s])
            assert rw[r] == acc, (d, r)
    # the rows' weights add up to the kept routing mass of every token (nothing is lost by aggregating)
    tot = np.zeros(T, np.float64)
    np.add.at(tot, rows, rw.astype(np.float64))
    assert np.allclose(tot, (w * kept).sum(-1, dtype=np.float64), atol=1e-5)

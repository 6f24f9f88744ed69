/*
 * cap_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, single-threaded CPU restatement of the five stages of CAP's
 * per-token routing-trace pipeline (arXiv 2607.05116, "Communication-Aware
 * Placement and Pruning for Efficient Mixture-of-Experts Inference"), written
 * from the paper (P:Lnnn = /root/reference/PAPER.md line nnn) and from the
 * readings listed in DESIGN.md section 3 (R1..R27).  It shares no code, header,
 * table or helper with the CUDA path under paper_2607_05116_b200/csrc/ and
 * neither imports the other.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may call it.
 *
 * Build: gcc -O2 -std=c11 -ffp-contract=off -fPIC -shared (see oracle/build.py).
 * -ffp-contract=off matters: every fp32 step below is one IEEE operation, the
 * only fused operations are the explicit fmaf() calls in expS.
 *
 * Pins (tests/test_oracle_pins.py, tests/test_oracle_placement_pins.py): every
 * function here is pinned by something other than itself -- closed forms,
 * brute force, library routines, hand-worked examples, the paper's Table III
 * "Default" value.  PARITY UNPINNED: capo_adjust_spectrum only -- P:L194 states
 * the goal of an adjustment step but no selection rule, so the rule is reading
 * R27 of DESIGN.md; it is pinned against R27's own hand example and properties,
 * not against the paper.  The one other reading that cannot be pinned against
 * the paper (which load definition Table IV uses, R6) is handled by exporting
 * both quantities.
 *
 * Functions: the five stages S1..S5 (capo_gate_topk, capo_coactivation,
 * capo_eval_placements, capo_prune, capo_dispatch_layout) and the consumers of
 * S2 in SURVEY.md 8(f): capo_coact_placement (p_ij + Algorithm 1),
 * capo_adjust_spectrum, capo_pairwise_objective (Eq. 2-3, Eq. 5),
 * capo_dispatch_rows (Fig. 2's one copy per device), capo_dispatch_row_weights
 * (the combine weight a_d of each row) and capo_prune_naive (the naive
 * expert-level baseline of P:L62 / Fig. 14).
 *
 * All arrays are HOST pointers, row-major, layouts as in include/cap.h.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define CAPO_OK 0
#define CAPO_EINVAL (-1)

/* ------------------------------------------------------------------------- *
 * expS / sigS: the reproducible fp32 exponential of DESIGN.md R-S1.3.
 * Only IEEE-exact fp32 operations (mul, add, fma, round-to-nearest-even,
 * divide), so that any conforming implementation returns identical bits.
 * Accuracy (pinned against libm exp in double in the tests): < 1 ulp.
 * ------------------------------------------------------------------------- */
static float capo_expS(float x)
{
    float t = x;
    if (t < -87.0f) t = -87.0f;
    if (t > 87.0f) t = 87.0f;
    float n = nearbyintf(t * 0x1.715476p+0f);      /* round-half-even of t*log2(e) */
    float r = fmaf(n, -0x1.62ep-1f, t);            /* Cody-Waite, ln2 high part    */
    r = fmaf(n, -0x1.0bfbe8p-15f, r);              /* ln2 low part                 */
    float p = 0x1.a01a02p-13f;                     /* 1/5040 */
    p = fmaf(p, r, 0x1.6c16c2p-10f);               /* 1/720  */
    p = fmaf(p, r, 0x1.111112p-7f);                /* 1/120  */
    p = fmaf(p, r, 0x1.555556p-5f);                /* 1/24   */
    p = fmaf(p, r, 0x1.555556p-3f);                /* 1/6    */
    p = fmaf(p, r, 0x1p-1f);                       /* 1/2    */
    p = fmaf(p, r, 1.0f);
    p = fmaf(p, r, 1.0f);
    /* exact scaling by 2^n, n in [-126,126] after the clamp */
    union { uint32_t u; float f; } s;
    s.u = (uint32_t)((int32_t)n + 127) << 23;
    return p * s.f;
}

static float capo_sigS(float x)
{
    return 1.0f / (1.0f + capo_expS(-x));
}

float capo_exp_s(float x) { return capo_expS(x); }
float capo_sig_s(float x) { return capo_sigS(x); }

/* ------------------------------------------------------------------------- *
 * S1  gate top-k.  P:L35-40 (sec. II-A, Eq. 1): "a gating network selects the
 * top-k experts for each token ... Gate_i(x) denotes the normalized routing
 * weight of the i-th selected expert".  Scoring function, tie rule, group-
 * limited routing: BASELINE.json north_star/configs, R1,R2,R14,R21.
 *
 * logits [L][T][E] fp32, bias [L][E] fp32 or NULL (sigmoid only)
 * idx    [L][T][k] int32 (slot 0 = best selection score), w [L][T][k] fp32
 * ------------------------------------------------------------------------- */
int capo_gate_topk(const float *logits, const float *bias, int32_t L, int64_t T,
                   int32_t E, int32_t k, int32_t scoring, int32_t renormalize,
                   int32_t n_group, int32_t topk_group, int32_t group_score,
                   float scale, int32_t *idx, float *w)
{
    if (L < 0 || T < 0 || E < 1 || E > 1024 || k < 1 || k > 16 || k > E) return CAPO_EINVAL;
    if (scoring != 0 && scoring != 1) return CAPO_EINVAL;
    if (scoring == 0 && bias != NULL) return CAPO_EINVAL;
    if (n_group < 1 || E % n_group != 0) return CAPO_EINVAL;
    if (n_group > 1) {
        if (topk_group < 1 || topk_group > n_group) return CAPO_EINVAL;
        if ((int64_t)k > (int64_t)topk_group * (E / n_group)) return CAPO_EINVAL;
        if (group_score != 0 && group_score != 1) return CAPO_EINVAL;
        if (group_score == 1 && E / n_group < 2) return CAPO_EINVAL;
    }
    float *c = (float *)malloc(sizeof(float) * (size_t)E);   /* selection score */
    float *s = (float *)malloc(sizeof(float) * (size_t)E);   /* unbiased sigmoid */
    uint8_t *elig = (uint8_t *)malloc((size_t)E);
    float *gs = (float *)malloc(sizeof(float) * (size_t)n_group);
    uint8_t *gsel = (uint8_t *)malloc((size_t)n_group);
    const int32_t gsz = E / n_group;

    for (int32_t l = 0; l < L; ++l) {
        const float *b = bias ? bias + (size_t)l * E : NULL;
        for (int64_t t = 0; t < T; ++t) {
            const float *x = logits + ((size_t)l * (size_t)T + (size_t)t) * (size_t)E;
            int32_t *oi = idx + ((size_t)l * (size_t)T + (size_t)t) * (size_t)k;
            float *ow = w + ((size_t)l * (size_t)T + (size_t)t) * (size_t)k;
            /* step 1: selection score c_e */
            for (int32_t e = 0; e < E; ++e) {
                if (scoring == 0) {
                    c[e] = x[e];             /* softmax is monotone: raw logit */
                } else {
                    s[e] = capo_sigS(x[e]);
                    c[e] = b ? s[e] + b[e] : s[e];
                }
                elig[e] = 1;
            }
            /* step 3: group-limited pre-selection */
            if (n_group > 1) {
                for (int32_t g = 0; g < n_group; ++g) {
                    const float *cg = c + (size_t)g * gsz;
                    if (group_score == 0) {
                        float m = cg[0];
                        for (int32_t j = 1; j < gsz; ++j) if (cg[j] > m) m = cg[j];
                        gs[g] = m;
                    } else {
                        /* fp32 sum of the two largest c_e of the group */
                        int32_t i1 = 0;
                        for (int32_t j = 1; j < gsz; ++j) if (cg[j] > cg[i1]) i1 = j;
                        int32_t i2 = -1;
                        for (int32_t j = 0; j < gsz; ++j) {
                            if (j == i1) continue;
                            if (i2 < 0 || cg[j] > cg[i2]) i2 = j;
                        }
                        gs[g] = cg[i1] + cg[i2];
                    }
                    gsel[g] = 0;
                }
                for (int32_t r = 0; r < topk_group; ++r) {
                    int32_t best = -1;
                    for (int32_t g = 0; g < n_group; ++g) {
                        if (gsel[g]) continue;
                        if (best < 0 || gs[g] > gs[best]) best = g;   /* ties -> lower g */
                    }
                    gsel[best] = 1;
                }
                for (int32_t e = 0; e < E; ++e) elig[e] = gsel[e / gsz];
            }
            /* step 4: k passes of linear arg-max, ties -> lower expert index */
            for (int32_t r = 0; r < k; ++r) {
                int32_t best = -1;
                for (int32_t e = 0; e < E; ++e) {
                    if (!elig[e]) continue;
                    if (best < 0 || c[e] > c[best]) best = e;
                }
                oi[r] = best;
                elig[best] = 0;
            }
            /* step 5: weights */
            if (scoring == 0) {
                if (renormalize) {
                    float raw[16];
                    for (int32_t r = 0; r < k; ++r) raw[r] = capo_expS(x[oi[r]] - x[oi[0]]);
                    float Z = raw[0];
                    for (int32_t r = 1; r < k; ++r) Z = Z + raw[r];
                    for (int32_t r = 0; r < k; ++r) {
                        float v = raw[r] / Z;
                        ow[r] = (scale == 1.0f) ? v : v * scale;
                    }
                } else {
                    /* full softmax probability of the selected experts
                       (tolerance-only mode, DESIGN.md R-S1.5) */
                    float m = x[0];
                    for (int32_t e = 1; e < E; ++e) if (x[e] > m) m = x[e];
                    double Zall = 0.0;
                    for (int32_t e = 0; e < E; ++e) Zall += (double)capo_expS(x[e] - m);
                    for (int32_t r = 0; r < k; ++r) {
                        float v = (float)((double)capo_expS(x[oi[r]] - m) / Zall);
                        ow[r] = (scale == 1.0f) ? v : v * scale;
                    }
                }
            } else {
                if (renormalize) {
                    float Z = s[oi[0]];
                    for (int32_t r = 1; r < k; ++r) Z = Z + s[oi[r]];
                    for (int32_t r = 0; r < k; ++r) {
                        float v = s[oi[r]] / Z;
                        ow[r] = (scale == 1.0f) ? v : v * scale;
                    }
                } else {
                    for (int32_t r = 0; r < k; ++r)
                        ow[r] = (scale == 1.0f) ? s[oi[r]] : s[oi[r]] * scale;
                }
            }
        }
    }
    free(c); free(s); free(elig); free(gs); free(gsel);
    return CAPO_OK;
}

/* ------------------------------------------------------------------------- *
 * S2  activation counts and co-activation.  P:L104 (sec. IV-A: "we collect
 * pairwise expert co-activation frequencies from inference-time routing
 * traces"), P:L148 ("the number of times they are selected together"),
 * P:L224 (placement runs on the pruned routing data -> optional kept mask).
 * counts[i] = #(token,slot) kept with expert i; C[i][j] = #tokens that keep
 * both i and j (i != j); C[i][i] = counts[i].  Plain triple loop over (t,a,b).
 * ------------------------------------------------------------------------- */
int capo_coactivation(const int32_t *idx, const uint8_t *kept, int32_t L, int64_t T,
                      int32_t k, int32_t E, int64_t *counts, int32_t *coact)
{
    if (L < 0 || T < 0 || E < 1 || k < 1 || k > 16) return CAPO_EINVAL;
    memset(counts, 0, sizeof(int64_t) * (size_t)L * (size_t)E);
    memset(coact, 0, sizeof(int32_t) * (size_t)L * (size_t)E * (size_t)E);
    for (int32_t l = 0; l < L; ++l) {
        int64_t *cnt = counts + (size_t)l * E;
        int32_t *C = coact + (size_t)l * E * E;
        for (int64_t t = 0; t < T; ++t) {
            size_t base = ((size_t)l * (size_t)T + (size_t)t) * (size_t)k;
            for (int32_t a = 0; a < k; ++a) {
                if (kept && !kept[base + a]) continue;
                int32_t i = idx[base + a];
                cnt[i] += 1;
                C[(size_t)i * E + i] += 1;
                for (int32_t b = 0; b < k; ++b) {
                    if (b == a) continue;
                    if (kept && !kept[base + b]) continue;
                    int32_t j = idx[base + b];
                    C[(size_t)i * E + j] += 1;
                }
            }
        }
    }
    return CAPO_OK;
}

/* ------------------------------------------------------------------------- *
 * S3  evaluation of P candidate placements.
 *  - P:L58 (sec. II-C): "each token is sent once to each device that hosts
 *    activated experts" -> per token the SET of devices, not the experts.
 *  - P:L152-158 (Eq. 2-3): cost 0 same device, 1 same node, c across nodes.
 *  - P:L186-188 (Eq. 4): imbalance = max_g L_g / mean_g L_g.
 *  - P:L196 (Fig. 6 x-axis): "average number of devices each token is routed
 *    to"; Table III fixes that this counts ALL devices (R4).
 *  - Table II: "Node per Token".
 * expert_dev [L][P][E], dev_node [D], token_src [L][T] or NULL (= t*D/T).
 * Scalar outputs [L][P]; load_pairs/recv_tokens [L][P][D]; tok_* [L][P][T].
 * Any output pointer may be NULL.
 * ------------------------------------------------------------------------- */
int capo_eval_placements(const int32_t *idx, const uint8_t *kept, const int32_t *token_src,
                         int32_t L, int64_t T, int32_t k, int32_t E,
                         const int32_t *expert_dev, int32_t P,
                         int32_t D, int32_t N, const int32_t *dev_node,
                         int32_t cost_local, int32_t cost_intra, int32_t cost_inter,
                         int64_t bytes_per_token,
                         int64_t *dev_visits, int64_t *remote_dev, int64_t *remote_intra,
                         int64_t *remote_inter, int64_t *node_visits, int64_t *remote_node,
                         int64_t *cost, int64_t *bytes,
                         int64_t *load_pairs, int64_t *recv_tokens,
                         double *imbalance, double *imbalance_recv,
                         uint8_t *tok_remote_dev, uint8_t *tok_remote_node)
{
    if (L < 0 || T < 0 || E < 1 || k < 1 || k > 16 || P < 0 || D < 1 || D > 64 || N < 1 || N > 64)
        return CAPO_EINVAL;
    for (int32_t d = 0; d < D; ++d)
        if (dev_node[d] < 0 || dev_node[d] >= N) return CAPO_EINVAL;
    for (int32_t l = 0; l < L; ++l) {
        for (int32_t p = 0; p < P; ++p) {
            const int32_t *pi = expert_dev + ((size_t)l * P + p) * (size_t)E;
            for (int32_t e = 0; e < E; ++e)
                if (pi[e] < 0 || pi[e] >= D) return CAPO_EINVAL;
            int64_t a_dev = 0, a_rdev = 0, a_intra = 0, a_inter = 0, a_node = 0, a_rnode = 0, a_local = 0;
            int64_t lp[64], rt[64];
            for (int32_t d = 0; d < D; ++d) { lp[d] = 0; rt[d] = 0; }
            for (int64_t t = 0; t < T; ++t) {
                size_t base = ((size_t)l * (size_t)T + (size_t)t) * (size_t)k;
                int32_t src = token_src ? token_src[(size_t)l * (size_t)T + (size_t)t]
                                        : (int32_t)(((int64_t)t * D) / T);
                int32_t srcn = dev_node[src];
                uint8_t indev[64], innode[64];
                memset(indev, 0, sizeof indev);
                memset(innode, 0, sizeof innode);
                for (int32_t sl = 0; sl < k; ++sl) {
                    if (kept && !kept[base + sl]) continue;
                    int32_t d = pi[idx[base + sl]];
                    lp[d] += 1;                       /* every kept pair is load */
                    indev[d] = 1;
                    innode[dev_node[d]] = 1;
                }
                int32_t rd = 0, rn = 0;
                for (int32_t d = 0; d < D; ++d) {
                    if (!indev[d]) continue;
                    a_dev += 1;
                    rt[d] += 1;
                    if (d == src) { a_local += 1; continue; }
                    rd += 1;
                    if (dev_node[d] == srcn) a_intra += 1; else a_inter += 1;
                }
                for (int32_t n = 0; n < N; ++n) {
                    if (!innode[n]) continue;
                    a_node += 1;
                    if (n != srcn) rn += 1;
                }
                a_rdev += rd;
                a_rnode += rn;
                if (tok_remote_dev) tok_remote_dev[((size_t)l * P + p) * (size_t)T + (size_t)t] = (uint8_t)rd;
                if (tok_remote_node) tok_remote_node[((size_t)l * P + p) * (size_t)T + (size_t)t] = (uint8_t)rn;
            }
            size_t o = (size_t)l * P + p;
            if (dev_visits) dev_visits[o] = a_dev;
            if (remote_dev) remote_dev[o] = a_rdev;
            if (remote_intra) remote_intra[o] = a_intra;
            if (remote_inter) remote_inter[o] = a_inter;
            if (node_visits) node_visits[o] = a_node;
            if (remote_node) remote_node[o] = a_rnode;
            if (cost) cost[o] = (int64_t)cost_local * a_local + (int64_t)cost_intra * a_intra
                                + (int64_t)cost_inter * a_inter;
            if (bytes) bytes[o] = a_rdev * bytes_per_token;
            int64_t mx = 0, sm = 0, mxr = 0, smr = 0;
            for (int32_t d = 0; d < D; ++d) {
                if (load_pairs) load_pairs[o * D + d] = lp[d];
                if (recv_tokens) recv_tokens[o * D + d] = rt[d];
                if (lp[d] > mx) mx = lp[d];
                sm += lp[d];
                if (rt[d] > mxr) mxr = rt[d];
                smr += rt[d];
            }
            /* Eq. 4: max / mean = max*D / sum; integer product exact, one divide */
            if (imbalance) imbalance[o] = sm ? (double)(mx * D) / (double)sm : 0.0;
            if (imbalance_recv) imbalance_recv[o] = smr ? (double)(mxr * D) / (double)smr : 0.0;
        }
    }
    return CAPO_OK;
}

/* ------------------------------------------------------------------------- *
 * S4  communication-aware pruning, P:L208-218 (sec. VI, Eq. 6 and the greedy
 * solver: "compute the ratio a_d/c_d for each device and retain devices in
 * descending order of this ratio until the target accuracy 1-p is
 * satisfied").  Heuristic: followed step by step, fp32, no reassociation.
 * Readings R7..R10: c_local = 0 -> ratio +inf (own device first),
 * keep while cum < 1-p, ties -> lower device id, p <= 0 is the identity.
 * expert_dev [L][E].  kept [L][T][k] out.  near_margin [L] out (nullable):
 * tokens whose deciding margin is below 1e-6 (R-S4.7).
 * ------------------------------------------------------------------------- */
int capo_prune(const int32_t *idx, const float *w, const int32_t *token_src,
               int32_t L, int64_t T, int32_t k, int32_t E,
               const int32_t *expert_dev, int32_t D, int32_t N, const int32_t *dev_node,
               int32_t cost_local, int32_t cost_intra, int32_t cost_inter,
               float p, uint8_t *kept, int64_t *near_margin)
{
    if (L < 0 || T < 0 || E < 1 || k < 1 || k > 16 || D < 1 || D > 64 || N < 1 || N > 64)
        return CAPO_EINVAL;
    if (!(p < 1.0f) || p != p) return CAPO_EINVAL;
    if (cost_local < 0 || cost_intra < 0 || cost_inter < 0) return CAPO_EINVAL;
    for (int32_t l = 0; l < L; ++l) {
        const int32_t *pi = expert_dev + (size_t)l * E;
        int64_t nm = 0;
        for (int64_t t = 0; t < T; ++t) {
            size_t base = ((size_t)l * (size_t)T + (size_t)t) * (size_t)k;
            if (p <= 0.0f) {                                  /* step 1: identity */
                for (int32_t s = 0; s < k; ++s) kept[base + s] = 1;
                continue;
            }
            int32_t src = token_src ? token_src[(size_t)l * (size_t)T + (size_t)t]
                                    : (int32_t)(((int64_t)t * D) / T);
            /* step 2: a_d in slot order */
            float a[64];
            uint8_t present[64], keepd[64];
            for (int32_t d = 0; d < D; ++d) { a[d] = 0.0f; present[d] = 0; keepd[d] = 0; }
            for (int32_t s = 0; s < k; ++s) {
                int32_t d = pi[idx[base + s]];
                a[d] = a[d] + w[base + s];
                present[d] = 1;
            }
            /* step 3: cost and ratio; step 4: order by ratio desc, ties lower d */
            int32_t order[64], m = 0;
            float ratio[64];
            for (int32_t d = 0; d < D; ++d) {
                if (!present[d]) continue;
                int32_t c = (d == src) ? cost_local
                          : (dev_node[d] == dev_node[src]) ? cost_intra : cost_inter;
                ratio[d] = (c == 0) ? INFINITY : a[d] / (float)c;
                order[m++] = d;
            }
            for (int32_t i = 1; i < m; ++i) {               /* stable insertion sort */
                int32_t d = order[i], j = i - 1;
                while (j >= 0 && ratio[order[j]] < ratio[d]) { order[j + 1] = order[j]; --j; }
                order[j + 1] = d;
            }
            /* step 5: keep while cum < target */
            float target = 1.0f - p;
            float cum = 0.0f;
            int near = 0;
            int32_t nk = 0;
            for (int32_t i = 0; i < m; ++i) {
                if (fabsf(cum - target) < 1e-6f) near = 1;
                if (cum >= target) break;
                keepd[order[i]] = 1;
                cum = cum + a[order[i]];
                nk = i + 1;
            }
            /* step 7: the ratio margin that decided kept-vs-dropped */
            if (nk < m) {
                float r1 = ratio[order[nk - 1]], r2 = ratio[order[nk]];
                if (isfinite(r1) && isfinite(r2) && (r1 - r2) < 1e-6f) near = 1;
            }
            nm += near;
            /* step 6 */
            for (int32_t s = 0; s < k; ++s) kept[base + s] = keepd[pi[idx[base + s]]];
        }
        if (near_margin) near_margin[l] = nm;
    }
    return CAPO_OK;
}

/* ------------------------------------------------------------------------- *
 * S5  dispatch layout, P:L58 (device-centric routing) + BASELINE.json (5):
 * stable counting sort of kept (token,slot) pairs i = t*k+s by destination
 * device pi(idx[i]).  Written as the definition: for each device in order,
 * scan the pairs in ascending i.
 * expert_dev [E].  sorted_pairs [>= n_kept], pair_pos [T*k] (nullable),
 * offsets [D+1].
 * ------------------------------------------------------------------------- */
int capo_dispatch_layout(const int32_t *idx, const uint8_t *kept, int64_t T, int32_t k,
                         int32_t E, const int32_t *expert_dev, int32_t D,
                         int32_t *sorted_pairs, int32_t *pair_pos, int64_t *offsets)
{
    if (T < 0 || E < 1 || k < 1 || k > 16 || D < 1 || D > 64) return CAPO_EINVAL;
    if (T * k >= ((int64_t)1 << 31)) return CAPO_EINVAL;
    int64_t n = T * k, pos = 0;
    if (pair_pos) for (int64_t i = 0; i < n; ++i) pair_pos[i] = -1;
    for (int32_t d = 0; d < D; ++d) {
        offsets[d] = pos;
        for (int64_t i = 0; i < n; ++i) {
            if (kept && !kept[i]) continue;
            if (expert_dev[idx[i]] != d) continue;
            sorted_pairs[pos] = (int32_t)i;
            if (pair_pos) pair_pos[i] = (int32_t)pos;
            ++pos;
        }
    }
    offsets[D] = pos;
    return CAPO_OK;
}

/* ------------------------------------------------------------------------- *
 * NEXT-1  co-activation probabilities and Algorithm 1.
 *
 * p_ij: "the ratio between the number of times they are selected
 * together and the total number of times either of them is selected" ->
 * reading R3 (Jaccard): p_ij = C_ij / (n_i + n_j - C_ij), 0 when the
 * denominator is 0, p_ii = 0 (never used: every sum below is over j != i or
 * over members of a group that e does not belong to).  Integers converted to
 * double exactly, one IEEE divide.
 *
 * Algorithm 1, followed line by line (capo_alg1 below):
 *   line 1   deg[i] = sum_{j != i} p_ij             (ascending j, fp64)
 *   line 2-3 G[g] = {} ; U = {all}
 *   line 4   pi = experts sorted by deg descending  (ties -> lower index, R23)
 *   line 5-7 for g = 1..k: seed G[g] with pi[g]
 *   line 8   while U not empty                      (starts at g = 1, R16)
 *   line 9-10  e* = argmax_{e in U} sum_{v in G[g]} p_ev   (sum in the order the
 *              members joined G[g]; ties -> lower index, R23)
 *   line 11-12 if that score is 0: e* = the r-th smallest element of U with
 *              r = rnd[step] mod |U| ("uniformly at random"; the random
 *              numbers are an INPUT, one per growth step, so that no generator
 *              is shared with the CUDA path; rnd == NULL reads as zeros)
 *   line 13  move e* from U to G[g]
 *   line 14  g = (g mod k) + 1
 * n must be a multiple of k ("each GPU hosts the same number of experts",
 * P:L160): the round-robin then fills every group to exactly n/k.
 *
 * Stage 2: "treat each GPU group as a coarse-grained unit, compute the
 * co-activation strength between groups, and apply the same grouping principle
 * again to assign GPU groups to nodes" -> reading R24: strength
 * W[a][b] = sum_{i in G[a]} sum_{j in G[b]} p_ij (i ascending outer, j
 * ascending inner, fp64), W[a][a] = 0; then capo_alg1 with n = D units, k = N.
 *
 * Outputs: expert_group [L][E] (stage 1), group_node [L][D] (stage 2), and the
 * placement expert_dev [L][E] on the regular topology dev_node[d] = d / (D/N):
 * group a becomes device group_node[a]*(D/N) + (rank at which a joined its node).
 * p_out [L][E][E] (nullable) receives the probabilities.
 * rnd [L][E + D] uint32 (nullable): stage 1 step s reads rnd[s], stage 2 step s
 * reads rnd[E + s].
 *
 * Pins (tests/test_oracle_pins.py): SURVEY worked example p_01 = 1/4, p_04 =
 * 2/3 by hand; k = 1, k = n closed forms; exact recovery of planted clusters
 * (block-diagonal C) and of planted node structure; an exact-rational
 * (fractions.Fraction) replay of the listing on tiny inputs; devices per token
 * below the sequential placement on the clustered trace (the paper's claim).
 * ------------------------------------------------------------------------- */
static void capo_alg1(int32_t n, int32_t k, const double *Pm, const uint32_t *rnd,
                      int32_t *grp, int32_t *ord)
{
    double *deg = (double *)malloc(sizeof(double) * (size_t)n);
    int32_t *pi = (int32_t *)malloc(sizeof(int32_t) * (size_t)n);
    int32_t *G = (int32_t *)malloc(sizeof(int32_t) * (size_t)n * (size_t)k); /* G[g][0..size) */
    int32_t *size = (int32_t *)calloc((size_t)k, sizeof(int32_t));
    uint8_t *inU = (uint8_t *)malloc((size_t)n);
    for (int32_t i = 0; i < n; ++i) {                       /* line 1 */
        double s = 0.0;
        for (int32_t j = 0; j < n; ++j)
            if (j != i) s += Pm[(size_t)i * n + j];
        deg[i] = s;
        inU[i] = 1;                                         /* line 3 */
        pi[i] = i;
    }
    for (int32_t a = 1; a < n; ++a) {                       /* line 4: stable insertion sort */
        int32_t x = pi[a];
        int32_t b = a - 1;
        while (b >= 0 && deg[pi[b]] < deg[x]) { pi[b + 1] = pi[b]; --b; }
        pi[b + 1] = x;
    }
    int32_t nU = n;
    for (int32_t g = 0; g < k; ++g) {                       /* lines 5-7 */
        int32_t s = pi[g];
        ord[s] = size[g];
        G[(size_t)g * n + size[g]++] = s;
        grp[s] = g;
        inU[s] = 0;
        --nU;
    }
    int32_t g = 0, step = 0;
    while (nU > 0) {                                        /* line 8 */
        int32_t best = -1;
        double bests = 0.0;
        for (int32_t e = 0; e < n; ++e) {                   /* lines 9-10 */
            if (!inU[e]) continue;
            double sc = 0.0;
            for (int32_t m = 0; m < size[g]; ++m) sc += Pm[(size_t)e * n + G[(size_t)g * n + m]];
            if (best < 0 || sc > bests) { best = e; bests = sc; }
        }
        if (bests == 0.0) {                                 /* lines 11-12 */
            uint32_t r = (rnd ? rnd[step] : 0u) % (uint32_t)nU;
            for (int32_t e = 0; e < n; ++e) {
                if (!inU[e]) continue;
                if (r == 0) { best = e; break; }
                --r;
            }
        }
        ord[best] = size[g];                                /* line 13 */
        G[(size_t)g * n + size[g]++] = best;
        grp[best] = g;
        inU[best] = 0;
        --nU;
        g = (g + 1) % k;                                    /* line 14 */
        ++step;
    }
    free(deg); free(pi); free(G); free(size); free(inU);
}

int capo_coact_placement(const int64_t *counts, const int32_t *coact, int32_t L, int32_t E,
                         int32_t D, int32_t N, const uint32_t *rnd, double *p_out,
                         int32_t *expert_group, int32_t *group_node, int32_t *expert_dev)
{
    if (L < 0 || E < 1 || D < 1 || N < 1 || E % D != 0 || D % N != 0) return CAPO_EINVAL;
    double *Pm = (double *)malloc(sizeof(double) * (size_t)E * (size_t)E);
    double *W = (double *)malloc(sizeof(double) * (size_t)D * (size_t)D);
    int32_t *ord = (int32_t *)malloc(sizeof(int32_t) * (size_t)E);
    int32_t *ord2 = (int32_t *)malloc(sizeof(int32_t) * (size_t)D);
    for (int32_t l = 0; l < L; ++l) {
        const int64_t *n = counts + (size_t)l * E;
        const int32_t *C = coact + (size_t)l * E * E;
        int32_t *grp = expert_group + (size_t)l * E;
        int32_t *gn = group_node + (size_t)l * D;
        for (int32_t i = 0; i < E; ++i)
            for (int32_t j = 0; j < E; ++j) {
                int64_t den = n[i] + n[j] - (int64_t)C[(size_t)i * E + j];
                Pm[(size_t)i * E + j] =
                    (i == j || den == 0) ? 0.0 : (double)C[(size_t)i * E + j] / (double)den;
            }
        if (p_out) memcpy(p_out + (size_t)l * E * E, Pm, sizeof(double) * (size_t)E * (size_t)E);
        capo_alg1(E, D, Pm, rnd ? rnd + (size_t)l * (size_t)(E + D) : NULL, grp, ord);
        for (int32_t a = 0; a < D; ++a)
            for (int32_t b = 0; b < D; ++b) {
                double s = 0.0;
                if (a != b)
                    for (int32_t i = 0; i < E; ++i) {
                        if (grp[i] != a) continue;
                        for (int32_t j = 0; j < E; ++j)
                            if (grp[j] == b) s += Pm[(size_t)i * E + j];
                    }
                W[(size_t)a * D + b] = s;
            }
        capo_alg1(D, N, W, rnd ? rnd + (size_t)l * (size_t)(E + D) + E : NULL, gn, ord2);
        for (int32_t e = 0; e < E; ++e)
            expert_dev[(size_t)l * E + e] = gn[grp[e]] * (D / N) + ord2[grp[e]];
    }
    free(Pm); free(W); free(ord); free(ord2);
    return CAPO_OK;
}

/* ------------------------------------------------------------------------- *
 * NEXT-3  the pairwise communication objective, Eq. 2-3
 * (P:L152-158), for P candidate placements, from the co-activation statistics
 * alone (no pass over the trace):
 *   C(pi) = sum_{i<j} p_ij d(pi(i), pi(j)),
 *   d = 0 same device, cost_intra (the paper's 1) same node, cost_inter (c) else.
 * Two weights: the integer co-activation counts C_ij (obj_count, int64, exact)
 * and the probabilities p_ij of P:L148 / R3 (obj_prob, fp64, summed over i
 * ascending, then j ascending).  Eq. 5: combined = lambda * obj_prob +
 * (1 - lambda) * B(pi) with B the caller's imbalance array (Eq. 4, an output
 * of S3); written only when imbalance != NULL.
 * expert_dev [L][P][E], dev_node [D]; outputs [L][P], any may be NULL.
 * Pins: all experts on one device -> 0; one expert per device on one node with
 * cost 1 -> sum_{i<j} C_ij = (sum_i (k-1) n_i) / 2 (S2's invariant); the
 * worked example by hand; the cluster-aligned placement scores below the
 * sequential one; brute force over pairs in Python.
 * ------------------------------------------------------------------------- */
int capo_pairwise_objective(const int64_t *counts, const int32_t *coact, int32_t L, int32_t E,
                            const int32_t *expert_dev, int32_t P, int32_t D, const int32_t *dev_node,
                            int32_t cost_intra, int32_t cost_inter, double lambda,
                            const double *imbalance, int64_t *obj_count, double *obj_prob,
                            double *combined)
{
    if (L < 0 || E < 1 || P < 0 || D < 1) return CAPO_EINVAL;
    for (int32_t l = 0; l < L; ++l) {
        const int64_t *n = counts + (size_t)l * E;
        const int32_t *C = coact + (size_t)l * E * E;
        for (int32_t p = 0; p < P; ++p) {
            const int32_t *pi = expert_dev + ((size_t)l * P + p) * E;
            int64_t oc = 0;
            double op = 0.0;
            for (int32_t i = 0; i < E; ++i)
                for (int32_t j = i + 1; j < E; ++j) {
                    int32_t di = pi[i], dj = pi[j];
                    int32_t d = di == dj ? 0 : (dev_node[di] == dev_node[dj] ? cost_intra : cost_inter);
                    int64_t c = C[(size_t)i * E + j];
                    int64_t den = n[i] + n[j] - c;
                    double pij = den == 0 ? 0.0 : (double)c / (double)den;
                    oc += c * (int64_t)d;
                    op += pij * (double)d;
                }
            size_t o = (size_t)l * P + p;
            if (obj_count) obj_count[o] = oc;
            if (obj_prob) obj_prob[o] = op;
            if (combined && imbalance) combined[o] = lambda * op + (1.0 - lambda) * imbalance[o];
        }
    }
    return CAPO_OK;
}

/* ------------------------------------------------------------------------- *
 * NEXT-4  device-centric dispatch rows.  P:L58 (sec.
 * II-C, Fig. 2): "each token is sent once to each device that hosts activated
 * experts" -- one row per (token, destination device), not per (token,
 * expert) as in S5 (R18).  Rows are grouped by device, ascending token inside
 * a device: rows_token[row_offsets[d] + r] = the r-th token (ascending) that
 * keeps at least one expert on d; row_offsets[D] = number of rows (= S3's
 * dev_visits; row_offsets[d+1]-row_offsets[d] = recv_tokens[d]).  pair_row[i]
 * (i = t*k+s, nullable) = the row that carries token t to the device of its
 * slot s, -1 for a pruned pair: the pointer the local weighted aggregation of
 * Fig. 2 needs.  Plain loops: devices outer, tokens inner.
 * ------------------------------------------------------------------------- */
int capo_dispatch_rows(const int32_t *idx, const uint8_t *kept, int64_t T, int32_t k, int32_t E,
                       const int32_t *expert_dev, int32_t D, int32_t *rows_token,
                       int32_t *pair_row, int64_t *row_offsets)
{
    if (T < 0 || k < 1 || E < 1 || D < 1) return CAPO_EINVAL;
    int64_t n = 0;
    if (pair_row)
        for (int64_t i = 0; i < T * k; ++i) pair_row[i] = -1;
    for (int32_t d = 0; d < D; ++d) {
        row_offsets[d] = n;
        for (int64_t t = 0; t < T; ++t) {
            int hit = 0;
            for (int32_t s = 0; s < k; ++s) {
                size_t i = (size_t)t * k + s;
                if (kept && !kept[i]) continue;
                if (expert_dev[idx[i]] != d) continue;
                hit = 1;
                if (pair_row) pair_row[i] = (int32_t)n;
            }
            if (hit) rows_token[n++] = (int32_t)t;
        }
    }
    row_offsets[D] = n;
    return CAPO_OK;
}

/* ------------------------------------------------------------------------- *
 * NEXT-2  the Adjustment Approach: "We start from
 * the communication-oriented placement ... and iteratively refine it through
 * expert swaps.  In each adjustment step, we swap a pair of experts between
 * high-load and low-load devices to reduce load imbalance while preserving as
 * much co-activation locality as possible."  The paper gives no selection
 * rule: PARITY UNPINNED AGAINST THE PAPER; the rule below is reading R27 and
 * the pins check it against its own stated properties and a hand example.
 *   load L_d = sum of n_e over the experts on d (R6, load_pairs);
 *   hot = device with the largest load, cold = with the smallest (ties -> lower id);
 *   candidates: a on hot, b on cold with 0 < n_a - n_b < L_hot - L_cold (both
 *     devices end strictly below L_hot: the imbalance cannot rise);
 *   choose the candidate with the smallest locality loss
 *     loss = aff(a, hot\a) + aff(b, cold\b) - aff(a, cold\b) - aff(b, hot\a),
 *     aff(x, S) = sum_{v in S} C_xv (integer co-activation counts, exact),
 *     ties -> lower a, then lower b;
 *   no candidate -> stop (the remaining spectrum entries repeat the last map).
 * expert_dev0 [L][E]; spectrum [L][S][E] = the map after each step; n_done [L];
 * swaps [L][S][2] = (a, b) of each step, -1 after the stop.
 * ------------------------------------------------------------------------- */
int capo_adjust_spectrum(const int64_t *counts, const int32_t *coact, int32_t L, int32_t E,
                         int32_t D, const int32_t *expert_dev0, int32_t S, int32_t *spectrum,
                         int32_t *n_done, int32_t *swaps)
{
    if (L < 0 || E < 1 || D < 1 || S < 0) return CAPO_EINVAL;
    int32_t *pi = (int32_t *)malloc(sizeof(int32_t) * (size_t)E);
    int64_t *load = (int64_t *)malloc(sizeof(int64_t) * (size_t)D);
    for (int32_t l = 0; l < L; ++l) {
        const int64_t *n = counts + (size_t)l * E;
        const int32_t *C = coact + (size_t)l * E * E;
        memcpy(pi, expert_dev0 + (size_t)l * E, sizeof(int32_t) * (size_t)E);
        int32_t done = S, stopped = 0;
        for (int32_t s = 0; s < S; ++s) {
            int32_t besta = -1, bestb = -1;
            if (!stopped) {
                for (int32_t d = 0; d < D; ++d) load[d] = 0;
                for (int32_t e = 0; e < E; ++e) load[pi[e]] += n[e];
                int32_t hot = 0, cold = 0;
                for (int32_t d = 1; d < D; ++d) {
                    if (load[d] > load[hot]) hot = d;
                    if (load[d] < load[cold]) cold = d;
                }
                int64_t bestloss = 0;
                for (int32_t a = 0; a < E; ++a) {
                    if (pi[a] != hot) continue;
                    for (int32_t b = 0; b < E; ++b) {
                        if (pi[b] != cold || hot == cold) continue;
                        int64_t delta = n[a] - n[b];
                        if (delta <= 0 || delta >= load[hot] - load[cold]) continue;
                        int64_t loss = 0;
                        for (int32_t v = 0; v < E; ++v) {
                            if (pi[v] == hot && v != a)
                                loss += (int64_t)C[(size_t)a * E + v] - (int64_t)C[(size_t)b * E + v];
                            if (pi[v] == cold && v != b)
                                loss += (int64_t)C[(size_t)b * E + v] - (int64_t)C[(size_t)a * E + v];
                        }
                        if (besta < 0 || loss < bestloss) { besta = a; bestb = b; bestloss = loss; }
                    }
                }
                if (besta < 0) { stopped = 1; done = s; }
                else { pi[besta] = cold; pi[bestb] = hot; }
            }
            memcpy(spectrum + ((size_t)l * S + s) * E, pi, sizeof(int32_t) * (size_t)E);
            if (swaps) {
                swaps[((size_t)l * S + s) * 2] = besta;
                swaps[((size_t)l * S + s) * 2 + 1] = bestb;
            }
        }
        if (n_done) n_done[l] = done;
    }
    free(pi); free(load);
    return CAPO_OK;
}

/* ------------------------------------------------------------------------- *
 * NEXT-4b  naive expert-level pruning.  P:L62 (sec. II-D): "a naive pruning strategy ...
 * selects the top-ranked experts for each token until their cumulative routing score
 * exceeds a predefined threshold"; P:L295 compares it with the communication-aware rule
 * at the same accuracy target 1-p (Fig. 14).  Restated as the one-expert-per-device,
 * uniform-cost case of capo_prune (Eq. 6 with c_d = 1): experts in descending routing
 * weight (ties -> lower expert id, R10), kept while the kept weight is < 1-p (the
 * crossing expert is kept, R9); p <= 0 keeps everything; near-margin as in R-S4.7.
 * Placement and topology play no role.
 * ------------------------------------------------------------------------- */
int capo_prune_naive(const int32_t *idx, const float *w, int32_t L, int64_t T, int32_t k,
                     float p, uint8_t *kept, int64_t *near_margin)
{
    if (L < 0 || T < 0 || k < 1 || k > 16) return CAPO_EINVAL;
    if (!(p < 1.0f) || p != p) return CAPO_EINVAL;
    for (int32_t l = 0; l < L; ++l) {
        int64_t nm = 0;
        for (int64_t t = 0; t < T; ++t) {
            size_t base = ((size_t)l * (size_t)T + (size_t)t) * (size_t)k;
            if (p <= 0.0f) {
                for (int32_t s = 0; s < k; ++s) kept[base + s] = 1;
                continue;
            }
            int32_t order[16];
            for (int32_t s = 0; s < k; ++s) order[s] = s;
            for (int32_t i = 1; i < k; ++i) {      /* insertion sort: weight desc, ties lower expert id */
                int32_t s = order[i], j = i - 1;
                while (j >= 0 && (w[base + order[j]] < w[base + s] ||
                                  (w[base + order[j]] == w[base + s] && idx[base + order[j]] > idx[base + s]))) {
                    order[j + 1] = order[j];
                    --j;
                }
                order[j + 1] = s;
            }
            float target = 1.0f - p, cum = 0.0f;
            int near = 0;
            int32_t nk = 0;
            for (int32_t s = 0; s < k; ++s) kept[base + s] = 0;
            for (int32_t i = 0; i < k; ++i) {
                if (fabsf(cum - target) < 1e-6f) near = 1;
                if (cum >= target) break;
                kept[base + order[i]] = 1;
                cum = cum + w[base + order[i]];
                nk = i + 1;
            }
            if (nk < k) {
                float r1 = w[base + order[nk - 1]], r2 = w[base + order[nk]];
                if ((r1 - r2) < 1e-6f) near = 1;
            }
            nm += near;
        }
        if (near_margin) near_margin[l] = nm;
    }
    return CAPO_OK;
}

/* ------------------------------------------------------------------------- *
 * NEXT-4c  combine weights of the dispatch rows.  P:L58 (sec. II-C, Fig. 2): a token is
 * "sent once to each device that hosts activated experts", the expert outputs are
 * "locally aggregated via a weighted summation" there, and one result per (token,
 * device) travels back.  The weight that row carries in the final combination is
 * a_d = sum of the routing weights of the token's kept experts on that device -- the
 * a_d of P:L212 (S4 step 2), in slot order, fp32.
 * pair_row [T*k]: row of pair i = t*k + s as written by capo_dispatch_rows (-1 = pruned).
 * row_w [n_rows] out.
 * ------------------------------------------------------------------------- */
int capo_dispatch_row_weights(const float *w, const int32_t *pair_row, int64_t T, int32_t k,
                              int64_t n_rows, float *row_w)
{
    if (T < 0 || k < 1 || k > 16 || n_rows < 0) return CAPO_EINVAL;
    for (int64_t r = 0; r < n_rows; ++r) row_w[r] = 0.0f;
    for (int64_t t = 0; t < T; ++t)
        for (int32_t s = 0; s < k; ++s) {
            int64_t i = t * k + s;
            int32_t r = pair_row[i];
            if (r < 0) continue;
            if ((int64_t)r >= n_rows) return CAPO_EINVAL;
            row_w[r] = row_w[r] + w[i];
        }
    return CAPO_OK;
}

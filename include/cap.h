/*
 * cap.h -- C ABI of the B200 (sm_100a) routing-trace hot path of CAP
 * (arXiv 2607.05116, "Communication-Aware Placement and Pruning for Efficient
 * Mixture-of-Experts Inference").  P:Lnnn = PAPER.md line nnn; Rn = reading n
 * in DESIGN.md section 3.
 *
 * Conventions (all entry points)
 *  - Every array pointer is a DEVICE pointer owned by the caller unless the
 *    comment says "host".  The structs (cap_gate_cfg, cap_topology,
 *    cap_eval_out) are read on the HOST at call time; the pointers inside them
 *    are device pointers.
 *  - The library never allocates, frees or synchronises device memory.  Work is enqueued on
 *    `stream` (a cudaStream_t passed as void*, NULL = default stream) and the
 *    call returns immediately.  Scratch comes from the caller's workspace `ws`
 *    of `ws_bytes` >= cap_workspace_bytes(...); it must stay untouched until the
 *    enqueued work has finished.  Calls with distinct workspaces are re-entrant.
 *  - Layouts are dense row-major with the dimensions written in brackets.
 *  - Return value: CAP_OK, or CAP_EINVAL (bad size / NULL / unsupported
 *    combination, detected on the host before anything is launched),
 *    CAP_EWORKSPACE (workspace too small), CAP_ECUDA (a launch failed;
 *    cap_last_cuda_error() returns the cudaError_t).
 *  - Values inside device arrays are not validated by the compute calls:
 *    expert_dev >= D, token_src >= D or non-finite logits give undefined but
 *    memory-safe results.  cap_validate_placements checks maps (synchronous).
 *  - T = 0 is valid: aggregate outputs are zeroed.
 *  - Limits: 1 <= E <= 1024, 1 <= k <= 16, k <= E, 1 <= D <= 64, 1 <= N <= 64,
 *    T*k < 2^31, L*T*k < 2^40.
 */
#ifndef CAP_H_
#define CAP_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define CAP_OK 0
#define CAP_EINVAL (-1)
#define CAP_EWORKSPACE (-2)
#define CAP_ECUDA (-3)

/* which_call values for cap_workspace_bytes */
#define CAP_CALL_GATE_TOPK 0
#define CAP_CALL_COACTIVATION 1
#define CAP_CALL_EVAL_PLACEMENTS 2
#define CAP_CALL_PRUNE 3
#define CAP_CALL_DISPATCH_LAYOUT 4
#define CAP_CALL_TRACE_FUSED 5
#define CAP_CALL_COACT_PLACEMENT 6   /* T, k, P ignored */
#define CAP_CALL_DISPATCH_ROWS 7     /* L, E, k, P ignored */
#define CAP_CALL_PRUNE_DISPATCH 8    /* P ignored */

/* Gate configuration (Eq. 1; scoring / group-limited routing / tie rule from
 * BASELINE.json, readings R1, R2, R14, R21). */
typedef struct {
    int32_t E;            /* experts */
    int32_t k;            /* experts selected per token */
    int32_t scoring;      /* 0 softmax (selection on the raw logit), 1 sigmoid (+bias) */
    int32_t renormalize;  /* 1: weights renormalised over the selected k */
    int32_t n_group;      /* 1 = no group-limited routing; else E % n_group == 0, n_group <= 32 */
    int32_t topk_group;   /* groups kept when n_group > 1 */
    int32_t group_score;  /* 0: max of the group; 1: fp32 sum of its two largest scores */
    float scale;          /* routed scaling factor applied to the weights (1.0 = none) */
} cap_gate_cfg;

/* Topology of a candidate placement (Eq. 3: d = 0 same device, 1 same node, c across nodes). */
typedef struct {
    int32_t D;               /* devices */
    int32_t N;               /* nodes */
    const int32_t *dev_node; /* [D] device ptr: node of each device, values in [0,N) */
    int32_t cost_local;      /* cost of staying on the token's own device (0, R7) */
    int32_t cost_intra;      /* cost of another device on the same node (1) */
    int32_t cost_inter;      /* cost of a device on another node (c) */
    int64_t bytes_per_token; /* bytes one token copy moves in one direction (R12) */
} cap_topology;

/* Outputs of the placement evaluation.  Any member may be NULL (not wanted). */
typedef struct {
    int64_t *dev_visits;    /* [L][P] sum over tokens of |Dev(t)|: "Device per Token" x T (Fig. 6, Table III) */
    int64_t *remote_dev;    /* [L][P] sum of |Dev(t) \ {src(t)}|: token copies sent by dispatch */
    int64_t *remote_intra;  /* [L][P] ... of which on the source's node */
    int64_t *remote_inter;  /* [L][P] ... of which on another node */
    int64_t *node_visits;   /* [L][P] sum of distinct nodes: "Node per Token" x T (Table II) */
    int64_t *remote_node;   /* [L][P] sum of distinct nodes other than the source's */
    int64_t *cost;          /* [L][P] cost_local*local + cost_intra*remote_intra + cost_inter*remote_inter */
    int64_t *bytes;         /* [L][P] remote_dev * bytes_per_token */
    int64_t *load_pairs;    /* [L][P][D] kept (token,expert) pairs computed on each device (L_g of Eq. 4, R6) */
    int64_t *recv_tokens;   /* [L][P][D] distinct tokens present on each device (local included) */
    double *imbalance;      /* [L][P] max_d load_pairs * D / sum_d load_pairs (Eq. 4), 0 if the sum is 0 */
    double *imbalance_recv; /* [L][P] same on recv_tokens */
    uint8_t *tok_remote_dev;  /* [L][P][T] |Dev(t) \ {src(t)}| per token */
    uint8_t *tok_remote_node; /* [L][P][T] distinct remote nodes per token */
} cap_eval_out;

/* S1 -- top-k gating (Eq. 1).
 * logits [L][T][E] fp32 (finite); bias [L][E] fp32 or NULL (sigmoid scoring only: selection
 * score = sigmoid(logit) + bias, weights from the unbiased sigmoid).
 * topk_idx [L][T][k] int32, slot 0 = largest selection score, ties -> lower expert index;
 * topk_w [L][T][k] fp32 routing weights (within 1e-6 of the definition).
 * EINVAL: bias with softmax, k > topk_group*E/n_group, n_group > 32, limits above. */
int cap_gate_topk(const float *logits, const float *bias, int32_t L, int64_t T,
                  const cap_gate_cfg *cfg, int32_t *topk_idx, float *topk_w,
                  void *ws, size_t ws_bytes, void *stream);

/* S2 -- activation counts and E x E co-activation (pruned trace P:L224).
 * topk_idx [L][T][k]: every row holds k DISTINCT ids in [0, E), as cap_gate_topk writes them (a repeated or
 * out-of-range id gives an undefined but memory-safe result); kept [L][T][k] uint8 or NULL (all kept).
 * counts [L][E] int64: kept (token,slot) pairs per expert.
 * coact [L][E][E] int32, full symmetric: tokens keeping both i and j; diagonal = counts. */
int cap_coactivation(const int32_t *topk_idx, const uint8_t *kept, int32_t L, int64_t T,
                     int32_t k, int32_t E, int64_t *counts, int32_t *coact,
                     void *ws, size_t ws_bytes, void *stream);

/* S3 -- score P candidate placements in one pass over the trace (Eq. 3, Eq. 4,
 * Fig. 6 axes, Tables II-IV).
 * token_src [L][T] int32 source device of each token, or NULL = floor(t*D/T) (R5).
 * expert_dev [L][P][E] int32 expert -> device maps, values in [0,D).
 * counts: optional [L][E] int64 from cap_coactivation on the SAME (topk_idx, kept); when
 * given, load_pairs is gathered from it instead of being recounted. */
int cap_eval_placements(const int32_t *topk_idx, const uint8_t *kept, const int32_t *token_src,
                        int32_t L, int64_t T, int32_t k, int32_t E,
                        const int32_t *expert_dev, int32_t P, const cap_topology *topo,
                        const int64_t *counts, const cap_eval_out *out,
                        void *ws, size_t ws_bytes, void *stream);

/* S4 -- communication-aware pruning under one placement (Eq. 6 + greedy).
 * Per token: a_d = sum of its weights on device d (slot order, fp32); c_d = cost_local /
 * cost_intra / cost_inter relative to token_src; devices kept by descending a_d/c_d (c_d = 0
 * first; ties -> lower device id) while the kept sum is < 1-p.  p <= 0 keeps everything.
 * Precondition: the weights of a token sum to 1 (renormalised gate, scale = 1): Eq. 6's 1-p is an
 * absolute share of the routing mass (reading R8).  With scaled or un-renormalised weights the call is
 * memory-safe but the stop rule no longer means "keep 1-p of the mass".
 * expert_dev [L][E].  kept [L][T][k] uint8 out.  after: optional S3 outputs (P = 1) of the
 * kept trace ("new volume and load").  near_margin [L] int64 or NULL: tokens whose deciding
 * comparison had a margin below 1e-6 (R-S4.7).  EINVAL unless p < 1. */
int cap_prune(const int32_t *topk_idx, const float *topk_w, const int32_t *token_src,
              int32_t L, int64_t T, int32_t k, int32_t E, const int32_t *expert_dev,
              const cap_topology *topo, float p, uint8_t *kept, const cap_eval_out *after,
              int64_t *near_margin, void *ws, size_t ws_bytes, void *stream);

/* S5 -- dispatch layout (P:L58 device-centric routing; BASELINE.json stage 5): stable
 * counting sort of the kept pairs i = t*k + s by destination device expert_dev[topk_idx[i]].
 * topk_idx [T][k]; kept [T][k] or NULL; expert_dev [E].
 * sorted_pairs [T*k] int32 (first offsets[D] entries valid): pair ids grouped by device,
 * ascending inside a device.  pair_pos [T*k] int32 or NULL: inverse (-1 if pruned).
 * offsets [D+1] int64: offsets[d] = kept pairs with device < d. */
int cap_dispatch_layout(const int32_t *topk_idx, const uint8_t *kept, int64_t T, int32_t k,
                        int32_t E, const int32_t *expert_dev, int32_t D, int32_t *sorted_pairs,
                        int32_t *pair_pos, int64_t *offsets, void *ws, size_t ws_bytes,
                        void *stream);

/* S4 followed by S5 under the same placement, in three launches instead of the six nodes of cap_prune +
 * cap_dispatch_layout_batched (at the BASELINE sizes both stages are launch-latency-bound).  Results are exactly
 * those of cap_prune(..., kept, after, near_margin, ...) followed by cap_dispatch_layout_batched(topk_idx, kept,
 * ..., expert_dev, D, sorted_pairs, pair_pos, offsets, ...): the pruning kernel (Eq. 6) also counts
 * the kept pairs per device of every 32 tokens, which is the histogram the stable counting sort starts
 * from; the sort's scan and scatter launches carry one extra block each that adds up / writes the after-metrics,
 * so no accumulator is zeroed and no separate histogram or finalize launch is needed.
 *   Arguments as in the two calls (expert_dev [L][E]: the chosen placement per layer; after, near_margin, pair_pos
 *   nullable).  Workspace: cap_workspace_bytes(CAP_CALL_PRUNE_DISPATCH, L, T, E, k, D, 0). */
int cap_prune_dispatch(const int32_t *topk_idx, const float *topk_w, const int32_t *token_src, int32_t L,
                       int64_t T, int32_t k, int32_t E, const int32_t *expert_dev, const cap_topology *topo,
                       float p, uint8_t *kept, const cap_eval_out *after, int64_t *near_margin,
                       int32_t *sorted_pairs, int32_t *pair_pos, int64_t *offsets, void *ws, size_t ws_bytes,
                       void *stream);

/* S5 for L layers in one call (three launches for all layers instead of three per layer: at the BASELINE sizes a
 * layer's sort is launch-latency-bound).  Per layer exactly cap_dispatch_layout: topk_idx / kept [L][T][k],
 * expert_dev [L][E] (one chosen placement per layer), sorted_pairs / pair_pos [L][T*k] (layer l's first
 * offsets[l][D] entries valid), offsets [L][D+1].  Workspace: cap_workspace_bytes(CAP_CALL_DISPATCH_LAYOUT, L, T,
 * E, k, D, 0) (for L = 1 that is cap_dispatch_layout's size). */
int cap_dispatch_layout_batched(const int32_t *topk_idx, const uint8_t *kept, int32_t L, int64_t T, int32_t k,
                                int32_t E, const int32_t *expert_dev, int32_t D, int32_t *sorted_pairs,
                                int32_t *pair_pos, int64_t *offsets, void *ws, size_t ws_bytes, void *stream);

/* S5 without a workspace, for callers that cannot allocate (CUDA graph capture, serving loops, harnesses
 * that forbid cudaMalloc).  Same result, bit for bit, as cap_dispatch_layout; the scratch is a static device
 * array of CAP_STATIC_SCRATCH_BYTES (4 MiB) inside the library, held by every GPU that loads it until exit.
 * Limit: cap_workspace_bytes(CAP_CALL_DISPATCH_LAYOUT, 1, T, E, k, D, 0) <= CAP_STATIC_SCRATCH_BYTES, i.e.
 * ceil128(ceil(T k / 256)) * D <= 524 256 -- e.g. T k <= 8.3 M pairs at D = 16, 2.0 M at D = 64; larger
 * sizes return CAP_EWORKSPACE (nothing is launched).  Calls no cudaMalloc / cudaFree; the array's device
 * address is resolved once per device (cudaGetSymbolAddress) on the first call made with that device
 * current -- make that call outside a stream capture.  All calls on a device share the array: it needs no
 * clearing between calls (each call writes what it reads), but calls that overlap on the GPU race on it --
 * order them on one stream or with an event.  Arguments as in cap_dispatch_layout. */
#define CAP_STATIC_SCRATCH_BYTES (4 * 1024 * 1024)
int cap_dispatch_layout_static(const int32_t *topk_idx, const uint8_t *kept, int64_t T, int32_t k,
                               int32_t E, const int32_t *expert_dev, int32_t D, int32_t *sorted_pairs,
                               int32_t *pair_pos, int64_t *offsets, void *stream);
/* CAP_STATIC_SCRATCH_BYTES as the loaded library was built. */
size_t cap_static_scratch_bytes(void);

/* S1 + S2 + S3 in one call over the logits (the measured pass).  Arguments as in the three
 * calls above; members of `out` may be NULL to skip an output; counts and coact are required
 * (CAP_EINVAL if NULL with L > 0: the fused kernel always produces them). */
int cap_trace_fused(const float *logits, const float *bias, int32_t L, int64_t T,
                    const cap_gate_cfg *cfg, int32_t *topk_idx, float *topk_w,
                    int64_t *counts, int32_t *coact, const int32_t *token_src,
                    const int32_t *expert_dev, int32_t P, const cap_topology *topo,
                    const cap_eval_out *out, void *ws, size_t ws_bytes, void *stream);

/* Introspection, host only (no launch, no device access): how cap_trace_fused would run these sizes
 * on the current device when token_src is NULL and no per-token output is asked for.
 *   plan[0] = 1 if the single fused S1+S2+S3 kernel serves them, 0 if the three staged kernels do;
 *   plan[1] = thread blocks per layer;  plan[2] = tokens per block (upper bound);
 *   plan[3] = largest number of tokens of ONE source device that a single block scores;
 *   plan[4] = tokens a block can count for one source before its bit-sliced counters are flushed
 *             (a "capacity flush": plan[3] > plan[4] means that branch runs);
 *   plan[5] = records a block can emit;  plan[6] = blocks per source device when block ranges are
 *             aligned to the source runs, else 0;  plan[7] = version of the fused kernel (0 if none).
 * Used by the tests to prove that a shape reaches a given branch.  CAP_EINVAL on invalid sizes. */
int cap_trace_fused_plan(int32_t L, int64_t T, const cap_gate_cfg *cfg, int32_t D, int32_t N, int32_t P,
                         int64_t plan[8]);

/* cap_trace_fused in two halves, for callers that overlap the end of S3 with the stages that follow
 * (S4 / S5 read topk_idx / topk_w, never the S3 outputs).  The candidate scoring (P:L64-66, P:L178,
 * P:L263) ends with a short launch that adds the per-block records up and writes `out`; _begin runs
 * everything before that launch and hands the launch back, _finish issues it on a stream of the
 * caller's choice:
 *     cap_trace_fused_begin(..., &pend, s);      topk_idx / topk_w / counts / coact final in order of s
 *     <event: s2 after s>   cap_trace_fused_finish(&pend, s2);    `out` final in order of s2
 *     cap_prune(..., s); cap_dispatch_layout(..., s);  <event: s after s2>
 * Arguments of _begin are those of cap_trace_fused (same checks, same results bit for bit).  `pend` is
 * plain host data owned by the caller (kind = 0: nothing owed -- the shape took a path that finishes
 * `out` itself --, _finish is then a no-op).  Between the halves `ws`, `counts`, `expert_dev`,
 * `topo->dev_node` and the `out` arrays must stay untouched; the ordering of s2 against s (and of the next
 * call that reuses `ws` against s2) is the caller's: the library adds no event.  A pending launch that is
 * never finished leaves `out` unwritten and leaks nothing. */
typedef struct cap_pending {
    int32_t kind;               /* 0 none, 1 decode launch of the bit-sliced S3 path */
    int32_t reserved;
    unsigned char blob[496];    /* launch parameters; opaque */
} cap_pending;
int cap_trace_fused_begin(const float *logits, const float *bias, int32_t L, int64_t T,
                          const cap_gate_cfg *cfg, int32_t *topk_idx, float *topk_w, int64_t *counts,
                          int32_t *coact, const int32_t *token_src, const int32_t *expert_dev, int32_t P,
                          const cap_topology *topo, const cap_eval_out *out, void *ws, size_t ws_bytes,
                          cap_pending *pend, void *stream);
int cap_trace_fused_finish(const cap_pending *pend, void *stream);

/* Co-activation driven expert placement: SURVEY 8(f) rank 1, the consumer of cap_coactivation's
 * outputs.  P:L148 defines the co-activation probability ("the ratio between the number of times
 * they are selected together and the total number of times either of them is selected"; reading R3:
 * p_ij = C_ij / (n_i + n_j - C_ij), 0 when the denominator is 0, p_ii = 0, fp64, one IEEE divide);
 * P:L106-144 is Algorithm 1 (weighted degrees, the D largest as seeds -- ties to the lower index,
 * R23 --, then round-robin growth from g = 1, each step taking the unassigned expert with the
 * largest sum of p to the group's members, summed in joining order, ties to the lower index; a zero
 * best score takes the r-th smallest unassigned expert, r = rnd[step] mod |U|); P:L162-164 applies
 * it again to the device groups with strength W[a][b] = sum_{i in G[a]} sum_{j in G[b]} p_ij
 * (ascending i outer, ascending j inner, R24) to form N node groups.
 *   counts [L][E] int64, coact [L][E][E] int32: as written by cap_coactivation / cap_trace_fused; coact
 *     must be symmetric, as those calls write it (the kernel reads rows where the definition reads
 *     columns); a non-symmetric matrix gives an undefined but memory-safe result.
 *   rnd [L][E + D] uint32, nullable (= zeros): stage 1 growth step s reads rnd[s], stage 2 step s
 *     reads rnd[E + s]; only consumed on the zero-score branch (line 12 of the listing).
 *   p_out [L][E][E] fp64, nullable: the probabilities.
 *   expert_group [L][E]: stage-1 group of each expert; group_node [L][D]: node of each group;
 *   expert_dev [L][E]: the placement on the regular topology dev_node[d] = d / (D/N): group a
 *     is device group_node[a] * (D/N) + (rank at which a joined its node group, seed = 0).
 * Requires E % D == 0 and D % N == 0 ("each GPU hosts the same number of experts"), else
 * CAP_EINVAL.  Workspace: cap_workspace_bytes(CAP_CALL_COACT_PLACEMENT, L, 0, E, 1, D, 0).
 * All outputs are reproducible bit for bit (fixed summation orders). */
int cap_coact_placement(const int64_t *counts, const int32_t *coact, int32_t L, int32_t E, int32_t D,
                        int32_t N, const uint32_t *rnd, double *p_out, int32_t *expert_group,
                        int32_t *group_node, int32_t *expert_dev, void *ws, size_t ws_bytes,
                        void *stream);

/* Adjustment Approach.  P:L194: "We start from the communication-oriented placement
 * produced by the Placement Approach and iteratively refine it through expert swaps.  In each adjustment
 * step, we swap a pair of experts between high-load and low-load devices to reduce load imbalance while
 * preserving as much co-activation locality as possible."  The paper states no selection rule; this call
 * implements reading R27 of DESIGN.md (parity unpinned against the paper, exact against the oracle):
 * load L_d = sum of counts over the experts on d; hot / cold = the device with the largest / smallest load
 * (ties to the lower id); candidates = (a on hot, b on cold) with 0 < n_a - n_b < L_hot - L_cold; the
 * candidate with the smallest loss = aff(a, hot\a) + aff(b, cold\b) - aff(a, cold\b) - aff(b, hot\a),
 * aff(x, S) = sum_{v in S} coact[x][v] (int64), is swapped (ties to the lower a, then the lower b); no
 * candidate stops the layer.
 *   expert_dev0 [L][E]: the starting maps (values clamped to [0, D)); S: number of steps;
 *   spectrum [L][S][E]: the map after each step (after a stop the last map is repeated) -- directly usable
 *     as the candidate array of cap_eval_placements / cap_pairwise_objective with P = S;
 *   n_done [L] int32, nullable: steps performed before the stop (S if none);
 *   swaps [L][S][2] int32, nullable: (a, b) of each step, (-1, -1) from the stop on.
 * counts / coact as written by cap_coactivation.  No workspace.  S = 0 or L = 0: nothing is written. */
int cap_adjust_spectrum(const int64_t *counts, const int32_t *coact, int32_t L, int32_t E, int32_t D,
                        const int32_t *expert_dev0, int32_t S, int32_t *spectrum, int32_t *n_done,
                        int32_t *swaps, void *stream);

/* Device-centric dispatch rows.  P:L58 (sec. II-C, Fig. 2): "each token is sent once
 * to each device that hosts activated experts" and aggregated there -- one row per (token, destination
 * device) instead of cap_dispatch_layout's one entry per (token, expert) pair (R18).
 *   rows_token [capacity >= T * min(k, D)] int32: token ids grouped by device, ascending token inside a
 *     device; rows_token[row_offsets[d] + r] = the r-th token that keeps at least one expert on device d.
 *   row_offsets [D + 1] int64: row_offsets[D] = number of rows (= dev_visits of cap_eval_placements for
 *     this map; row_offsets[d + 1] - row_offsets[d] = recv_tokens[d]).
 *   pair_row [T * k] int32, nullable: for pair i = t * k + s the row that carries token t to the device of
 *     its slot s (what the local weighted aggregation of Fig. 2 indexes), -1 for a pruned pair.
 * topk_idx [T][k], kept [T][k] nullable (= all kept), expert_dev [E] as in cap_dispatch_layout; one layer
 * per call.  T = 0 is valid (offsets zeroed).  Workspace: cap_workspace_bytes(CAP_CALL_DISPATCH_ROWS, 1, T,
 * E, k, D, 0).  Out-of-range experts / devices are clamped (memory-safe, result undefined). */
int cap_dispatch_rows(const int32_t *topk_idx, const uint8_t *kept, int64_t T, int32_t k, int32_t E,
                      const int32_t *expert_dev, int32_t D, int32_t *rows_token, int32_t *pair_row,
                      int64_t *row_offsets, void *ws, size_t ws_bytes, void *stream);

/* Combine weights of the dispatch rows.  P:L58: the outputs of a token's experts on one
 * device are "locally aggregated via a weighted summation" and one result per (token, device) row returns; the
 * weight of that row is a_d of P:L212 -- the fp32 sum, in slot order, of the routing weights of the token's kept
 * experts on the device.
 *   topk_w [T][k] fp32; pair_row [T*k] int32 as written by cap_dispatch_rows (-1 = pruned pair);
 *   n_rows = row_offsets[D] of that call (the caller reads it back, or passes the capacity T * min(k, D));
 *   row_w [n_rows] fp32 out: row_w[pair_row[i]] = sum over the pairs of that row.  Rows >= n_rows are skipped.
 * Bit-exact against the oracle (single IEEE adds in a fixed order).  No workspace. */
int cap_dispatch_row_weights(const float *topk_w, const int32_t *pair_row, int64_t T, int32_t k, int64_t n_rows,
                             float *row_w, void *stream);

/* Naive expert-level pruning (the baseline of Fig. 14 / P:L295): per token the experts
 * in descending routing weight (ties -> lower expert id) are kept while the kept weight is < 1 - p (the crossing
 * expert is kept; p <= 0 keeps everything) -- cap_prune's rule with one expert per device and c_d = 1, so that the
 * two can be compared at the same accuracy target.  No placement, no topology.
 *   topk_idx, topk_w [L][T][k]; kept [L][T][k] uint8 out; near_margin [L] int64 or NULL (as in cap_prune).
 * Same precondition as cap_prune: a token's weights sum to 1.  EINVAL unless p < 1.  No workspace. */
int cap_prune_naive(const int32_t *topk_idx, const float *topk_w, int32_t L, int64_t T, int32_t k, float p,
                    uint8_t *kept, int64_t *near_margin, void *stream);

/* Pairwise communication objective of P:L152-158 (Eq. 2-3) for P candidate placements, computed from
 * the co-activation statistics alone: C(pi) = sum_{i<j} w_ij d(pi(i), pi(j)) with
 * d = 0 on the same device, topo->cost_intra (the paper's 1) on the same node, topo->cost_inter (the
 * paper's c) across nodes (cost_local is not used), for two weights:
 *   obj_count [L][P] int64: w_ij = C_ij (exact);
 *   obj_prob  [L][P] fp64:  w_ij = p_ij = C_ij / (n_i + n_j - C_ij) (R3; 0 when the denominator
 *     is 0).  Summation order is the kernel's (fixed, so results repeat run to run); the definition's
 *     i-then-j order differs by at most (E^2 / 2) ulp relative, all terms being non-negative: compare
 *     with relative tolerance 1e-10.
 *   combined  [L][P] fp64, nullable: Eq. 5, lambda * obj_prob + (1 - lambda) * imbalance, with
 *     imbalance [L][P] fp64 (B(pi) of Eq. 4, e.g. cap_eval_out.imbalance); CAP_EINVAL if combined is
 *     given without imbalance.
 * counts [L][E] int64 and coact [L][E][E] int32 as written by cap_coactivation; expert_dev [L][P][E]
 * (values outside [0, D) are clamped: memory-safe, result undefined).  Any output may be NULL.  No
 * workspace. */
int cap_pairwise_objective(const int64_t *counts, const int32_t *coact, int32_t L, int32_t E,
                           const int32_t *expert_dev, int32_t P, const cap_topology *topo, double lambda,
                           const double *imbalance, int64_t *obj_count, double *obj_prob, double *combined,
                           void *stream);

/* Bytes of workspace the given call needs for these sizes (0 on invalid sizes). */
size_t cap_workspace_bytes(int which_call, int32_t L, int64_t T, int32_t E, int32_t k,
                           int32_t D, int32_t P);

/* Synchronous check that every expert_dev[l][p][e] lies in [0,D).  Returns CAP_OK, or
 * CAP_EINVAL if a value is out of range, or CAP_ECUDA.  Blocks on `stream`. */
int cap_validate_placements(const int32_t *expert_dev, int32_t L, int32_t P, int32_t E,
                            int32_t D, void *stream);

/* cudaError_t of the last failed launch on the calling thread (0 if none). */
int cap_last_cuda_error(void);

/* Number of kernels the library has launched since it was loaded (all threads). */
int64_t cap_launch_count(void);

/* Profiling aid (not part of the data path; not thread-safe).  cap_kernel_timer_arm(tag, slot)
 * makes the next launch of the kernel tagged `tag` ("gate_topk", "coact", "eval", "eval_finalize",
 * "eval_table", "eval_decode", "masked_counts", "prune", "dispatch_hist", "dispatch_scan",
 * "dispatch_scatter", "trace_fused", "coact_placement", "objective", "rows_hist", "rows_scan", "rows_scatter", "adjust")
 * record a CUDA event pair, owned by the library, around itself on its stream; up to 128 arms
 * may be pending, slot in [0,4096).  cap_kernel_timer_ms(slot) returns the elapsed device time
 * in milliseconds once that work has completed (the caller synchronises), or -1. */
int cap_kernel_timer_arm(const char *tag, int slot);
float cap_kernel_timer_ms(int slot);

/* Profiling aid, synchronous, host pointers where noted: builds the candidate tables once, then
 * launches ONLY the fused S1+S2+S3 kernel of cap_trace_fused n_rep times back to back on `stream`
 * (launch i reads logits_list[i % n_list], so that inputs larger than L2 can be rotated) between two
 * library-owned CUDA events, and stores the average device time per launch in *avg_ms (host).
 * logits_list is a HOST array of n_list device pointers.  The outputs are left un-finalised (the
 * accumulators hold n_rep passes).  CAP_EINVAL when the configuration is not served by the fused
 * kernel (it is for softmax scoring with renormalisation, no group limit, k <= 8, E in {64,128,256},
 * token_src NULL, candidates fitting one table).  Other arguments as in cap_trace_fused. */
int cap_profile_fused_kernel(const float *const *logits_list, int32_t n_list, int32_t n_rep, int32_t L,
                             int64_t T, const cap_gate_cfg *cfg, int32_t *topk_idx, float *topk_w,
                             int64_t *counts, int32_t *coact, const int32_t *expert_dev, int32_t P,
                             const cap_topology *topo, const cap_eval_out *out, void *ws, size_t ws_bytes,
                             void *stream, float *avg_ms);

/* Library version string (static storage). */
const char *cap_version(void);

#ifdef __cplusplus
}
#endif
#endif /* CAP_H_ */

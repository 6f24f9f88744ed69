// S4 -- communication-aware pruning (Eq. 6 and its greedy solver), fused with the
// evaluation of the pruned trace under the same placement ("new volume and load").  One thread per
// token, everything in registers (fully unrolled over the k slots, no indexed local arrays):
//   1. aggregate the slot weights per destination device in slot order (fp32, single IEEE adds),
//   2. price each device by topology relative to the token's source (readings R7, R13),
//   3. rank the devices by a_d / c_d descending, ties -> lower device id (R10),
//   4. keep devices in rank order while the kept weight is below 1 - p (R8, R9),
//   5. kept[t][s] = 1 iff the slot's device was kept; near-margin tokens are counted (R-S4.7).
// When the caller wants the after-metrics, the same thread also adds the token's kept device set
// into the block's evaluation accumulators (distinct devices / nodes, local, same-node, received
// tokens per device, kept pairs per expert), which are flushed with a few atomics per block; the
// block that finishes last in its layer (ticket in a spare accumulator slot) turns the sums into the
// caller's outputs (eval_finalize_one), so cap_prune with after-metrics is one memset and ONE kernel.
#include <math_constants.h>

#include "cap_eval_final.cuh"
#include "cap_internal.cuh"
#include "cap_prune_core.cuh"

namespace cap {

struct PruneParams {
    const int32_t *idx;
    const float *w;
    const int32_t *token_src;
    const int32_t *expert_dev;   // [L][E]
    const int32_t *dev_node;
    uint8_t *kept;
    unsigned long long *near_margin;   // [L * near_stride] or NULL
    int32_t near_stride;
    FinalParams fin;              // used when acc != NULL
    // evaluation of the kept trace (all NULL when not wanted)
    unsigned long long *acc;      // [L][ACC_N]
    unsigned long long *recv;     // [L][D]
    unsigned long long *ldirect;  // [L][64] kept pairs per device
    uint8_t *tok_rdev, *tok_rnode;   // [L][T] or NULL
    int64_t T;
    int32_t k, E, D, N, cost_local, cost_intra, cost_inter, vec, vec2, small;
    float p;
    // cap_prune_dispatch: kept pairs per device of every warp's 32 tokens -> histogram rows of S5, the block's sums
    // -> part (plain stores; no accumulator has to be zeroed, no ticket)
    int *hist;                    // [L][...] rows of hist_stride sub-chunks, layers hist_layer apart; or NULL
    int64_t hist_stride, hist_layer;
    uint32_t *part;               // [L][gridDim.x][PD_PART]
};

constexpr int PR_THREADS = 128;
constexpr int PR_WARPS = PR_THREADS / 32;

template <int KMAX>
__global__ void __launch_bounds__(PR_THREADS) prune_kernel(PruneParams prm)
{
    extern __shared__ int s_map[];     // [E] expert -> device, [64] device -> node
    __shared__ unsigned long long s_nodemask[64];
    __shared__ unsigned long long s_acc[ACC_N];
    __shared__ unsigned long long s_lp[64];
    __shared__ unsigned int s_cnt[PR_WARPS][64];   // per warp and device: tokens received << 16 | kept pairs
    __shared__ int s_last;
    const int layer = blockIdx.y;
    const int E = prm.E, D = prm.D, k = prm.k;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int *s_dn = s_map + E;
    const bool fusedm = prm.hist != nullptr;
    const bool want_eval = prm.acc != nullptr || fusedm;
    pdl_launch_dependents();
    pdl_wait();
    // this thread's token (vector path): in flight while the maps are staged
    const int64_t tq = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    int4 q_i0 = make_int4(0, 0, 0, 0), q_i1 = q_i0;
    float4 q_w0 = make_float4(0.f, 0.f, 0.f, 0.f), q_w1 = q_w0;
    if (KMAX == 8 && prm.vec && tq < prm.T) {
        const int64_t qb = ((int64_t)layer * prm.T + tq) * k;
        q_i0 = __ldg(reinterpret_cast<const int4 *>(prm.idx + qb));
        q_i1 = __ldg(reinterpret_cast<const int4 *>(prm.idx + qb) + 1);
        q_w0 = __ldg(reinterpret_cast<const float4 *>(prm.w + qb));
        q_w1 = __ldg(reinterpret_cast<const float4 *>(prm.w + qb) + 1);
    }
    for (int i = threadIdx.x; i < E; i += blockDim.x) s_map[i] = prm.expert_dev[(size_t)layer * E + i];
    if (threadIdx.x < 64) {
        s_dn[threadIdx.x] = (int)threadIdx.x < D ? prm.dev_node[threadIdx.x] : 0;
        s_nodemask[threadIdx.x] = 0ull;
    }
    static_assert(PR_WARPS * 64 == 2 * PR_THREADS, "two counters per thread");
    (&s_cnt[0][0])[threadIdx.x] = 0u;
    (&s_cnt[0][0])[threadIdx.x + PR_THREADS] = 0u;
    if (threadIdx.x < ACC_N) s_acc[threadIdx.x] = 0ull;
    __syncthreads();
    // devices of every node: one shared-memory OR per device (from the staged copy)
    if ((int)threadIdx.x < D) {
        const int n = s_dn[threadIdx.x];
        if ((unsigned)n < (unsigned)prm.N) atomicOr(&s_nodemask[n], 1ull << threadIdx.x);
    }
    __syncthreads();

    const int64_t T = prm.T;
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    int near = 0;
    unsigned a_dev = 0, a_loc = 0, a_same = 0, a_node = 0, a_rnode = 0;
    if (t < T) {
        const int64_t base = ((int64_t)layer * T + t) * k;
        int e[KMAX], d[KMAX];
        float wv[KMAX];
        if (KMAX == 8 && prm.vec) {
            const int4 i0 = q_i0, i1 = q_i1;
            const float4 w0 = q_w0, w1 = q_w1;
            e[0] = i0.x; e[1] = i0.y; e[2] = i0.z; e[3] = i0.w;
            e[4 % KMAX] = i1.x; e[5 % KMAX] = i1.y; e[6 % KMAX] = i1.z; e[7 % KMAX] = i1.w;
            wv[0] = w0.x; wv[1] = w0.y; wv[2] = w0.z; wv[3] = w0.w;
            wv[4 % KMAX] = w1.x; wv[5 % KMAX] = w1.y; wv[6 % KMAX] = w1.z; wv[7 % KMAX] = w1.w;
        } else if (KMAX % 2 == 0 && prm.vec2) {
            // even k, 8-byte aligned arrays: 64-bit loads (k = 10: 5 + 5 instead of 10 + 10)
#pragma unroll
            for (int s = 0; s < KMAX; s += 2) {
                int2 v = make_int2(0, 0);
                float2 u = make_float2(0.f, 0.f);
                if (s < k) {
                    v = __ldg(reinterpret_cast<const int2 *>(prm.idx + base + s));
                    u = __ldg(reinterpret_cast<const float2 *>(prm.w + base + s));
                }
                e[s] = v.x; e[(s + 1) % KMAX] = v.y;
                wv[s] = u.x; wv[(s + 1) % KMAX] = u.y;
            }
        } else {
#pragma unroll
            for (int s = 0; s < KMAX; ++s) {
                e[s] = s < k ? __ldg(prm.idx + base + s) : 0;
                wv[s] = s < k ? __ldg(prm.w + base + s) : 0.0f;
            }
        }
#pragma unroll
        for (int s = 0; s < KMAX; ++s) {
            const int ee = (unsigned)e[s] < (unsigned)E ? e[s] : 0;
            d[s] = s_map[ee] & 63;
        }
        // source device of the token (reading A5): explicit, or contiguous blocks floor(t D / T); the 32-bit
        // quotient is exact whenever T D < 2^32 (one short division instead of a 64-bit one)
        const int src = prm.token_src ? (prm.token_src[(int64_t)layer * T + t] & 63)
                        : prm.small ? (int)(((unsigned)t * (unsigned)D) / (unsigned)T) : (int)((t * D) / T);
        unsigned long long keepmask = 0ull;
        PruneRuns<KMAX> runs;
        if (prm.p <= 0.0f) {
#pragma unroll
            for (int s = 0; s < KMAX; ++s)
                if (s < k) keepmask |= 1ull << d[s];
            if (want_eval) prune_runs_only<KMAX>(d, k, runs);
        } else {
            keepmask = prune_token<KMAX>(d, wv, k, src, s_dn, prm.cost_local, prm.cost_intra, prm.cost_inter, prm.p,
                                         near, runs);
        }
        // kept mask per slot
        if (KMAX == 8 && k == 8 && prm.vec) {
            unsigned lo = 0, hi = 0;
#pragma unroll
            for (int s = 0; s < 4; ++s) {
                lo |= (unsigned)((keepmask >> d[s]) & 1ull) << (8 * s);
                hi |= (unsigned)((keepmask >> d[(4 + s) % KMAX]) & 1ull) << (8 * s);
            }
            *reinterpret_cast<uint2 *>(prm.kept + base) = make_uint2(lo, hi);
        } else {
#pragma unroll
            for (int s = 0; s < KMAX; ++s)
                if (s < k) prm.kept[base + s] = (uint8_t)((keepmask >> d[s]) & 1ull);
        }
        // evaluation of the kept trace under this placement (P = 1)
        if (want_eval) {
            const int srcn = s_dn[src];
            // nodes the kept devices sit on: one mask test per node (N <= 8) instead of a map look-up and a 64-bit
            // shift per slot
            unsigned nodebits = 0u;
            for (int n = 0; n < prm.N; ++n) nodebits |= (keepmask & s_nodemask[n]) ? (1u << n) : 0u;
#pragma unroll
            for (int i = 0; i < KMAX; ++i) {
                const uint32_t r = runs.run[i];
                const int dd = (int)(r & 63u);
                if (r != 0u && ((keepmask >> dd) & 1ull))
                    atomicAdd(&s_cnt[warp][dd], 0x10000u | ((r >> 8) & 0xffu));   // one token, run-length pairs
            }
            a_dev = __popcll(keepmask);
            a_loc = (unsigned)((keepmask >> src) & 1ull);
            a_same = __popcll(keepmask & s_nodemask[srcn]);
            a_node = __popc(nodebits);
            a_rnode = a_node - ((nodebits >> srcn) & 1u);
            if (prm.tok_rdev) prm.tok_rdev[(int64_t)layer * T + t] = (uint8_t)(a_dev - a_loc);
            if (prm.tok_rnode) prm.tok_rnode[(int64_t)layer * T + t] = (uint8_t)a_rnode;
        }
    }
    if (fusedm) {
        const unsigned b = __ballot_sync(0xffffffffu, near != 0);
        if (lane == 0 && b) atomicAdd(&s_acc[ACC_NEAR], (unsigned long long)__popc(b));
        // this warp's 32 tokens are sub-chunk `sub` of S5
        __syncwarp();
        const int64_t sub = (int64_t)blockIdx.x * PR_WARPS + warp;
        int *h = prm.hist + (int64_t)layer * prm.hist_layer;
        if (lane < D) h[(int64_t)lane * prm.hist_stride + sub] = (int)(s_cnt[warp][lane] & 0xffffu);
        if (lane + 32 < D) h[(int64_t)(lane + 32) * prm.hist_stride + sub] = (int)(s_cnt[warp][lane + 32] & 0xffffu);
    } else if (prm.near_margin) {
        const unsigned b = __ballot_sync(0xffffffffu, near != 0);
        if (lane == 0 && b) atomicAdd(&prm.near_margin[(size_t)layer * prm.near_stride], (unsigned long long)__popc(b));
    }
    if (want_eval) {
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) {
            a_dev += __shfl_xor_sync(0xffffffffu, a_dev, off);
            a_loc += __shfl_xor_sync(0xffffffffu, a_loc, off);
            a_same += __shfl_xor_sync(0xffffffffu, a_same, off);
            a_node += __shfl_xor_sync(0xffffffffu, a_node, off);
            a_rnode += __shfl_xor_sync(0xffffffffu, a_rnode, off);
        }
        if (lane == 0) {
            atomicAdd(&s_acc[ACC_DEV], (unsigned long long)a_dev);
            atomicAdd(&s_acc[ACC_LOCAL], (unsigned long long)a_loc);
            atomicAdd(&s_acc[ACC_SAMENODE], (unsigned long long)a_same);
            atomicAdd(&s_acc[ACC_NODE], (unsigned long long)a_node);
            atomicAdd(&s_acc[ACC_RNODE], (unsigned long long)a_rnode);
        }
        __syncthreads();
        if (fusedm) {
            uint32_t *pp = prm.part + ((size_t)layer * gridDim.x + blockIdx.x) * PD_PART;
            if (threadIdx.x < ACC_N) pp[threadIdx.x] = (uint32_t)s_acc[threadIdx.x];
            if (threadIdx.x < 64) {
                unsigned rc = 0;
#pragma unroll
                for (int w2 = 0; w2 < PR_WARPS; ++w2) rc += s_cnt[w2][threadIdx.x] >> 16;
                pp[ACC_N + threadIdx.x] = rc;
            }
            return;
        }
        if (threadIdx.x < ACC_N && s_acc[threadIdx.x])
            atomicAdd(&prm.acc[(size_t)layer * ACC_N + threadIdx.x], s_acc[threadIdx.x]);
        if (threadIdx.x < 64) {
            // the block's tokens received / kept pairs per device
            unsigned rc = 0, pr = 0;
#pragma unroll
            for (int w2 = 0; w2 < PR_WARPS; ++w2) {
                const unsigned v = s_cnt[w2][threadIdx.x];
                rc += v >> 16;
                pr += v & 0xffffu;
            }
            if ((int)threadIdx.x < D && rc) atomicAdd(&prm.recv[(size_t)layer * D + threadIdx.x], (unsigned long long)rc);
            if (pr) atomicAdd(&prm.ldirect[(size_t)layer * 64 + threadIdx.x], (unsigned long long)pr);
        }
        // last block of the layer: all sums are in L2, finish the outputs
        __threadfence();
        __syncthreads();
        if (threadIdx.x == 0)
            s_last = atomicAdd(&prm.acc[(size_t)layer * ACC_N + ACC_TICKET], 1ull) == (unsigned long long)gridDim.x - 1ull;
        __syncthreads();
        if (s_last && threadIdx.x < 32) {
            __threadfence();
            eval_finalize_one(prm.fin, layer, (int)threadIdx.x, s_lp);
        }
    }
}

// Prune and, when `after` is given, evaluate the kept trace (P = 1): ws is the evaluation workspace.
int launch_prune(const int32_t *idx, const float *w, const int32_t *token_src, int32_t L,
                 int64_t T, int32_t k, int32_t E, const int32_t *expert_dev,
                 const cap_topology &topo, float p, uint8_t *kept, int64_t *near_margin,
                 const cap_eval_out *after, void *ws, cudaStream_t st)
{
    if (L == 0) return CAP_OK;
    // with the after-metrics the near-margin count rides in the evaluation accumulators (one memset for
    // everything, written out by the finalize kernel); without them it is counted in place
    if (near_margin && (!after || T == 0) &&
        cudaMemsetAsync(near_margin, 0, sizeof(int64_t) * (size_t)L, st) != cudaSuccess)
        return check_launch("memset near_margin");
    PruneParams prm;
    prm.acc = prm.recv = prm.ldirect = nullptr;
    prm.tok_rdev = prm.tok_rnode = nullptr;
    prm.hist = nullptr;
    prm.hist_stride = prm.hist_layer = 0;
    prm.part = nullptr;
    if (after) {
        CAP_TRY(eval_zero_ws(L, E, topo.D, 1, true, ws, st));
        EvalWs ew = eval_ws_carve(ws, L, E, topo.D, 1);
        prm.acc = ew.acc;
        prm.recv = ew.recv;
        prm.ldirect = ew.ldirect;
        prm.tok_rdev = after->tok_remote_dev;
        prm.tok_rnode = after->tok_remote_node;
        prm.fin = make_final_params(L, E, 1, expert_dev, topo, reinterpret_cast<const int64_t *>(ew.mcounts), *after, ws,
                                    T > 0 ? near_margin : nullptr);
        prm.fin.load_direct = ew.ldirect;
    }
    if (T > 0) {
        prm.idx = idx;
        prm.w = w;
        prm.token_src = token_src;
        prm.expert_dev = expert_dev;
        prm.dev_node = topo.dev_node;
        prm.kept = kept;
        prm.near_margin = reinterpret_cast<unsigned long long *>(near_margin);
        prm.near_stride = 1;
        if (after && near_margin) {
            prm.near_margin = prm.acc + ACC_NEAR;
            prm.near_stride = ACC_N;
        }
        prm.T = T;
        prm.k = k;
        prm.E = E;
        prm.D = topo.D;
        prm.N = topo.N;
        prm.cost_local = topo.cost_local;
        prm.cost_intra = topo.cost_intra;
        prm.cost_inter = topo.cost_inter;
        prm.p = p;
        prm.small = (unsigned long long)T * (unsigned long long)topo.D < (1ull << 32);
        prm.vec = k == 8 && ((reinterpret_cast<uintptr_t>(idx) | reinterpret_cast<uintptr_t>(w)) & 15u) == 0 &&
                  (reinterpret_cast<uintptr_t>(kept) & 7u) == 0;
        prm.vec2 = (k & 1) == 0 && ((reinterpret_cast<uintptr_t>(idx) | reinterpret_cast<uintptr_t>(w)) & 7u) == 0;
        dim3 grid((unsigned)((T + PR_THREADS - 1) / PR_THREADS), (unsigned)L);
        const size_t smem = sizeof(int) * ((size_t)E + 64);
        {
            KernelTimerScope ts("prune", st);
            // the unrolled O(K^2) select chains are sized by the template: k = 10 (config 5) in <12>, not <16>
            if (k <= 4) launch_pdl(prune_kernel<4>, grid, dim3(PR_THREADS), smem, st, prm);
            else if (k <= 8) launch_pdl(prune_kernel<8>, grid, dim3(PR_THREADS), smem, st, prm);
            else if (k <= 10) launch_pdl(prune_kernel<10>, grid, dim3(PR_THREADS), smem, st, prm);
            else if (k <= 12) launch_pdl(prune_kernel<12>, grid, dim3(PR_THREADS), smem, st, prm);
            else launch_pdl(prune_kernel<16>, grid, dim3(PR_THREADS), smem, st, prm);
        }
        note_launch();
        CAP_TRY(check_launch("prune_kernel"));
    }
    if (after && T == 0) {
        EvalWs ew = eval_ws_carve(ws, L, E, topo.D, 1);
        return launch_eval_finalize(L, E, 1, expert_dev, topo, reinterpret_cast<const int64_t *>(ew.mcounts), *after,
                                    ws, st, nullptr);
    }
    return CAP_OK;
}

// ---- cap_prune_dispatch: S4 + S5 in three launches ----------------------------------------------------------
// ws: [evaluation sums of P = 1 (eval_ws_carve)] [hist | base | device totals per layer] [per-block partials]
static int64_t pd_stride(int64_t T) { return dispatch_stride_subs((T + 31) / 32); }

size_t prune_dispatch_ws_bytes(int32_t L, int64_t T, int32_t k, int32_t E, int32_t D)
{
    const int64_t stride = pd_stride(T);
    const size_t ll = (size_t)(L < 1 ? 1 : L);
    return eval_ws_bytes(L, 0, E, k, D, 1) + 256 + ll * (size_t)(2 * stride * D + 64) * sizeof(int) + 256 +
           ll * (size_t)(stride / PR_WARPS) * PD_PART * sizeof(uint32_t) + 256 +
           ll * (size_t)PD_MAXRB * PD_PART * sizeof(unsigned long long);
}

int launch_prune_dispatch(const int32_t *idx, const float *w, const int32_t *token_src, int32_t L, int64_t T,
                          int32_t k, int32_t E, const int32_t *expert_dev, const cap_topology &topo, float p,
                          uint8_t *kept, int64_t *near_margin, const cap_eval_out *after, int32_t *sorted_pairs,
                          int32_t *pair_pos, int64_t *offsets, void *ws, cudaStream_t st)
{
    if (L == 0) return CAP_OK;
    const int D = topo.D;
    if (T == 0) {
        // nothing to prune or to lay out: the stand-alone calls handle the empty outputs
        CAP_TRY(launch_prune(idx, w, token_src, L, T, k, E, expert_dev, topo, p, kept, near_margin, after, ws, st));
        return launch_dispatch_batched(idx, kept, L, T, k, E, expert_dev, D, sorted_pairs, pair_pos, offsets, ws, st);
    }
    const int64_t stride = pd_stride(T);
    const int64_t nblk = stride / PR_WARPS;
    EvalWs ew = eval_ws_carve(ws, L, E, D, 1);
    uintptr_t a = reinterpret_cast<uintptr_t>(ws) + eval_ws_bytes(L, 0, E, k, D, 1);
    a = (a + 255) & ~(uintptr_t)255;
    int *hist = reinterpret_cast<int *>(a);
    a += (size_t)L * (size_t)(2 * stride * D + 64) * sizeof(int);
    a = (a + 255) & ~(uintptr_t)255;
    uint32_t *part = reinterpret_cast<uint32_t *>(a);
    a += (size_t)L * (size_t)nblk * PD_PART * sizeof(uint32_t);
    a = (a + 255) & ~(uintptr_t)255;
    unsigned long long *red = reinterpret_cast<unsigned long long *>(a);

    PruneParams prm;
    prm.acc = prm.recv = prm.ldirect = nullptr;
    prm.tok_rdev = after ? after->tok_remote_dev : nullptr;
    prm.tok_rnode = after ? after->tok_remote_node : nullptr;
    prm.fin = FinalParams{};
    prm.idx = idx;
    prm.w = w;
    prm.token_src = token_src;
    prm.expert_dev = expert_dev;
    prm.dev_node = topo.dev_node;
    prm.kept = kept;
    prm.near_margin = nullptr;
    prm.near_stride = 0;
    prm.T = T;
    prm.k = k;
    prm.E = E;
    prm.D = D;
    prm.N = topo.N;
    prm.cost_local = topo.cost_local;
    prm.cost_intra = topo.cost_intra;
    prm.cost_inter = topo.cost_inter;
    prm.p = p;
    prm.small = (unsigned long long)T * (unsigned long long)D < (1ull << 32);
    prm.vec = k == 8 && ((reinterpret_cast<uintptr_t>(idx) | reinterpret_cast<uintptr_t>(w)) & 15u) == 0 &&
              (reinterpret_cast<uintptr_t>(kept) & 7u) == 0;
    prm.vec2 = (k & 1) == 0 && ((reinterpret_cast<uintptr_t>(idx) | reinterpret_cast<uintptr_t>(w)) & 7u) == 0;
    prm.hist = hist;
    prm.hist_stride = stride;
    prm.hist_layer = 2 * stride * D + 64;
    prm.part = part;
    const dim3 grid((unsigned)nblk, (unsigned)L);       // padding blocks (no tokens) zero their hist entries
    const size_t smem = sizeof(int) * ((size_t)E + 64);
    {
        KernelTimerScope ts("prune", st);
        // programmatic edge kept under capture (measured: config 3 step 66.5 -> 59.0 us): the kernel's launch and the
        // staging of its maps overlap the tail of whatever precedes it in the stream; it waits before its first read
        if (k <= 4) launch_pdl_edge(prune_kernel<4>, grid, dim3(PR_THREADS), smem, st, prm);
        else if (k <= 8) launch_pdl_edge(prune_kernel<8>, grid, dim3(PR_THREADS), smem, st, prm);
        else if (k <= 10) launch_pdl_edge(prune_kernel<10>, grid, dim3(PR_THREADS), smem, st, prm);   // config 5: 32 comparators per network instead of 42
        else if (k <= 12) launch_pdl_edge(prune_kernel<12>, grid, dim3(PR_THREADS), smem, st, prm);
        else launch_pdl_edge(prune_kernel<16>, grid, dim3(PR_THREADS), smem, st, prm);
    }
    note_launch();
    CAP_TRY(check_launch("prune_kernel"));
    DsReduce rd;
    rd.part = part;
    rd.red = red;
    rd.per_rb = (int32_t)((nblk + PD_MAXRB - 1) / PD_MAXRB < 64 ? 64 : (nblk + PD_MAXRB - 1) / PD_MAXRB);
    rd.nrb = (int32_t)((nblk + rd.per_rb - 1) / rd.per_rb);
    rd.acc = ew.acc;
    rd.recv = ew.recv;
    rd.nblk = nblk;
    cap_eval_out none = {};
    FinalParams fin = make_final_params(L, E, 1, expert_dev, topo, nullptr, after ? *after : none, ws, near_margin);
    return launch_dispatch_tail(idx, kept, L, T * k, E, expert_dev, D, sorted_pairs, pair_pos, offsets, hist, stride, k,
                                rd, &fin, st);
}

}  // namespace cap

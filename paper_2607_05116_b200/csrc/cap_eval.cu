// S3 -- evaluation of P candidate placements in one pass over the trace (Eq. 3, Eq. 4,
// Fig. 6 axes, Tables II-IV).  Generic kernel: a block stages a chunk of candidate maps in
// shared memory transposed ([expert][candidate] bytes, so a warp's 32 candidates read 32
// consecutive bytes), one thread owns one candidate and walks the block's tokens, building the
// token's device set as a 64-bit mask.  Scalar totals live in registers, per-device token
// counts in a shared-memory column private to the thread; both are flushed once per block.
#include "cap_eval_final.cuh"
#include "cap_internal.cuh"

namespace cap {

size_t eval_ws_bytes(int32_t L, int64_t T, int32_t E, int32_t k, int32_t D, int32_t P)
{
    size_t n = (size_t)L * P * ACC_N + (size_t)L * P * D + (size_t)L * E + (size_t)L * 64;
    return n * sizeof(unsigned long long) + 512 + eval_fast_ws_bytes(L, T, k, E, D, P);
}

EvalWs eval_ws_carve(void *ws, int32_t L, int32_t E, int32_t D, int32_t P)
{
    uintptr_t a = (reinterpret_cast<uintptr_t>(ws) + 255) & ~(uintptr_t)255;
    EvalWs w;
    w.acc = reinterpret_cast<unsigned long long *>(a);
    w.recv = w.acc + (size_t)L * P * ACC_N;
    w.mcounts = w.recv + (size_t)L * P * D;
    w.ldirect = w.mcounts + (size_t)L * E;
    return w;
}

constexpr int EV_TT = 64;   // tokens staged per step

struct EvalParams {
    const int32_t *idx;
    const uint8_t *kept;
    const int32_t *token_src;
    const int32_t *expert_dev;   // [L][P][E]
    const int32_t *dev_node;     // [D]
    unsigned long long *acc;     // [L][P][ACC_N]
    unsigned long long *recv;    // [L][P][D]
    uint8_t *tok_rdev;           // [L][P][T] or NULL
    uint8_t *tok_rnode;
    int64_t T;
    int64_t tok_per_block;
    int32_t k, E, P, D, N, PC;
};

__global__ void __launch_bounds__(256) eval_generic_kernel(EvalParams prm)
{
    extern __shared__ unsigned char smraw[];
    const int PC = prm.PC, E = prm.E, D = prm.D, N = prm.N, k = prm.k;
    // shared layout
    unsigned long long *nodemask = reinterpret_cast<unsigned long long *>(smraw);   // [64]
    int *s_idx = reinterpret_cast<int *>(nodemask + 64);                             // [EV_TT][k]
    int *s_src = s_idx + EV_TT * 16;                                                 // [EV_TT]
    int *recv_s = s_src + EV_TT;                                                     // [D][PC]
    unsigned char *s_kept = reinterpret_cast<unsigned char *>(recv_s + (size_t)D * PC);  // [EV_TT][16]
    unsigned char *s_dn = s_kept + EV_TT * 16;                                       // [64]
    unsigned char *mapT = s_dn + 64;                                                 // [E][PC]
    unsigned char *s_tok = mapT + (size_t)E * PC;                                    // [2][PC][EV_TT] (optional)

    const int layer = blockIdx.z;
    const int p0 = blockIdx.y * PC;
    const int p = p0 + threadIdx.x;
    const bool valid_p = threadIdx.x < PC && p < prm.P;
    const int64_t T = prm.T;
    const int32_t *idx = prm.idx + (int64_t)layer * T * k;
    const uint8_t *kept = prm.kept ? prm.kept + (int64_t)layer * T * k : nullptr;
    const int32_t *tsrc = prm.token_src ? prm.token_src + (int64_t)layer * T : nullptr;
    const int32_t *maps = prm.expert_dev + ((int64_t)layer * prm.P) * E;

    // ---- stage maps (transposed), node masks, zero counters ------------------------------------
    if (threadIdx.x < 64)
        s_dn[threadIdx.x] = ((int)threadIdx.x < D) ? (unsigned char)(prm.dev_node[threadIdx.x] & 63) : 0;
    for (int i = threadIdx.x; i < E * PC; i += blockDim.x) {
        int pp = i / E, e = i - pp * E;          // coalesced read of map rows
        int v = (p0 + pp < prm.P) ? maps[(int64_t)(p0 + pp) * E + e] : 0;
        mapT[(size_t)e * PC + pp] = (unsigned)v < (unsigned)D ? (unsigned char)v : (unsigned char)0;   // memory-safe on garbage
    }
    for (int i = threadIdx.x; i < D * PC; i += blockDim.x) recv_s[i] = 0;
    __syncthreads();
    if (threadIdx.x < 64) {
        unsigned long long m = 0ull;              // devices of node threadIdx.x, from the shared copy
        if ((int)threadIdx.x < N)
            for (int d = 0; d < D; ++d)
                if (s_dn[d] == (int)threadIdx.x) m |= 1ull << d;
        nodemask[threadIdx.x] = m;
    }
    __syncthreads();

    unsigned long long a_dev = 0, a_local = 0, a_same = 0, a_node = 0, a_rnode = 0;
    const int64_t t0 = (int64_t)blockIdx.x * prm.tok_per_block;
    const int64_t t1 = min(T, t0 + prm.tok_per_block);
    const bool want_tok = prm.tok_rdev != nullptr || prm.tok_rnode != nullptr;

    for (int64_t tb = t0; tb < t1; tb += EV_TT) {
        const int nt = (int)min((int64_t)EV_TT, t1 - tb);
        __syncthreads();
        for (int i = threadIdx.x; i < nt * k; i += blockDim.x) {
            int tt = i / k, s = i - tt * k;
            const int e = idx[(tb + tt) * k + s];
            s_idx[tt * 16 + s] = (unsigned)e < (unsigned)E ? e : 0;
            s_kept[tt * 16 + s] = kept ? kept[(tb + tt) * k + s] : 1;
        }
        for (int i = threadIdx.x; i < nt; i += blockDim.x)
            s_src[i] = tsrc ? (tsrc[tb + i] & 63) : (int)(((tb + i) * D) / T);   // & 63: memory-safe on garbage
        __syncthreads();
        if (valid_p) {
            for (int tt = 0; tt < nt; ++tt) {
                unsigned long long mask = 0ull;
                for (int s = 0; s < k; ++s) {
                    if (s_kept[tt * 16 + s]) {
                        int d = mapT[(size_t)s_idx[tt * 16 + s] * PC + threadIdx.x];
                        mask |= 1ull << d;
                    }
                }
                const int src = s_src[tt];
                const int sn = s_dn[src];
                const int dv = __popcll(mask);
                const int loc = (int)((mask >> src) & 1ull);
                const int same = __popcll(mask & nodemask[sn]);
                int nv = 0;
                for (int n = 0; n < N; ++n) nv += (mask & nodemask[n]) != 0ull;
                const int rn = nv - (same != 0);
                a_dev += dv;
                a_local += loc;
                a_same += same;
                a_node += nv;
                a_rnode += rn;
                unsigned long long m = mask;
                while (m) {
                    int d = __ffsll((long long)m) - 1;
                    recv_s[d * PC + threadIdx.x] += 1;
                    m &= m - 1;
                }
                if (want_tok) {
                    s_tok[(size_t)threadIdx.x * EV_TT + tt] = (unsigned char)(dv - loc);
                    s_tok[(size_t)(PC + threadIdx.x) * EV_TT + tt] = (unsigned char)rn;
                }
            }
        }
        if (want_tok) {
            __syncthreads();
            // rows of nt consecutive bytes per candidate
            for (int i = threadIdx.x; i < PC * nt; i += blockDim.x) {
                int pp = i / nt, tt = i - pp * nt;
                if (p0 + pp < prm.P) {
                    size_t o = ((size_t)layer * prm.P + (p0 + pp)) * (size_t)T + (size_t)(tb + tt);
                    if (prm.tok_rdev) prm.tok_rdev[o] = s_tok[(size_t)pp * EV_TT + tt];
                    if (prm.tok_rnode) prm.tok_rnode[o] = s_tok[(size_t)(PC + pp) * EV_TT + tt];
                }
            }
        }
    }
    if (valid_p) {
        unsigned long long *acc = prm.acc + ((size_t)layer * prm.P + p) * ACC_N;
        atomicAdd(&acc[ACC_DEV], a_dev);
        atomicAdd(&acc[ACC_LOCAL], a_local);
        atomicAdd(&acc[ACC_SAMENODE], a_same);
        atomicAdd(&acc[ACC_NODE], a_node);
        atomicAdd(&acc[ACC_RNODE], a_rnode);
        unsigned long long *rv = prm.recv + ((size_t)layer * prm.P + p) * D;
        for (int d = 0; d < D; ++d) {
            int v = recv_s[d * PC + threadIdx.x];
            if (v) atomicAdd(&rv[d], (unsigned long long)v);
        }
    }
}

// kept pairs per expert (only when the caller did not pass counts)
__global__ void __launch_bounds__(256)
masked_counts_kernel(const int32_t *__restrict__ idx, const uint8_t *__restrict__ kept, int64_t T,
                     int k, int E, unsigned long long *__restrict__ counts, int64_t tok_per_block)
{
    extern __shared__ int cnt[];
    const int layer = blockIdx.y;
    idx += (int64_t)layer * T * k;
    if (kept) kept += (int64_t)layer * T * k;
    for (int i = threadIdx.x; i < E; i += blockDim.x) cnt[i] = 0;
    __syncthreads();
    const int64_t i0 = (int64_t)blockIdx.x * tok_per_block * k;
    const int64_t i1 = min(T * k, i0 + tok_per_block * k);
    for (int64_t i = i0 + threadIdx.x; i < i1; i += blockDim.x)
        if ((!kept || kept[i]) && (unsigned)idx[i] < (unsigned)E) atomicAdd(&cnt[idx[i]], 1);
    __syncthreads();
    for (int i = threadIdx.x; i < E; i += blockDim.x)
        if (cnt[i]) atomicAdd(&counts[(size_t)layer * E + i], (unsigned long long)cnt[i]);
}

constexpr int FIN_WARPS = 4;
__global__ void __launch_bounds__(32 * FIN_WARPS) eval_finalize_kernel(FinalParams f)
{
    __shared__ unsigned long long s_lp[FIN_WARPS][64];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int o = blockIdx.x * FIN_WARPS + warp;
    pdl_launch_dependents();
    pdl_wait();
    if (o >= f.L * f.P) return;
    eval_finalize_one(f, o, lane, s_lp[warp]);
}

FinalParams make_final_params(int32_t L, int32_t E, int32_t P, const int32_t *expert_dev, const cap_topology &topo,
                              const int64_t *counts, const cap_eval_out &out, void *ws, int64_t *near_out)
{
    EvalWs w = eval_ws_carve(ws, L, E, topo.D, P);
    FinalParams f;
    f.acc = w.acc;
    f.recv = w.recv;
    f.counts = reinterpret_cast<const long long *>(counts);
    f.load_direct = nullptr;
    f.expert_dev = expert_dev;
    f.out = out;
    f.near_out = reinterpret_cast<long long *>(near_out);
    f.L = L;
    f.P = P;
    f.E = E;
    f.D = topo.D;
    f.cost_local = topo.cost_local;
    f.cost_intra = topo.cost_intra;
    f.cost_inter = topo.cost_inter;
    f.bytes_per_token = topo.bytes_per_token;
    return f;
}

// last step of every S3 path: per-candidate sums, costs, load_pairs from the counts, imbalance
int launch_eval_finalize(int32_t L, int32_t E, int32_t P, const int32_t *expert_dev, const cap_topology &topo,
                         const int64_t *counts, const cap_eval_out &out, void *ws, cudaStream_t st,
                         int64_t *near_out)
{
    const FinalParams f = make_final_params(L, E, P, expert_dev, topo, counts, out, ws, near_out);
    const int n = L * P;
    {
        KernelTimerScope ts("eval_finalize", st);
        launch_pdl(eval_finalize_kernel, dim3((unsigned)((n + FIN_WARPS - 1) / FIN_WARPS)), dim3(32 * FIN_WARPS), 0, st, f);
    }
    note_launch();
    return check_launch("eval_finalize_kernel");
}

// zero the accumulators of the evaluation workspace (acc, recv and, if wanted, mcounts)
int eval_zero_ws(int32_t L, int32_t E, int32_t D, int32_t P, bool with_mcounts, void *ws, cudaStream_t st)
{
    EvalWs w = eval_ws_carve(ws, L, E, D, P);
    const size_t zero_bytes = sizeof(unsigned long long) *
                              ((size_t)L * P * ACC_N + (size_t)L * P * D + (with_mcounts ? (size_t)L * E + (size_t)L * 64 : 0));
    if (cudaMemsetAsync(w.acc, 0, zero_bytes, st) != cudaSuccess) return check_launch("memset eval ws");
    return CAP_OK;
}

static size_t eval_smem_bytes(int E, int D, int PC, bool want_tok)
{
    return 64 * 8 + sizeof(int) * (EV_TT * 16 + EV_TT) + sizeof(int) * (size_t)D * PC + EV_TT * 16 + 64 +
           (size_t)E * PC + (want_tok ? 2 * (size_t)PC * EV_TT : 0) + 16;
}

int launch_eval(const int32_t *idx, const uint8_t *kept, const int32_t *token_src, int32_t L,
                int64_t T, int32_t k, int32_t E, const int32_t *expert_dev, int32_t P,
                int64_t /*layer_stride_maps*/, const cap_topology &topo, const int64_t *counts,
                const cap_eval_out &out, void *ws, cudaStream_t st)
{
    if (L == 0 || P == 0) return CAP_OK;
    const int D = topo.D;
    EvalWs w = eval_ws_carve(ws, L, E, D, P);
    CAP_TRY(eval_zero_ws(L, E, D, P, counts == nullptr, ws, st));

    const bool want_tok = out.tok_remote_dev || out.tok_remote_node;
    if (T > 0) {
        if (!counts) {
            int64_t want = (2 * (int64_t)sm_count() + L - 1) / L;
            int64_t tpb = (T + want - 1) / want;
            if (tpb < 1024) tpb = 1024;
            dim3 grid((unsigned)((T + tpb - 1) / tpb), (unsigned)L);
            {
                KernelTimerScope ts("masked_counts", st);
                masked_counts_kernel<<<grid, 256, sizeof(int) * (size_t)E, st>>>(idx, kept, T, k, E, w.mcounts, tpb);
            }
            note_launch();
            CAP_TRY(check_launch("masked_counts_kernel"));
        }
        bool fast = false;
        if (!want_tok) {
            CAP_TRY(launch_eval_fast(idx, kept, L, T, k, E, expert_dev, P, topo,
                                     counts ? counts : reinterpret_cast<const int64_t *>(w.mcounts), out, ws, st, &fast,
                                     token_src));
            if (fast) return CAP_OK;         // the decode kernel of the fast path writes the outputs itself
        }
        int PC = 256;
        while (PC > 32 && eval_smem_bytes(E, D, PC, want_tok) > 200 * 1024) PC >>= 1;
        if (P < PC) PC = ((P + 31) / 32) * 32;
        const size_t smem = eval_smem_bytes(E, D, PC, want_tok);
        // per device and cheap: set on every launch (a per-process flag would leave a second GPU without the opt-in)
        cudaFuncSetAttribute(eval_generic_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 220 * 1024);
        const int pchunks = (P + PC - 1) / PC;
        int64_t want = (2 * (int64_t)sm_count() + (int64_t)pchunks * L - 1) / ((int64_t)pchunks * L);
        if (want < 1) want = 1;
        int64_t tpb = (T + want - 1) / want;
        tpb = ((tpb + EV_TT - 1) / EV_TT) * EV_TT;
        if (tpb < 4 * EV_TT) tpb = 4 * EV_TT;
        EvalParams prm;
        prm.idx = idx;
        prm.kept = kept;
        prm.token_src = token_src;
        prm.expert_dev = expert_dev;
        prm.dev_node = topo.dev_node;
        prm.acc = w.acc;
        prm.recv = w.recv;
        prm.tok_rdev = out.tok_remote_dev;
        prm.tok_rnode = out.tok_remote_node;
        prm.T = T;
        prm.tok_per_block = tpb;
        prm.k = k;
        prm.E = E;
        prm.P = P;
        prm.D = D;
        prm.N = topo.N;
        prm.PC = PC;
        dim3 grid((unsigned)((T + tpb - 1) / tpb), (unsigned)pchunks, (unsigned)L);
        if (!fast) {
            {
                KernelTimerScope ts("eval", st);
                eval_generic_kernel<<<grid, PC < 64 ? 64 : PC, smem, st>>>(prm);
            }
            note_launch();
            CAP_TRY(check_launch("eval_generic_kernel"));
        }
    }
    return launch_eval_finalize(L, E, P, expert_dev, topo, counts ? counts : reinterpret_cast<const int64_t *>(w.mcounts), out, ws, st);
}

}  // namespace cap

// Last step of every S3 path (Eq. 3 costs, Eq. 4 imbalance): from the accumulated
// per-candidate sums to the caller's outputs.  A device function, so that kernels whose last block
// knows that the sums are complete (cap_prune) can finish the job without another launch.
#pragma once
#include "cap_internal.cuh"

namespace cap {

struct FinalParams {
    const unsigned long long *acc, *recv;
    const long long *counts;            // [L][E]
    const unsigned long long *load_direct;   // [L][64] pairs per device counted directly (P = 1), or NULL
    const int32_t *expert_dev;          // [L][P][E]
    cap_eval_out out;
    int32_t L, P, E, D;
    int32_t cost_local, cost_intra, cost_inter;
    long long bytes_per_token;
    long long *near_out;                // [L] <- acc[ACC_NEAR] (cap_prune with P = 1), or NULL
};

FinalParams make_final_params(int32_t L, int32_t E, int32_t P, const int32_t *expert_dev, const cap_topology &topo,
                              const int64_t *counts, const cap_eval_out &out, void *ws, int64_t *near_out);

// One warp finishes (layer, candidate) o: lanes stride over the experts (coalesced map and count
// reads), per-device sums in lp (shared memory, 64 entries of this warp), then over the devices.
// Reads go to L2 (__ldcg): the sums may have been produced by other blocks of the same launch.
// lp_ready: lp[0..63] already holds the pairs per device (the caller counted them itself).
__device__ __forceinline__ void eval_finalize_one(const FinalParams &f, int o, int lane, unsigned long long *lp,
                                                  bool lp_ready = false)
{
    const int layer = o / f.P;
    // every global load of this candidate goes out first (independent: one L2 round trip for all of them)
    const long long r0 = lane < f.D ? (long long)__ldcg(f.recv + (size_t)o * f.D + lane) : 0ll;
    const long long r1 = lane + 32 < f.D ? (long long)__ldcg(f.recv + (size_t)o * f.D + lane + 32) : 0ll;
    const unsigned long long *a = f.acc + (size_t)o * ACC_N;
    const unsigned long long av = lane < ACC_N ? __ldcg(a + lane) : 0ull;
    if (lp_ready) {
        __syncwarp();
    } else if (f.load_direct) {
        lp[lane] = __ldcg(f.load_direct + (size_t)o * 64 + lane);
        lp[lane + 32] = __ldcg(f.load_direct + (size_t)o * 64 + lane + 32);
    } else {
        lp[lane] = 0ull;
        lp[lane + 32] = 0ull;
        __syncwarp();
        // load_pairs[d] = sum of the (kept) counts of the experts placed on d
        const int32_t *pi = f.expert_dev + (size_t)o * f.E;
        const long long *cnt = f.counts + (size_t)layer * f.E;
        for (int e = lane; e < f.E; e += 32) {
            const int d = pi[e];
            const long long c = __ldcg(cnt + e);
            if (d >= 0 && d < f.D && c) atomicAdd(&lp[d], (unsigned long long)c);
        }
    }
    __syncwarp();
    long long mx = 0, sm = 0, mxr = 0, smr = 0;
    for (int d = lane; d < f.D; d += 32) {
        const long long l = (long long)lp[d];
        const long long r = d < 32 ? r0 : r1;
        if (f.out.load_pairs) f.out.load_pairs[(size_t)o * f.D + d] = l;
        if (f.out.recv_tokens) f.out.recv_tokens[(size_t)o * f.D + d] = r;
        mx = max(mx, l);
        sm += l;
        mxr = max(mxr, r);
        smr += r;
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, off));
        mxr = max(mxr, __shfl_xor_sync(0xffffffffu, mxr, off));
        sm += __shfl_xor_sync(0xffffffffu, sm, off);
        smr += __shfl_xor_sync(0xffffffffu, smr, off);
    }
    const long long dv = (long long)__shfl_sync(0xffffffffu, av, ACC_DEV), loc = (long long)__shfl_sync(0xffffffffu, av, ACC_LOCAL),
                    same = (long long)__shfl_sync(0xffffffffu, av, ACC_SAMENODE);
    const long long a_node = (long long)__shfl_sync(0xffffffffu, av, ACC_NODE), a_rnode = (long long)__shfl_sync(0xffffffffu, av, ACC_RNODE),
                    a_near = (long long)__shfl_sync(0xffffffffu, av, ACC_NEAR);
    if (lane != 0) return;
    const long long rdev = dv - loc, intra = same - loc, inter = dv - same;
    if (f.near_out) f.near_out[o] = a_near;
    if (f.out.dev_visits) f.out.dev_visits[o] = dv;
    if (f.out.remote_dev) f.out.remote_dev[o] = rdev;
    if (f.out.remote_intra) f.out.remote_intra[o] = intra;
    if (f.out.remote_inter) f.out.remote_inter[o] = inter;
    if (f.out.node_visits) f.out.node_visits[o] = a_node;
    if (f.out.remote_node) f.out.remote_node[o] = a_rnode;
    if (f.out.cost)
        f.out.cost[o] = (long long)f.cost_local * loc + (long long)f.cost_intra * intra +
                        (long long)f.cost_inter * inter;
    if (f.out.bytes) f.out.bytes[o] = rdev * f.bytes_per_token;
    if (f.out.imbalance) f.out.imbalance[o] = sm ? __ddiv_rn((double)(mx * f.D), (double)sm) : 0.0;
    if (f.out.imbalance_recv)
        f.out.imbalance_recv[o] = smr ? __ddiv_rn((double)(mxr * f.D), (double)smr) : 0.0;
}

}  // namespace cap

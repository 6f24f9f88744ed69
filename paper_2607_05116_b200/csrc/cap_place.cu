// cap_coact_placement: co-activation probabilities p_ij (reading R3: Jaccard) and
// Algorithm 1 of the paper in both stages: experts -> D device groups,
// then device groups -> N node groups (reading R24 for the group strength).
//
// The method is E - D dependent greedy steps per layer (each an arg-max over the unassigned
// experts followed by a rank-1 update of one group's scores), so the parallelism is
//   - one CTA per layer (the 48-58 layers of configs 2 and 4 fill a third of the SMs),
//   - one thread per expert inside the CTA: a step is one coalesced read of a row of the
//     (transposed) probability matrix from L2, one warp-shuffle arg-max and one __syncthreads.
// Every fp64 value is produced by the same IEEE operations in the same order as the definition
// (ascending-j degree sums, scores summed in joining order), so all outputs are reproducible
// bit for bit; the "uniformly at random" branch of line 12 consumes caller-supplied numbers.
#include <climits>

#include "cap_internal.cuh"

namespace cap {
namespace {

struct Best {
    double v;
    int e;
};

__device__ __forceinline__ Best better(Best a, Best b)   // larger score, ties -> lower index (R23)
{
    return (b.v > a.v || (b.v == a.v && b.e < a.e)) ? b : a;
}

__device__ __forceinline__ Best warp_best(Best x)
{
#pragma unroll
    for (int o = 16; o; o >>= 1) {
        Best y;
        y.v = __shfl_xor_sync(0xffffffffu, x.v, o);
        y.e = __shfl_xor_sync(0xffffffffu, x.e, o);
        x = better(x, y);
    }
    return x;
}

struct PlaceSmem {
    double deg[1024];
    int grp[1024], ord[1024], members[1024];
    int grp2[64], ord2[64], seeds[64], gsize[64];
    double pv[2][32];
    int pe[2][32];
    int wcnt[32];
    int pick;
};

// Algorithm 1 on n units and k groups.  MT[m * n + e] = M[e][m] (so that a step reads one
// contiguous row); score is [k][n] scratch in global memory, each element touched by one thread.
__device__ void alg1(int n, int k, const double *MT, double *score, const uint32_t *rnd, int *grp, int *ord,
                     PlaceSmem &sm)
{
    const int e = threadIdx.x, lane = e & 31, wid = e >> 5, nw = blockDim.x >> 5;
    double d = 0.0;
    if (e < n) {                                              // line 1: ascending j, j != e
        for (int j = 0; j < n; ++j)
            if (j != e) d += MT[(size_t)j * n + e];
        sm.deg[e] = d;
    }
    __syncthreads();
    bool inU = e < n;
    if (e < n) {                                              // line 4 as a rank; lines 5-7
        int rank = 0;
        for (int j = 0; j < n; ++j) {
            double dj = sm.deg[j];
            rank += (dj > d || (dj == d && j < e)) ? 1 : 0;
        }
        if (rank < k) {
            grp[e] = rank;
            ord[e] = 0;
            sm.seeds[rank] = e;
            sm.gsize[rank] = 1;
            inU = false;
        }
    }
    __syncthreads();
    if (e < n)
        for (int g = 0; g < k; ++g) score[(size_t)g * n + e] = 0.0 + MT[(size_t)sm.seeds[g] * n + e];
    const int steps = n - k;
    for (int step = 0; step < steps; ++step) {                // line 8
        const int g = step % k, par = step & 1;               // line 14
        Best b;
        b.v = inU ? score[(size_t)g * n + e] : -1.0;
        b.e = inU ? e : INT_MAX;
        b = warp_best(b);                                     // lines 9-10
        if (lane == 0) {
            sm.pv[par][wid] = b.v;
            sm.pe[par][wid] = b.e;
        }
        __syncthreads();
        Best c;
        c.v = lane < nw ? sm.pv[par][lane] : -1.0;
        c.e = lane < nw ? sm.pe[par][lane] : INT_MAX;
        c = warp_best(c);
        int pick = c.e;
        if (c.v == 0.0) {                                     // lines 11-12 (block-uniform branch)
            uint32_t r = (rnd ? rnd[step] : 0u) % (uint32_t)(steps - step);
            unsigned bal = __ballot_sync(0xffffffffu, inU);
            if (lane == 0) sm.wcnt[wid] = __popc(bal);
            __syncthreads();
            int pre = __popc(bal & ((1u << lane) - 1u));
            for (int w = 0; w < wid; ++w) pre += sm.wcnt[w];
            if (inU && pre == (int)r) sm.pick = e;
            __syncthreads();
            pick = sm.pick;
        }
        if (e == pick) {                                      // line 13
            inU = false;
            grp[e] = g;
            ord[e] = sm.gsize[g];
            sm.gsize[g] += 1;
        }
        if (inU) score[(size_t)g * n + e] += MT[(size_t)pick * n + e];
    }
    __syncthreads();
}

__global__ void __launch_bounds__(1024, 1)
place_kernel(const int64_t *__restrict__ counts, const int32_t *__restrict__ coact, int E, int D, int N,
             const uint32_t *__restrict__ rnd, double *p_out, double *wsP, double *wsS, double *wsW,
             int32_t *expert_group, int32_t *group_node, int32_t *expert_dev)
{
    __shared__ PlaceSmem sm;
    const int l = blockIdx.x, tid = threadIdx.x;
    const int64_t *n = counts + (size_t)l * E;
    const int32_t *C = coact + (size_t)l * E * E;
    double *pT = wsP + (size_t)l * E * E;
    double *score = wsS + (size_t)l * D * E;
    double *WT = wsW + (size_t)l * D * D;
    double *po = p_out ? p_out + (size_t)l * E * E : nullptr;
    const uint32_t *r1 = rnd ? rnd + (size_t)l * (E + D) : nullptr;

    // p_ij = C_ij / (n_i + n_j - C_ij): exact int -> double conversions, one IEEE divide (R3)
    for (int q = tid; q < E * E; q += blockDim.x) {
        int i = q / E, j = q - i * E;
        long long c = C[q];
        long long den = n[i] + n[j] - c;
        double v = (i == j || den == 0) ? 0.0 : __ddiv_rn((double)c, (double)den);
        if (po) po[q] = v;
        pT[(size_t)j * E + i] = v;
    }
    __syncthreads();
    alg1(E, D, pT, score, r1, sm.grp, sm.ord, sm);

    // stage 2 (R24): W[a][b] = sum over i in G[a] (ascending), j in G[b] (ascending) of p_ij
    const int m = E / D;
    if (tid < D) {
        int r = 0;
        for (int e = 0; e < E; ++e)
            if (sm.grp[e] == tid) sm.members[tid * m + r++] = e;
    }
    __syncthreads();
    for (int q = tid; q < D * D; q += blockDim.x) {
        int a = q / D, b = q - a * D;
        double s = 0.0;
        if (a != b)
            for (int x = 0; x < m; ++x) {
                int i = sm.members[a * m + x];
                for (int y = 0; y < m; ++y) s += pT[(size_t)sm.members[b * m + y] * E + i];
            }
        WT[(size_t)b * D + a] = s;
    }
    __syncthreads();
    alg1(D, N, WT, score, r1 ? r1 + E : nullptr, sm.grp2, sm.ord2, sm);

    if (tid < E) {
        int g = sm.grp[tid];
        expert_group[(size_t)l * E + tid] = g;
        expert_dev[(size_t)l * E + tid] = sm.grp2[g] * (D / N) + sm.ord2[g];
    }
    if (tid < D) group_node[(size_t)l * D + tid] = sm.grp2[tid];
}

}  // namespace

size_t place_ws_bytes(int32_t L, int32_t E, int32_t D)
{
    return (size_t)L * ((size_t)E * E + (size_t)D * E + (size_t)D * D) * sizeof(double) + 256;
}

int launch_place(const int64_t *counts, const int32_t *coact, int32_t L, int32_t E, int32_t D, int32_t N,
                 const uint32_t *rnd, double *p_out, int32_t *expert_group, int32_t *group_node,
                 int32_t *expert_dev, void *ws, cudaStream_t st)
{
    if (L == 0) return CAP_OK;
    double *wsP = (double *)(((uintptr_t)ws + 255) & ~(uintptr_t)255);
    double *wsS = wsP + (size_t)L * E * E;
    double *wsW = wsS + (size_t)L * D * E;
    int threads = ((E > 64 ? E : 64) + 31) & ~31;
    KernelTimerScope kt("coact_placement", st);
    place_kernel<<<L, threads, 0, st>>>(counts, coact, E, D, N, rnd, p_out, wsP, wsS, wsW, expert_group,
                                        group_node, expert_dev);
    note_launch();
    return check_launch("place_kernel");
}

}  // namespace cap

extern "C" int cap_coact_placement(const int64_t *counts, const int32_t *coact, int32_t L, int32_t E, int32_t D,
                                   int32_t N, const uint32_t *rnd, double *p_out, int32_t *expert_group,
                                   int32_t *group_node, int32_t *expert_dev, void *ws, size_t ws_bytes,
                                   void *stream)
{
    if (L < 0 || L > 65535 || E < 1 || E > 1024 || D < 1 || D > 64 || N < 1 || N > 64) return CAP_EINVAL;
    if (E % D != 0 || D % N != 0) return CAP_EINVAL;
    if (L > 0 && (!counts || !coact || !expert_group || !group_node || !expert_dev)) return CAP_EINVAL;
    if (!ws || ws_bytes < cap::place_ws_bytes(L, E, D)) return CAP_EWORKSPACE;
    return cap::launch_place(counts, coact, L, E, D, N, rnd, p_out, expert_group, group_node, expert_dev, ws,
                             (cudaStream_t)stream);
}

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

// Arg-max of non-negative doubles over a warp, ties -> lowest lane (= lowest index, R23).  The bit
// pattern of a non-negative double orders like the value, so the maximum is two 32-bit REDUX
// operations (high word, then low word among the lanes that hold the largest high word) and one
// ballot.  Lanes outside U pass hi = -1.  Returns the winning lane; *mh / *ml = the maximum's words.
__device__ __forceinline__ int warp_argmax(int hi, unsigned lo, int *mh, unsigned *ml)
{
    int h = __reduce_max_sync(0xffffffffu, hi);
    unsigned l = __reduce_max_sync(0xffffffffu, hi == h ? lo : 0u);
    unsigned bal = __ballot_sync(0xffffffffu, hi == h && lo == l);
    *mh = h;
    *ml = l;
    return __ffs(bal) - 1;
}

struct PlaceSmem {
    long long cnt[1024];
    double deg[1024];
    int grp[1024], ord[1024], members[1024];
    int grp2[64], ord2[64], seeds[64], gsize[64];
    int ph[2][32];
    unsigned pl[2][32];
    int pe[2][32];
    int wcnt[32];
    int pick;
};

// File-scope shared state: every access below is then a direct shared-memory access.  With the struct and
// the score rows passed as pointers the compiler formed generic addresses, which costs a read of the CTA's
// cluster rank (S2R SR_CgaCtaId) inside every greedy step.
__shared__ PlaceSmem sm;
extern __shared__ double sscore[];

// Algorithm 1 on n units and k groups.  MT[m * n + e] = M[e][m] (so that a step reads one
// contiguous row); score is [k][n] scratch in global memory, each element touched by one thread.
// The scores of groups g < gs live in shared memory (sscore), the rest in global memory (score):
// a global store does not allocate in L1, so a global score costs an L2 round trip per step.
template <bool STAGE2>
__device__ __forceinline__ void alg1(int n, int k, const double *MT, double *score, int gs, const uint32_t *rnd)
{
    int *const grp = STAGE2 ? sm.grp2 : sm.grp;
    int *const ord = STAGE2 ? sm.ord2 : sm.ord;
    const int e = threadIdx.x, lane = e & 31, wid = e >> 5;
    double d = 0.0;
    if (e < n) {                                              // line 1: ascending j, j != e
#pragma unroll 16
        for (int j = 0; j < n; ++j) {
            double x = MT[(size_t)j * n + e];
            if (j != e) d += x;
        }
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
        for (int g = 0; g < k; ++g) {
            double x = 0.0 + MT[(size_t)sm.seeds[g] * n + e];
            if (g < gs) sscore[g * n + e] = x;
            else score[(size_t)g * n + e] = x;
        }
    const int steps = n - k;
    // The rank-1 update of group g's scores (line 13's effect on line 9) is next needed k steps later, so
    // the row of MT loaded in step s is added in step s + depth (depth = 4 when k >= 5, 1 when k >= 2,
    // 0 when k = 1): a step is ~300 cycles, an L2 row read ~800, and this takes the read off the step's
    // dependent chain without changing any operand or the order of the additions to a score.
    const int depth = k >= 5 ? 4 : (k >= 2 ? 1 : 0);
    double m0 = 0.0, m1 = 0.0, m2 = 0.0, m3 = 0.0;
    int g0 = -1, g1 = -1, g2 = -1, g3 = -1;                   // oldest first
    // only the warps that own units take part in the greedy loop (named barrier 1 over nwa warps); the
    // others wait at the __syncthreads() after it
    const int nwa = (n + 31) >> 5;
    int g = 0;
    for (int step = 0; wid < nwa && step < steps; ++step, g = (g + 1 == k) ? 0 : g + 1) {   // lines 8, 14
        const int par = step & 1;
        double v = 0.0;
        if (inU) v = g < gs ? sscore[g * n + e] : score[(size_t)g * n + e];
        int mh, wh;
        unsigned ml, wl;
        int src = warp_argmax(inU ? __double2hiint(v) : -1, (unsigned)__double2loint(v), &mh, &ml);   // lines 9-10
        if (lane == 0) {
            sm.ph[par][wid] = mh;
            sm.pl[par][wid] = ml;
            sm.pe[par][wid] = (wid << 5) + src;
        }
        asm volatile("bar.sync 1, %0;" ::"r"(nwa * 32) : "memory");
        int src2 = warp_argmax(lane < nwa ? sm.ph[par][lane] : -1, lane < nwa ? sm.pl[par][lane] : 0u, &wh, &wl);
        int pick = sm.pe[par][src2];
        if (wh == 0 && wl == 0u) {                            // lines 11-12 (block-uniform branch)
            uint32_t r = (rnd ? rnd[step] : 0u) % (uint32_t)(steps - step);
            unsigned bal = __ballot_sync(0xffffffffu, inU);
            if (lane == 0) sm.wcnt[wid] = __popc(bal);
            asm volatile("bar.sync 1, %0;" ::"r"(nwa * 32) : "memory");
            int pre = __popc(bal & ((1u << lane) - 1u));
            for (int w = 0; w < wid; ++w) pre += sm.wcnt[w];
            if (inU && pre == (int)r) sm.pick = e;
            asm volatile("bar.sync 1, %0;" ::"r"(nwa * 32) : "memory");
            pick = sm.pick;
        }
        if (e == pick) {                                      // line 13
            inU = false;
            grp[e] = g;
            ord[e] = sm.gsize[g];
            sm.gsize[g] += 1;
        }
        if (e < n) {
            double mnew = MT[(size_t)pick * n + e];
            double ma;
            int ga;
            if (depth == 4) {
                ma = m0; ga = g0;
                m0 = m1; g0 = g1;
                m1 = m2; g1 = g2;
                m2 = m3; g2 = g3;
                m3 = mnew; g3 = g;
            } else if (depth == 1) {
                ma = m3; ga = g3;
                m3 = mnew; g3 = g;
            } else {
                ma = mnew; ga = g;
            }
            if (ga >= 0) {
                if (ga < gs) sscore[ga * n + e] += ma;
                else score[(size_t)ga * n + e] += ma;
            }
        }
    }
    __syncthreads();
}

__global__ void __launch_bounds__(1024, 1)
place_kernel(const int64_t *__restrict__ counts, const int32_t *__restrict__ coact, int E, int D, int N,
             const uint32_t *__restrict__ rnd, double *p_out, double *wsP, double *wsS, double *wsW,
             int32_t *expert_group, int32_t *group_node, int32_t *expert_dev, int gs1)
{
    const int l = blockIdx.x, tid = threadIdx.x;
    const int64_t *n = counts + (size_t)l * E;
    const int32_t *C = coact + (size_t)l * E * E;
    double *pT = wsP + (size_t)l * E * E;
    double *score = wsS + (size_t)l * D * E;
    double *WT = wsW + (size_t)l * D * D;
    double *po = p_out ? p_out + (size_t)l * E * E : nullptr;
    const uint32_t *r1 = rnd ? rnd + (size_t)l * (E + D) : nullptr;

    // p_ij = C_ij / (n_i + n_j - C_ij): exact int -> double conversions, one IEEE divide (R3)
    for (int e = tid; e < E; e += blockDim.x) sm.cnt[e] = n[e];
    __syncthreads();
#pragma unroll 4
    for (int q = tid; q < E * E; q += blockDim.x) {
        int i = q / E, j = q - i * E;
        long long c = C[q];
        long long den = sm.cnt[i] + sm.cnt[j] - c;
        double v = (i == j || den == 0) ? 0.0 : __ddiv_rn((double)c, (double)den);
        if (po) po[q] = v;
        pT[q] = v;                           // coact is symmetric (cap.h), so p is its own transpose
    }
    __syncthreads();
    alg1<false>(E, D, pT, score, gs1, r1);

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
#pragma unroll 8
                for (int y = 0; y < m; ++y) s += pT[(size_t)sm.members[b * m + y] * E + i];
            }
        WT[(size_t)b * D + a] = s;
    }
    __syncthreads();
    alg1<true>(D, N, WT, score, N, r1 ? r1 + E : nullptr);

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
    // at least 512 threads: the E^2 prologue (probabilities, degrees' operands) is latency-bound and wants
    // the memory-level parallelism; threads beyond E only take part in the barriers of the greedy loop
    int threads = ((E > 512 ? E : 512) + 31) & ~31;
    // shared-memory score rows: as many groups as fit in 192 KB beside the static 30 KB
    int gs1 = (int)((size_t)196608 / ((size_t)E * sizeof(double)));
    if (gs1 > D) gs1 = D;
    size_t dyn = (size_t)gs1 * E * sizeof(double);
    if (dyn < (size_t)N * D * sizeof(double)) dyn = (size_t)N * D * sizeof(double);
    // per device and cheap: set on every launch (a per-process flag would leave a second GPU without the opt-in)
    if (cudaFuncSetAttribute(place_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 196608) != cudaSuccess)
        return check_launch("place_kernel attribute");
    KernelTimerScope kt("coact_placement", st);
    place_kernel<<<L, threads, dyn, st>>>(counts, coact, E, D, N, rnd, p_out, wsP, wsS, wsW, expert_group,
                                          group_node, expert_dev, gs1);
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

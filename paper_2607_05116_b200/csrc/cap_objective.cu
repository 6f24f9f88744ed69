// cap_pairwise_objective: the paper's communication objective C(pi) = sum_{i<j} p_ij d(pi(i), pi(j))
// (Eq. 2-3) for P candidate placements from the co-activation statistics alone, with the
// integer counts C_ij (exact int64) and the probabilities p_ij (R3, fp64) as weights, plus Eq. 5's
// scalarisation with a caller-supplied imbalance.
//
// Work is P * E^2 / 2 pair evaluations over an E x E matrix that stays in L2 (1 MB of int32 at E = 512):
// a block scores PC (8, fewer for small P) candidates per pass over the matrix (coalesced row-major reads, the (device,
// node) codes of its candidates in shared memory), so the matrix is read P / 8 times from L2 and once
// from HBM.  Bound: fp64 / integer ALU (one divide per pair and block, 8 select-multiply-adds).
#include "cap_internal.cuh"

namespace cap {
namespace {

constexpr int OBJ_THREADS = 512;

template <int PC>   // candidates per block
__global__ void __launch_bounds__(OBJ_THREADS)
objective_kernel(const int64_t *__restrict__ counts, const int32_t *__restrict__ coact, int E,
                 const int32_t *__restrict__ expert_dev, int P, int D, const int32_t *__restrict__ dev_node,
                 int cost_intra, int cost_inter, double lambda, const double *__restrict__ imbalance,
                 int64_t *obj_count, double *obj_prob, double *combined)
{
    __shared__ uint16_t code[PC][1024];      // device | node << 8 of every expert under each candidate
    __shared__ long long cnt[1024];
    __shared__ long long rc[OBJ_THREADS / 32][PC];
    __shared__ double rp[OBJ_THREADS / 32][PC];
    const int l = blockIdx.y, p0 = blockIdx.x * PC, tid = threadIdx.x;
    const int np = min(PC, P - p0);
    const int32_t *C = coact + (size_t)l * E * E;
    for (int q = tid; q < PC * E; q += OBJ_THREADS) {
        int c = q / E, e = q - c * E;
        int d = c < np ? expert_dev[((size_t)l * P + p0 + c) * E + e] : 0;
        d = min(max(d, 0), D - 1);           // memory-safe on garbage maps
        code[c][e] = (uint16_t)(d | (dev_node[d] << 8));
    }
    for (int e = tid; e < E; e += OBJ_THREADS) cnt[e] = counts[(size_t)l * E + e];
    __syncthreads();

    long long ac[PC];
    double ap[PC];
#pragma unroll
    for (int c = 0; c < PC; ++c) {
        ac[c] = 0;
        ap[c] = 0.0;
    }
    // Upper triangle only, folded so that every folded row has E - 1 entries: folded row r holds row r's
    // E - 1 - r entries (j > r) followed by row E - 1 - r's r entries; contiguous runs, so the reads stay
    // coalesced.  Latency-bound L2 reads: the loads of four iterations are issued together.
    const int W1 = E - 1, R = (E + 1) >> 1;
#pragma unroll 4
    for (int q = tid; q < R * W1; q += OBJ_THREADS) {
        int r = q / W1, cc = q - r * W1;
        int i, j;
        if (cc < W1 - r) {
            i = r;
            j = r + 1 + cc;
        } else {
            i = W1 - r;
            j = i + 1 + (cc - (W1 - r));
        }
        bool ok = cc < W1 - r || 2 * r != W1;   // odd E: the middle row is its own partner, count it once
        long long c = ok ? C[(size_t)i * E + j] : 0;
        if (c == 0) continue;                // c = 0 means p_ij = 0 as well
        long long den = cnt[i] + cnt[j] - c;
        double pij = den == 0 ? 0.0 : __ddiv_rn((double)c, (double)den);
#pragma unroll
        for (int k = 0; k < PC; ++k) {
            unsigned a = code[k][i], b = code[k][j];
            int d = a == b ? 0 : ((a >> 8) == (b >> 8) ? cost_intra : cost_inter);
            ac[k] += c * d;
            ap[k] += pij * (double)d;
        }
    }
    const int lane = tid & 31, wid = tid >> 5;
#pragma unroll
    for (int k = 0; k < PC; ++k) {
        long long x = ac[k];
        double y = ap[k];
#pragma unroll
        for (int o = 16; o; o >>= 1) {
            x += __shfl_xor_sync(0xffffffffu, x, o);
            y += __shfl_xor_sync(0xffffffffu, y, o);
        }
        if (lane == 0) {
            rc[wid][k] = x;
            rp[wid][k] = y;
        }
    }
    __syncthreads();
    if (tid < np) {
        long long x = 0;
        double y = 0.0;
        for (int w = 0; w < OBJ_THREADS / 32; ++w) {
            x += rc[w][tid];
            y += rp[w][tid];
        }
        size_t o = (size_t)l * P + p0 + tid;
        if (obj_count) obj_count[o] = x;
        if (obj_prob) obj_prob[o] = y;
        if (combined && imbalance) combined[o] = lambda * y + (1.0 - lambda) * imbalance[o];
    }
}

}  // namespace
}  // namespace cap

extern "C" int cap_pairwise_objective(const int64_t *counts, const int32_t *coact, int32_t L, int32_t E,
                                      const int32_t *expert_dev, int32_t P, const cap_topology *topo, double lambda,
                                      const double *imbalance, int64_t *obj_count, double *obj_prob,
                                      double *combined, void *stream)
{
    using namespace cap;
    if (L < 0 || L > 65535 || E < 1 || E > 1024 || P < 0 || !topo) return CAP_EINVAL;
    if (topo->D < 1 || topo->D > 64 || topo->N < 1 || topo->N > 64 || !topo->dev_node) return CAP_EINVAL;
    if (topo->cost_intra < 0 || topo->cost_inter < 0) return CAP_EINVAL;
    if ((int64_t)L * P > 0 && (!counts || !coact || !expert_dev)) return CAP_EINVAL;
    if (combined && !imbalance) return CAP_EINVAL;
    if (L == 0 || P == 0) return CAP_OK;
    cudaStream_t st = (cudaStream_t)stream;
    KernelTimerScope kt("objective", st);
    // 8 candidates per block amortise the pass over the matrix; fewer when that would leave SMs idle
    const long long want = sm_count();
    int pc = 8;
    while (pc > 1 && (long long)((P + pc - 1) / pc) * L < want) pc >>= 1;
#define CAP_OBJ_LAUNCH(PCV)                                                                                      \
    objective_kernel<PCV><<<dim3((P + PCV - 1) / PCV, L), OBJ_THREADS, 0, st>>>(                                  \
        counts, coact, E, expert_dev, P, topo->D, topo->dev_node, topo->cost_intra, topo->cost_inter, lambda,    \
        imbalance, obj_count, obj_prob, combined)
    if (pc == 8) CAP_OBJ_LAUNCH(8);
    else if (pc == 4) CAP_OBJ_LAUNCH(4);
    else if (pc == 2) CAP_OBJ_LAUNCH(2);
    else CAP_OBJ_LAUNCH(1);
#undef CAP_OBJ_LAUNCH
    note_launch();
    return check_launch("objective_kernel");
}

// cap_adjust_spectrum: the Adjustment Approach of P:L194 (reading R27 in DESIGN.md): S dependent swap
// steps per layer, each moving one expert from the most loaded to the least loaded device and one back,
// chosen among the load-reducing pairs by the smallest loss of co-activation locality (integer, exact).
// One CTA per layer, one thread per expert; per step: shared-memory load histogram, hot / cold pick,
// ballot-compacted member lists (ascending), per-member affinities to both devices, one thread per
// candidate pair, block arg-min on (loss, pair index).  Latency-bound like Algorithm 1; all integer.
#include <climits>

#include "cap_internal.cuh"

namespace cap {
namespace {

struct AdjSmem {
    int pi[1024];
    int hotm[1024], coldm[1024];                 // members, ascending
    long long affH[1024], affC[1024];            // by expert id: sum of C to the hot / cold members (v != x)
    unsigned long long load[64];
    int wcH[32], wcC[32];
    long long rl[32];
    int rq[32];
    int hot, cold, nH, nC, bestq;
};

__global__ void __launch_bounds__(1024, 1)
adjust_kernel(const int64_t *__restrict__ counts, const int32_t *__restrict__ coact, int E, int D,
              const int32_t *__restrict__ pi0, int S, int32_t *spectrum, int32_t *n_done, int32_t *swaps)
{
    __shared__ AdjSmem sm;
    const int l = blockIdx.x, e = threadIdx.x, lane = e & 31, wid = e >> 5, nw = blockDim.x >> 5;
    const int32_t *C = coact + (size_t)l * E * E;
    const long long ne = e < E ? counts[(size_t)l * E + e] : 0;
    if (e < E) sm.pi[e] = min(max(pi0[(size_t)l * E + e], 0), D - 1);
    int done = S;
    bool stopped = false;
    for (int s = 0; s < S; ++s) {
        int besta = -1, bestb = -1;
        if (!stopped) {                                          // block-uniform
            if (e < 64) sm.load[e] = 0ull;
            __syncthreads();
            if (e < E) atomicAdd(&sm.load[sm.pi[e]], (unsigned long long)ne);
            __syncthreads();
            if (e == 0) {
                int hot = 0, cold = 0;
                for (int d = 1; d < D; ++d) {
                    if (sm.load[d] > sm.load[hot]) hot = d;
                    if (sm.load[d] < sm.load[cold]) cold = d;
                }
                sm.hot = hot;
                sm.cold = cold;
            }
            __syncthreads();
            const int hot = sm.hot, cold = sm.cold;
            const int mine = e < E ? sm.pi[e] : -1;
            const bool isH = mine == hot, isC = mine == cold && hot != cold;
            unsigned bh = __ballot_sync(0xffffffffu, isH), bcl = __ballot_sync(0xffffffffu, isC);
            if (lane == 0) {
                sm.wcH[wid] = __popc(bh);
                sm.wcC[wid] = __popc(bcl);
            }
            __syncthreads();
            int ph = __popc(bh & ((1u << lane) - 1u)), pc = __popc(bcl & ((1u << lane) - 1u));
            int th = 0, tc = 0;
            for (int w = 0; w < nw; ++w) {
                if (w < wid) {
                    ph += sm.wcH[w];
                    pc += sm.wcC[w];
                }
                th += sm.wcH[w];
                tc += sm.wcC[w];
            }
            if (isH) sm.hotm[ph] = e;
            if (isC) sm.coldm[pc] = e;
            if (e == 0) {
                sm.nH = th;
                sm.nC = tc;
            }
            __syncthreads();
            const int nH = sm.nH, nC = sm.nC;
            if (isH || isC) {                                    // affinities of the members
                long long ah = 0, ac = 0;
                for (int x = 0; x < nH; ++x) {
                    int v = sm.hotm[x];
                    if (v != e) ah += C[(size_t)e * E + v];
                }
                for (int x = 0; x < nC; ++x) {
                    int v = sm.coldm[x];
                    if (v != e) ac += C[(size_t)e * E + v];
                }
                sm.affH[e] = ah;
                sm.affC[e] = ac;
            }
            __syncthreads();
            const long long gap = (long long)(sm.load[hot] - sm.load[cold]);
            long long bl = LLONG_MAX;
            int bq = INT_MAX;
            for (int q = e; q < nH * nC; q += blockDim.x) {      // q ascending = (a, b) lexicographic
                int a = sm.hotm[q / nC], b = sm.coldm[q % nC];
                long long delta = counts[(size_t)l * E + a] - counts[(size_t)l * E + b];
                if (delta <= 0 || delta >= gap) continue;
                long long cab = C[(size_t)a * E + b], cba = C[(size_t)b * E + a];
                // aff(a, hot\a) + aff(b, cold\b) - aff(a, cold\b) - aff(b, hot\a)
                long long loss = sm.affH[a] + sm.affC[b] - (sm.affC[a] - cab) - (sm.affH[b] - cba);
                if (loss < bl) {
                    bl = loss;
                    bq = q;
                }
            }
#pragma unroll
            for (int o = 16; o; o >>= 1) {
                long long ol = __shfl_xor_sync(0xffffffffu, bl, o);
                int oq = __shfl_xor_sync(0xffffffffu, bq, o);
                if (ol < bl || (ol == bl && oq < bq)) {
                    bl = ol;
                    bq = oq;
                }
            }
            if (lane == 0) {
                sm.rl[wid] = bl;
                sm.rq[wid] = bq;
            }
            __syncthreads();
            if (e == 0) {
                long long xl = LLONG_MAX;
                int xq = INT_MAX;
                for (int w = 0; w < nw; ++w)
                    if (sm.rl[w] < xl || (sm.rl[w] == xl && sm.rq[w] < xq)) {
                        xl = sm.rl[w];
                        xq = sm.rq[w];
                    }
                sm.bestq = xq;
                if (xq != INT_MAX) {
                    int a = sm.hotm[xq / nC], b = sm.coldm[xq % nC];
                    sm.pi[a] = cold;
                    sm.pi[b] = hot;
                }
            }
            __syncthreads();
            if (sm.bestq == INT_MAX) {
                stopped = true;
                done = s;
            } else {
                besta = sm.hotm[sm.bestq / nC];
                bestb = sm.coldm[sm.bestq % nC];
            }
        }
        if (e < E) spectrum[((size_t)l * S + s) * E + e] = sm.pi[e];
        if (swaps && e == 0) {
            swaps[((size_t)l * S + s) * 2] = besta;
            swaps[((size_t)l * S + s) * 2 + 1] = bestb;
        }
        __syncthreads();
    }
    if (n_done && e == 0) n_done[l] = done;
}

}  // namespace
}  // namespace cap

extern "C" int cap_adjust_spectrum(const int64_t *counts, const int32_t *coact, int32_t L, int32_t E, int32_t D,
                                   const int32_t *expert_dev0, int32_t S, int32_t *spectrum, int32_t *n_done,
                                   int32_t *swaps, void *stream)
{
    using namespace cap;
    if (L < 0 || L > 65535 || E < 1 || E > 1024 || D < 1 || D > 64 || S < 0) return CAP_EINVAL;
    if ((int64_t)L * S > 0 && (!counts || !coact || !expert_dev0 || !spectrum)) return CAP_EINVAL;
    if (L == 0 || S == 0) return CAP_OK;
    cudaStream_t st = (cudaStream_t)stream;
    int threads = ((E > 64 ? E : 64) + 31) & ~31;
    KernelTimerScope kt("adjust", st);
    adjust_kernel<<<L, threads, 0, st>>>(counts, coact, E, D, expert_dev0, S, spectrum, n_done, swaps);
    note_launch();
    return check_launch("adjust_kernel");
}

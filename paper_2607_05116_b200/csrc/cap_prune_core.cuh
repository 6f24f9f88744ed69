// S4, the per-token part (Eq. 6 and its greedy solver; readings R7-R10, R13), shared by the kernels
// of cap_prune.cu and cap_prune_dispatch.cu.  One thread per token, everything in registers, no branches that
// depend on the token (the warp's tokens diverge everywhere: selects only):
//   1. the slots are put in (device, slot) order by a sorting network; a running sum over that order gives every
//      device's weight at the LAST slot of its run, added in slot order (fp32, single IEEE adds);
//   2. each device is priced by topology relative to the token's source (R7, R13): ratio = a_d / c_d;
//   3. a second network orders the devices by ratio descending, ties -> lower device id (R10);
//   4. devices are kept in that order while the kept weight is below 1 - p (R8, R9); near-margin tokens
//      are flagged (R-S4.7).
// Round 1 ranked the devices by counting (k^2 / 2 comparisons) and picked the r-th by k selects per rank
// (k^2 more): 5.3 k instructions per token at k = 10 (ncu, profiles/r2d_s4s5.md).  The networks are Batcher's
// merge exchange, valid for every size: 5 / 19 / 32 / 42 / 63 comparators for 4 / 8 / 10 / 12 / 16 slots.
#pragma once
#include <math_constants.h>

#include "cap_internal.cuh"

namespace cap {

// Batcher's merge exchange for N elements; ce(i, j) with i < j must leave the element that comes first at i.
// Fully unrolled: every index is a compile-time constant, the arrays stay in registers.
template <int N, typename F>
__device__ __forceinline__ void sort_network(F ce)
{
#pragma unroll
    for (int p = 1; p < N; p <<= 1) {
#pragma unroll
        for (int k = p; k >= 1; k >>= 1) {
#pragma unroll
            for (int j = k % p; j + k < N; j += 2 * k) {
#pragma unroll
                for (int i = 0; i < (k < N - j - k ? k : N - j - k); ++i)
                    if ((i + j) / (2 * p) == (i + j + k) / (2 * p)) ce(i + j, i + j + k);
            }
        }
    }
}

// What a token's slots look like in (device, slot) order, kept for the counting that follows the decision:
// run[i] = device | run length << 8 | 0x10000 at the last slot of a device's run, 0 elsewhere.
template <int KMAX>
struct PruneRuns {
    uint32_t run[KMAX];
};

// d[s]: device of slot s (0..63) for s < k; wv[s]: its routing weight.  Returns the kept device set and the
// near-margin flag; runs receives the token's device runs.
template <int KMAX>
__device__ __forceinline__ unsigned long long prune_token(const int (&d)[KMAX], const float (&wv)[KMAX], int k, int src,
                                                          const int *s_dn, int cost_local, int cost_intra,
                                                          int cost_inter, float p, int &near, PruneRuns<KMAX> &runs)
{
    // When every non-zero cost is a power of two (all BASELINE configs: 0 / 1 / 4, 0 / 1 / 1) a_d / c_d is the
    // product with the exact reciprocal: both are the correctly rounded value of the same real number, so the bits
    // are those of the IEEE division the oracle does (ncu: the eight divisions were 112 of 1 690 instructions per
    // token).  Uniform branch; any other cost takes the division.
    const bool recip_ok = (cost_local & (cost_local - 1)) == 0 && (cost_intra & (cost_intra - 1)) == 0 &&
                          (cost_inter & (cost_inter - 1)) == 0 && cost_local >= 0 && cost_intra >= 0 && cost_inter >= 0;
    const float r_local = cost_local > 0 ? __fdiv_rn(1.0f, (float)cost_local) : 0.0f;
    const float r_intra = cost_intra > 0 ? __fdiv_rn(1.0f, (float)cost_intra) : 0.0f;
    const float r_inter = cost_inter > 0 ? __fdiv_rn(1.0f, (float)cost_inter) : 0.0f;
    // 1. (device, slot) order; absent slots (s >= k) behind every device
    uint32_t key[KMAX];
    float a[KMAX];
#pragma unroll
    for (int s = 0; s < KMAX; ++s) {
        key[s] = ((uint32_t)(s < k ? (d[s] & 63) : 64 + s) << 4) | (uint32_t)s;
        a[s] = wv[s];
    }
    sort_network<KMAX>([&](int i, int j) {
        const bool sw = key[i] > key[j];
        const uint32_t ki = key[i], kj = key[j];
        const float ai = a[i], aj = a[j];
        key[i] = sw ? kj : ki;
        key[j] = sw ? ki : kj;
        a[i] = sw ? aj : ai;
        a[j] = sw ? ai : aj;
    });
    int len[KMAX];
    len[0] = 1;
#pragma unroll
    for (int i = 1; i < KMAX; ++i) {
        const bool same = (key[i] >> 4) == (key[i - 1] >> 4);
        a[i] = same ? __fadd_rn(a[i - 1], a[i]) : a[i];
        len[i] = same ? len[i - 1] + 1 : 1;
    }
    // 2. the devices (last slot of each run) and their cost ratios as ordered keys; 0 = not a device
    const int srcn = s_dn[src];
    uint32_t hi[KMAX], lo[KMAX];
    int m = 0;
#pragma unroll
    for (int i = 0; i < KMAX; ++i) {
        const int dd = (int)(key[i] >> 4) & 63;
        const bool last = i == KMAX - 1 ? true : (key[i] >> 4) != (key[i + 1] >> 4);
        const bool rep = last & (key[i] < (64u << 4));
        const bool is_loc = dd == src, is_same = s_dn[dd] == srcn;
        const int c = is_loc ? cost_local : is_same ? cost_intra : cost_inter;
        float ratio;
        if (recip_ok) {
            const float rc = is_loc ? r_local : is_same ? r_intra : r_inter;
            ratio = (c == 0) ? CUDART_INF_F : __fmul_rn(a[i], rc);
        } else {
            ratio = (c == 0) ? CUDART_INF_F : __fdiv_rn(a[i], (float)c);
        }
        hi[i] = rep ? okey(ratio) : 0u;
        lo[i] = (uint32_t)(63 - dd);
        runs.run[i] = rep ? ((uint32_t)dd | ((uint32_t)len[i] << 8) | 0x10000u) : 0u;
        m += rep ? 1 : 0;
    }
    // 3. larger ratio first, equal ratios: lower device id first
    sort_network<KMAX>([&](int i, int j) {
        const bool sw = (hi[i] < hi[j]) | ((hi[i] == hi[j]) & (lo[i] < lo[j]));
        const uint32_t hi_i = hi[i], hi_j = hi[j], lo_i = lo[i], lo_j = lo[j];
        const float ai = a[i], aj = a[j];
        hi[i] = sw ? hi_j : hi_i;
        hi[j] = sw ? hi_i : hi_j;
        lo[i] = sw ? lo_j : lo_i;
        lo[j] = sw ? lo_i : lo_j;
        a[i] = sw ? aj : ai;
        a[j] = sw ? ai : aj;
    });
    // 4. greedy in that order
    const float target = __fsub_rn(1.0f, p);
    float cum = 0.0f, r_last = 0.0f, r_cut = 0.0f;
    bool stopped = false;
    unsigned long long keepmask = 0ull;
#pragma unroll
    for (int r = 0; r < KMAX; ++r) {
        const float Ar = a[r], Rr = unkey(hi[r]);
        const int dr = 63 - (int)lo[r];
        const bool act = (r < m) & !stopped;
        const bool reached = cum >= target;
        near |= (int)(act & (fabsf(__fsub_rn(cum, target)) < 1e-6f));
        const bool stop_now = act & reached, keep_now = act & !reached;
        r_cut = stop_now ? Rr : r_cut;
        keepmask |= keep_now ? (1ull << dr) : 0ull;
        cum = keep_now ? __fadd_rn(cum, Ar) : cum;
        r_last = keep_now ? Rr : r_last;
        stopped = stopped | stop_now;
    }
    if (stopped && r_last != CUDART_INF_F && r_cut != CUDART_INF_F && __fsub_rn(r_last, r_cut) < 1e-6f) near = 1;
    return keepmask;
}

// The runs of a token whose decision is "keep everything" (p <= 0): only the (device, slot) order is needed.
template <int KMAX>
__device__ __forceinline__ void prune_runs_only(const int (&d)[KMAX], int k, PruneRuns<KMAX> &runs)
{
    uint32_t key[KMAX];
#pragma unroll
    for (int s = 0; s < KMAX; ++s) key[s] = ((uint32_t)(s < k ? (d[s] & 63) : 64 + s) << 4) | (uint32_t)s;
    sort_network<KMAX>([&](int i, int j) {
        const uint32_t ki = key[i], kj = key[j];
        key[i] = min(ki, kj);
        key[j] = max(ki, kj);
    });
    int len = 1;
#pragma unroll
    for (int i = 0; i < KMAX; ++i) {
        const int dd = (int)(key[i] >> 4) & 63;
        const bool last = i == KMAX - 1 ? true : (key[i] >> 4) != (key[i + 1] >> 4);
        const bool rep = last & (key[i] < (64u << 4));
        runs.run[i] = rep ? ((uint32_t)dd | ((uint32_t)len << 8) | 0x10000u) : 0u;
        len = last ? 1 : len + 1;
    }
}

}  // namespace cap

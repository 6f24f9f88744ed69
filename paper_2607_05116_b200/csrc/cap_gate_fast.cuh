// S1 fast path (softmax scoring, renormalised weights, no group limit, k <= 8): one THREAD per
// token.  The token's logits row sits in shared memory (staged by TMA); the thread streams it in
// groups of 8, sorts each group with a 19-comparator network and merges it into a running sorted
// top-8 list (half-cleaner + bitonic merge), all on 32-bit integer keys with min/max only.
//
// Keys.  key = order-preserving image of the logit with its low IB = log2(E) bits replaced by
// (E-1-e): larger key = larger logit, equal truncated logits -> lower expert index first, so one
// 32-bit comparator orders (value, index) pairs.  Truncation can only mis-order two experts whose
// keys agree in all upper 32-IB bits; the thread therefore also tracks the 9th largest key and,
// if any two neighbours among the top 9 share their upper bits, redoes that token with exact
// full-precision comparisons (k passes of arg-max).  The result is always the exact top-k with
// ties toward the lower index (reading R2), the fast path is taken for all but ~0.1% of tokens.
#pragma once
#include "cap_internal.cuh"

namespace cap {

#define CAP_CE(a, b)                         \
    do {                                     \
        const uint32_t _h = max((a), (b));   \
        (b) = min((a), (b));                 \
        (a) = _h;                            \
    } while (0)

// sort 8 keys descending: optimal 19-comparator network
__device__ __forceinline__ void sort8_desc(uint32_t (&g)[8])
{
    CAP_CE(g[0], g[1]); CAP_CE(g[2], g[3]); CAP_CE(g[4], g[5]); CAP_CE(g[6], g[7]);
    CAP_CE(g[0], g[2]); CAP_CE(g[1], g[3]); CAP_CE(g[4], g[6]); CAP_CE(g[5], g[7]);
    CAP_CE(g[1], g[2]); CAP_CE(g[5], g[6]); CAP_CE(g[0], g[4]); CAP_CE(g[3], g[7]);
    CAP_CE(g[1], g[5]); CAP_CE(g[2], g[6]);
    CAP_CE(g[1], g[4]); CAP_CE(g[3], g[6]);
    CAP_CE(g[2], g[4]); CAP_CE(g[3], g[5]);
    CAP_CE(g[3], g[4]);
}

// r (sorted desc) <- top 8 of r U g (g sorted desc); r9 <- max(r9, largest discarded key)
__device__ __forceinline__ void merge8_desc(uint32_t (&r)[8], const uint32_t (&g)[8], uint32_t &r9)
{
    uint32_t lo = r9;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const uint32_t a = r[i], b = g[7 - i];
        r[i] = max(a, b);
        lo = max(lo, min(a, b));
    }
    r9 = lo;
    CAP_CE(r[0], r[4]); CAP_CE(r[1], r[5]); CAP_CE(r[2], r[6]); CAP_CE(r[3], r[7]);
    CAP_CE(r[0], r[2]); CAP_CE(r[1], r[3]); CAP_CE(r[4], r[6]); CAP_CE(r[5], r[7]);
    CAP_CE(r[0], r[1]); CAP_CE(r[2], r[3]); CAP_CE(r[4], r[5]); CAP_CE(r[6], r[7]);
}

template <int E>
struct GateBits {
    static constexpr int IB = E <= 64 ? 6 : E <= 128 ? 7 : E <= 256 ? 8 : E <= 512 ? 9 : 10;
    static constexpr uint32_t MASK = (1u << IB) - 1u;
};

// key of logit x for expert e (e a compile-time constant after unrolling)
template <int E>
__device__ __forceinline__ uint32_t gate_key(float x, int e)
{
    const float c = __fadd_rn(x, 0.0f);                  // -0 -> +0 (IEEE: they compare equal)
    const uint32_t b = __float_as_uint(c);
    const uint32_t o = b ^ ((uint32_t)((int32_t)b >> 31) | 0x80000000u);
    return (o | GateBits<E>::MASK) ^ (uint32_t)e;        // low bits = MASK - e
}

// Exact top-k of one row by k passes of arg-max on full keys (ties -> lower index).
// Returns the k indices packed one per byte (E <= 256), slot 0 in the low byte.
template <int E>
__device__ __noinline__ unsigned long long gate_select_exact(const float *row, int k)
{
    unsigned long long packed = 0ull;
    uint32_t used[(E + 31) / 32];
#pragma unroll
    for (int i = 0; i < (E + 31) / 32; ++i) used[i] = 0u;
    for (int s = 0; s < k; ++s) {
        uint32_t bk = 0u;
        int bi = 0;
        for (int e = 0; e < E; ++e) {
            const uint32_t key = okey(row[e]);
            const bool free_ = !((used[e >> 5] >> (e & 31)) & 1u);
            if (free_ && key > bk) { bk = key; bi = e; }
        }
        packed |= (unsigned long long)bi << (8 * s);
        used[bi >> 5] |= 1u << (bi & 31);
    }
    return packed;
}

// Top-k selection of one token.  row: E floats in shared memory, 16-byte aligned.
// sel[0..k) = expert indices in descending score order.
template <int E>
__device__ __forceinline__ void gate_select(const float *row, int k, int (&sel)[8])
{
    static_assert(E % 8 == 0, "E must be a multiple of 8");
    constexpr int IB = GateBits<E>::IB;
    uint32_t r[8];
    uint32_t r9 = 0u;
#pragma unroll
    for (int gi = 0; gi < E / 8; ++gi) {
        const float4 va = *reinterpret_cast<const float4 *>(row + gi * 8);
        const float4 vb = *reinterpret_cast<const float4 *>(row + gi * 8 + 4);
        uint32_t g[8];
        g[0] = gate_key<E>(va.x, gi * 8 + 0); g[1] = gate_key<E>(va.y, gi * 8 + 1);
        g[2] = gate_key<E>(va.z, gi * 8 + 2); g[3] = gate_key<E>(va.w, gi * 8 + 3);
        g[4] = gate_key<E>(vb.x, gi * 8 + 4); g[5] = gate_key<E>(vb.y, gi * 8 + 5);
        g[6] = gate_key<E>(vb.z, gi * 8 + 6); g[7] = gate_key<E>(vb.w, gi * 8 + 7);
        sort8_desc(g);
        if (gi == 0) {
#pragma unroll
            for (int i = 0; i < 8; ++i) r[i] = g[i];
        } else {
            merge8_desc(r, g, r9);
        }
    }
    // neighbours among the top 9 that agree in every bit above the index field are ambiguous
    bool amb = ((r[7] ^ r9) >> IB) == 0u;
#pragma unroll
    for (int i = 0; i < 7; ++i) amb |= ((r[i] ^ r[i + 1]) >> IB) == 0u;
    if (E == 8) amb = false;   // no 9th key
    static_assert(E <= 256, "packed fallback indices are one byte each");
    if (amb) {
        const unsigned long long pk = gate_select_exact<E>(row, k);
#pragma unroll
        for (int i = 0; i < 8; ++i) sel[i] = (int)((pk >> (8 * i)) & 0xffull);
    } else {
#pragma unroll
        for (int i = 0; i < 8; ++i) sel[i] = (int)(GateBits<E>::MASK - (r[i] & GateBits<E>::MASK));
    }
}

// Renormalised softmax weights of the selected experts (DESIGN.md R-S1.3): r_s = expS(x_s - x_0),
// Z summed in slot order, w_s = r_s / Z (* scale).
__device__ __forceinline__ void gate_weights_softmax(const float *row, int k, const int (&sel)[8],
                                                     float scale, float (&w)[8])
{
    const float x0 = row[sel[0]];
    float Z = 0.0f;
#pragma unroll
    for (int s = 0; s < 8; ++s) {
        if (s < k) {
            const float rs = exp_s(__fsub_rn(row[sel[s]], x0));
            w[s] = rs;
            Z = s == 0 ? rs : __fadd_rn(Z, rs);
        }
    }
#pragma unroll
    for (int s = 0; s < 8; ++s) {
        if (s < k) {
            float v = __fdiv_rn(w[s], Z);
            if (scale != 1.0f) v = __fmul_rn(v, scale);
            w[s] = v;
        }
    }
}

}  // namespace cap

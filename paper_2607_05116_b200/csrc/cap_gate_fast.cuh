// S1 fast path (softmax scoring, renormalised weights, no group limit, k <= 8): a PAIR of threads
// per token.  The token's logits row sits in shared memory (staged by TMA); each thread streams its
// half of the row in groups of 8, sorts each group with a 19-comparator network and merges it into a running sorted
// top-8 list (half-cleaner + bitonic merge), all on 32-bit keys with fp32 min/max only.
//
// Keys.  key = the logit's own bit pattern with its low BYTE replaced by the element's position
// (one PRMT per element, no sign transform: fp32 min/max already order the patterns).  A payload can
// only decide a comparison between two keys that agree in all upper 24 bits; the thread therefore
// also tracks the 9th largest key and, if any two neighbours among the top 9 share their upper bits
// -- or one of them is a zero, whose two signs are distinct patterns but compare equal (reading R2) --
// the warp redoes that token with exact full-precision comparisons (k rounds of warp-wide arg-max).
// The result is always the exact top-k with ties toward the lower index; the fast path alone serves
// all but ~0.2% of the tokens of the paper-shaped traces.
#pragma once
#include "cap_async.cuh"
#include "cap_internal.cuh"

namespace cap {

__device__ __forceinline__ float kmax(float a, float b)
{
    float r;
    asm("max.f32 %0, %1, %2;" : "=f"(r) : "f"(a), "f"(b));
    return r;
}
__device__ __forceinline__ float kmin(float a, float b)
{
    float r;
    asm("min.f32 %0, %1, %2;" : "=f"(r) : "f"(a), "f"(b));
    return r;
}
__device__ __forceinline__ float kmax3(float a, float b, float c)
{
    float r;
    asm("max.f32 %0, %1, %2, %3;" : "=f"(r) : "f"(a), "f"(b), "f"(c));
    return r;
}

#define CAP_CE(a, b)                         \
    do {                                     \
        const float _h = kmax((a), (b));     \
        (b) = kmin((a), (b));                \
        (a) = _h;                            \
    } while (0)

// sort 8 keys descending: optimal 19-comparator network
__device__ __forceinline__ void sort8_desc(float (&g)[8])
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
__device__ __forceinline__ void merge8_desc(float (&r)[8], const float (&g)[8], float &r9)
{
    float lo = r9;
#pragma unroll
    for (int i = 0; i < 8; i += 2) {
        const float a0 = r[i], b0 = g[7 - i], a1 = r[i + 1], b1 = g[6 - i];
        r[i] = kmax(a0, b0);
        r[i + 1] = kmax(a1, b1);
        lo = kmax3(lo, kmin(a0, b0), kmin(a1, b1));
    }
    r9 = lo;
    CAP_CE(r[0], r[4]); CAP_CE(r[1], r[5]); CAP_CE(r[2], r[6]); CAP_CE(r[3], r[7]);
    CAP_CE(r[0], r[2]); CAP_CE(r[1], r[3]); CAP_CE(r[4], r[6]); CAP_CE(r[5], r[7]);
    CAP_CE(r[0], r[1]); CAP_CE(r[2], r[3]); CAP_CE(r[4], r[5]); CAP_CE(r[6], r[7]);
}

// key of the logit x at position pos of the thread's half row (pos a compile-time constant after
// unrolling): the low byte of the pattern is replaced by pos
__device__ __forceinline__ float gate_key(float x, int pos)
{
    const uint32_t pay = 0x03020100u + 0x04040404u * (uint32_t)(pos >> 2);
    return __uint_as_float(__byte_perm(__float_as_uint(x), pay, 0x3214u + (uint32_t)(pos & 3)));
}

// Exact top-k of one row, computed by the WHOLE warp (all 32 lanes must call it with the same row):
// lane l holds experts [l E/32, (l+1) E/32) as full 32-bit keys; k rounds of {warp max of the lanes'
// best keys, warp min over the owners' indices} so that ties go to the lower expert index.
template <int E>
__device__ __noinline__ void gate_select_exact_warp(uint32_t row_smem, int lane, int k, int (&sel)[8])
{
    constexpr int VPL = E / 32;
    uint32_t key[VPL];
#pragma unroll
    for (int j = 0; j < VPL; ++j) {
        float x;
        asm volatile("ld.shared.f32 %0, [%1];" : "=f"(x) : "r"(row_smem + (uint32_t)(lane * VPL + j) * 4u));
        key[j] = okey(x);
    }
#pragma unroll
    for (int s = 0; s < 8; ++s) {
        int wi = 0;
        if (s < k) {
            uint32_t bk = 0u;
            int bi = 0x7fffffff;
#pragma unroll
            for (int j = 0; j < VPL; ++j)
                if (key[j] > bk) { bk = key[j]; bi = lane * VPL + j; }
            const uint32_t m = __reduce_max_sync(0xffffffffu, bk);
            wi = __reduce_min_sync(0xffffffffu, bk == m ? bi : 0x7fffffff);
#pragma unroll
            for (int j = 0; j < VPL; ++j)
                if (lane * VPL + j == wi) key[j] = 0u;
        }
        sel[s] = wi;
    }
}

// Top-k selection of one token by a PAIR of lanes (lane and lane ^ 16): lane half h streams experts
// [h E/2, (h+1) E/2) of the row with half-relative index immediates, the two sorted lists are then
// rebased to full indices and merged (both lanes end with the same result).
// row: E floats in shared memory, dense (4E-byte rows, tile base 128-byte aligned).  To keep the
// 128-bit row reads bank-conflict free without padding, lane t reads 16-byte chunk c of its half at
// chunk position c ^ (t & 7): the keys then carry the index payload of position c, and since the
// payload never decides a comparison whose outcome is kept (equal upper bits -> exact fallback),
// the true index is recovered afterwards as payload ^ 4 (t & 7).
// sel[0..8) = expert indices, descending score.
template <int E>
__device__ __forceinline__ void gate_select_pair(const float *row, int h, int t7, int k, int (&sel)[8])
{
    static_assert(E % 16 == 0 && E >= 32 && E <= 256, "E must be a multiple of 16 in [32, 256]");
    constexpr int H = E / 2;
    const uint32_t hb = smem_u32(row + h * H) | ((uint32_t)t7 << 4);   // 128-byte aligned | swizzle
    float r[8];
    float r9 = __uint_as_float(0xff800000u);                           // -inf: below every finite key
#pragma unroll
    for (int gi = 0; gi < H / 8; ++gi) {
        float4 va, vb;
        asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];"
                     : "=f"(va.x), "=f"(va.y), "=f"(va.z), "=f"(va.w)
                     : "r"(hb ^ (uint32_t)(gi * 32)));
        asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];"
                     : "=f"(vb.x), "=f"(vb.y), "=f"(vb.z), "=f"(vb.w)
                     : "r"(hb ^ (uint32_t)(gi * 32 + 16)));
        float g[8];
        g[0] = gate_key(va.x, gi * 8 + 0); g[1] = gate_key(va.y, gi * 8 + 1);
        g[2] = gate_key(va.z, gi * 8 + 2); g[3] = gate_key(va.w, gi * 8 + 3);
        g[4] = gate_key(vb.x, gi * 8 + 4); g[5] = gate_key(vb.y, gi * 8 + 5);
        g[6] = gate_key(vb.z, gi * 8 + 6); g[7] = gate_key(vb.w, gi * 8 + 7);
        sort8_desc(g);
        if (gi == 0) {
#pragma unroll
            for (int i = 0; i < 8; ++i) r[i] = g[i];
        } else {
            merge8_desc(r, g, r9);
        }
    }
    // payload (position in the half row) -> full expert index: undo the chunk swizzle (XOR of bits
    // 2..4), then add h E/2 (position < E/2 <= 128, so the sum stays inside the byte)
    const uint32_t swz = (uint32_t)t7 << 2;
    const uint32_t adj = (uint32_t)(h * H);
    float g[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        r[i] = __uint_as_float((__float_as_uint(r[i]) ^ swz) + adj);
        g[i] = __shfl_xor_sync(0xffffffffu, r[i], 16);
    }
    r9 = kmax(r9, __shfl_xor_sync(0xffffffffu, r9, 16));               // its payload is never decoded
    merge8_desc(r, g, r9);
    // ambiguous: neighbours among the top 9 that agree in every bit above the payload, or a zero
    // among them (+0 and -0 are different patterns that must compare equal)
    uint32_t u[9];
#pragma unroll
    for (int i = 0; i < 8; ++i) u[i] = __float_as_uint(r[i]);
    u[8] = __float_as_uint(r9);
    bool amb = false;
#pragma unroll
    for (int i = 0; i < 8; ++i) amb |= ((u[i] ^ u[i + 1]) >> 8) == 0u;
#pragma unroll
    for (int i = 0; i < 9; ++i) amb |= (u[i] & 0x7fffff00u) == 0u;
#pragma unroll
    for (int i = 0; i < 8; ++i) sel[i] = (int)(u[i] & 0xffu);
    // ambiguous tokens (rare): the whole warp redoes them one at a time with exact comparisons
    const int lane = (int)(threadIdx.x & 31u);
    unsigned todo = __ballot_sync(0xffffffffu, amb) & 0xffffu;     // one lane of each pair
    const uint32_t row_s = smem_u32(row);
    while (todo) {
        const int src = __ffs((int)todo) - 1;
        todo &= todo - 1u;
        const uint32_t rs = __shfl_sync(0xffffffffu, row_s, src);
        int ex[8];
        gate_select_exact_warp<E>(rs, lane, k, ex);
        if ((lane & 15) == src) {
#pragma unroll
            for (int i = 0; i < 8; ++i) sel[i] = ex[i];
        }
    }
}

// Renormalised softmax weights (DESIGN.md R-S1.3): r_s = expS(x_s - x_0), Z summed in slot order,
// w_s = r_s / Z (* scale).  Lane half h evaluates slots 4h..4h+3, the pair exchanges them, both sum
// Z in slot order; w[0..4) = weights of slots 4h..4h+3.
__device__ __forceinline__ void gate_weights_softmax_pair(const float *row, int h, int k,
                                                          const int (&sel)[8], float scale, float (&w)[4])
{
    const float x0 = row[sel[0]];
    float mine[4], other[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const int s = h ? 4 + j : j;
        const int e = h ? sel[4 + j] : sel[j];
        mine[j] = s < k ? exp_s(__fsub_rn(row[e], x0)) : 0.0f;
        other[j] = __shfl_xor_sync(0xffffffffu, mine[j], 16);
    }
    float Z = h ? other[0] : mine[0];
#pragma unroll
    for (int s = 1; s < 8; ++s) {
        const float rs = (s < 4) ? (h ? other[s & 3] : mine[s & 3]) : (h ? mine[s & 3] : other[s & 3]);
        if (s < k) Z = __fadd_rn(Z, rs);
    }
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        float v = __fdiv_rn(mine[j], Z);
        if (scale != 1.0f) v = __fmul_rn(v, scale);
        w[j] = v;
    }
}

}  // namespace cap

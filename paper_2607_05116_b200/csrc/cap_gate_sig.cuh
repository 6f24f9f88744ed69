// S1 fast path for sigmoid scoring with a selection bias and group-limited routing (Eq. 1;
// BASELINE.json config 4, reading R14: groups = contiguous blocks of 32 experts, group score = max or
// fp32 sum of the top-2 biased scores, top `topk_group` groups, then top-k inside them by the biased
// score, weights from the unbiased sigmoid, renormalised).  A PAIR of lanes per token, as in
// cap_gate_fast.cuh: lane half h streams experts [h E/2, (h+1) E/2) = E/64 groups from the staged row.
//
// Two-level precision.  The reference selection score is c = sigS(x) + b with the reproducible sigS of
// DESIGN.md R-S1.3 (~30 instructions and an IEEE divide per expert).  Here every expert gets the CHEAP
// score a = 1 / (1 + 2^(-x log2 e)) + b from the special-function unit (|a - c| <= GS_EPS, derivation in
// DESIGN.md 6.9), packed into a 32-bit key whose low byte is the expert's position (|key - a| < 256 ulp).
// Per group the keys go through the sort-8 / merge-8 networks into a sorted top-8 list, group scores come
// from the two list heads, the selected groups' lists are merged.  Every decision that the approximate
// keys cannot certify -- a selected and an unselected group closer than GS_THRG, two neighbours among
// the top k+1 keys closer than two key steps, a key below 0.25 among them -- sends the token to
// gate_select_exact_sig_warp, which the whole warp runs with the reference arithmetic.  The result is
// therefore always the oracle's (ties toward the lower group / expert included); the cheap path alone
// serves ~99 % of the tokens of the config-4 trace.
#pragma once
#include "cap_gate_fast.cuh"

namespace cap {

constexpr float GS_EPS = 2.0e-6f;       // |cheap score - reference score|, bound derived in DESIGN.md 6.9 (~4e-7) x 5
constexpr float GS_THRG = 1.4e-4f;      // group scores (sums of two keys): 2 * (2 * (GS_EPS + 256 ulp(1.0)) + rounding)
constexpr uint32_t GS_SENT = 0xff000000u;   // list filler (-1.7e38): stays finite under the payload arithmetic

// 1 / (1 + 2^(-x log2 e)) on the special-function unit: FMUL, MUFU.EX2, FADD, MUFU.RCP.  The raw .ftz
// instructions, not __expf / __fdividef: without fast-math those carry denormal-range fix-ups (14 instructions
// per expert instead of 4).  Saturation is right by construction: 2^(+big) = inf -> 1/inf = 0, 2^(-big) = 0 -> 1.
__device__ __forceinline__ float gs_cheap_sigmoid(float x)
{
    float e, r;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(e) : "f"(__fmul_rn(x, -1.4426950408889634f)));
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(__fadd_rn(1.0f, e)));
    return r;
}

// key of the cheap score: low byte <- byte j of the payload word (positions of four consecutive experts)
__device__ __forceinline__ float gs_key_rt(float x, float b, uint32_t pay, int j)
{
    return __uint_as_float(__byte_perm(__float_as_uint(__fadd_rn(gs_cheap_sigmoid(x), b)), pay, 0x3214u + (uint32_t)j));
}

// Exact selection of one token by the WHOLE warp (all lanes call it with the same row): lane l holds
// experts [l E/32, (l+1) E/32), a group of 32 experts = 32 / (E/32) consecutive lanes.  Follows the
// oracle step by step: c = sigS(x) + b, group scores, topk_group rounds (ties -> lower group), k rounds
// of arg-max (ties -> lower expert).  bias_g = 0 means "no bias".
template <int E>
__device__ __noinline__ void gate_select_exact_sig_warp(uint32_t row_smem, const float *bias_g, int lane, int k,
                                                        int topk_group, int group_score, int (&sel)[8])
{
    constexpr int VPL = E / 32, LPG = 32 / VPL;
    constexpr unsigned FULL = 0xffffffffu;
    uint32_t key[VPL];
#pragma unroll
    for (int j = 0; j < VPL; ++j) {
        float x;
        asm volatile("ld.shared.f32 %0, [%1];" : "=f"(x) : "r"(row_smem + (uint32_t)(lane * VPL + j) * 4u));
        const float s = sig_s(x);
        key[j] = okey(bias_g ? __fadd_rn(s, __ldg(bias_g + lane * VPL + j)) : s);
    }
    // two largest keys of the group: inside the lane, then across the LPG lanes of the group
    uint32_t m1 = 0u, m2 = 0u;
#pragma unroll
    for (int j = 0; j < VPL; ++j) {
        m2 = max(m2, min(m1, key[j]));
        m1 = max(m1, key[j]);
    }
#pragma unroll
    for (int o = 1; o < LPG; o <<= 1) {
        const uint32_t o1 = __shfl_xor_sync(FULL, m1, o), o2 = __shfl_xor_sync(FULL, m2, o);
        m2 = max(min(m1, o1), max(m2, o2));
        m1 = max(m1, o1);
    }
    const int grp = lane / LPG;
    uint32_t gk = group_score == 1 ? okey(__fadd_rn(unkey(m1), unkey(m2))) : m1;
    if (lane % LPG != 0) gk = 0u;                        // one holder lane per group
    uint32_t selmask = 0u;
    for (int r = 0; r < topk_group; ++r) {
        const uint32_t m = __reduce_max_sync(FULL, gk);
        const int wg = __reduce_min_sync(FULL, (gk == m && lane % LPG == 0) ? grp : 0x7fffffff);
        if ((unsigned)wg < 32u) selmask |= 1u << wg;
        if (grp == wg) gk = 0u;
    }
    if (!((selmask >> grp) & 1u)) {
#pragma unroll
        for (int j = 0; j < VPL; ++j) key[j] = 0u;
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
            const uint32_t m = __reduce_max_sync(FULL, bk);
            wi = __reduce_min_sync(FULL, bk == m ? bi : 0x7fffffff);
            if ((unsigned)wi >= (unsigned)E) wi = 0;     // garbage rows (NaN): stay in range
#pragma unroll
            for (int j = 0; j < VPL; ++j)
                if (lane * VPL + j == wi) key[j] = 0u;
        }
        sel[s] = wi;
    }
}

// Selection of one token by a pair of lanes.  row: E floats in shared memory (tile base 1024-byte aligned,
// dense rows); bias_g: the layer's E selection biases in global memory (16-byte aligned) or 0.  Reads are
// XOR-swizzled per lane inside every 128-byte block (= one group of 32 experts), for the row and for the
// bias alike, so the payload is the position ^ (t7 << 2); it is undone once at the end.
template <int E>
__device__ __forceinline__ void gate_select_sig_pair(const float *row, const float *bias_g, int h, int t7, int k,
                                                     int topk_group, int group_score, int (&sel)[8])
{
    static_assert(E == 64 || E == 128 || E == 256, "groups of 32 experts, E/64 groups per lane");
    constexpr int H = E / 2, G = H / 32;
    const uint32_t hb = smem_u32(row + h * H) | ((uint32_t)t7 << 4);
    const float sent = __uint_as_float(GS_SENT);
    float lst[G][8], l9[G];
#pragma unroll
    for (int g = 0; g < G; ++g) {
        // The four 8-expert sub-blocks of a group are a ROLLED loop (runtime payload word): fully unrolled, the
        // selection is ~6 000 instructions (96 KB), which 12 warps at different positions cannot keep in the
        // 32 KB instruction cache -- ncu showed 57 % of the stall samples as no_inst.
        float r[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) r[i] = sent;
        float r9 = sent;
#pragma unroll 1
        for (int sb = 0; sb < 4; ++sb) {
            const uint32_t off = (uint32_t)(g * 128 + sb * 32);
            float4 va, vb, ba = make_float4(0.f, 0.f, 0.f, 0.f), bb = ba;
            asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];"
                         : "=f"(va.x), "=f"(va.y), "=f"(va.z), "=f"(va.w) : "r"(hb ^ off));
            asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];"
                         : "=f"(vb.x), "=f"(vb.y), "=f"(vb.z), "=f"(vb.w) : "r"(hb ^ (off + 16u)));
            if (bias_g) {
                const char *bp = reinterpret_cast<const char *>(bias_g + h * H);
                ba = __ldg(reinterpret_cast<const float4 *>(bp + (off ^ ((uint32_t)t7 << 4))));
                bb = __ldg(reinterpret_cast<const float4 *>(bp + ((off + 16u) ^ ((uint32_t)t7 << 4))));
            }
            // payload words: bytes = positions p0..p0+3 and p0+4..p0+7 of the lane's half row
            const uint32_t payA = 0x03020100u + 0x01010101u * (uint32_t)(g * 32 + sb * 8);
            const uint32_t payB = payA + 0x04040404u;
            float q[8];
            q[0] = gs_key_rt(va.x, ba.x, payA, 0); q[1] = gs_key_rt(va.y, ba.y, payA, 1);
            q[2] = gs_key_rt(va.z, ba.z, payA, 2); q[3] = gs_key_rt(va.w, ba.w, payA, 3);
            q[4] = gs_key_rt(vb.x, bb.x, payB, 0); q[5] = gs_key_rt(vb.y, bb.y, payB, 1);
            q[6] = gs_key_rt(vb.z, bb.z, payB, 2); q[7] = gs_key_rt(vb.w, bb.w, payB, 3);
            sort8_desc(q);
            merge8_desc(r, q, r9);          // the first merge meets the fillers
        }
#pragma unroll
        for (int i = 0; i < 8; ++i) lst[g][i] = r[i];
        l9[g] = r9;
    }
    // ---- group scores of all E/32 groups (own and partner's), selection of the topk_group best ----
    float gsc[G], osc[G];
#pragma unroll
    for (int g = 0; g < G; ++g) {
        gsc[g] = group_score == 1 ? __fadd_rn(lst[g][0], lst[g][1]) : lst[g][0];
        osc[g] = __shfl_xor_sync(0xffffffffu, gsc[g], 16);
    }
    bool amb = false;
    float smin = 3.0e38f, umax = sent;          // weakest selected / strongest unselected group score
    bool gsel[G];
#pragma unroll
    for (int g = 0; g < G; ++g) {
        int rank = 0;
#pragma unroll
        for (int g2 = 0; g2 < G; ++g2) {
            if (g2 != g) rank += (gsc[g2] > gsc[g] || (gsc[g2] == gsc[g] && g2 < g)) ? 1 : 0;
            // partner's group g2 has the lower global id iff this lane is half 1
            rank += (osc[g2] > gsc[g] || (osc[g2] == gsc[g] && h == 1)) ? 1 : 0;
        }
        gsel[g] = rank < topk_group;
        if (gsel[g]) smin = kmin(smin, gsc[g]);
        else umax = kmax(umax, gsc[g]);
    }
    smin = kmin(smin, __shfl_xor_sync(0xffffffffu, smin, 16));
    umax = kmax(umax, __shfl_xor_sync(0xffffffffu, umax, 16));
    amb |= !(smin - umax >= GS_THRG);          // also catches NaN scores
    // ---- merge the selected groups' lists (unselected ones enter as fillers: branch-free) ----
    float r[8];
    float r9 = sent;
#pragma unroll
    for (int g = 0; g < G; ++g) {
        float q[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) q[i] = gsel[g] ? lst[g][i] : sent;
        const float q9 = gsel[g] ? l9[g] : sent;
        if (g == 0) {
#pragma unroll
            for (int i = 0; i < 8; ++i) r[i] = q[i];
            r9 = q9;
        } else {
            merge8_desc(r, q, r9);
            r9 = kmax(r9, q9);
        }
    }
    // payload -> full expert index (undo the swizzle, add the half's base), then the partner's list
    const uint32_t swz = (uint32_t)t7 << 2, adj = (uint32_t)(h * H);
    float q[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        r[i] = __uint_as_float((__float_as_uint(r[i]) ^ swz) + adj);
        q[i] = __shfl_xor_sync(0xffffffffu, r[i], 16);
    }
    r9 = kmax(r9, __shfl_xor_sync(0xffffffffu, r9, 16));
    merge8_desc(r, q, r9);
    // ---- can the keys certify the order of the top k and the cut below it? ----
    uint32_t u[9];
#pragma unroll
    for (int i = 0; i < 8; ++i) u[i] = __float_as_uint(r[i]);
    u[8] = __float_as_uint(r9);
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        if (i < k) {
            // positive keys >= 0.25: one key step (256 ulp >= 7.6e-6) exceeds 2 GS_EPS, so a difference of two
            // steps or more between the truncated patterns proves the order of the reference scores
            amb |= (u[i] >> 8) - (u[i + 1] >> 8) < 2u;
            amb |= (int32_t)u[i + 1] < 0x3e800000;          // next key below 0.25, negative or a filler
        }
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) sel[i] = (int)(u[i] & 0xffu) & (E - 1);
    // ---- ambiguous tokens: the whole warp redoes them one at a time with the reference arithmetic ----
    const int lane = (int)(threadIdx.x & 31u);
    amb |= __shfl_xor_sync(0xffffffffu, amb ? 1 : 0, 16) != 0;
    unsigned todo = __ballot_sync(0xffffffffu, amb) & 0xffffu;
    const uint32_t row_s = smem_u32(row);
    while (todo) {
        const int src = __ffs((int)todo) - 1;
        todo &= todo - 1u;
        const uint32_t rs = __shfl_sync(0xffffffffu, row_s, src);
        int ex[8];
        gate_select_exact_sig_warp<E>(rs, bias_g, lane, k, topk_group, group_score, ex);
        if ((lane & 15) == src) {
#pragma unroll
            for (int i = 0; i < 8; ++i) sel[i] = ex[i];
        }
    }
}

// Renormalised sigmoid weights (oracle step 5): s_r = sigS(x of slot r) without the bias, Z summed in slot
// order, w_r = s_r / Z (* scale).  Lane half h evaluates slots 4h..4h+3; w[0..4) = their weights.
__device__ __forceinline__ void gate_weights_sigmoid_pair(const float *row, int h, int k, const int (&sel)[8],
                                                          float scale, float (&w)[4])
{
    float mine[4], other[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const int s = h ? 4 + j : j;
        const int e = h ? sel[4 + j] : sel[j];
        mine[j] = s < k ? sig_s(row[e]) : 0.0f;
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

// S1 -- top-k gating (Eq. 1).  Generic exact kernel: one warp per token, each lane
// holds VPL router scores as order-preserving integer keys in registers; selection is k rounds
// of {warp max of the lanes' best keys, warp min over the owners' expert indices} so that ties
// go to the lower expert index by construction.  Rows are read once with 128-bit loads.
#include "cap_internal.cuh"

namespace cap {

struct GateParams {
    const float *logits;
    const float *bias;
    int32_t *idx;
    float *w;
    int64_t LT;   // L*T tokens
    int64_t T;
    int32_t E, k, scoring, renormalize, n_group, topk_group, group_score;
    float scale;
    int vec;      // 1: rows are 16-byte aligned and E % 4 == 0
};

// expert index of register j of a lane: chunks of CW consecutive experts, chunk c -> lane c%32
template <int VPL>
__device__ __forceinline__ int expert_of(int lane, int j)
{
    constexpr int CW = VPL >= 4 ? 4 : VPL;
    return (j / CW) * (32 * CW) + lane * CW + (j % CW);
}

template <int VPL>
__global__ void __launch_bounds__(256) gate_topk_kernel(GateParams prm)
{
    constexpr unsigned FULL = 0xffffffffu;
    constexpr int CW = VPL >= 4 ? 4 : VPL;
    const int lane = threadIdx.x & 31;
    const int64_t warp0 = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int64_t nwarps = ((int64_t)gridDim.x * blockDim.x) >> 5;
    const int E = prm.E, k = prm.k;

    for (int64_t tok = warp0; tok < prm.LT; tok += nwarps) {
        const float *row = prm.logits + tok * E;
        const int64_t layer = tok / prm.T;
        float xv[VPL];
        uint32_t key[VPL];
        // ---- load the row -----------------------------------------------------------------
        bool loaded = false;
        if constexpr (CW == 4) {
            if (prm.vec) {
#pragma unroll
                for (int c = 0; c < VPL / 4; ++c) {
                    int e0 = c * 128 + lane * 4;
                    float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
                    if (e0 < E) v = __ldg(reinterpret_cast<const float4 *>(row + e0));
                    xv[c * 4 + 0] = v.x;
                    xv[c * 4 + 1] = v.y;
                    xv[c * 4 + 2] = v.z;
                    xv[c * 4 + 3] = v.w;
                }
                loaded = true;
            }
        }
        if (!loaded) {
#pragma unroll
            for (int j = 0; j < VPL; ++j) {
                int e = expert_of<VPL>(lane, j);
                xv[j] = (e < E) ? __ldg(row + e) : 0.f;
            }
        }
        // ---- selection scores as keys ---------------------------------------------------------
        uint32_t rowmax_key = 0;   // raw-logit row maximum (softmax without renormalisation)
#pragma unroll
        for (int j = 0; j < VPL; ++j) {
            int e = expert_of<VPL>(lane, j);
            if (e < E) {
                float c;
                if (prm.scoring == 0) {
                    c = xv[j];
                } else {
                    float s = sig_s(xv[j]);
                    c = prm.bias ? __fadd_rn(s, __ldg(prm.bias + layer * E + e)) : s;
                }
                key[j] = okey(c);
                rowmax_key = max(rowmax_key, okey(xv[j]));
            } else {
                key[j] = 0u;
            }
        }
        // ---- group-limited pre-selection ------------------------------------------------------
        if (prm.n_group > 1) {
            const int gsz = E / prm.n_group;
            uint32_t gk = 0u;       // lane g holds the key of group g's score
            // Segmented path: with 4 consecutive experts per register block and group sizes that divide 128,
            // a register block lies inside one group and a group occupies gsz / 4 consecutive lanes of one
            // block: top-2 per block in registers, then a butterfly inside the lane segment (all groups at
            // once) instead of one warp-wide reduction per group.
            const int seg = gsz >> 2;
            const bool segmented = CW == 4 && (gsz & 3) == 0 && gsz <= 128 && (128 % gsz) == 0;
            if (segmented) {
                if constexpr (CW == 4) {
                    const int gb = (lane * gsz) >> 7, gl = ((lane * gsz) & 127) >> 2;   // block / first lane of group `lane`
#pragma unroll
                    for (int c = 0; c < VPL / 4; ++c) {
                        const uint32_t a = key[4 * c], b = key[4 * c + 1], cc = key[4 * c + 2], d = key[4 * c + 3];
                        const uint32_t h1 = max(a, b), l1 = min(a, b), h2 = max(cc, d), l2 = min(cc, d);
                        uint32_t m1 = max(h1, h2), m2 = max(min(h1, h2), max(l1, l2));   // two largest elements
                        for (int o = 1; o < seg; o <<= 1) {
                            const uint32_t o1 = __shfl_xor_sync(FULL, m1, o), o2 = __shfl_xor_sync(FULL, m2, o);
                            m2 = max(min(m1, o1), max(m2, o2));
                            m1 = max(m1, o1);
                        }
                        const uint32_t score = prm.group_score == 1 ? okey(__fadd_rn(unkey(m1), unkey(m2))) : m1;
                        const uint32_t v = __shfl_sync(FULL, score, gl & 31);
                        if (lane < prm.n_group && gb == c) gk = v;
                    }
                }
            } else
            for (int g = 0; g < prm.n_group; ++g) {
                const int lo = g * gsz, hi = lo + gsz;
                uint32_t lm = 0u;
                int li = 0x7fffffff;
#pragma unroll
                for (int j = 0; j < VPL; ++j) {
                    int e = expert_of<VPL>(lane, j);
                    if (e >= lo && e < hi && key[j] > lm) { lm = key[j]; li = e; }
                }
                uint32_t g1 = __reduce_max_sync(FULL, lm);
                uint32_t score_key = g1;
                if (prm.group_score == 1) {
                    int w1 = __reduce_min_sync(FULL, (lm == g1) ? li : 0x7fffffff);
                    uint32_t lm2 = 0u;
#pragma unroll
                    for (int j = 0; j < VPL; ++j) {
                        int e = expert_of<VPL>(lane, j);
                        if (e >= lo && e < hi && e != w1 && key[j] > lm2) lm2 = key[j];
                    }
                    uint32_t g2 = __reduce_max_sync(FULL, lm2);
                    score_key = okey(__fadd_rn(unkey(g1), unkey(g2)));
                }
                if (lane == g) gk = score_key;
            }
            uint32_t selmask = 0u;
            for (int r = 0; r < prm.topk_group; ++r) {
                uint32_t m = __reduce_max_sync(FULL, gk);
                int wl = __reduce_min_sync(FULL, (gk == m && lane < prm.n_group) ? lane : 0x7fffffff);
                selmask |= 1u << wl;
                if (lane == wl) gk = 0u;
            }
#pragma unroll
            for (int j = 0; j < VPL; ++j) {
                int e = expert_of<VPL>(lane, j);
                if (e < E && !((selmask >> (e / gsz)) & 1u)) key[j] = 0u;
            }
        }
        // ---- k rounds of arg-max, ties -> lower expert index -----------------------------------
        uint32_t bk = 0u;
        int bi = 0x7fffffff;
#pragma unroll
        for (int j = 0; j < VPL; ++j)
            if (key[j] > bk) { bk = key[j]; bi = expert_of<VPL>(lane, j); }
        int selidx = 0;
        for (int r = 0; r < k; ++r) {
            uint32_t m = __reduce_max_sync(FULL, bk);
            int wi = __reduce_min_sync(FULL, (bk == m) ? bi : 0x7fffffff);
            if (lane == r) selidx = wi;
            if (bk == m && bi == wi) {
                bk = 0u;
                bi = 0x7fffffff;
#pragma unroll
                for (int j = 0; j < VPL; ++j) {
                    int e = expert_of<VPL>(lane, j);
                    if (e == wi) key[j] = 0u;
                    if (key[j] > bk) { bk = key[j]; bi = e; }
                }
            }
        }
        // ---- routing weights (lanes 0..k-1 hold one slot each) ---------------------------------
        const bool mine = lane < k;
        const float xs = mine ? __ldg(row + selidx) : 0.f;
        float wv;
        if (prm.scoring == 0) {
            if (prm.renormalize) {
                float x0 = __shfl_sync(FULL, xs, 0);
                float r = mine ? exp_s(__fsub_rn(xs, x0)) : 0.f;
                float Z = __shfl_sync(FULL, r, 0);
                for (int s = 1; s < k; ++s) Z = __fadd_rn(Z, __shfl_sync(FULL, r, s));
                wv = __fdiv_rn(r, Z);
            } else {
                uint32_t mk = __reduce_max_sync(FULL, rowmax_key);
                float m = unkey(mk);
                double part = 0.0;
#pragma unroll
                for (int j = 0; j < VPL; ++j) {
                    int e = expert_of<VPL>(lane, j);
                    if (e < E) part += (double)exp_s(__fsub_rn(xv[j], m));
                }
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(FULL, part, o);
                wv = (float)((double)exp_s(__fsub_rn(xs, m)) / part);
            }
        } else {
            float s = mine ? sig_s(xs) : 0.f;
            if (prm.renormalize) {
                float Z = __shfl_sync(FULL, s, 0);
                for (int q = 1; q < k; ++q) Z = __fadd_rn(Z, __shfl_sync(FULL, s, q));
                wv = __fdiv_rn(s, Z);
            } else {
                wv = s;
            }
        }
        if (prm.scale != 1.0f) wv = __fmul_rn(wv, prm.scale);
        if (mine) {
            prm.idx[tok * k + lane] = selidx;
            prm.w[tok * k + lane] = wv;
        }
    }
}

template <int VPL>
static int launch_vpl(const GateParams &prm, cudaStream_t st)
{
    const int threads = 256;
    int64_t warps_needed = prm.LT;
    int64_t blocks = (warps_needed + 7) / 8;
    int64_t cap_blocks = (int64_t)sm_count() * 8;
    if (blocks > cap_blocks) blocks = cap_blocks;
    if (blocks < 1) blocks = 1;
    {
        KernelTimerScope ts("gate_topk", st);
        gate_topk_kernel<VPL><<<(unsigned)blocks, threads, 0, st>>>(prm);
    }
    note_launch();
    return check_launch("gate_topk_kernel");
}

int launch_gate_topk(const float *logits, const float *bias, int32_t L, int64_t T,
                     const cap_gate_cfg &cfg, int32_t *idx, float *w, cudaStream_t st)
{
    bool fast = false;
    CAP_TRY(launch_gate_fast(logits, bias, L, T, cfg, idx, w, st, &fast));
    if (fast) return CAP_OK;
    CAP_TRY(launch_gate_sig(logits, bias, L, T, cfg, idx, w, st, &fast));
    if (fast) return CAP_OK;
    CAP_TRY(launch_gate_wide(logits, bias, L, T, cfg, idx, w, st, &fast));
    if (fast) return CAP_OK;
    GateParams prm;
    prm.logits = logits;
    prm.bias = bias;
    prm.idx = idx;
    prm.w = w;
    prm.LT = (int64_t)L * T;
    prm.T = T > 0 ? T : 1;
    prm.E = cfg.E;
    prm.k = cfg.k;
    prm.scoring = cfg.scoring;
    prm.renormalize = cfg.renormalize;
    prm.n_group = cfg.n_group;
    prm.topk_group = cfg.topk_group;
    prm.group_score = cfg.group_score;
    prm.scale = cfg.scale;
    prm.vec = (cfg.E % 4 == 0) && ((reinterpret_cast<uintptr_t>(logits) & 15u) == 0);
    if (prm.LT == 0) return CAP_OK;
    const int E = cfg.E;
    if (E <= 32) return launch_vpl<1>(prm, st);
    if (E <= 64) return launch_vpl<2>(prm, st);
    if (E <= 128) return launch_vpl<4>(prm, st);
    if (E <= 256) return launch_vpl<8>(prm, st);
    if (E <= 512) return launch_vpl<16>(prm, st);
    return launch_vpl<32>(prm, st);
}

}  // namespace cap

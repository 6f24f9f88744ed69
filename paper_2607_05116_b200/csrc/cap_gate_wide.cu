// S1 fast path for wide routers (Eq. 1; BASELINE.json config 5: E = 512, top-10): softmax scoring,
// renormalised weights, no group limit, k <= 10, E = 512.  Same ring as cap_gate_fast.cu -- persistent blocks,
// producer warps stream 16-token tiles of logits (32 KB) into shared memory with TMA bulk copies -- but a token
// gets FOUR lanes and a tile two warps (8 tokens each): with two lanes per token and one warp per tile only as
// many warps worked as the ring has stages (6), and ncu showed the kernel waiting, not issuing.  Each lane
// streams a quarter row (128 logits): groups of 8 are sorted by the 19-comparator network and merged into a
// running sorted top-12 (half-cleaner against the lower part of the list + pruned bitonic merge), in a rolled loop
// (unrolled it would not fit the instruction cache); the four lists are merged by two butterfly steps.
// Keys are the logits' own bit patterns with the low byte replaced by the position in the quarter row (fp32
// min / max order them); for the cross-lane merges the low NINE bits become the expert index.  A payload can
// only decide a comparison between keys that agree in all upper bits: if two neighbours among the 11 largest
// agree in their upper 23 bits, or one of them is a zero, the warp redoes the token with exact comparisons
// (k rounds of warp-wide arg-max, ties to the lower index), so the result is always the exact top-k.  The
// generic warp-per-token kernel it replaces here ran 1.8 k warp instructions per token (ncu,
// profiles/r2d_step.md); this one ~0.4 k.
#include "cap_async.cuh"
#include "cap_gate_fast.cuh"

namespace cap {

constexpr int GW_E = 512;
constexpr int GW_NP = 2;                       // producer warps
constexpr int GW_NC = 12;                      // consumer warps
constexpr int GW_THREADS = 32 * (GW_NC + GW_NP);
constexpr int GW_NST = 6;                      // stages of 16 tokens x 2 KB
constexpr int GW_TILE = 16;

struct GateWideParams {
    const float *logits;
    int32_t *idx;
    float *w;
    int64_t LT;
    int64_t tiles_per_cta;
    int32_t k;
    float scale;
};

// r[0..11] (sorted descending) <- the 12 largest of r[0..11] and g (8 keys, sorted descending).  It is the
// merge of a sorted 16-list with a sorted 8-list (half-cleaner r[8 + i] = max(r[8 + i], g[7 - i]), then a bitonic
// merge over distances 8, 4, 2, 1) with r[12..15] = -inf, written out with everything that only feeds positions
// 12..15 left out: the half-cleaner moves g[3..0] into those four positions (t), the distance-4 stage keeps only
// the maxima of (8..11, 12..15), the last two stages skip them: 56 min / max instead of 72.  k <= 10 needs the 11
// largest keys.
__device__ __forceinline__ void merge8_into12(float (&r)[16], const float (&g)[8])
{
    float t0 = g[3], t1 = g[2], t2 = g[1], t3 = g[0];
    r[8] = kmax(r[8], g[7]); r[9] = kmax(r[9], g[6]); r[10] = kmax(r[10], g[5]); r[11] = kmax(r[11], g[4]);
    CAP_CE(r[0], r[8]); CAP_CE(r[1], r[9]); CAP_CE(r[2], r[10]); CAP_CE(r[3], r[11]);
    CAP_CE(r[4], t0); CAP_CE(r[5], t1); CAP_CE(r[6], t2); CAP_CE(r[7], t3);
    CAP_CE(r[0], r[4]); CAP_CE(r[1], r[5]); CAP_CE(r[2], r[6]); CAP_CE(r[3], r[7]);
    r[8] = kmax(r[8], t0); r[9] = kmax(r[9], t1); r[10] = kmax(r[10], t2); r[11] = kmax(r[11], t3);
    CAP_CE(r[0], r[2]); CAP_CE(r[1], r[3]); CAP_CE(r[4], r[6]); CAP_CE(r[5], r[7]);
    CAP_CE(r[8], r[10]); CAP_CE(r[9], r[11]);
    CAP_CE(r[0], r[1]); CAP_CE(r[2], r[3]); CAP_CE(r[4], r[5]); CAP_CE(r[6], r[7]);
    CAP_CE(r[8], r[9]); CAP_CE(r[10], r[11]);
}

// exact top-k (k <= 16) of one row of 512 logits by the whole warp: lane l holds experts [16 l, 16 l + 16)
__device__ __noinline__ void gate_select_exact_warp16(uint32_t row_smem, int lane, int k, int (&sel)[16])
{
    uint32_t key[16];
#pragma unroll
    for (int j = 0; j < 16; ++j) {
        float x;
        asm volatile("ld.shared.f32 %0, [%1];" : "=f"(x) : "r"(row_smem + (uint32_t)(lane * 16 + j) * 4u));
        key[j] = okey(x);
    }
#pragma unroll 1
    for (int s = 0; s < 16; ++s) {
        int wi = 0;
        if (s < k) {
            uint32_t bk = 0u;
            int bi = 0x7fffffff;
#pragma unroll
            for (int j = 0; j < 16; ++j)
                if (key[j] > bk) { bk = key[j]; bi = lane * 16 + j; }
            const uint32_t m = __reduce_max_sync(0xffffffffu, bk);
            wi = __reduce_min_sync(0xffffffffu, bk == m ? bi : 0x7fffffff);
#pragma unroll
            for (int j = 0; j < 16; ++j)
                if (lane * 16 + j == wi) key[j] = 0u;
        }
#pragma unroll
        for (int i = 0; i < 16; ++i)
            if (i == s) sel[i] = wi;
    }
}

// Lanes l, l ^ 8, l ^ 16, l ^ 24 share token l & 7 of the warp's eight; quarter qd = l >> 3 streams experts
// [128 qd, 128 qd + 128) of the row (2 KB, 512-byte aligned quarters; lane t reads 16-byte chunk c of its quarter
// at chunk position c ^ (t & 7), as in cap_gate_fast.cuh).  All four lanes end with the same list.
__device__ __forceinline__ void gate_select_quad512(const float *row, int qd, int t7, int k, int (&sel)[16])
{
    const uint32_t hb = (smem_u32(row) + (uint32_t)qd * 512u) | ((uint32_t)t7 << 4);
    float r[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) r[i] = __uint_as_float(0xff800000u);          // -inf: below every finite key
#pragma unroll 1
    for (int gi = 0; gi < 16; ++gi) {
        float4 va, vb;
        asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];"
                     : "=f"(va.x), "=f"(va.y), "=f"(va.z), "=f"(va.w)
                     : "r"(hb ^ (uint32_t)(gi * 32)));
        asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];"
                     : "=f"(vb.x), "=f"(vb.y), "=f"(vb.z), "=f"(vb.w)
                     : "r"(hb ^ (uint32_t)(gi * 32 + 16)));
        // position gi * 8 + j in the low byte (one byte permute per element)
        const uint32_t p0 = 0x03020100u + 0x04040404u * (uint32_t)(2 * gi), p1 = p0 + 0x04040404u;
        float g[8];
        g[0] = __uint_as_float(__byte_perm(__float_as_uint(va.x), p0, 0x3214u));
        g[1] = __uint_as_float(__byte_perm(__float_as_uint(va.y), p0, 0x3215u));
        g[2] = __uint_as_float(__byte_perm(__float_as_uint(va.z), p0, 0x3216u));
        g[3] = __uint_as_float(__byte_perm(__float_as_uint(va.w), p0, 0x3217u));
        g[4] = __uint_as_float(__byte_perm(__float_as_uint(vb.x), p1, 0x3214u));
        g[5] = __uint_as_float(__byte_perm(__float_as_uint(vb.y), p1, 0x3215u));
        g[6] = __uint_as_float(__byte_perm(__float_as_uint(vb.z), p1, 0x3216u));
        g[7] = __uint_as_float(__byte_perm(__float_as_uint(vb.w), p1, 0x3217u));
        sort8_desc(g);
        merge8_into12(r, g);                  // r[12..15] stay -inf
    }
    // low nine bits <- expert index: undo the chunk swizzle (XOR of position bits 2..4), add 128 qd
    const uint32_t swz = (uint32_t)t7 << 2, qbits = (uint32_t)qd << 7;
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        const uint32_t u = __float_as_uint(r[i]);
        r[i] = __uint_as_float((u & 0xfffffe00u) | qbits | ((u & 0x7fu) ^ swz));
    }
    // two butterfly steps over the four quarters: the partner's list reversed, element-wise max, bitonic merge
#pragma unroll
    for (int off = 8; off <= 16; off <<= 1) {
        float gp[16];
#pragma unroll
        for (int i = 0; i < 16; ++i) gp[i] = __shfl_xor_sync(0xffffffffu, r[15 - i], off);
#pragma unroll
        for (int i = 0; i < 16; ++i) r[i] = kmax(r[i], gp[i]);
#pragma unroll
        for (int s = 8; s >= 1; s >>= 1) {
#pragma unroll
            for (int i = 0; i < 16; ++i)
                if ((i & s) == 0) CAP_CE(r[i], r[i + s]);
        }
    }
    // ambiguous: neighbours among the 11 largest that agree in every bit above the payload, or a zero among them
    bool amb = false;
#pragma unroll
    for (int i = 0; i < 10; ++i) amb |= ((__float_as_uint(r[i]) ^ __float_as_uint(r[i + 1])) >> 9) == 0u;
#pragma unroll
    for (int i = 0; i < 11; ++i) amb |= (__float_as_uint(r[i]) & 0x7ffffe00u) == 0u;
#pragma unroll
    for (int i = 0; i < 16; ++i) sel[i] = (int)(__float_as_uint(r[i]) & 0x1ffu);
    const int lane = (int)(threadIdx.x & 31u);
    unsigned todo = __ballot_sync(0xffffffffu, amb) & 0xffu;       // one lane of each quad
    const uint32_t row_s = smem_u32(row);
    while (todo) {
        const int src = __ffs((int)todo) - 1;
        todo &= todo - 1u;
        const uint32_t rs = __shfl_sync(0xffffffffu, row_s, src);
        int ex[16];
        gate_select_exact_warp16(rs, lane, k, ex);
        if ((lane & 7) == src) {
#pragma unroll
            for (int i = 0; i < 16; ++i) sel[i] = ex[i];
        }
    }
}

// Renormalised softmax weights (DESIGN.md R-S1.3): r_s = expS(x_s - x_0), Z summed in slot order, w_s = r_s / Z
// (* scale).  Quarter lane qd evaluates slots 4 qd .. 4 qd + 3; w[0..4) = their weights.
__device__ __forceinline__ void gate_weights_softmax_quad16(const float *row, int qd, int k, const int (&sel)[16],
                                                            float scale, float (&w)[4])
{
    const float x0 = row[sel[0]];
    const int lane = (int)(threadIdx.x & 31u);
    float mine[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        int e = 0;
#pragma unroll
        for (int s = 0; s < 16; ++s) e = (s == 4 * qd + j) ? sel[s] : e;
        mine[j] = 4 * qd + j < k ? exp_s(__fsub_rn(row[e], x0)) : 0.0f;
    }
    float Z = 0.0f;
#pragma unroll
    for (int s = 0; s < 16; ++s) {
        const float rs = __shfl_sync(0xffffffffu, mine[s & 3], (lane & 7) | ((s >> 2) << 3));
        if (s == 0) Z = rs;
        else if (s < k) Z = __fadd_rn(Z, rs);
    }
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        float v = __fdiv_rn(mine[j], Z);
        if (scale != 1.0f) v = __fmul_rn(v, scale);
        w[j] = v;
    }
}

__global__ void __launch_bounds__(GW_THREADS) gate_wide_kernel(GateWideParams q)
{
    extern __shared__ __align__(1024) unsigned char gw_sm[];
    __shared__ uint64_t full_bar[GW_NST], empty_bar[GW_NST];
    // use number of every stage (more consumer warps than stages: a warp first waits until the stage is in ITS use,
    // then on the barrier's parity; cap_gate_sig.cu)
    __shared__ uint32_t stage_use[GW_NST];
    constexpr int ROWB = GW_E * 4;
    constexpr int STAGEB = GW_TILE * ROWB;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int s = 0; s < GW_NST; ++s) {
            mbar_init(&full_bar[s], 1);
            mbar_init(&empty_bar[s], 2);            // the two warps of a tile
            stage_use[s] = 0xffffffffu;
        }
        mbar_fence_init();
    }
    __syncthreads();
    const int64_t ntiles = (q.LT + GW_TILE - 1) / GW_TILE;
    const int64_t tile0 = (int64_t)blockIdx.x * q.tiles_per_cta;
    int64_t nt = ntiles - tile0;
    if (nt > q.tiles_per_cta) nt = q.tiles_per_cta;
    if (nt <= 0) return;

    if (warp < GW_NP) {
        if (lane == 0) {
            for (int64_t j = warp; j < nt; j += GW_NP) {
                const int st = (int)(j % GW_NST);
                if (j >= GW_NST) mbar_wait(&empty_bar[st], (uint32_t)(((j / GW_NST) - 1) & 1));
                const int64_t tok0 = (tile0 + j) * GW_TILE;
                const int rows = (int)min((int64_t)GW_TILE, q.LT - tok0);
                st_release_shared(&stage_use[st], (uint32_t)(j / GW_NST));
                mbar_expect_tx(&full_bar[st], (uint32_t)rows * ROWB);
                bulk_g2s(gw_sm + (size_t)st * STAGEB, q.logits + tok0 * GW_E, (uint32_t)rows * ROWB, &full_bar[st]);
            }
        }
    } else {
        // consumers: warps 2m and 2m + 1 share tiles m, m + NC / 2, ...; each takes eight of the tile's tokens
        const int c = warp - GW_NP;
        const int k = q.k;
        const int sub = c & 1, qd = lane >> 3, tl = lane & 7;
        for (int64_t j = c >> 1; j < nt; j += GW_NC / 2) {
            const int st = (int)(j % GW_NST);
            const uint32_t use = (uint32_t)(j / GW_NST);
            while (ld_acquire_shared(&stage_use[st]) != use) __nanosleep(32);
            mbar_wait(&full_bar[st], use & 1u);
            const int64_t tok = (tile0 + j) * GW_TILE + 8 * sub + tl;
            const bool valid = tok < q.LT;
            // rows past the end of a ragged last tile were not written: those lanes redo row 0
            const float *row =
                reinterpret_cast<const float *>(gw_sm + (size_t)st * STAGEB + (valid ? 8 * sub + tl : 0) * ROWB);
            int sel[16];
            float wv[4];
            gate_select_quad512(row, qd, tl, k, sel);
            gate_weights_softmax_quad16(row, qd, k, sel, q.scale, wv);
            if (valid) {
#pragma unroll
                for (int jj = 0; jj < 4; ++jj) {
                    const int s = 4 * qd + jj;
                    int e = 0;
#pragma unroll
                    for (int i = 0; i < 16; ++i) e = (i == s) ? sel[i] : e;
                    if (s < k) {
                        q.idx[tok * k + s] = e;
                        q.w[tok * k + s] = wv[jj];
                    }
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty_bar[st]);
        }
    }
}

int launch_gate_wide(const float *logits, const float *bias, int32_t L, int64_t T, const cap_gate_cfg &cfg,
                     int32_t *idx, float *w, cudaStream_t st, bool *used)
{
    *used = false;
    if (cfg.scoring != 0 || cfg.renormalize != 1 || cfg.n_group != 1 || bias != nullptr) return CAP_OK;
    if (cfg.E != GW_E || cfg.k > 10) return CAP_OK;
    if (reinterpret_cast<uintptr_t>(logits) & 15u) return CAP_OK;
    GateWideParams prm;
    prm.logits = logits;
    prm.idx = idx;
    prm.w = w;
    prm.LT = (int64_t)L * T;
    prm.k = cfg.k;
    prm.scale = cfg.scale;
    prm.tiles_per_cta = 0;
    *used = true;
    if (prm.LT == 0) return CAP_OK;
    constexpr int STAGEB = GW_TILE * GW_E * 4;
    cudaFuncSetAttribute(gate_wide_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, GW_NST * STAGEB + 1024);
    const int64_t ntiles = (prm.LT + GW_TILE - 1) / GW_TILE;
    int64_t grid = sm_count();
    if (grid > ntiles) grid = ntiles;
    prm.tiles_per_cta = (ntiles + grid - 1) / grid;
    grid = (ntiles + prm.tiles_per_cta - 1) / prm.tiles_per_cta;
    {
        KernelTimerScope ts("gate_topk", st);
        gate_wide_kernel<<<(unsigned)grid, GW_THREADS, (size_t)GW_NST * STAGEB, st>>>(prm);
    }
    note_launch();
    return check_launch("gate_wide_kernel");
}

}  // namespace cap

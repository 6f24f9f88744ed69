// cap_trace_fused, single-launch kernel (round 2): S1 (gate top-k) + S2 (counts / co-activation) + S3
// (scoring of P candidate placements) AND every reduction behind them in ONE cooperative launch
// (BASELINE.json north_star; Eq. 1, P:L104 / L148, P:L58 / Eq. 3 / Eq. 4).
//
// What changed against cap_fused.cu (kept as the fallback for the shapes this kernel does not take):
//   * no table kernel: the S3 warps build the one-hot code tables in shared memory straight from the
//     caller's expert -> device maps while the first logits tiles are in flight;
//   * no decode / finalize kernels and no pre-zeroed accumulators: a block leaves its co-activation
//     accumulator (TMEM) and its decoded per-run counters as plain partial results in the workspace,
//     one grid-wide barrier follows, then every block reduces its slice of the partials and finishes
//     its share of the candidates (costs, bytes, load_pairs, imbalance);
//   * S3 threads own 16-byte table columns and a warp owns whole tokens (32 / C tokens per load for a
//     row of C chunks), device codes and node codes are separate tables served by separate warps of
//     the same code: every row load is one conflict-free LDS.128 wavefront set, and the layout is the
//     one a TMEM-resident table needs (tcgen05.ld 32x32b.x4);
//   * more S1 warps (the block is 704 threads: 1 producer, 1 tensor-core warp, C_dev/4 + C_node/4
//     scoring warps, the rest S1).
// Roles are handed over through mbarriers exactly as before: TMA producer -> S1 (logits ring), S1 ->
// tensor-core warp (one-hot tiles), S1 -> S3 (row descriptors of 64-token blocks).
#include <cooperative_groups.h>

#include <cstdio>
#include <cstdlib>

#include "cap_async.cuh"
#include "cap_eval_fast.cuh"
#include "cap_gate_fast.cuh"
#include "cap_tc.cuh"

namespace cg = cooperative_groups;

namespace cap {

constexpr int F2_TILE = 16;          // tokens per S1 tile (two lanes per token)
constexpr int F2_BT = 64;            // tokens per S3 block = tokens per MMA tile
constexpr int F2_TPB = F2_BT / F2_TILE;
constexpr int F2_OB = 4;             // descriptor blocks in flight between S1 and S3
constexpr int F2_MAXST = 24;         // logits ring stages
constexpr int F2_THREADS = 704;      // 22 warps
constexpr int F2_MAXRUNBLK = 29;     // 64-token blocks per run: <= 31 CSA rounds of 8 inputs < 256
constexpr int F2_NPL = 11;           // planes of a run after its 8 partial counters were added
constexpr int F2_CG = 4;             // candidates a block finishes per round of phase 1
constexpr int F2_MAXSLOTS = 4096;    // records per layer the finishing phase can index

struct F2Params {
    const float *logits;
    int32_t *idx;
    float *w;
    long long *counts;            // [L][E]
    int *coact;                   // [L][E][E]
    const int32_t *maps;          // [L][P][E]
    const int32_t *dev_node;      // [D]
    cap_eval_out out;
    int *partC;                   // [L][nblk][EP * EP] raw accumulator images
    uint32_t *partCnt;            // [L][nblk][E]
    uint32_t *recs;               // [L][nblk][maxrec][ncnt]
    int32_t *rec_src;             // [L][nblk][maxrec], -1 = unused
    int64_t T, tiles_per_cta;
    int32_t cps;
    float scale;
    int32_t k, D, N, P, WD, WN, Cd, Cn, nwd, nwn, nst, maxrec, ncnt, ndev;
    int32_t cost_local, cost_intra, cost_inter;
    long long bytes_per_token;
};

struct F2Smem {
    uint32_t ring, tiles, tabD, tabN, offs, xch, total;
};

__host__ __device__ inline F2Smem f2_smem_layout(int E, int EP, int Cd, int Cn, int nwd, int nwn, int nst)
{
    F2Smem m;
    uint32_t o = 0;
    m.ring = o;
    o += (uint32_t)nst * F2_TILE * E * 4;
    m.tiles = o;
    o += 2u * EP * F2_BT;
    m.tabD = o;                                   // rows of 16 Cd bytes, 512-byte aligned
    o += (uint32_t)E * Cd * 16;
    m.tabN = o;
    o += (uint32_t)E * Cn * 16;
    m.offs = o;                                   // [F2_OB][64 tokens][2 classes][8 slots] row descriptors
    o += (uint32_t)F2_OB * F2_BT * 16 * 4;
    m.xch = o;                                    // plane exchange of the flush, then the planes to decode
    const uint32_t hd = (uint32_t)(nwd / 2 > 0 ? nwd / 2 : 0), hn = (uint32_t)(nwn / 2 > 0 ? nwn / 2 : 0);
    uint32_t x = (hd + hn) * 32u * F2_NPL * 16u;
    const uint32_t fin = (uint32_t)(Cd + Cn) * 16u * F2_NPL;
    if (x < fin) x = fin;
    o += x;
    m.total = o;
    return m;
}

__device__ __forceinline__ void st_release_cta(uint32_t *p, uint32_t v)
{
    asm volatile("st.release.cta.shared::cta.u32 [%0], %1;" ::"r"(smem_u32(p)), "r"(v) : "memory");
}
__device__ __forceinline__ uint32_t ld_acquire_cta(const uint32_t *p)
{
    uint32_t v;
    asm volatile("ld.acquire.cta.shared::cta.u32 %0, [%1];" : "=r"(v) : "r"(smem_u32(p)) : "memory");
    return v;
}
__device__ __forceinline__ uint4 ld_acquire_cta_v4(const uint32_t *p)
{
    // four relaxed loads and one acquire fence: the counters are written with st.release by single writers
    uint4 v;
    asm volatile("ld.relaxed.cta.shared::cta.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w)
                 : "r"(smem_u32(p))
                 : "memory");
    asm volatile("fence.acq_rel.cta;" ::: "memory");
    return v;
}

__device__ __forceinline__ void f2_bar(int id, int nthreads)
{
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

// ---- table build: one item = (expert e, 16 consecutive candidates) --------------------------------------
template <int WD, int WN>
__device__ __forceinline__ void f2_build_items(const int32_t *__restrict__ maps, const unsigned char *node_of, int E,
                                               int P, int D, int Cd, int Cn, unsigned char *tabD, unsigned char *tabN,
                                               int t3, int ns3)
{
    constexpr int DWORDS = 16 * WD / 32;          // device-code words of an item (4 .. 32)
    constexpr int NWORDS = 16 * WN / 32;          // node-code words of an item (1, 2, 4)
    const int padD = Cd * 128 / WD, padN = Cn * 128 / WN;     // candidates a row has room for
    const int np16 = ((padD > padN ? padD : padN) + 15) / 16;
    const int nitems = E * np16;
    for (int it = t3; it < nitems; it += ns3) {
        const int p16 = it / E, e = it - p16 * E;
        const int p0 = p16 * 16;
        int dv[16];
#pragma unroll
        for (int j = 0; j < 16; ++j) dv[j] = (p0 + j < P) ? maps[(size_t)(p0 + j) * E + e] : -1;
        uint32_t dw[DWORDS], nw[NWORDS];
#pragma unroll
        for (int j = 0; j < DWORDS; ++j) dw[j] = 0u;
#pragma unroll
        for (int j = 0; j < NWORDS; ++j) nw[j] = 0u;
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            const int d = dv[j];
            if ((unsigned)d < (unsigned)D) {
                if (WD == 64) {
                    dw[2 * j] |= d < 32 ? 1u << d : 0u;
                    dw[2 * j + 1] |= d >= 32 ? 1u << (d - 32) : 0u;
                } else {
                    dw[(j * WD) / 32] |= 1u << (((j * WD) % 32) + d);
                }
                nw[(j * WN) / 32] |= 1u << (((j * WN) % 32) + (node_of[d] & (WN - 1)));
            }
        }
        if (p0 < padD) {
            const int c0 = p0 * WD / 128;
            unsigned char *row = tabD + (size_t)e * Cd * 16;
#pragma unroll
            for (int q = 0; q < DWORDS / 4; ++q)
                if (c0 + q < Cd)
                    *reinterpret_cast<uint4 *>(row + 16 * ((c0 + q) ^ (e & (Cd - 1)))) =
                        make_uint4(dw[4 * q], dw[4 * q + 1], dw[4 * q + 2], dw[4 * q + 3]);
        }
        if (p0 < padN) {
            const int w0 = p0 * WN / 32;
            unsigned char *row = tabN + (size_t)e * Cn * 16;
#pragma unroll
            for (int q = 0; q < NWORDS; ++q) {
                const int wq = w0 + q;
                if ((wq >> 2) < Cn) *reinterpret_cast<uint32_t *>(row + 16 * ((wq >> 2) ^ (e & (Cn - 1))) + 4 * (wq & 3)) = nw[q];
            }
        }
    }
}

__device__ __noinline__ void f2_build_tables(const int32_t *__restrict__ maps, const unsigned char *node_of, int E, int P,
                                             int D, int WD, int WN, int Cd, int Cn, unsigned char *tabD,
                                             unsigned char *tabN, int t3, int ns3)
{
#define F2_B(wd, wn) f2_build_items<wd, wn>(maps, node_of, E, P, D, Cd, Cn, tabD, tabN, t3, ns3)
    switch (WD * 16 + WN) {
    case 8 * 16 + 2: F2_B(8, 2); break;
    case 8 * 16 + 4: F2_B(8, 4); break;
    case 8 * 16 + 8: F2_B(8, 8); break;
    case 16 * 16 + 2: F2_B(16, 2); break;
    case 16 * 16 + 4: F2_B(16, 4); break;
    case 16 * 16 + 8: F2_B(16, 8); break;
    case 32 * 16 + 2: F2_B(32, 2); break;
    case 32 * 16 + 4: F2_B(32, 4); break;
    case 32 * 16 + 8: F2_B(32, 8); break;
    case 64 * 16 + 2: F2_B(64, 2); break;
    case 64 * 16 + 4: F2_B(64, 4); break;
    default: F2_B(64, 8); break;
    }
#undef F2_B
}

// ---- bit-sliced helpers on 16-byte columns ----------------------------------------------------------------
#define F2_CSA4(S, Cy, A, B, X)                    \
    do {                                           \
        CAP_CSA((S).x, (Cy).x, (A).x, (B).x, (X).x); \
        CAP_CSA((S).y, (Cy).y, (A).y, (B).y, (X).y); \
        CAP_CSA((S).z, (Cy).z, (A).z, (B).z, (X).z); \
        CAP_CSA((S).w, (Cy).w, (A).w, (B).w, (X).w); \
    } while (0)

// OR of the eight table rows of one token at this lane's 16-byte column (descriptors: absolute shared
// addresses of the rows with the row's swizzle seed in the chunk bits; cx = this lane's chunk << 4)
__device__ __forceinline__ uint4 f2_token_mask(const uint32_t *od, uint32_t cx)
{
    const uint4 oa = *reinterpret_cast<const uint4 *>(od);
    const uint4 ob = *reinterpret_cast<const uint4 *>(od + 4);
    uint4 v[8];
#define F2_LD(i, a) \
    asm("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v[i].x), "=r"(v[i].y), "=r"(v[i].z), "=r"(v[i].w) : "r"((a) ^ cx))
    F2_LD(0, oa.x); F2_LD(1, oa.y); F2_LD(2, oa.z); F2_LD(3, oa.w);
    F2_LD(4, ob.x); F2_LD(5, ob.y); F2_LD(6, ob.z); F2_LD(7, ob.w);
#undef F2_LD
    uint4 m;
#define F2_OR(F) m.F = lop_or3(lop_or3(lop_or3(v[0].F, v[1].F, v[2].F), v[3].F, v[4].F), lop_or3(v[5].F, v[6].F, v[7].F), 0u)
    F2_OR(x); F2_OR(y); F2_OR(z); F2_OR(w);
#undef F2_OR
    return m;
}

// a (np planes) += b (np planes), result has np + 1 planes (bit-sliced ripple add)
__device__ __forceinline__ void f2_add_planes(uint4 (&a)[F2_NPL], const uint4 (&b)[F2_NPL], int np)
{
    uint4 cy = make_uint4(0u, 0u, 0u, 0u);
#pragma unroll
    for (int p = 0; p < F2_NPL; ++p) {
        if (p <= np) {
            const uint4 x = p < np ? b[p] : make_uint4(0u, 0u, 0u, 0u);
            uint4 s, c;
            F2_CSA4(s, c, a[p], x, cy);
            a[p] = s;
            cy = c;
        }
    }
}

template <int E>
__global__ void __launch_bounds__(F2_THREADS, 1) trace_fused2_kernel(const F2Params q)
{
    extern __shared__ __align__(1024) unsigned char f2_sm[];
    __shared__ uint64_t full_bar[F2_MAXST], empty_bar[F2_MAXST];
    __shared__ uint64_t offs_full[F2_OB];
    __shared__ uint64_t tile_full[2], mma_done[2];
    // progress counters of the two back edges (S3 -> S1: descriptor blocks consumed by each scoring warp;
    // tensor-core warp -> S1: one-hot tile buffers recycled).  Plain monotonic counters instead of parity
    // barriers: an S1 warp visits only every ns1w-th tile, so it can be several phases ahead of a barrier
    // it has never waited on, which a parity wait cannot tell from "already complete".
    __shared__ __align__(16) uint32_t s3_prog[16];
    __shared__ uint32_t s_recycled;
    __shared__ uint64_t acc_done;
    __shared__ uint32_t s_tmem;
    __shared__ unsigned char s_node[64];
    constexpr int EP = E <= 128 ? 128 : 256;
    constexpr uint32_t LBO = 128u, SBO = (F2_BT / 16) * 128u;
    constexpr uint32_t NCOLS = EP == 128 ? 128u : 512u;
    constexpr uint32_t IDESC = (2u << 4) | ((uint32_t)(EP >> 3) << 17) | (8u << 24);
    constexpr int TILE_BYTES = F2_TILE * E * 4;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int nthr = blockDim.x;
    const int layer = blockIdx.y, blk = blockIdx.x, nblk = gridDim.x;
    const int nst = q.nst, k = q.k, D = q.D;
    const int ns3w = q.nwd + q.nwn, ns3 = ns3w * 32;
    const int s1w0 = 2 + ns3w;                           // first S1 warp
    const int ns1w = (nthr >> 5) - s1w0;
    const F2Smem lay = f2_smem_layout(E, EP, q.Cd, q.Cn, q.nwd, q.nwn, nst);
    unsigned char *ring = f2_sm + lay.ring;
    unsigned char *tiles = f2_sm + lay.tiles;
    unsigned char *tabD = f2_sm + lay.tabD;
    unsigned char *tabN = f2_sm + lay.tabN;
    uint32_t *offs = reinterpret_cast<uint32_t *>(f2_sm + lay.offs);
    uint4 *xch = reinterpret_cast<uint4 *>(f2_sm + lay.xch);

    // ---- this block's token range [t0, t1) of one layer (same two splits as cap_fused.cu) ----
    const int64_t T = q.T;
    int64_t t0, t1;
    if (q.cps > 0) {
        const int srcd = blk / q.cps, jj = blk % q.cps;
        const int64_t b0 = ((int64_t)srcd * T + D - 1) / D, b1 = ((int64_t)(srcd + 1) * T + D - 1) / D;
        const int64_t nts = (b1 - b0 + F2_TILE - 1) / F2_TILE;
        const int64_t base = nts / q.cps, rem = nts % q.cps;
        const int64_t ts = jj * base + (jj < rem ? jj : rem), tn = base + (jj < rem ? 1 : 0);
        t0 = min(b1, b0 + ts * F2_TILE);
        t1 = min(b1, t0 + tn * F2_TILE);
    } else {
        t0 = min(T, (int64_t)blk * q.tiles_per_cta * F2_TILE);
        t1 = min(T, t0 + q.tiles_per_cta * F2_TILE);
    }
    const int nt = (int)((t1 - t0 + F2_TILE - 1) / F2_TILE);
    const int ntp = ((nt + F2_TPB - 1) / F2_TPB) * F2_TPB;      // with ghost tiles: whole 64-token blocks
    const int nb = ntp / F2_TPB;
    const float *logits = q.logits + (size_t)layer * T * E;
    int32_t *gidx = q.idx + (size_t)layer * T * k;
    float *gw = q.w + (size_t)layer * T * k;
    const size_t pslot = (size_t)layer * nblk + blk;           // this block's partial-result slot
    int *partC = q.partC + pslot * (size_t)(EP * EP);
    uint32_t *partCnt = q.partCnt + pslot * E;
    const size_t slot0 = pslot * q.maxrec;

    // ---- set-up ----
    if (tid == 0) {
        for (int s = 0; s < nst; ++s) {
            mbar_init(&full_bar[s], 1);
            mbar_init(&empty_bar[s], 1);
        }
        for (int s = 0; s < F2_OB; ++s) mbar_init(&offs_full[s], F2_TPB);
        for (int s = 0; s < 2; ++s) {
            mbar_init(&tile_full[s], F2_TPB);
            mbar_init(&mma_done[s], 1);
        }
        for (int s = 0; s < 16; ++s) s3_prog[s] = s < ns3w ? 0u : 0x7fffffffu;
        s_recycled = 0u;
        mbar_init(&acc_done, 1);
        mbar_fence_init();
    }
    if (warp == 1) tmem_alloc(&s_tmem, NCOLS);
    {
        uint4 *z = reinterpret_cast<uint4 *>(tiles);
        for (int i = tid; i < 2 * EP * F2_BT / 16; i += nthr) z[i] = make_uint4(0u, 0u, 0u, 0u);
    }
    if (tid < 64) s_node[tid] = tid < D ? (unsigned char)(q.dev_node[tid] & 63) : 0;
    if (tid >= 64 && tid < 64 + q.maxrec) q.rec_src[slot0 + (tid - 64)] = -1;
    proxy_fence_async();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = s_tmem;

    if (warp == 0) {
        // ================= producer =================
        if (lane == 0) {
            for (int j = 0; j < nt; ++j) {
                const int st = j % nst;
                if (j >= nst) mbar_wait_relaxed(&empty_bar[st], (uint32_t)(((j / nst) - 1) & 1), 128);
                const int64_t tok0 = t0 + (int64_t)j * F2_TILE;
                const int rows = (int)min((int64_t)F2_TILE, t1 - tok0);
                mbar_expect_tx(&full_bar[st], (uint32_t)rows * E * 4);
                bulk_g2s(ring + (size_t)st * TILE_BYTES, logits + tok0 * E, (uint32_t)rows * E * 4, &full_bar[st]);
            }
        }
    } else if (warp == 1) {
        // ================= tensor-core warp: C += A^T A on the one-hot tiles =================
        for (int m = 0; m < nb; ++m) {
            const int tb = m & 1;
            unsigned char *tile = tiles + (size_t)tb * EP * F2_BT;
            mbar_wait_relaxed(&tile_full[tb], (uint32_t)((m >> 1) & 1), 128);
            tc_fence_after();
            if (lane == 0) {
                const uint32_t base = smem_u32(tile);
#pragma unroll
                for (int j = 0; j < F2_BT / 32; ++j) {
                    const uint64_t bd = umma_desc(base + j * 2 * LBO, LBO, SBO);
                    umma_i8(tmem, bd, bd, IDESC, (uint32_t)((m | j) != 0));
                    if (EP == 256) {
                        const uint64_t a1 = umma_desc(base + 16 * SBO + j * 2 * LBO, LBO, SBO);
                        umma_i8(tmem + 256u, a1, bd, IDESC, (uint32_t)((m | j) != 0));
                    }
                }
                umma_commit(&mma_done[tb]);
                if (m == nb - 1) umma_commit(&acc_done);
            }
            __syncwarp();
            if (m + 2 < nb) {
                mbar_wait(&mma_done[tb], (uint32_t)((m >> 1) & 1));
                uint4 *z = reinterpret_cast<uint4 *>(tile);
                for (int i = lane; i < EP * F2_BT / 16; i += 32) z[i] = make_uint4(0u, 0u, 0u, 0u);
                proxy_fence_async();
                __syncwarp();
                if (lane == 0) st_release_cta(&s_recycled, (uint32_t)(m + 1));
            }
        }
    } else if (warp >= s1w0) {
        // ================= S1: gate top-k, two lanes per token =================
        const int c = warp - s1w0;
        const int h = lane >> 4, tl = lane & 15;
        const uint32_t tabD_s = smem_u32(tabD), tabN_s = smem_u32(tabN);
        const uint32_t rowD = (uint32_t)q.Cd * 16u, rowN = (uint32_t)q.Cn * 16u;
        const uint32_t mD = (uint32_t)q.Cd - 1u, mN = (uint32_t)q.Cn - 1u;
        for (int j = c; j < ntp; j += ns1w) {
            const bool ghost = j >= nt;
            const int st = j % nst;
            const int64_t tok = t0 + (int64_t)j * F2_TILE + tl;
            const bool valid = !ghost && tok < t1;
            int sel[8];
#pragma unroll
            for (int i = 0; i < 8; ++i) sel[i] = 0;
            if (!ghost) {
                const int u = j / nst;
                if (u >= 1) mbar_wait(&empty_bar[st], (uint32_t)((u - 1) & 1));
                mbar_wait(&full_bar[st], (uint32_t)(u & 1));
                const float *row = reinterpret_cast<const float *>(ring + (size_t)st * TILE_BYTES +
                                                                   (size_t)(tok < t1 ? tl : 0) * E * 4);
                float wv[4];
                gate_select_pair<E>(row, h, tl & 7, k, sel);
                gate_weights_softmax_pair(row, h, k, sel, q.scale, wv);
                if (valid) {
                    if (k == 8) {
                        *reinterpret_cast<int4 *>(gidx + tok * 8 + 4 * h) =
                            h ? make_int4(sel[4], sel[5], sel[6], sel[7]) : make_int4(sel[0], sel[1], sel[2], sel[3]);
                        *reinterpret_cast<float4 *>(gw + tok * 8 + 4 * h) = make_float4(wv[0], wv[1], wv[2], wv[3]);
                    } else {
#pragma unroll
                        for (int jj = 0; jj < 4; ++jj) {
                            const int s = 4 * h + jj;
                            if (s < k) {
                                gidx[tok * k + s] = h ? sel[4 + jj] : sel[jj];
                                gw[tok * k + s] = wv[jj];
                            }
                        }
                    }
                }
            }
            // ---- row descriptors for S3: slots past k repeat slot 0 (OR is idempotent); tokens past the
            //      range point at row 0 and are masked out by their index ----
            const int b = j / F2_TPB, ob = b % F2_OB;
            if (b >= F2_OB) {
                // every scoring warp must have finished block b - F2_OB (it used this descriptor slot)
                for (;;) {
                    const uint4 p0 = ld_acquire_cta_v4(&s3_prog[0]), p1 = ld_acquire_cta_v4(&s3_prog[4]),
                                p2 = ld_acquire_cta_v4(&s3_prog[8]), p3 = ld_acquire_cta_v4(&s3_prog[12]);
                    const uint32_t m0 = min(min(min(p0.x, p0.y), min(p0.z, p0.w)), min(min(p1.x, p1.y), min(p1.z, p1.w)));
                    const uint32_t m1 = min(min(min(p2.x, p2.y), min(p2.z, p2.w)), min(min(p3.x, p3.y), min(p3.z, p3.w)));
                    if (min(m0, m1) >= (uint32_t)(b - F2_OB + 1)) break;
                    __nanosleep(40);
                }
            }
            {
                uint32_t od[4], on[4];
#pragma unroll
                for (int jj = 0; jj < 4; ++jj) {
                    const int s = 4 * h + jj;
                    const uint32_t e = (uint32_t)(valid ? (s < k ? (h ? sel[4 + jj] : sel[jj]) : sel[0]) : 0);
                    od[jj] = tabD_s + e * rowD + ((e & mD) << 4);
                    on[jj] = tabN_s + e * rowN + ((e & mN) << 4);
                }
                const int slot = (j % F2_TPB) * F2_TILE + tl;
                uint32_t *op = offs + ((size_t)ob * F2_BT + slot) * 16 + 4 * h;
                *reinterpret_cast<uint4 *>(op) = make_uint4(od[0], od[1], od[2], od[3]);
                *reinterpret_cast<uint4 *>(op + 8) = make_uint4(on[0], on[1], on[2], on[3]);
            }
            // ---- one-hot bytes for the co-activation MMA ----
            const int tb = b & 1;
            if (b >= 2)
                while (ld_acquire_cta(&s_recycled) < (uint32_t)(b - 1)) __nanosleep(40);
            if (valid) {
                const int tp = (j % F2_TPB) * F2_TILE + tl;
                unsigned char *col = tiles + (size_t)tb * EP * F2_BT + (tp >> 4) * LBO + (tp & 15);
#pragma unroll
                for (int jj = 0; jj < 4; ++jj) {
                    const int s = 4 * h + jj;
                    const int e = h ? sel[4 + jj] : sel[jj];
                    if (s < k) col[(e >> 3) * SBO + (e & 7) * 16] = 1;
                }
            }
            proxy_fence_async();
            __syncwarp();
            if (lane == 0) {
                mbar_arrive(&offs_full[ob]);
                mbar_arrive(&tile_full[tb]);
                if (!ghost) mbar_arrive(&empty_bar[st]);
            }
        }
        // ---- drain the co-activation accumulator into this block's partial image (plain stores):
        //      image[(half * EP + col) * 128 + row % 128] = C[row][col], lanes = consecutive rows ----
        if (c < 4) {
            const int quad = warp & 3;
            if (nb > 0) {
                mbar_wait_relaxed(&acc_done, 0u, 64);
                tc_fence_after();
            }
#pragma unroll 1
            for (int hh = 0; hh < EP / 128; ++hh) {
                const int r = hh * 128 + quad * 32 + lane;
#pragma unroll 1
                for (int cb = 0; cb < EP / 32; ++cb) {
                    if (cb * 32 >= E || hh * 128 + quad * 32 >= E) continue;
                    uint32_t v[32];
                    if (nb > 0) {
                        tmem_ld32(tmem + ((uint32_t)(quad * 32) << 16) + (uint32_t)(hh * 256 + cb * 32), v);
                    } else {
#pragma unroll
                        for (int j = 0; j < 32; ++j) v[j] = 0u;
                    }
                    int *pp = partC + ((size_t)(hh * EP + cb * 32)) * 128 + quad * 32 + lane;
#pragma unroll
                    for (int j = 0; j < 32; ++j) pp[(size_t)j * 128] = (int)v[j];
                    if ((r >> 5) == cb && r < E) {
                        uint32_t d = 0u;
#pragma unroll
                        for (int j = 0; j < 32; ++j) d = (r & 31) == j ? v[j] : d;
                        partCnt[r] = d;
                    }
                }
            }
        }
    } else {
        // ================= S3: bit-sliced candidate scoring =================
        const int w3 = warp - 2;
        const int t3 = tid - 64;
        f2_build_tables(q.maps + (size_t)layer * q.P * E, s_node, E, q.P, D, q.WD, q.WN, q.Cd, q.Cn, tabD, tabN, t3, ns3);
        f2_bar(1, ns3);
        const int cls = w3 < q.nwd ? 0 : 1;
        const int a = cls ? w3 - q.nwd : w3;               // warp within its class
        const int nwc = cls ? q.nwn : q.nwd;               // warps of the class = C / 4
        const int C = cls ? q.Cn : q.Cd;                   // 16-byte chunks per row
        const int TPW = 32 / C;                            // tokens per load
        const int tk = lane / C, cc = lane - tk * C;
        const uint32_t cx = (uint32_t)cc << 4;
        const int tokw = a * 8 * TPW + tk;                 // + i * TPW: token of input i inside a block
        const int64_t cap_run = (int64_t)F2_MAXRUNBLK * F2_BT;
        uint4 pl[F2_NPL];
#pragma unroll
        for (int p = 0; p < F2_NPL; ++p) pl[p] = make_uint4(0u, 0u, 0u, 0u);
        int nrec = 0, src = 0;
        int64_t rend = t0;
        bool have_run = false;

        auto flush = [&]() {
            // (1) the TPW lanes of a warp that share a chunk: butterfly over the token bits of the lane id
            int np = 8;
            for (int off = C; off < 32; off <<= 1) {
                uint4 o[F2_NPL];
#pragma unroll
                for (int p = 0; p < F2_NPL; ++p) {
                    o[p].x = __shfl_xor_sync(0xffffffffu, pl[p].x, off);
                    o[p].y = __shfl_xor_sync(0xffffffffu, pl[p].y, off);
                    o[p].z = __shfl_xor_sync(0xffffffffu, pl[p].z, off);
                    o[p].w = __shfl_xor_sync(0xffffffffu, pl[p].w, off);
                }
                f2_add_planes(pl, o, np);
                ++np;
            }
            // (2) the warps of a class: tree through shared memory (both classes keep the same barrier count)
            const int xbase = cls ? (q.nwd / 2) * 32 * F2_NPL : 0;
            for (int half = 4; half >= 1; half >>= 1) {
                const bool act = 2 * half <= nwc;
                if (act && a >= half && a < 2 * half) {
#pragma unroll
                    for (int p = 0; p < F2_NPL; ++p) xch[xbase + ((a - half) * F2_NPL + p) * 32 + lane] = pl[p];
                }
                f2_bar(1, ns3);
                if (act && a < half) {
                    uint4 o[F2_NPL];
#pragma unroll
                    for (int p = 0; p < F2_NPL; ++p) o[p] = xch[xbase + (a * F2_NPL + p) * 32 + lane];
                    f2_add_planes(pl, o, np);
                }
                if (act) ++np;
                f2_bar(1, ns3);
            }
            // (3) warp 0 of each class leaves the run's planes as [plane][word] (device words, then node words)
            uint32_t *fin = reinterpret_cast<uint32_t *>(xch);
            const int nwords = (q.Cd + q.Cn) * 4;
            if (a == 0 && tk == 0) {
                const int wb = (cls ? q.Cd * 4 : 0) + cc * 4;
#pragma unroll
                for (int p = 0; p < F2_NPL; ++p)
                    *reinterpret_cast<uint4 *>(fin + (size_t)p * nwords + wb) = pl[p];
            }
            f2_bar(1, ns3);
            // (4) every S3 thread decodes counters: counter i = bit (i & 31) of word i >> 5
            {
                uint32_t *rec = q.recs + (slot0 + nrec) * (size_t)q.ncnt;
                for (int i = t3; i < q.ncnt; i += ns3) {
                    const int wi = i >> 5, bit = i & 31;
                    uint32_t v = 0u;
#pragma unroll
                    for (int p = 0; p < F2_NPL; ++p) v |= ((fin[(size_t)p * nwords + wi] >> bit) & 1u) << p;
                    rec[i] = v;
                }
                if (t3 == 0) q.rec_src[slot0 + nrec] = src;
            }
            f2_bar(1, ns3);
            ++nrec;
#pragma unroll
            for (int p = 0; p < F2_NPL; ++p) pl[p] = make_uint4(0u, 0u, 0u, 0u);
        };

        for (int b = 0; b < nb; ++b) {
            const int ob = b % F2_OB;
            mbar_wait_relaxed(&offs_full[ob], (uint32_t)((b / F2_OB) & 1), 64);
            const int64_t bt0 = t0 + (int64_t)b * F2_BT;
            const int64_t bend = min(bt0 + F2_BT, t1);
            const uint32_t *obuf = offs + ((size_t)ob * F2_BT + tokw) * 16 + cls * 8;
            int64_t cur = bt0;
            while (cur < bend) {
                if (cur >= rend) {
                    if (have_run) flush();
                    src = (int)((cur * D) / T);
                    const int64_t bnd = ((int64_t)(src + 1) * T + D - 1) / D;
                    rend = min(bnd, cur + cap_run);
                    have_run = true;
                }
                const int64_t seg = min(bend, rend);
                const bool whole = cur == bt0 && seg == bt0 + F2_BT;
                uint4 x0, x1, x2, x3, fA, fB;
#define F2_LOAD(X, I)                                                        \
    do {                                                                     \
        X = f2_token_mask(obuf + (size_t)(I) * TPW * 16, cx);                \
        if (!whole) {                                                        \
            const int64_t tkn = bt0 + tokw + (I) * TPW;                      \
            if (tkn < cur || tkn >= seg) X = make_uint4(0u, 0u, 0u, 0u);     \
        }                                                                    \
    } while (0)
#define F2_HALF(OUT4)                                  \
    do {                                               \
        uint4 tA, tB, s;                               \
        F2_CSA4(s, tA, pl[0], x0, x1);                 \
        F2_CSA4(s, tB, s, x2, x3);                     \
        pl[0] = s;                                     \
        F2_CSA4(pl[1], OUT4, pl[1], tA, tB);           \
    } while (0)
                F2_LOAD(x0, 0); F2_LOAD(x1, 1); F2_LOAD(x2, 2); F2_LOAD(x3, 3);
                F2_HALF(fA);
                F2_LOAD(x0, 4); F2_LOAD(x1, 5); F2_LOAD(x2, 6); F2_LOAD(x3, 7);
                F2_HALF(fB);
                {
                    uint4 e8;
                    F2_CSA4(pl[2], e8, pl[2], fA, fB);
#pragma unroll
                    for (int p = 3; p < 8; ++p) {
                        uint4 cy;
                        cy.x = pl[p].x & e8.x; cy.y = pl[p].y & e8.y; cy.z = pl[p].z & e8.z; cy.w = pl[p].w & e8.w;
                        pl[p].x ^= e8.x; pl[p].y ^= e8.y; pl[p].z ^= e8.z; pl[p].w ^= e8.w;
                        e8 = cy;
                    }
                }
#undef F2_LOAD
#undef F2_HALF
                cur = seg;
            }
            __syncwarp();
            if (lane == 0) st_release_cta(&s3_prog[w3], (uint32_t)(b + 1));
        }
        if (have_run) flush();
    }

    // ================= every partial result of the layer is in the workspace =================
    tc_fence_before();
    __threadfence();
    cg::this_grid().sync();
    if (warp == 1) tmem_dealloc(tmem, NCOLS);

    // ---- phase 1a: expert counts of the whole layer (shared memory), written out by block 0 ----
    uint32_t *cnt_s = reinterpret_cast<uint32_t *>(f2_sm);                     // [E]
    unsigned long long *lp_s = reinterpret_cast<unsigned long long *>(f2_sm + 4096);   // [F2_CG][64]
    unsigned long long *rv_s = lp_s + F2_CG * 64;                              // [F2_CG][64] received tokens
    unsigned long long *sc_s = rv_s + F2_CG * 64;                              // [F2_CG][8] scalar sums
    signed char *src_s = reinterpret_cast<signed char *>(sc_s + F2_CG * 8);    // [nslots]
    const int nslots = nblk * q.maxrec;
    {
        const uint32_t *pc = q.partCnt + (size_t)layer * nblk * E;
        for (int e = tid; e < E; e += nthr) {
            uint32_t s = 0u;
#pragma unroll 4
            for (int b = 0; b < nblk; ++b) s += __ldcg(pc + (size_t)b * E + e);
            cnt_s[e] = s;
            if (blk == 0) q.counts[(size_t)layer * E + e] = (long long)s;
        }
        const int32_t *rs = q.rec_src + (size_t)layer * nslots;
        for (int i = tid; i < nslots; i += nthr) src_s[i] = (signed char)__ldcg(rs + i);
    }
    // ---- phase 1b: this block's slice of the co-activation matrix: sum of the partial images ----
    {
        const int total4 = E * E / 4;
        const int per = (total4 + nblk - 1) / nblk;
        const int v0 = blk * per, v1 = min(total4, v0 + per);
        const int4 *pc4 = reinterpret_cast<const int4 *>(q.partC + (size_t)layer * nblk * (size_t)(EP * EP));
        int4 *out4 = reinterpret_cast<int4 *>(q.coact + (size_t)layer * E * E);
        for (int v = v0 + tid; v < v1; v += nthr) {
            // output element o = col * E + row (C is symmetric); image index ((row / 128) * EP + col) * 128 + row % 128
            const int o = v * 4, col = o / E, row = o - col * E;
            const size_t f4 = (((size_t)(row >> 7) * EP + col) * 128 + (row & 127)) >> 2;
            int4 s = make_int4(0, 0, 0, 0);
#pragma unroll 4
            for (int b = 0; b < nblk; ++b) {
                const int4 x = __ldcg(pc4 + (size_t)b * (EP * EP / 4) + f4);
                s.x += x.x; s.y += x.y; s.z += x.z; s.w += x.w;
            }
            out4[v] = s;
        }
    }
    __syncthreads();
    // ---- phase 1c: finish this block's candidates p = blk, blk + nblk, ... (F2_CG at a time) ----
    const int WD = q.WD, WN = q.WN, P = q.P, N = q.N;
    const uint32_t *recs = q.recs + (size_t)layer * nslots * (size_t)q.ncnt;
    const int ncand = P > blk ? (P - blk + nblk - 1) / nblk : 0;
    for (int c0 = 0; c0 < ncand; c0 += F2_CG) {
        const int ng = min(F2_CG, ncand - c0);
        for (int i = tid; i < F2_CG * (64 + 64 + 8); i += nthr) lp_s[i] = 0ull;
        __syncthreads();
        // received tokens per device, local / same-node sums: one thread per (candidate, record, device slot)
        {
            const int per_c = nslots * WD;
            for (int i = tid; i < ng * per_c; i += nthr) {
                const int g = i / per_c, r2 = i - g * per_c;
                const int slot = r2 / WD, d = r2 - slot * WD;
                const int p = blk + (c0 + g) * nblk;
                const int sr = src_s[slot];
                uint32_t v = 0u;
                if (sr >= 0 && d < D) v = __ldcg(recs + (size_t)slot * q.ncnt + (size_t)p * WD + d);
                const bool loc = sr >= 0 && d == sr;
                const bool same = sr >= 0 && d < D && s_node[d] == s_node[sr];
                if (v) atomicAdd(&rv_s[g * 64 + d], (unsigned long long)v);
                // lanes of one warp may span two candidates only when per_c is not a multiple of 32: add per thread then
                if ((per_c & 31) == 0) {
                    const uint32_t sl = __reduce_add_sync(0xffffffffu, loc ? v : 0u);
                    const uint32_t ss = __reduce_add_sync(0xffffffffu, same ? v : 0u);
                    const uint32_t sa = __reduce_add_sync(0xffffffffu, v);
                    if (lane == 0) {
                        atomicAdd(&sc_s[g * 8 + 0], (unsigned long long)sa);
                        atomicAdd(&sc_s[g * 8 + 1], (unsigned long long)sl);
                        atomicAdd(&sc_s[g * 8 + 2], (unsigned long long)ss);
                    }
                } else if (v) {
                    atomicAdd(&sc_s[g * 8 + 0], (unsigned long long)v);
                    if (loc) atomicAdd(&sc_s[g * 8 + 1], (unsigned long long)v);
                    if (same) atomicAdd(&sc_s[g * 8 + 2], (unsigned long long)v);
                }
            }
            const int per_n = nslots * WN;
            for (int i = tid; i < ng * per_n; i += nthr) {
                const int g = i / per_n, r2 = i - g * per_n;
                const int slot = r2 / WN, n = r2 - slot * WN;
                const int p = blk + (c0 + g) * nblk;
                const int sr = src_s[slot];
                uint32_t v = 0u;
                if (sr >= 0 && n < N) v = __ldcg(recs + (size_t)slot * q.ncnt + q.ndev + (size_t)p * WN + n);
                if (v) {
                    atomicAdd(&sc_s[g * 8 + 3], (unsigned long long)v);
                    if (n != (s_node[sr] & (WN - 1))) atomicAdd(&sc_s[g * 8 + 4], (unsigned long long)v);
                }
            }
            // load_pairs[d] = sum of the counts of the experts placed on d
            for (int i = tid; i < ng * E; i += nthr) {
                const int g = i / E, e = i - g * E;
                const int p = blk + (c0 + g) * nblk;
                const int d = q.maps[((size_t)layer * P + p) * E + e];
                const uint32_t cv = cnt_s[e];
                if ((unsigned)d < (unsigned)D && cv) atomicAdd(&lp_s[g * 64 + d], (unsigned long long)cv);
            }
        }
        __syncthreads();
        if (warp < ng) {
            const int g = warp;
            const int p = blk + (c0 + g) * nblk;
            const size_t o = (size_t)layer * P + p;
            long long mx = 0, sm = 0, mxr = 0, smr = 0;
            for (int d = lane; d < D; d += 32) {
                const long long l = (long long)lp_s[g * 64 + d];
                const long long r = (long long)rv_s[g * 64 + d];
                if (q.out.load_pairs) q.out.load_pairs[o * D + d] = l;
                if (q.out.recv_tokens) q.out.recv_tokens[o * D + d] = r;
                mx = max(mx, l);
                sm += l;
                mxr = max(mxr, r);
                smr += r;
            }
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) {
                mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, off));
                mxr = max(mxr, __shfl_xor_sync(0xffffffffu, mxr, off));
                sm += __shfl_xor_sync(0xffffffffu, sm, off);
                smr += __shfl_xor_sync(0xffffffffu, smr, off);
            }
            if (lane == 0) {
                const long long dv = (long long)sc_s[g * 8 + 0], loc = (long long)sc_s[g * 8 + 1],
                                same = (long long)sc_s[g * 8 + 2], a_node = (long long)sc_s[g * 8 + 3],
                                a_rnode = (long long)sc_s[g * 8 + 4];
                const long long rdev = dv - loc, intra = same - loc, inter = dv - same;
                if (q.out.dev_visits) q.out.dev_visits[o] = dv;
                if (q.out.remote_dev) q.out.remote_dev[o] = rdev;
                if (q.out.remote_intra) q.out.remote_intra[o] = intra;
                if (q.out.remote_inter) q.out.remote_inter[o] = inter;
                if (q.out.node_visits) q.out.node_visits[o] = a_node;
                if (q.out.remote_node) q.out.remote_node[o] = a_rnode;
                if (q.out.cost)
                    q.out.cost[o] = (long long)q.cost_local * loc + (long long)q.cost_intra * intra +
                                    (long long)q.cost_inter * inter;
                if (q.out.bytes) q.out.bytes[o] = rdev * q.bytes_per_token;
                if (q.out.imbalance) q.out.imbalance[o] = sm ? __ddiv_rn((double)(mx * D), (double)sm) : 0.0;
                if (q.out.imbalance_recv) q.out.imbalance_recv[o] = smr ? __ddiv_rn((double)(mxr * D), (double)smr) : 0.0;
            }
        }
        __syncthreads();
    }
}

// ---- host side ------------------------------------------------------------------------------------------
struct F2Geom {
    int WD, WN, Cd, Cn, nwd, nwn, nst, EP, cps, maxrec, ncnt, ndev, nblk, nthreads;
    int64_t tiles_per_cta, tpc;
    size_t smem;
    size_t partC_ints, partCnt_words, rec_words, rec_slots;
};

static int pow2_ceil(int v)
{
    int p = 1;
    while (p < v) p <<= 1;
    return p;
}

static bool f2_geom(int32_t L, int64_t T, int32_t k, int32_t E, int32_t D, int32_t N, int32_t P, F2Geom *g)
{
#define F2_FAIL(why) do { if (getenv("CAP_DEBUG")) fprintf(stderr, "f2_geom: %s\n", why); return false; } while (0)
    if (getenv("CAP_NO_FUSED2")) F2_FAIL("disabled");
    if (E != 64 && E != 128 && E != 256) F2_FAIL("E");
    if (k > 8 || L < 1 || T < 1 || P < 1 || D < 1 || D > 64 || N < 1 || N > 8) F2_FAIL("sizes");
    g->WD = D <= 8 ? 8 : D <= 16 ? 16 : D <= 32 ? 32 : 64;
    g->WN = N <= 2 ? 2 : N <= 4 ? 4 : 8;
    const int cd = ((int64_t)P * g->WD + 127) / 128, cn = ((int64_t)P * g->WN + 127) / 128;
    if (cd > 32 || cn > 8) F2_FAIL("row too long");
    g->Cd = pow2_ceil(cd < 4 ? 4 : cd);
    g->Cn = pow2_ceil(cn < 4 ? 4 : cn);
    g->nwd = g->Cd / 4;
    g->nwn = g->Cn / 4;
    g->EP = E <= 128 ? 128 : 256;
    g->nthreads = F2_THREADS;
    if (2 + g->nwd + g->nwn + 4 > F2_THREADS / 32) F2_FAIL("warps");
    const size_t budget = 222 * 1024;
    int n = 16;
    for (; n >= 4; n -= 1)
        if (f2_smem_layout(E, g->EP, g->Cd, g->Cn, g->nwd, g->nwn, n).total <= budget) break;
    if (n < 4) F2_FAIL("smem");
    g->nst = n;
    g->smem = f2_smem_layout(E, g->EP, g->Cd, g->Cn, g->nwd, g->nwn, n).total;
    const int64_t ltiles = (T + F2_TILE - 1) / F2_TILE;
    int64_t want = sm_count() / L;
    if (want < 1) F2_FAIL("more layers than SMs");        // every block of the launch must be resident
    const int64_t cap_run = (int64_t)F2_MAXRUNBLK * F2_BT;
    g->cps = 0;
    if (D <= want && T / D >= 4 * F2_BT) {
        g->cps = (int)(want / D);
        const int64_t per_src = (T + D - 1) / D;
        const int64_t nts = (per_src + F2_TILE - 1) / F2_TILE;
        g->tiles_per_cta = (nts + g->cps - 1) / g->cps;
        g->nblk = g->cps * D;
        g->tpc = g->tiles_per_cta * F2_TILE;
        g->maxrec = (int)((g->tpc + cap_run - 1) / cap_run);
    } else {
        g->tiles_per_cta = (ltiles + want - 1) / want;
        g->nblk = (int)((ltiles + g->tiles_per_cta - 1) / g->tiles_per_cta);
        g->tpc = g->tiles_per_cta * F2_TILE;
        int64_t srcb = ((g->tpc - 1) * D) / T + 1;
        if (srcb > D - 1) srcb = D - 1;
        g->maxrec = (int)((g->tpc + cap_run - 1) / cap_run + srcb + 1);
    }
    if ((int64_t)g->nblk * L > sm_count()) F2_FAIL("grid");
    if (g->maxrec > 600) F2_FAIL("records");
    if ((int64_t)g->nblk * g->maxrec > F2_MAXSLOTS) F2_FAIL("slots");
    g->ndev = g->Cd * 128;
    g->ncnt = (g->Cd + g->Cn) * 128;
    g->rec_slots = (size_t)L * g->nblk * g->maxrec;
    g->rec_words = g->rec_slots * (size_t)g->ncnt;
    g->partC_ints = (size_t)L * g->nblk * (size_t)g->EP * g->EP;
    g->partCnt_words = (size_t)L * g->nblk * E;
    // phase 1 reuses the front of the dynamic shared memory: counts, per-round sums, record sources
    if (4096 + F2_CG * (64 + 64 + 8) * 8 + (size_t)g->nblk * g->maxrec + 64 > g->smem) F2_FAIL("phase-1 smem");
    return true;
#undef F2_FAIL
}

size_t fused2_ws_bytes(int32_t L, int64_t T, int32_t k, int32_t E, int32_t D, int32_t P)
{
    size_t best = 0;
    for (int N = 2; N <= 8; N *= 2) {
        F2Geom g;
        if (!f2_geom(L, T, k, E, D, N, P, &g)) continue;
        const size_t b = g.partC_ints * 4 + 256 + g.partCnt_words * 4 + 256 + g.rec_words * 4 + 256 + g.rec_slots * 4 + 256;
        if (b > best) best = b;
    }
    return best;
}

bool fused2_plan(int32_t L, int64_t T, const cap_gate_cfg &cfg, int32_t D, int32_t N, int32_t P, int64_t *plan)
{
    if (cfg.scoring != 0 || cfg.renormalize != 1 || cfg.n_group != 1 || cfg.k > 8) return false;
    F2Geom g;
    if (!f2_geom(L, T, cfg.k, cfg.E, D, N, P, &g)) return false;
    const int64_t per_src = (T + D - 1) / D;
    plan[0] = 1;
    plan[1] = g.nblk;
    plan[2] = g.tpc;
    plan[3] = g.tpc < per_src ? g.tpc : per_src;
    plan[4] = (int64_t)F2_MAXRUNBLK * F2_BT;
    plan[5] = g.maxrec;
    plan[6] = g.cps;
    plan[7] = 2;
    return true;
}

template <int E>
static int launch_f2_e(const F2Params &prm, const F2Geom &g, int L, cudaStream_t st)
{
    cudaFuncSetAttribute(trace_fused2_kernel<E>, cudaFuncAttributeMaxDynamicSharedMemorySize, 225 * 1024);
    if (getenv("CAP_DEBUG")) {
        int nb = -1;
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, trace_fused2_kernel<E>, g.nthreads, g.smem);
        fprintf(stderr, "fused2: grid %d x %d, %d threads, %zu B smem, nst %d, Cd %d Cn %d, maxrec %d, occupancy %d (%s)\n",
                g.nblk, L, g.nthreads, g.smem, g.nst, g.Cd, g.Cn, g.maxrec, nb, cudaGetErrorString(cudaGetLastError()));
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)g.nblk, (unsigned)L);
    cfg.blockDim = dim3((unsigned)g.nthreads);
    cfg.dynamicSmemBytes = g.smem;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeCooperative;
    at[0].val.cooperative = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    {
        KernelTimerScope ts("trace_fused", st);
        cudaLaunchKernelEx(&cfg, trace_fused2_kernel<E>, prm);
    }
    note_launch();
    return check_launch("trace_fused2_kernel");
}

static bool f2_args_ok(const float *logits, const float *bias, const cap_gate_cfg &cfg, int32_t *idx, float *w,
                       int64_t *counts, int32_t *coact, const int32_t *token_src, const cap_eval_out &out,
                       int32_t L, int64_t T, int32_t P)
{
    if (cfg.scoring != 0 || cfg.renormalize != 1 || cfg.n_group != 1 || cfg.k > 8 || bias != nullptr) return false;
    if (token_src != nullptr || out.tok_remote_dev || out.tok_remote_node) return false;
    if (!counts || !coact || L < 1 || T < 1 || P < 1) return false;
    if ((reinterpret_cast<uintptr_t>(logits) | reinterpret_cast<uintptr_t>(idx) | reinterpret_cast<uintptr_t>(w) |
         reinterpret_cast<uintptr_t>(coact)) & 15u)
        return false;
    return true;
}

// ws_f2: the region of the workspace reserved for this kernel (256-byte aligned)
int launch_trace_fused2(const float *logits, const float *bias, int32_t L, int64_t T, const cap_gate_cfg &cfg,
                        int32_t *idx, float *w, int64_t *counts, int32_t *coact, const int32_t *token_src,
                        const int32_t *expert_dev, int32_t P, const cap_topology &topo, const cap_eval_out &out,
                        void *ws_f2, cudaStream_t st, bool *used)
{
    *used = false;
    if (!f2_args_ok(logits, bias, cfg, idx, w, counts, coact, token_src, out, L, T, P)) return CAP_OK;
    F2Geom g;
    if (!f2_geom(L, T, cfg.k, cfg.E, topo.D, topo.N, P, &g)) return CAP_OK;
    uintptr_t a = (reinterpret_cast<uintptr_t>(ws_f2) + 255) & ~(uintptr_t)255;
    F2Params prm = {};
    prm.partC = reinterpret_cast<int *>(a);
    a = (a + g.partC_ints * 4 + 255) & ~(uintptr_t)255;
    prm.partCnt = reinterpret_cast<uint32_t *>(a);
    a = (a + g.partCnt_words * 4 + 255) & ~(uintptr_t)255;
    prm.recs = reinterpret_cast<uint32_t *>(a);
    a = (a + g.rec_words * 4 + 255) & ~(uintptr_t)255;
    prm.rec_src = reinterpret_cast<int32_t *>(a);
    prm.logits = logits;
    prm.idx = idx;
    prm.w = w;
    prm.counts = reinterpret_cast<long long *>(counts);
    prm.coact = coact;
    prm.maps = expert_dev;
    prm.dev_node = topo.dev_node;
    prm.out = out;
    prm.T = T;
    prm.tiles_per_cta = g.tiles_per_cta;
    prm.cps = g.cps;
    prm.scale = cfg.scale;
    prm.k = cfg.k;
    prm.D = topo.D;
    prm.N = topo.N;
    prm.P = P;
    prm.WD = g.WD;
    prm.WN = g.WN;
    prm.Cd = g.Cd;
    prm.Cn = g.Cn;
    prm.nwd = g.nwd;
    prm.nwn = g.nwn;
    prm.nst = g.nst;
    prm.maxrec = g.maxrec;
    prm.ncnt = g.ncnt;
    prm.ndev = g.ndev;
    prm.cost_local = topo.cost_local;
    prm.cost_intra = topo.cost_intra;
    prm.cost_inter = topo.cost_inter;
    prm.bytes_per_token = topo.bytes_per_token;
    int rc;
    switch (cfg.E) {
    case 64: rc = launch_f2_e<64>(prm, g, L, st); break;
    case 128: rc = launch_f2_e<128>(prm, g, L, st); break;
    default: rc = launch_f2_e<256>(prm, g, L, st); break;
    }
    CAP_TRY(rc);
    *used = true;
    return CAP_OK;
}

}  // namespace cap

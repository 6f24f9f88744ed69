// cap_trace_fused fast path: S1 (gate top-k) + S2 (counts / co-activation) + S3 (scoring of P candidate
// placements) in ONE persistent, warp-specialised kernel that reads the logits exactly once
// (BASELINE.json north_star, L104/L148, L58/Eq. 3/Eq. 4).  One block per SM, roles:
//   warp 0        producer: TMA bulk copies of 16-token logits tiles into a shared-memory ring, and
//                 the one-hot code table of cap_eval_fast.cuh (prebuilt by eval_table_kernel)
//   warp 1        tensor-core warp: issues tcgen05.mma.kind::i8 on the one-hot tiles (C += A^T A in
//                 TMEM), recycles the tile buffers
//   warps 2..9    S1: two lanes per token selection network (cap_gate_fast.cuh); besides top-k
//                 indices / weights to HBM they leave (a) the token's table-row offsets in a
//                 shared-memory ring for S3 and (b) its one-hot bytes in the current MMA tile
//                 (when their tiles are done, four of them drain the TMEM accumulator into the
//                 global matrix, one lane quadrant each)
//   warps 10..    S3: bit-sliced candidate scoring (cap_eval_fast.cuh) fed from the offsets ring.
// Everything is handed over through mbarriers; only run flushes use a named barrier among the S3
// warps.  Records / decode / finalize are those of the standalone S3 path.
#include <cstdio>
#include <cstdlib>

#include "cap_async.cuh"
#include "cap_eval_fast.cuh"
#include "cap_gate_fast.cuh"
#include "cap_tc.cuh"

namespace cap {

constexpr int FU_NC = 8;            // S1 warps
constexpr int FU_S3W0 = 2 + FU_NC;  // first S3 warp
constexpr int FU_TILE = 16;         // tokens per S1 tile
constexpr int FU_MT = 64;           // tokens per MMA tile (4 S1 tiles, 2 MMAs of K = 32)
constexpr int FU_OB = 4;            // S3 offset blocks in the ring
constexpr int FU_MAXST = 12;        // logits ring stages (<= 4 FU_OB - 3: an S1 warp can never be two phases ahead of offs_empty)
constexpr int FU_MAXTHREADS = 896;
constexpr int FU_KP = 8;            // offsets per token (k <= 8, padded with the zero row)

// Optional per-warp timeline (build with -DCAP_FU_TRACE; read back with cap_debug_fused_trace): clock64
// stamps relative to the block's entry at role milestones, plus cycles spent waiting on each hand-over.
// -DCAP_FU_NO_S1 / -DCAP_FU_NO_S3 compile the S1 selection / the S3 scoring out (outputs are then wrong):
// the ablation builds behind the decomposition quoted in profiles/r1c_fused.md and DESIGN.md 6.3.
#ifdef CAP_FU_TRACE
__device__ unsigned long long g_fu_trace[160 * 24 * 8];
#define FU_TR(ev, val)                                                                        \
    do {                                                                                      \
        if (lane == 0 && blockIdx.x < 160 && warp < 24)                                       \
            g_fu_trace[((size_t)blockIdx.x * 24 + warp) * 8 + (ev)] = (unsigned long long)(val); \
    } while (0)
#define FU_NOW() ((long long)clock64() - tr_t0)
#define FU_WAIT_BEGIN() const long long tr_w0 = clock64()
#define FU_WAIT_END(acc) (acc) += clock64() - tr_w0
#else
#define FU_TR(ev, val) do { } while (0)
#define FU_NOW() 0
#define FU_WAIT_BEGIN() do { } while (0)
#define FU_WAIT_END(acc) do { } while (0)
#endif

struct FusedParams {
    const float *logits;
    int32_t *idx;
    float *w;
    unsigned long long *counts;   // [L][E], zeroed
    int *coact;                   // [L][E][E], zeroed
    const uint32_t *table;        // [L][E + 1][RS * 4]
    int32_t *rec_src;             // [L][ncta_t][maxrec]
    uint32_t *rec_planes;         // [L][ncta_t][maxrec][W][EF_RECW]
    int64_t T;
    int64_t tiles_per_cta;        // real 16-token tiles per block (uniform split)
    int32_t cps;                  // > 0: blocks per source device, block ranges aligned to the source runs
    float scale;
    int32_t k, D, pack64;
    int32_t R, RS, S, logS, maxrec, NPR, ncta_t, nst, ns3w;
};

struct FusedSmem {
    // byte offsets into the dynamic shared memory
    uint32_t table, xch, tiles, offs, ring, total;
};

__host__ __device__ inline FusedSmem fused_smem_layout(int E, int EP, int RS, int R, int S, int nst)
{
    FusedSmem m;
    uint32_t o = 0;
    m.ring = o;                                   // 128-byte aligned rows for the swizzled reads
    o += (uint32_t)nst * FU_TILE * E * 4;
    m.tiles = o;
    o += 2u * EP * FU_MT;
    m.table = o;
    o += (uint32_t)(E + 1) * RS * 16;
    m.offs = o;
    o += (uint32_t)FU_OB * EF_PASSES * S * FU_KP * 4;
    m.xch = o;                                    // level 0 of the sub-slot tree is the largest exchange
    o += (uint32_t)(S / 2 > 0 ? S / 2 : 1) * R * EF_BT * 16;
    m.total = o;
    return m;
}

__device__ __forceinline__ void named_bar_sync(int id, int nthreads)
{
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

// bit-sliced a += b; b has np planes of 2 words (the rest are zero)
__device__ __forceinline__ void fu_add_planes(uint2 (&a)[EF_NPL], const uint2 *b, int stride, int np)
{
    uint2 carry = make_uint2(0u, 0u);
#pragma unroll
    for (int p = 0; p < EF_NPL; ++p) {
        const uint2 x = p < np ? b[(size_t)p * stride] : make_uint2(0u, 0u);
        uint2 s, c;
        CAP_CSA(s.x, c.x, a[p].x, x.x, carry.x);
        CAP_CSA(s.y, c.y, a[p].y, x.y, carry.y);
        a[p] = s;
        carry = c;
    }
}

// OR of the FU_KP table rows of one token at this thread's 8-byte column
__device__ __forceinline__ uint2 fu_token_mask(const unsigned char *tblc, const uint32_t *op)
{
    const uint4 oa = *reinterpret_cast<const uint4 *>(op);
    const uint4 ob = *reinterpret_cast<const uint4 *>(op + 4);
    const uint2 v0 = *reinterpret_cast<const uint2 *>(tblc + oa.x);
    const uint2 v1 = *reinterpret_cast<const uint2 *>(tblc + oa.y);
    const uint2 v2 = *reinterpret_cast<const uint2 *>(tblc + oa.z);
    const uint2 v3 = *reinterpret_cast<const uint2 *>(tblc + oa.w);
    const uint2 v4 = *reinterpret_cast<const uint2 *>(tblc + ob.x);
    const uint2 v5 = *reinterpret_cast<const uint2 *>(tblc + ob.y);
    const uint2 v6 = *reinterpret_cast<const uint2 *>(tblc + ob.z);
    const uint2 v7 = *reinterpret_cast<const uint2 *>(tblc + ob.w);
    uint2 m;
    m.x = lop_or3(lop_or3(lop_or3(v0.x, v1.x, v2.x), v3.x, v4.x), lop_or3(v5.x, v6.x, v7.x), 0u);
    m.y = lop_or3(lop_or3(lop_or3(v0.y, v1.y, v2.y), v3.y, v4.y), lop_or3(v5.y, v6.y, v7.y), 0u);
    return m;
}

// half a Harley-Seal block: four token masks into planes 0/1, carry of weight 4 out
#define CAP_FU_HALF(F, X0, X1, X2, X3, OUT4)            \
    do {                                                \
        uint32_t tA, tB, s;                             \
        CAP_CSA(s, tA, pl[0].F, (X0).F, (X1).F);        \
        CAP_CSA(s, tB, s, (X2).F, (X3).F);              \
        pl[0].F = s;                                    \
        CAP_CSA(pl[1].F, OUT4, pl[1].F, tA, tB);        \
    } while (0)
// weight-4 carries of the two halves into plane 2, weight-8 carry rippled into planes 3..EF_BT-1
#define CAP_FU_TOP(F, FA, FB)                           \
    do {                                                \
        uint32_t e8;                                    \
        CAP_CSA(pl[2].F, e8, pl[2].F, FA, FB);          \
        _Pragma("unroll") for (int p = 3; p < EF_BT; ++p) { \
            const uint32_t c = pl[p].F & e8;            \
            pl[p].F ^= e8;                              \
            e8 = c;                                     \
        }                                               \
    } while (0)

template <int E>
__global__ void __launch_bounds__(FU_MAXTHREADS, 1) trace_fused_kernel(FusedParams q)
{
    extern __shared__ __align__(1024) unsigned char fu_sm[];
    __shared__ uint64_t full_bar[FU_MAXST], empty_bar[FU_MAXST];
    __shared__ uint64_t offs_full[FU_OB], offs_empty[FU_OB];
    __shared__ uint64_t tile_full[2], tile_ready[2], mma_done[2];
    __shared__ uint64_t tbl_bar, acc_done;
    __shared__ uint32_t s_tmem;
    constexpr int EP = E <= 128 ? 128 : 256;
    constexpr uint32_t LBO = 128u, SBO = (FU_MT / 16) * 128u;
    constexpr uint32_t NCOLS = EP == 128 ? 128u : 512u;
    constexpr uint32_t IDESC = (2u << 4) | ((uint32_t)(EP >> 3) << 17) | (8u << 24);
    constexpr int TILE_BYTES = FU_TILE * E * 4;
    constexpr int MT_TILES = FU_MT / FU_TILE;          // S1 tiles per MMA tile
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
#ifdef CAP_FU_TRACE
    const long long tr_t0 = clock64();
    long long tr_wa = 0, tr_wb = 0, tr_wc = 0;
#endif
    const int layer = blockIdx.y;
    const int S = q.S, R = q.R, nst = q.nst, k = q.k;
    const int BT = EF_PASSES * S;                       // tokens per S3 block
    const int TPB = BT / FU_TILE;                       // S1 tiles per S3 block
    const FusedSmem lay = fused_smem_layout(E, EP, q.RS, R, S, nst);
    unsigned char *ring = fu_sm + lay.ring;
    unsigned char *tiles = fu_sm + lay.tiles;
    unsigned char *tbl = fu_sm + lay.table;
    uint32_t *offs = reinterpret_cast<uint32_t *>(fu_sm + lay.offs);
    uint2 *xch = reinterpret_cast<uint2 *>(fu_sm + lay.xch);
    const int rowb = q.RS * 16;
    const uint32_t zero_row = (uint32_t)E * rowb;
    const int ns3 = q.ns3w * 32;

    // ---- this block's token range [t0, t1) of one layer, in 16-token tiles from t0 ----
    // uniform split: equal tile counts; aligned split (cps > 0): the tokens of each source device
    // (default token_src: contiguous blocks, reading A5) are shared by cps blocks, so that a block
    // scores a single run and flushes its counters once
    const int64_t T = q.T;
    int64_t t0, t1;
    if (q.cps > 0) {
        const int srcd = (int)blockIdx.x / q.cps, jj = (int)blockIdx.x % q.cps;
        const int64_t b0 = ((int64_t)srcd * T + q.D - 1) / q.D, b1 = ((int64_t)(srcd + 1) * T + q.D - 1) / q.D;
        const int64_t nts = (b1 - b0 + FU_TILE - 1) / FU_TILE;
        const int64_t base = nts / q.cps, rem = nts % q.cps;
        const int64_t ts = jj * base + (jj < rem ? jj : rem), tn = base + (jj < rem ? 1 : 0);
        t0 = min(b1, b0 + ts * FU_TILE);
        t1 = min(b1, t0 + tn * FU_TILE);
    } else {
        t0 = min(T, (int64_t)blockIdx.x * q.tiles_per_cta * FU_TILE);
        t1 = min(T, t0 + q.tiles_per_cta * FU_TILE);
    }
    const int nt = (int)((t1 - t0 + FU_TILE - 1) / FU_TILE);
    const int pad = TPB > MT_TILES ? TPB : MT_TILES;
    const int ntp = ((nt + pad - 1) / pad) * pad;       // with ghost tiles: whole S3 blocks and MMA tiles
    const int nb = ntp / TPB, nm = ntp / MT_TILES;
    const float *logits = q.logits + (size_t)layer * T * E;
    int32_t *gidx = q.idx + (size_t)layer * T * k;
    float *gw = q.w + (size_t)layer * T * k;

    // ---- set-up ----
    if (tid == 0) {
        for (int s = 0; s < nst; ++s) {
            mbar_init(&full_bar[s], 1);
            mbar_init(&empty_bar[s], 1);
        }
        for (int s = 0; s < FU_OB; ++s) {
            mbar_init(&offs_full[s], TPB);
            mbar_init(&offs_empty[s], q.ns3w);
        }
        for (int s = 0; s < 2; ++s) {
            mbar_init(&tile_full[s], MT_TILES);
            mbar_init(&tile_ready[s], 1);
            mbar_init(&mma_done[s], 1);
        }
        mbar_init(&tbl_bar, 1);
        mbar_init(&acc_done, 1);
        mbar_fence_init();
    }
    if (warp == 1) tmem_alloc(&s_tmem, NCOLS);
    {
        uint4 *z = reinterpret_cast<uint4 *>(tiles);
        for (int i = tid; i < 2 * EP * FU_MT / 16; i += blockDim.x) z[i] = make_uint4(0u, 0u, 0u, 0u);
    }
    proxy_fence_async();
    tc_fence_before();
    pdl_launch_dependents();
    // No grid-dependency wait here: the predecessor (eval_table_kernel) produces the code table and clears the
    // accumulators, which this kernel consumes late -- the table when S3 starts, the cleared outputs at the flush
    // and the drain.  The logits stream and the selection depend on nothing it writes, so they start while it
    // still runs; pdl_wait() sits at the three consumers below.
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = s_tmem;
    FU_TR(1, FU_NOW());

    if (warp == 0) {
        // ================= producer =================
        if (lane == 0 && nt > 0) {
            auto issue = [&](int j) {
                const int st = j % nst;
                const int64_t tok0 = t0 + (int64_t)j * FU_TILE;
                const int rows = (int)min((int64_t)FU_TILE, t1 - tok0);
                mbar_expect_tx(&full_bar[st], (uint32_t)rows * E * 4);
                bulk_g2s(ring + (size_t)st * TILE_BYTES, logits + tok0 * E, (uint32_t)rows * E * 4, &full_bar[st]);
            };
            const int npre = nt < nst ? nt : nst;
            for (int j = 0; j < npre; ++j) issue(j);          // the first ring needs no free-stage wait
            // the logits are on their way: now the code table, the first thing the predecessor produced
            pdl_wait();
            mbar_expect_tx(&tbl_bar, (uint32_t)(E + 1) * rowb);
            bulk_g2s(tbl, q.table + (size_t)layer * (E + 1) * q.RS * 4, (uint32_t)(E + 1) * rowb, &tbl_bar);
            for (int j = npre; j < nt; ++j) {
                mbar_wait_relaxed(&empty_bar[j % nst], (uint32_t)(((j / nst) - 1) & 1), 256);
                issue(j);
            }
        }
        FU_TR(2, FU_NOW());
    } else if (warp == 1) {
        // ================= tensor-core warp =================
        for (int m = 0; m < nm; ++m) {
            const int tb = m & 1;
            unsigned char *tile = tiles + (size_t)tb * EP * FU_MT;
            mbar_wait_relaxed(&tile_full[tb], (uint32_t)((m >> 1) & 1), 256);
            tc_fence_after();
            if (lane == 0) {
                const uint32_t base = smem_u32(tile);
#pragma unroll
                for (int j = 0; j < FU_MT / 32; ++j) {
                    const uint64_t bd = umma_desc(base + j * 2 * LBO, LBO, SBO);
                    umma_i8(tmem, bd, bd, IDESC, (uint32_t)((m | j) != 0));
                    if (EP == 256) {
                        const uint64_t a1 = umma_desc(base + 16 * SBO + j * 2 * LBO, LBO, SBO);
                        umma_i8(tmem + 256u, a1, bd, IDESC, (uint32_t)((m | j) != 0));
                    }
                }
                umma_commit(&mma_done[tb]);
                if (m == nm - 1) umma_commit(&acc_done);
            }
            __syncwarp();
            if (m + 2 < nm) {
                // recycle the buffer for MMA tile m + 2: wait until the tensor core has read it, clear it
                mbar_wait(&mma_done[tb], (uint32_t)((m >> 1) & 1));
                uint4 *z = reinterpret_cast<uint4 *>(tile);
                for (int i = lane; i < EP * FU_MT / 16; i += 32) z[i] = make_uint4(0u, 0u, 0u, 0u);
                proxy_fence_async();
                __syncwarp();
                if (lane == 0) mbar_arrive(&tile_ready[tb]);
            }
        }
        FU_TR(2, FU_NOW());
    } else if (warp < FU_S3W0) {
        // ================= S1: gate top-k, two lanes per token =================
        const int c = warp - 2;
        const int h = lane >> 4, tl = lane & 15;
        for (int j = c; j < ntp; j += FU_NC) {
            const bool ghost = j >= nt;
            const int st = j % nst;
            const int64_t tok = t0 + (int64_t)j * FU_TILE + tl;
            const bool valid = !ghost && tok < t1;
            int sel[8];
#pragma unroll
            for (int i = 0; i < 8; ++i) sel[i] = 0;
            if (!ghost) {
                // this warp alternates on a stage with one other warp: first make sure that warp's
                // tile (the previous use of the stage) has been consumed, then wait for ours
                const int u = j / nst;
                FU_WAIT_BEGIN();
                if (u >= 1) mbar_wait(&empty_bar[st], (uint32_t)((u - 1) & 1));
                mbar_wait(&full_bar[st], (uint32_t)(u & 1));
                FU_WAIT_END(tr_wa);
                const float *row = reinterpret_cast<const float *>(ring + (size_t)st * TILE_BYTES +
                                                                   (size_t)(tok < t1 ? tl : 0) * E * 4);
                float wv[4];
#ifdef CAP_FU_NO_S1      // ablation build: no selection arithmetic (arbitrary distinct experts)
#pragma unroll
                for (int i = 0; i < 8; ++i) sel[i] = (tl * 8 + i + j) & (E - 1);
                wv[0] = wv[1] = wv[2] = wv[3] = row[h];
#else
                gate_select_pair<E>(row, h, tl & 7, k, sel);
                gate_weights_softmax_pair(row, h, k, sel, q.scale, wv);
#endif
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
            // ---- table-row offsets for S3 ----
            const int b = j / TPB, ob = b % FU_OB;
            {
                FU_WAIT_BEGIN();
                if (b >= FU_OB) mbar_wait(&offs_empty[ob], (uint32_t)(((b / FU_OB) - 1) & 1));
                FU_WAIT_END(tr_wb);
            }
            {
                uint4 o4;
                uint32_t ov[4];
#pragma unroll
                for (int jj = 0; jj < 4; ++jj) {
                    const int s = 4 * h + jj;
                    const int e = h ? sel[4 + jj] : sel[jj];
                    ov[jj] = (valid && s < k) ? (uint32_t)e * rowb : zero_row;
                }
                o4 = make_uint4(ov[0], ov[1], ov[2], ov[3]);
                const int slot = (j % TPB) * FU_TILE + tl;
                *reinterpret_cast<uint4 *>(offs + ((size_t)ob * BT + slot) * FU_KP + 4 * h) = o4;
            }
            // ---- one-hot bytes for the co-activation MMA ----
            const int m = j / MT_TILES, tb = m & 1;
            {
                FU_WAIT_BEGIN();
                if (m >= 2) mbar_wait(&tile_ready[tb], (uint32_t)(((m >> 1) - 1) & 1));
                FU_WAIT_END(tr_wc);
            }
            if (valid) {
                const int tp = (j % MT_TILES) * FU_TILE + tl;
                unsigned char *col = tiles + (size_t)tb * EP * FU_MT + (tp >> 4) * LBO + (tp & 15);
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
        FU_TR(2, FU_NOW());
        FU_TR(5, tr_wa);
        FU_TR(6, tr_wb);
        FU_TR(7, tr_wc);
        // ---- drain the co-activation accumulator: S1 warps 0..3, one TMEM lane quadrant each ----
        if (c < 4 && nm > 0) {
            pdl_wait();                 // counts / coact were cleared by the predecessor
            mbar_wait_relaxed(&acc_done, 0u, 128);
            FU_TR(3, FU_NOW());
            tc_fence_after();
            const int quad = warp & 3;
            int *C = q.coact + (size_t)layer * E * E;
            unsigned long long *cnt = q.counts + (size_t)layer * E;
#pragma unroll 1
            for (int hh = 0; hh < EP / 128; ++hh) {
                const int r = hh * 128 + quad * 32 + lane;
#pragma unroll 1
                for (int cb = 0; cb < EP / 32; ++cb) {
                    uint32_t v[32];
                    tmem_ld32(tmem + ((uint32_t)(quad * 32) << 16) + (uint32_t)(hh * 256 + cb * 32), v);
                    const bool rok = r < E;
                    if (q.pack64) {
                        int *cp = C + (size_t)(cb * 32) * E + (r & ~1);
#pragma unroll
                        for (int j = 0; j < 32; j += 2) {
                            const uint32_t p0 = __shfl_xor_sync(0xffffffffu, v[j], 1);
                            const uint32_t p1 = __shfl_xor_sync(0xffffffffu, v[j + 1], 1);
                            const int jj = j + (lane & 1);
                            const unsigned long long pk = (lane & 1) ? ((unsigned long long)v[j + 1] << 32) | p1
                                                                     : ((unsigned long long)p0 << 32) | v[j];
                            if (rok && cb * 32 + jj < E)
                                asm volatile("red.global.add.u64 [%0], %1;" ::"l"(cp + (size_t)jj * E), "l"(pk) : "memory");
                        }
                    } else {
                        int *cp = C + (size_t)(cb * 32) * E + r;
#pragma unroll
                        for (int j = 0; j < 32; ++j)
                            if (rok && cb * 32 + j < E)
                                asm volatile("red.global.add.s32 [%0], %1;" ::"l"(cp + (size_t)j * E), "r"(v[j]) : "memory");
                    }
                    if (rok && (r >> 5) == cb) {
                        uint32_t d = 0u;
#pragma unroll
                        for (int j = 0; j < 32; ++j) d = (r & 31) == j ? v[j] : d;
                        atomicAdd(&cnt[r], (unsigned long long)d);
                    }
                }
            }
        }
    } else {
        // ================= S3: bit-sliced candidate scoring =================
        // a thread owns one 8-byte column (2 words) of one token sub-slot: twice the threads of a 16-byte
        // split, half the registers each -- more row loads in flight per SM (the loop waits on LDS latency)
        const int t3 = tid - FU_S3W0 * 32;
        const int R2 = 2 * R;
        const bool active = t3 < R2 * S;
        // (sub-slot, column) of this thread: whole warps own 32 consecutive columns of one sub-slot (one
        // row segment per load: no bank conflicts); the R % 32 remaining columns are packed behind them
        const int Rm = R2 & ~31, Rr = R2 - Rm;
        int sub = 0, col = 0;
        if (active) {
            if (t3 < Rm * S) {
                sub = (t3 >> 5) % S;
                col = ((t3 >> 5) / S) * 32 + (t3 & 31);
            } else {
                const int tt = t3 - Rm * S;
                sub = tt / Rr;
                col = Rm + tt - sub * Rr;
            }
        }
        const unsigned char *tblc = tbl + col * 8;
        const int D = q.D;
        const size_t slot0 = ((size_t)layer * q.ncta_t + blockIdx.x) * q.maxrec;
        const int64_t cap_run = (int64_t)(EF_MAXBLK - 2) * BT;
        if (nt > 0) mbar_wait(&tbl_bar, 0u);
        uint2 pl[EF_NPL];
#pragma unroll
        for (int p = 0; p < EF_NPL; ++p) pl[p] = make_uint2(0u, 0u);
        int nrec = 0, src = 0;
        int64_t rend = t0;               // end of the current run (none yet)
        bool have_run = false;

        auto flush = [&]() {
            pdl_wait();                 // the record headers were reset by the predecessor
            // add the S sub-slots in the bit-sliced domain (tree through shared memory), write the record
            for (int lvl = 0; lvl < q.logS; ++lvl) {
                const int half = S >> (lvl + 1);
                const int stride = half * R2;
                const int np = EF_BT + lvl;
                if (active && sub >= half && sub < 2 * half) {
#pragma unroll
                    for (int p = 0; p < EF_NPL; ++p)
                        if (p < np) xch[(size_t)p * stride + (sub - half) * R2 + col] = pl[p];
                }
                named_bar_sync(1, ns3);
                if (active && sub < half) fu_add_planes(pl, xch + sub * R2 + col, stride, np);
                named_bar_sync(1, ns3);
            }
            FU_TR(6, FU_NOW());
            if (active && sub == 0) {
                // word-major record: the planes of a word are one 64-byte run (what the decode kernel reads)
                uint32_t *rp = q.rec_planes + ((slot0 + nrec) * (size_t)(R * 4) + (size_t)col * 2) * EF_RECW;
                uint32_t v[EF_RECW];
#pragma unroll
                for (int p = 0; p < EF_RECW; ++p) v[p] = (p < EF_NPL && p < q.NPR) ? pl[p < EF_NPL ? p : 0].x : 0u;
                ef_store_word_planes(rp, v);
#pragma unroll
                for (int p = 0; p < EF_RECW; ++p) v[p] = (p < EF_NPL && p < q.NPR) ? pl[p < EF_NPL ? p : 0].y : 0u;
                ef_store_word_planes(rp + EF_RECW, v);
            }
            if (t3 == 0) q.rec_src[slot0 + nrec] = src;
            ++nrec;
#pragma unroll
            for (int p = 0; p < EF_NPL; ++p) pl[p] = make_uint2(0u, 0u);
        };

        for (int b = 0; b < nb; ++b) {
            const int ob = b % FU_OB;
            {
                FU_WAIT_BEGIN();
                mbar_wait_relaxed(&offs_full[ob], (uint32_t)((b / FU_OB) & 1), 128);
                FU_WAIT_END(tr_wa);
            }
            const int64_t bt0 = t0 + (int64_t)b * BT;
            const int64_t bend = min(bt0 + BT, t1);
            const uint32_t *obuf = offs + ((size_t)ob * BT + sub) * FU_KP;
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
                const bool whole = cur == bt0 && seg == bend;     // tokens past t1 carry the zero row
#ifdef CAP_FU_NO_S3      // ablation build: no candidate scoring
                if (false) {
#else
                if (active) {
#endif
                    uint2 x0, x1, x2, x3;
                    uint32_t fAx, fAy, fBx, fBy;
#define CAP_FU_LOAD(X, PS)                                                               \
    do {                                                                                 \
        X = fu_token_mask(tblc, obuf + (size_t)(PS) * S * FU_KP);                        \
        if (!whole) {                                                                    \
            const int64_t tk = bt0 + (PS) * S + sub;                                     \
            if (tk < cur || tk >= seg) X = make_uint2(0u, 0u);                           \
        }                                                                                \
    } while (0)
                    CAP_FU_LOAD(x0, 0); CAP_FU_LOAD(x1, 1); CAP_FU_LOAD(x2, 2); CAP_FU_LOAD(x3, 3);
                    CAP_FU_HALF(x, x0, x1, x2, x3, fAx); CAP_FU_HALF(y, x0, x1, x2, x3, fAy);
                    CAP_FU_LOAD(x0, 4); CAP_FU_LOAD(x1, 5); CAP_FU_LOAD(x2, 6); CAP_FU_LOAD(x3, 7);
                    CAP_FU_HALF(x, x0, x1, x2, x3, fBx); CAP_FU_HALF(y, x0, x1, x2, x3, fBy);
                    CAP_FU_TOP(x, fAx, fBx); CAP_FU_TOP(y, fAy, fBy);
#undef CAP_FU_LOAD
                }
                cur = seg;
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&offs_empty[ob]);
        }
        FU_TR(2, FU_NOW());
        FU_TR(5, tr_wa);
        if (have_run) flush();
        FU_TR(3, FU_NOW());
    }
    FU_TR(4, FU_NOW());
    tc_fence_before();
    __syncthreads();
    FU_TR(0, FU_NOW());
    if (warp == 1) tmem_dealloc(tmem, NCOLS);
}

// ---- host side ------------------------------------------------------------------------------------------
struct FusedGeom {
    EvalFastGeom g;      // table / column geometry of the S3 part; ncta_t, maxrec, rec_* hold the fused values
    int nst, ns3w, nthreads, EP, cps;
    int64_t tiles_per_cta;
    size_t smem;
};

static bool fused_geom(int32_t L, int64_t T, int32_t k, int32_t E, int32_t D, int32_t N, int32_t P, FusedGeom *f)
{
#define FG_FAIL(why) do { if (getenv("CAP_DEBUG")) fprintf(stderr, "fused_geom: %s\n", why); return false; } while (0)
    if (E != 64 && E != 128 && E != 256) FG_FAIL("E");
    if (k > 8 || L < 1 || T < 1 || P < 1) FG_FAIL("sizes");
    EvalFastGeom &g = f->g;
    if (!eval_fast_geom(L, T, k, E, D, N, P, sm_count(), 150 * 1024, &g)) FG_FAIL("eval geom");
    if (g.PC != 1 || g.S < 4) FG_FAIL("PC/S");
    f->EP = E <= 128 ? 128 : 256;
    // fewer token sub-slots (S) shrink the offsets ring and the exchange area: trade them for ring stages
    const size_t budget = 224 * 1024;
    int nst = 0, bestS = 0, bestLog = 0, bestNst = 0;
    for (int S = g.S, lg = g.logS; S >= 4; S /= 2, lg -= 1) {
        int n = FU_MAXST;
        for (; n >= 8; n -= 4)
            if (fused_smem_layout(E, f->EP, g.RS, g.R, S, n).total <= budget) break;
        if (n < 8) continue;
        if (32 * (FU_S3W0 + (2 * g.R * S + 31) / 32) > FU_MAXTHREADS) continue;
        if (bestS == 0) { bestS = S; bestLog = lg; bestNst = n; }          // most sub-slots that fit at all
        if (n >= 12 && S >= 8) { bestS = S; bestLog = lg; bestNst = n; break; }   // double-buffered S1 warps
    }
    if (bestS == 0) FG_FAIL("smem");
    g.S = bestS;
    g.logS = bestLog;
    nst = bestNst;
    f->ns3w = (2 * g.R * g.S + 31) / 32;
    f->nthreads = 32 * (FU_S3W0 + f->ns3w);
    if (f->nthreads > FU_MAXTHREADS) FG_FAIL("threads");
    f->nst = nst;
    f->smem = fused_smem_layout(E, f->EP, g.RS, g.R, g.S, nst).total;
    const int64_t ltiles = (T + FU_TILE - 1) / FU_TILE;
    int64_t want = sm_count() / L;
    if (want < 1) want = 1;
    const int64_t BT = (int64_t)EF_PASSES * g.S;
    const int64_t cap_run = (int64_t)(EF_MAXBLK - 2) * BT;
    f->cps = 0;
    if (D <= want && T / D >= 4 * BT) {
        // aligned split: want / D blocks per source device, one run per block
        f->cps = (int)(want / D);
        const int64_t per_src = (T + D - 1) / D;                            // tokens of the largest source
        const int64_t nts = (per_src + FU_TILE - 1) / FU_TILE;
        f->tiles_per_cta = (nts + f->cps - 1) / f->cps;
        g.ncta_t = f->cps * D;
        const int64_t tpc = f->tiles_per_cta * FU_TILE;
        g.maxrec = (int)((tpc + cap_run - 1) / cap_run + 1);
        g.tpc = tpc;
    } else {
        f->tiles_per_cta = (ltiles + want - 1) / want;
        g.ncta_t = (int)((ltiles + f->tiles_per_cta - 1) / f->tiles_per_cta);
        if (g.ncta_t > 65535) return false;
        const int64_t tpc = f->tiles_per_cta * FU_TILE;
        int64_t srcb = ((tpc - 1) * D) / T + 1;
        if (srcb > D - 1) srcb = D - 1;
        g.maxrec = (int)((tpc + cap_run - 1) / cap_run + srcb + 1);
        g.tpc = tpc;
    }
    g.NPR = EF_BT + g.logS;
    g.rec_slots = (size_t)L * g.ncta_t * g.maxrec;
    g.rec_words = g.rec_slots * (size_t)EF_RECW * g.W;
    g.table_words = (size_t)L * (E + 1) * g.RS * 4;
    return true;
}

size_t fused_ws_bytes(int32_t L, int64_t T, int32_t k, int32_t E, int32_t D, int32_t P)
{
    size_t best = 0;
    for (int N = 2; N <= 8; N *= 2) {
        FusedGeom f;
        if (!fused_geom(L, T, k, E, D, N, P, &f)) continue;
        const size_t b = f.g.rec_slots * 4 + 256 + f.g.rec_words * 4 + 256 + f.g.table_words * 4 + 256;
        if (b > best) best = b;
    }
    return best;
}

// cap_trace_fused_plan: the geometry above in numbers (host only)
bool fused_plan(int32_t L, int64_t T, const cap_gate_cfg &cfg, int32_t D, int32_t N, int32_t P, int64_t *plan)
{
    for (int i = 0; i < 8; ++i) plan[i] = 0;
    if (cfg.scoring != 0 || cfg.renormalize != 1 || cfg.n_group != 1 || cfg.k > 8) return false;
    if (fused2_plan(L, T, cfg, D, N, P, plan)) return true;
    FusedGeom f;
    if (!fused_geom(L, T, cfg.k, cfg.E, D, N, P, &f)) return false;
    const int64_t BT = (int64_t)EF_PASSES * f.g.S;
    const int64_t per_src = (T + D - 1) / D;
    plan[0] = 1;
    plan[1] = f.g.ncta_t;
    plan[2] = f.g.tpc;
    plan[3] = f.g.tpc < per_src ? f.g.tpc : per_src;
    plan[4] = (int64_t)(EF_MAXBLK - 2) * BT;
    plan[5] = f.g.maxrec;
    plan[6] = f.cps;
    plan[7] = 1;
    return true;
}

template <int E>
static int launch_fused_e(const FusedParams &prm, const FusedGeom &f, int L, cudaStream_t st)
{
    // per device and cheap: set on every launch (a per-process flag would leave a second GPU without the opt-in)
    cudaFuncSetAttribute(trace_fused_kernel<E>, cudaFuncAttributeMaxDynamicSharedMemorySize, 225 * 1024);
    {
        KernelTimerScope ts("trace_fused", st);
        launch_pdl_edge(trace_fused_kernel<E>, dim3((unsigned)f.g.ncta_t, (unsigned)L), dim3(f.nthreads), f.smem, st, prm);
    }
    note_launch();
    return check_launch("trace_fused_kernel");
}

// nrep > 0: profiling mode -- after the table build, launch ONLY the fused kernel nrep times back to
// back (input i = logits_list[i % nlist]) between two events and return the average in *avg_ms.
static int fused_core(const float *const *logits_list, int nlist, int nrep, float *avg_ms, int32_t L, int64_t T,
                      const cap_gate_cfg &cfg, int32_t *idx, float *w, int64_t *counts, int32_t *coact,
                      const int32_t *expert_dev, int32_t P, const cap_topology &topo, const cap_eval_out &out,
                      void *ws, cudaStream_t st, bool *used)
{
    *used = false;
    FusedGeom f;
    if (!fused_geom(L, T, cfg.k, cfg.E, topo.D, topo.N, P, &f)) return CAP_OK;
    const int E = cfg.E;
    EvalFastWs fw = eval_fast_ws_carve(ws, L, E, topo.D, P, f.g);
    // every buffer the pass accumulates into is cleared by the table kernel itself (no memset nodes)
    const EfFill fills[3] = {
        {counts, sizeof(int64_t) * (size_t)L * E, 0u},
        {coact, sizeof(int32_t) * (size_t)L * E * E, 0u},
        {fw.rec_src, f.g.rec_slots * 4, 0xffffffffu},
    };
    CAP_TRY(ef_launch_table(f.g, fw, expert_dev, topo.dev_node, L, E, P, topo.D, st, fills, 3));
    FusedParams prm;
    prm.logits = logits_list[0];
    prm.idx = idx;
    prm.w = w;
    prm.counts = reinterpret_cast<unsigned long long *>(counts);
    prm.coact = coact;
    prm.table = fw.table;
    prm.rec_src = fw.rec_src;
    prm.rec_planes = fw.rec_planes;
    prm.T = T;
    prm.tiles_per_cta = f.tiles_per_cta;
    prm.cps = f.cps;
    prm.scale = cfg.scale;
    prm.k = cfg.k;
    prm.D = topo.D;
    prm.pack64 = (E % 2 == 0) && (reinterpret_cast<uintptr_t>(coact) & 7u) == 0;
    prm.R = f.g.R;
    prm.RS = f.g.RS;
    prm.S = f.g.S;
    prm.logS = f.g.logS;
    prm.maxrec = f.g.maxrec;
    prm.NPR = f.g.NPR;
    prm.ncta_t = f.g.ncta_t;
    prm.nst = f.nst;
    prm.ns3w = f.ns3w;
    cudaEvent_t ea = nullptr, eb = nullptr;
    if (nrep > 0) {
        if (cudaEventCreate(&ea) != cudaSuccess || cudaEventCreate(&eb) != cudaSuccess) return check_launch("event");
        cudaEventRecord(ea, st);
    }
    const int reps = nrep > 0 ? nrep : 1;
    for (int i = 0; i < reps; ++i) {
        prm.logits = logits_list[i % nlist];
        int rc;
        switch (E) {
        case 64: rc = launch_fused_e<64>(prm, f, L, st); break;
        case 128: rc = launch_fused_e<128>(prm, f, L, st); break;
        default: rc = launch_fused_e<256>(prm, f, L, st); break;
        }
        CAP_TRY(rc);
    }
    if (nrep > 0) {
        cudaEventRecord(eb, st);
        if (cudaEventSynchronize(eb) != cudaSuccess) return check_launch("event sync");
        float ms = 0.0f;
        cudaEventElapsedTime(&ms, ea, eb);
        cudaEventDestroy(ea);
        cudaEventDestroy(eb);
        if (avg_ms) *avg_ms = ms / (float)nrep;
        *used = true;
        return CAP_OK;        // accumulators hold nrep passes: profiling only, outputs are not finalised
    }
    CAP_TRY(ef_launch_decode(f.g, fw, L, T, E, P, topo, expert_dev, counts, out, st));
    *used = true;
    return CAP_OK;
}

static bool fused_args_ok(const float *logits, const float *bias, const cap_gate_cfg &cfg, int32_t *idx, float *w,
                          int64_t *counts, int32_t *coact, const int32_t *token_src, const cap_eval_out &out,
                          int32_t L, int64_t T, int32_t P)
{
    if (cfg.scoring != 0 || cfg.renormalize != 1 || cfg.n_group != 1 || cfg.k > 8 || bias != nullptr) return false;
    if (token_src != nullptr || out.tok_remote_dev || out.tok_remote_node) return false;
    if (!counts || !coact || L < 1 || T < 1 || P < 1) return false;
    if ((reinterpret_cast<uintptr_t>(logits) | reinterpret_cast<uintptr_t>(idx) | reinterpret_cast<uintptr_t>(w)) & 15u)
        return false;
    return true;
}

int launch_trace_fused_fast(const float *logits, const float *bias, int32_t L, int64_t T, const cap_gate_cfg &cfg,
                            int32_t *idx, float *w, int64_t *counts, int32_t *coact, const int32_t *token_src,
                            const int32_t *expert_dev, int32_t P, const cap_topology &topo,
                            const cap_eval_out &out, void *ws, cudaStream_t st, bool *used)
{
    *used = false;
    CAP_TRY(launch_trace_fused2(logits, bias, L, T, cfg, idx, w, counts, coact, token_src, expert_dev, P, topo, out,
                                eval_fast_region(ws, L, cfg.E, topo.D, P), st, used));
    if (*used) return CAP_OK;
    if (!fused_args_ok(logits, bias, cfg, idx, w, counts, coact, token_src, out, L, T, P)) return CAP_OK;
    return fused_core(&logits, 1, 0, nullptr, L, T, cfg, idx, w, counts, coact, expert_dev, P, topo, out, ws, st, used);
}

int profile_trace_fused_kernel(const float *const *logits_list, int nlist, int nrep, float *avg_ms, int32_t L,
                               int64_t T, const cap_gate_cfg &cfg, int32_t *idx, float *w, int64_t *counts,
                               int32_t *coact, const int32_t *expert_dev, int32_t P, const cap_topology &topo,
                               const cap_eval_out &out, void *ws, cudaStream_t st, bool *used)
{
    *used = false;
    {
        // the single-launch kernel: a launch is the whole call, so the profile times nrep complete calls
        int64_t plan[8];
        if (nrep > 0 && fused2_plan(L, T, cfg, topo.D, topo.N, P, plan)) {
            cudaEvent_t ea = nullptr, eb = nullptr;
            if (cudaEventCreate(&ea) != cudaSuccess || cudaEventCreate(&eb) != cudaSuccess) return check_launch("event");
            void *reg = eval_fast_region(ws, L, cfg.E, topo.D, P);
            bool u2 = false;
            CAP_TRY(launch_trace_fused2(logits_list[0], nullptr, L, T, cfg, idx, w, counts, coact, nullptr, expert_dev,
                                        P, topo, out, reg, st, &u2));
            if (u2) {
                cudaEventRecord(ea, st);
                for (int i = 0; i < nrep; ++i)
                    CAP_TRY(launch_trace_fused2(logits_list[i % nlist], nullptr, L, T, cfg, idx, w, counts, coact, nullptr,
                                                expert_dev, P, topo, out, reg, st, &u2));
                cudaEventRecord(eb, st);
                if (cudaEventSynchronize(eb) != cudaSuccess) return check_launch("event sync");
                float ms = 0.0f;
                cudaEventElapsedTime(&ms, ea, eb);
                cudaEventDestroy(ea);
                cudaEventDestroy(eb);
                if (avg_ms) *avg_ms = ms / (float)nrep;
                *used = true;
                return CAP_OK;
            }
            cudaEventDestroy(ea);
            cudaEventDestroy(eb);
        }
    }
    for (int i = 0; i < nlist; ++i)
        if (!fused_args_ok(logits_list[i], nullptr, cfg, idx, w, counts, coact, nullptr, out, L, T, P)) return CAP_OK;
    return fused_core(logits_list, nlist, nrep, avg_ms, L, T, cfg, idx, w, counts, coact, expert_dev, P, topo, out,
                      ws, st, used);
}

}  // namespace cap

#ifdef CAP_FU_TRACE
extern "C" int cap_debug_fused_trace(unsigned long long *host_out, int n)
{
    if (n > 160 * 24 * 8) n = 160 * 24 * 8;
    return (int)cudaMemcpyFromSymbol(host_out, cap::g_fu_trace, sizeof(unsigned long long) * (size_t)n);
}
#endif

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
constexpr int F2_MAXST = 16;         // logits ring stages
constexpr int F2_THREADS = 640;      // 20 warps: 96 registers per thread (the scoring loop needs ~90)
constexpr int F2_MAXRUNBLK = 29;     // 64-token blocks per run: <= 31 CSA rounds of 8 inputs < 256
constexpr int F2_NPL = 11;           // planes of a run after its 8 partial counters were added
constexpr int F2_CG = 4;             // candidates a block finishes per round of phase 1
constexpr int F2_MAXSLOTS = 4096;    // records per layer the finishing phase can index

// Optional per-warp timeline (build with -DCAP_F2_TRACE, read back with cap_debug_f2_trace): clock64 stamps
// relative to the block's entry at role milestones.  Not compiled into the product library.
#ifdef CAP_F2_TRACE
__device__ unsigned long long g_f2_trace[160 * 24 * 32];
#define F2_TR(ev)                                                                              \
    do {                                                                                       \
        if ((threadIdx.x & 31) == 0 && blockIdx.x + gridDim.x * blockIdx.y < 160 && (threadIdx.x >> 5) < 24) { \
            unsigned long long gt_;                                                            \
            asm volatile("mov.u64 %0, %globaltimer;" : "=l"(gt_));                             \
            g_f2_trace[((size_t)(blockIdx.x + gridDim.x * blockIdx.y) * 24 + (threadIdx.x >> 5)) * 32 + (ev)] = gt_; \
        }                                                                                      \
    } while (0)
#else
#define F2_TR(ev) do { } while (0)
#endif

struct F2Params {
    const float *logits;
    int32_t *idx;
    float *w;
    long long *counts;            // [L][E]
    int *coact;                   // [L][E][E]
    const int32_t *maps;          // [L][P][E]
    const int32_t *dev_node;      // [D]
    cap_eval_out out;
    uint32_t *recs;               // [L][nblk][maxrec][ncnt]
    int32_t *rec_src;             // [L][nblk][maxrec], -1 = unused
    unsigned char *gtab;          // [L][E * (Cd + Cn) * 16] code tables (device rows, then node rows), shared-memory layout
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
    // the blocks of a layer share the work: block b builds items [b * chunk, (b + 1) * chunk) of the layer's
    // table in the workspace (every SM reading all P * E map entries itself costs ~6 us: the same 128 KB
    // requested by 148 SMs at once)
    const int chunk = (nitems + (int)gridDim.x - 1) / (int)gridDim.x;
    const int i_lo = (int)blockIdx.x * chunk, i_hi = min(nitems, i_lo + chunk);
    for (int it = i_lo + t3; it < i_hi; it += ns3) {
        const int p16 = it / E, e = it - p16 * E;
        const int p0 = p16 * 16;
        int dv[16];
#pragma unroll
        for (int j = 0; j < 16; ++j) dv[j] = __ldg(maps + (size_t)min(p0 + j, P - 1) * E + e);   // clamped: no branch
#pragma unroll
        for (int j = 0; j < 16; ++j) dv[j] = (p0 + j < P) ? dv[j] : -1;
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
    uint4 v0, v1, v2, v3, m;
#define F2_LD(V, a) \
    asm("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(V.x), "=r"(V.y), "=r"(V.z), "=r"(V.w) : "r"((a) ^ cx))
    F2_LD(v0, oa.x); F2_LD(v1, oa.y); F2_LD(v2, oa.z); F2_LD(v3, oa.w);
    m.x = lop_or3(v0.x, v1.x, lop_or3(v2.x, v3.x, 0u));
    m.y = lop_or3(v0.y, v1.y, lop_or3(v2.y, v3.y, 0u));
    m.z = lop_or3(v0.z, v1.z, lop_or3(v2.z, v3.z, 0u));
    m.w = lop_or3(v0.w, v1.w, lop_or3(v2.w, v3.w, 0u));
    F2_LD(v0, ob.x); F2_LD(v1, ob.y); F2_LD(v2, ob.z); F2_LD(v3, ob.w);
#undef F2_LD
    m.x = lop_or3(lop_or3(m.x, v0.x, v1.x), v2.x, v3.x);
    m.y = lop_or3(lop_or3(m.y, v0.y, v1.y), v2.y, v3.y);
    m.z = lop_or3(lop_or3(m.z, v0.z, v1.z), v2.z, v3.z);
    m.w = lop_or3(lop_or3(m.w, v0.w, v1.w), v2.w, v3.w);
    return m;
}

// a (np planes) += b (np planes, plane p fetched by FETCH(p)), result has np + 1 planes (bit-sliced ripple
// add, one plane of b live at a time)
#define F2_ADD_PLANES(A, NP, FETCH)                                        \
    do {                                                                   \
        uint4 cy_ = make_uint4(0u, 0u, 0u, 0u);                            \
        _Pragma("unroll") for (int p = 0; p < F2_NPL; ++p) {               \
            if (p <= (NP)) {                                               \
                uint4 x_ = make_uint4(0u, 0u, 0u, 0u);                     \
                if (p < (NP)) x_ = FETCH(p);                               \
                uint4 s_, c_;                                              \
                F2_CSA4(s_, c_, (A)[p], x_, cy_);                          \
                (A)[p] = s_;                                               \
                cy_ = c_;                                                  \
            }                                                              \
        }                                                                  \
    } while (0)

// ---- block-shared state (static shared memory) ---------------------------------------------------------
struct F2Shared {
    uint64_t full_bar[F2_MAXST], empty_bar[F2_MAXST];   // logits ring
    uint64_t offs_full[F2_OB];                          // S1 -> S3: a 64-token descriptor block is complete
    uint64_t tile_full[2], mma_done[2];                 // S1 -> tensor-core warp, tensor core -> its warp
    uint64_t acc_done, tbl_bar;
    // progress counters of the two back edges (S3 -> S1: descriptor blocks consumed by each scoring warp;
    // tensor-core warp -> S1: one-hot tile buffers recycled).  Plain monotonic counters instead of parity
    // barriers: an S1 warp visits only every ns1w-th tile, so it can be several phases ahead of a barrier
    // it has never waited on, which a parity wait cannot tell from "already complete".
    alignas(16) uint32_t s3_prog[16];
    uint32_t recycled;
    uint32_t tile_ctr;                                  // next 16-token tile an S1 warp takes
    uint32_t tmem;
    long long t0, t1;                                   // this block's token range of its layer
    int nt, ntp, nb;                                    // 16-token tiles, tiles with ghosts, 64-token blocks
    unsigned char node[64];                             // node of each device
};

template <int E>
struct F2Const {
    static constexpr int EP = E <= 128 ? 128 : 256;
    static constexpr uint32_t LBO = 128u, SBO = (F2_BT / 16) * 128u;
    static constexpr uint32_t NCOLS = EP == 128 ? 128u : 512u;
    static constexpr uint32_t IDESC = (2u << 4) | ((uint32_t)(EP >> 3) << 17) | (8u << 24);
    static constexpr int TILE_BYTES = F2_TILE * E * 4;
};

// ================= producer: TMA bulk copies of 16-token logits tiles into the ring =================
template <int E>
__device__ __noinline__ void f2_role_producer(const F2Params &q, F2Shared &sh, unsigned char *sm, int first)
{
    const F2Smem lay = f2_smem_layout(E, F2Const<E>::EP, q.Cd, q.Cn, q.nwd, q.nwn, q.nst);
    unsigned char *ring = sm + lay.ring;
    const int nst = q.nst, nt = sh.nt;
    const long long t0 = sh.t0, t1 = sh.t1;
    const float *logits = q.logits + (size_t)blockIdx.y * q.T * E;
    for (int j = first; j < nt; ++j) {
        const int st = j % nst;
        if (j >= nst) mbar_wait_relaxed(&sh.empty_bar[st], (uint32_t)(((j / nst) - 1) & 1), 128);
        const long long tok0 = t0 + (long long)j * F2_TILE;
        const int rows = (int)min((long long)F2_TILE, t1 - tok0);
        mbar_expect_tx(&sh.full_bar[st], (uint32_t)rows * E * 4);
        bulk_g2s(ring + (size_t)st * F2Const<E>::TILE_BYTES, logits + tok0 * E, (uint32_t)rows * E * 4, &sh.full_bar[st]);
    }
}

// ================= tensor-core warp: C += A^T A on the one-hot tiles =================
template <int E>
__device__ __noinline__ void f2_role_mma(const F2Params &q, F2Shared &sh, unsigned char *sm)
{
    using K = F2Const<E>;
    const F2Smem lay = f2_smem_layout(E, K::EP, q.Cd, q.Cn, q.nwd, q.nwn, q.nst);
    unsigned char *tiles = sm + lay.tiles;
    const int lane = threadIdx.x & 31;
    const int nb = sh.nb;
    const uint32_t tmem = sh.tmem;
    for (int m = 0; m < nb; ++m) {
        const int tb = m & 1;
        unsigned char *tile = tiles + (size_t)tb * K::EP * F2_BT;
        mbar_wait_relaxed(&sh.tile_full[tb], (uint32_t)((m >> 1) & 1), 128);
        tc_fence_after();
        if (lane == 0) {
            const uint32_t base = smem_u32(tile);
#pragma unroll
            for (int j = 0; j < F2_BT / 32; ++j) {
                const uint64_t bd = umma_desc(base + j * 2 * K::LBO, K::LBO, K::SBO);
                umma_i8(tmem, bd, bd, K::IDESC, (uint32_t)((m | j) != 0));
                if (K::EP == 256) {
                    const uint64_t a1 = umma_desc(base + 16 * K::SBO + j * 2 * K::LBO, K::LBO, K::SBO);
                    umma_i8(tmem + 256u, a1, bd, K::IDESC, (uint32_t)((m | j) != 0));
                }
            }
            umma_commit(&sh.mma_done[tb]);
            if (m == nb - 1) umma_commit(&sh.acc_done);
        }
        __syncwarp();
        if (m + 2 < nb) {
            // recycle the buffer for block m + 2: wait until the tensor core has read it, clear it
            mbar_wait(&sh.mma_done[tb], (uint32_t)((m >> 1) & 1));
            uint4 *z = reinterpret_cast<uint4 *>(tile);
            for (int i = lane; i < K::EP * F2_BT / 16; i += 32) z[i] = make_uint4(0u, 0u, 0u, 0u);
            proxy_fence_async();
            __syncwarp();
            if (lane == 0) st_release_cta(&sh.recycled, (uint32_t)(m + 1));
        }
    }
}

// ================= S1: gate top-k, two lanes per token; c = index among the ns1w S1 warps =================
template <int E>
__device__ __noinline__ void f2_role_s1(const F2Params &q, F2Shared &sh, unsigned char *sm, int c, int ns1w)
{
    using K = F2Const<E>;
    const F2Smem lay = f2_smem_layout(E, K::EP, q.Cd, q.Cn, q.nwd, q.nwn, q.nst);
    unsigned char *ring = sm + lay.ring;
    unsigned char *tiles = sm + lay.tiles;
    uint32_t *offs = reinterpret_cast<uint32_t *>(sm + lay.offs);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int layer = blockIdx.y;
    const int nst = q.nst, k = q.k;
    const long long t0 = sh.t0, t1 = sh.t1;
    const int nt = sh.nt, ntp = sh.ntp, nb = sh.nb;
    int32_t *gidx = q.idx + (size_t)layer * q.T * k;
    float *gw = q.w + (size_t)layer * q.T * k;
    const int h = lane >> 4, tl = lane & 15;
    const uint32_t tabD_s = smem_u32(sm + lay.tabD), tabN_s = smem_u32(sm + lay.tabN);
    const uint32_t rowD = (uint32_t)q.Cd * 16u, rowN = (uint32_t)q.Cn * 16u;
    const uint32_t mD = (uint32_t)q.Cd - 1u, mN = (uint32_t)q.Cn - 1u;
    // tiles are handed out dynamically (in increasing order): the S1 warps of the four scheduler partitions
    // stay equally loaded whatever their number
    for (;;) {
        int j = 0;
        if (lane == 0) j = (int)atomicAdd(&sh.tile_ctr, 1u);
        j = __shfl_sync(0xffffffffu, j, 0);
        if (j >= ntp) break;
        const bool ghost = j >= nt;
        const int st = j % nst;
        const long long tok = t0 + (long long)j * F2_TILE + tl;
        const bool valid = !ghost && tok < t1;
        int sel[8];
        float wv[4];
#pragma unroll
        for (int i = 0; i < 8; ++i) sel[i] = 0;
        wv[0] = wv[1] = wv[2] = wv[3] = 0.0f;
        if (!ghost) {
            // this warp shares a stage with other warps: first make sure the previous use of the stage has
            // been consumed (so that the parity below is this use's), then wait for the data
            const int u = j / nst;
            if (u >= 1) mbar_wait(&sh.empty_bar[st], (uint32_t)((u - 1) & 1));
            mbar_wait(&sh.full_bar[st], (uint32_t)(u & 1));
            const float *row = reinterpret_cast<const float *>(ring + (size_t)st * K::TILE_BYTES +
                                                               (size_t)(tok < t1 ? tl : 0) * E * 4);
            if (j < ns1w) F2_TR(1);
            else if (j < 2 * ns1w) F2_TR(10);
            gate_select_pair<E>(row, h, tl & 7, k, sel);
            if (j >= ns1w && j < 2 * ns1w) F2_TR(11);
            gate_weights_softmax_pair(row, h, k, sel, q.scale, wv);
            if (j < ns1w) F2_TR(2);
            else if (j < 2 * ns1w) F2_TR(12);
        }
        // ---- row descriptors for S3: slots past k repeat slot 0 (OR is idempotent); tokens past the
        //      range point at row 0 and are masked out by their index ----
        const int b = j / F2_TPB, ob = b % F2_OB;
        if (b >= F2_OB) {
            // every scoring warp must have finished block b - F2_OB (it used this descriptor slot)
            for (;;) {
                const uint4 p0 = ld_acquire_cta_v4(&sh.s3_prog[0]), p1 = ld_acquire_cta_v4(&sh.s3_prog[4]),
                            p2 = ld_acquire_cta_v4(&sh.s3_prog[8]), p3 = ld_acquire_cta_v4(&sh.s3_prog[12]);
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
            while (ld_acquire_cta(&sh.recycled) < (uint32_t)(b - 1)) __nanosleep(40);
        if (valid) {
            const int tp = (j % F2_TPB) * F2_TILE + tl;
            unsigned char *col = tiles + (size_t)tb * K::EP * F2_BT + (tp >> 4) * K::LBO + (tp & 15);
#pragma unroll
            for (int jj = 0; jj < 4; ++jj) {
                const int s = 4 * h + jj;
                const int e = h ? sel[4 + jj] : sel[jj];
                if (s < k) col[(e >> 3) * K::SBO + (e & 7) * 16] = 1;
            }
        }
        proxy_fence_async();
        __syncwarp();
        if (lane == 0) {
            mbar_arrive(&sh.offs_full[ob]);
            mbar_arrive(&sh.tile_full[tb]);
            if (!ghost) mbar_arrive(&sh.empty_bar[st]);
        }
        // top-k indices and weights to HBM last: the proxy fence above must not wait for these stores
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
        if (j >= ns1w && j < 2 * ns1w) F2_TR(13);
    }
    F2_TR(3);
    // ---- drain the co-activation accumulator: reductions straight into the layer's matrix, which the
    //      blocks cleared before the first grid barrier (64-bit packed: two int32 counters per reduction,
    //      coalesced through the symmetry C[r][c] = C[c][r]); the diagonal is the activation count ----
    if (c < 4 && nb > 0) {
        const uint32_t tmem = sh.tmem;
        const int quad = warp & 3;
        mbar_wait_relaxed(&sh.acc_done, 0u, 64);
        tc_fence_after();
        int *C = q.coact + (size_t)layer * E * E;
        unsigned long long *cnt = reinterpret_cast<unsigned long long *>(q.counts) + (size_t)layer * E;
#pragma unroll 1
        for (int hh = 0; hh < K::EP / 128; ++hh) {
            const int r = hh * 128 + quad * 32 + lane;
#pragma unroll 1
            for (int cb = 0; cb < K::EP / 32; ++cb) {
                if (cb * 32 >= E || hh * 128 + quad * 32 >= E) continue;
                uint32_t v[32];
                tmem_ld32(tmem + ((uint32_t)(quad * 32) << 16) + (uint32_t)(hh * 256 + cb * 32), v);
                const bool rok = r < E;
                int *cp = C + (size_t)(cb * 32) * E + (r & ~1);
#pragma unroll
                for (int j = 0; j < 32; j += 2) {
                    const uint32_t p0 = __shfl_xor_sync(0xffffffffu, v[j], 1);
                    const uint32_t p1 = __shfl_xor_sync(0xffffffffu, v[j + 1], 1);
                    const int jj = j + (lane & 1);
                    const unsigned long long pk = (lane & 1) ? ((unsigned long long)v[j + 1] << 32) | p1
                                                             : ((unsigned long long)p0 << 32) | v[j];
                    if (rok && cb * 32 + jj < E && pk)
                        asm volatile("red.global.add.u64 [%0], %1;" ::"l"(cp + (size_t)jj * E), "l"(pk) : "memory");
                }
                if (rok && (r >> 5) == cb) {
                    uint32_t d = 0u;
#pragma unroll
                    for (int j = 0; j < 32; ++j) d = (r & 31) == j ? v[j] : d;
                    if (d) atomicAdd(&cnt[r], (unsigned long long)d);
                }
            }
        }
    }
}

// ================= S3: bit-sliced candidate scoring; w3 = index among the scoring warps =================
// flush of one run: add the 8 partial counters of every bit position (lanes of a warp that share a chunk,
// then the warps of a class), decode the sums, write the record
struct F2Planes8 {
    uint4 p[8];
};
__device__ __forceinline__ void f2_flush(const F2Params &q, const F2Planes8 &in, uint4 *xch, int cls, int a, int nwc, int C,
                                      int lane, int t3, int ns3, size_t rec_slot, int src)
{
    const int tk = lane / C, cc = lane - tk * C;
    uint4 pl[F2_NPL];
#pragma unroll
    for (int p = 0; p < F2_NPL; ++p) pl[p] = p < 8 ? in.p[p < 8 ? p : 0] : make_uint4(0u, 0u, 0u, 0u);
    // (1) the lanes of a warp that share a chunk: butterfly over the token bits of the lane id
    int np = 8;
    for (int off = C; off < 32; off <<= 1) {
#define F2_FETCH_SHFL(p)                                                                                      \
    make_uint4(__shfl_xor_sync(0xffffffffu, pl[p].x, off), __shfl_xor_sync(0xffffffffu, pl[p].y, off),        \
               __shfl_xor_sync(0xffffffffu, pl[p].z, off), __shfl_xor_sync(0xffffffffu, pl[p].w, off))
        F2_ADD_PLANES(pl, np, F2_FETCH_SHFL);
#undef F2_FETCH_SHFL
        ++np;
    }
    F2_TR(9);
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
#define F2_FETCH_XCH(p) xch[xbase + (a * F2_NPL + (p)) * 32 + lane]
            F2_ADD_PLANES(pl, np, F2_FETCH_XCH);
#undef F2_FETCH_XCH
        }
        if (act) ++np;
        f2_bar(1, ns3);
    }
    F2_TR(10);
    // (3) warp 0 of each class leaves the run's planes as [plane][word] (device words, then node words)
    uint32_t *fin = reinterpret_cast<uint32_t *>(xch);
    const int nwords = (q.Cd + q.Cn) * 4;
    if (a == 0 && tk == 0) {
        const int wb = (cls ? q.Cd * 4 : 0) + cc * 4;
#pragma unroll
        for (int p = 0; p < F2_NPL; ++p) *reinterpret_cast<uint4 *>(fin + (size_t)p * nwords + wb) = pl[p];
    }
    f2_bar(1, ns3);
    F2_TR(11);
    // (4) every S3 thread decodes counters: counter i = bit (i & 31) of word i >> 5
    {
        uint32_t *rec = q.recs + rec_slot * (size_t)q.ncnt;
        for (int i = t3; i < q.ncnt; i += ns3) {
            const int wi = i >> 5, bit = i & 31;
            uint32_t v = 0u;
#pragma unroll
            for (int p = 0; p < F2_NPL; ++p) v |= ((fin[(size_t)p * nwords + wi] >> bit) & 1u) << p;
            rec[i] = v;
        }
        if (t3 == 0) q.rec_src[rec_slot] = src;
    }
    F2_TR(12);
    f2_bar(1, ns3);
}

template <int E>
__device__ __noinline__ void f2_role_s3(const F2Params &q, F2Shared &sh, unsigned char *sm, int w3)
{
    const F2Smem lay = f2_smem_layout(E, F2Const<E>::EP, q.Cd, q.Cn, q.nwd, q.nwn, q.nst);
    uint32_t *offs = reinterpret_cast<uint32_t *>(sm + lay.offs);
    uint4 *xch = reinterpret_cast<uint4 *>(sm + lay.xch);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int ns3 = (q.nwd + q.nwn) * 32;
    const int t3 = threadIdx.x - ((int)blockDim.x - ns3);
    const int D = q.D;
    const long long T = q.T, t0 = sh.t0, t1 = sh.t1;
    const int nb = sh.nb;
    const int cls = w3 < q.nwd ? 0 : 1;
    const int a = cls ? w3 - q.nwd : w3;               // warp within its class
    const int nwc = cls ? q.nwn : q.nwd;               // warps of the class = C / 4
    const int C = cls ? q.Cn : q.Cd;                   // 16-byte chunks per row
    const int TPW = 32 / C;                            // tokens per load
    const int tk = lane / C, cc = lane - tk * C;
    const uint32_t cx = (uint32_t)cc << 4;
    const int tokw = a * 8 * TPW + tk;                 // + i * TPW: token of input i inside a block
    const long long cap_run = (long long)F2_MAXRUNBLK * F2_BT;
    const size_t slot0 = ((size_t)blockIdx.y * gridDim.x + blockIdx.x) * q.maxrec;
    F2Planes8 cnt;                                     // planes a lane counts in (inputs < 256 per run)
#define pl8 cnt.p
#pragma unroll
    for (int p = 0; p < 8; ++p) pl8[p] = make_uint4(0u, 0u, 0u, 0u);
    int nrec = 0, src = 0;
    long long rend = t0;
    bool have_run = false;
    (void)warp;

    mbar_wait(&sh.tbl_bar, 0u);
    for (int b = 0; b < nb; ++b) {
        const int ob = b % F2_OB;
        mbar_wait_relaxed(&sh.offs_full[ob], (uint32_t)((b / F2_OB) & 1), 64);
        if (b == 0) F2_TR(2);
        if (b < 8) F2_TR(16 + 2 * b);
        const long long bt0 = t0 + (long long)b * F2_BT;
        const long long bend = min(bt0 + F2_BT, t1);
        const uint32_t *obuf = offs + ((size_t)ob * F2_BT + tokw) * 16 + cls * 8;
        long long cur = bt0;
        while (cur < bend) {
            if (cur >= rend) {
                if (have_run) {
                    f2_flush(q, cnt, xch, cls, a, nwc, C, lane, t3, ns3, slot0 + nrec, src);
                    ++nrec;
#pragma unroll
                    for (int p = 0; p < 8; ++p) pl8[p] = make_uint4(0u, 0u, 0u, 0u);
                }
                src = (int)((cur * D) / T);
                const long long bnd = ((long long)(src + 1) * T + D - 1) / D;
                rend = min(bnd, cur + cap_run);
                have_run = true;
            }
            const long long seg = min(bend, rend);
            const bool whole = cur == bt0 && seg == bt0 + F2_BT;
            uint4 fA, fB;
#define F2_LOAD(X, I)                                                        \
    do {                                                                     \
        X = f2_token_mask(obuf + (size_t)(I) * TPW * 16, cx);                \
        if (!whole) {                                                        \
            const long long tkn = bt0 + tokw + (I) * TPW;                    \
            if (tkn < cur || tkn >= seg) X = make_uint4(0u, 0u, 0u, 0u);     \
        }                                                                    \
    } while (0)
#define F2_HALF(OUT4, I0)                              \
    do {                                               \
        uint4 tA, tB, s, xa, xb;                       \
        F2_LOAD(xa, (I0));                             \
        F2_LOAD(xb, (I0) + 1);                         \
        F2_CSA4(s, tA, pl8[0], xa, xb);                \
        F2_LOAD(xa, (I0) + 2);                         \
        F2_LOAD(xb, (I0) + 3);                         \
        F2_CSA4(s, tB, s, xa, xb);                     \
        pl8[0] = s;                                    \
        F2_CSA4(pl8[1], OUT4, pl8[1], tA, tB);         \
    } while (0)
            F2_HALF(fA, 0);
            F2_HALF(fB, 4);
            {
                uint4 e8;
                F2_CSA4(pl8[2], e8, pl8[2], fA, fB);
#pragma unroll
                for (int p = 3; p < 8; ++p) {
                    uint4 cy;
                    cy.x = pl8[p].x & e8.x; cy.y = pl8[p].y & e8.y; cy.z = pl8[p].z & e8.z; cy.w = pl8[p].w & e8.w;
                    pl8[p].x ^= e8.x; pl8[p].y ^= e8.y; pl8[p].z ^= e8.z; pl8[p].w ^= e8.w;
                    e8 = cy;
                }
            }
#undef F2_LOAD
#undef F2_HALF
            cur = seg;
        }
        __syncwarp();
        if (lane == 0) st_release_cta(&sh.s3_prog[w3], (uint32_t)(b + 1));
        if (b < 8) F2_TR(17 + 2 * b);
    }
    F2_TR(3);
    if (have_run) f2_flush(q, cnt, xch, cls, a, nwc, C, lane, t3, ns3, slot0 + nrec, src);
    F2_TR(4);
#undef pl8
}

// ================= after the grid barrier: reductions of the layer's partial results =================
template <int E>
__device__ __noinline__ void f2_phase1(const F2Params &q, F2Shared &sh, unsigned char *sm)
{
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, nthr = blockDim.x;
    const int layer = blockIdx.y, blk = blockIdx.x, nblk = gridDim.x;
    const int D = q.D;
    // ---- expert counts of the layer (complete in global memory since the grid barrier) and the sources of
    //      the layer's records, staged in shared memory ----
    // 32-bit sums: every total is bounded by T k < 2^31 (cap.h limits)
    uint32_t *cnt_s = reinterpret_cast<uint32_t *>(sm);                        // [E]
    uint32_t *lp_s = reinterpret_cast<uint32_t *>(sm + 4096);                  // [F2_CG][64] pairs per device
    uint32_t *rv_s = lp_s + F2_CG * 64;                                        // [F2_CG][64] received tokens
    uint32_t *sc_s = rv_s + F2_CG * 64;                                        // [F2_CG][8] scalar sums
    signed char *src_s = reinterpret_cast<signed char *>(sc_s + F2_CG * 8);    // [nslots]
    const int nslots = nblk * q.maxrec;
    for (int e = tid; e < E; e += nthr) cnt_s[e] = (uint32_t)__ldcg(q.counts + (size_t)layer * E + e);
    {
        const int32_t *rs = q.rec_src + (size_t)layer * nslots;
        for (int i = tid; i < nslots; i += nthr) src_s[i] = (signed char)__ldcg(rs + i);
    }
    __syncthreads();
    F2_TR(7);
    // ---- 1c: finish this block's candidates p = blk, blk + nblk, ... (F2_CG at a time) ----
    const int WD = q.WD, WN = q.WN, P = q.P, N = q.N;
    const uint32_t *recs = q.recs + (size_t)layer * nslots * (size_t)q.ncnt;
    const int ncand = P > blk ? (P - blk + nblk - 1) / nblk : 0;
    for (int c0 = 0; c0 < ncand; c0 += F2_CG) {
        const int ng = min(F2_CG, ncand - c0);
        for (int i = tid; i < F2_CG * (64 + 64 + 8); i += nthr) lp_s[i] = 0u;
        __syncthreads();
        // received tokens per device, local / same-node sums: thread = (slot group sg, candidate g, device d);
        // a thread walks the record slots sg, sg + SG, ... with every load in flight, then adds its sums
        {
            const int ncol = ng * WD;
            const int SG = max(1, nthr / ncol);
            const int sg = tid / ncol, col = tid - sg * ncol;
            const int g = col / WD, d = col - g * WD;
            if (sg < SG && d < D) {
                const int p = blk + (c0 + g) * nblk;
                const uint32_t *rp = recs + (size_t)p * WD + d;
                const int nd = sh.node[d];
                uint32_t sv = 0u, sl = 0u, ss = 0u;
#pragma unroll 8
                for (int slot = sg; slot < nslots; slot += SG) {
                    const int sr = src_s[slot];
                    const uint32_t v = __ldcg(rp + (size_t)slot * q.ncnt);     // unused slots hold stale data: masked
                    const uint32_t vm = sr >= 0 ? v : 0u;
                    sv += vm;
                    sl += (sr == d) ? vm : 0u;
                    ss += (sr >= 0 && sh.node[sr < 0 ? 0 : sr] == nd) ? vm : 0u;
                }
                if (sv) {
                    atomicAdd(&rv_s[g * 64 + d], sv);
                    atomicAdd(&sc_s[g * 8 + 0], sv);
                }
                if (sl) atomicAdd(&sc_s[g * 8 + 1], sl);
                if (ss) atomicAdd(&sc_s[g * 8 + 2], ss);
            }
            const int ncoln = ng * WN;
            const int SGn = max(1, nthr / ncoln);
            const int sgn = tid / ncoln, coln = tid - sgn * ncoln;
            const int gn = coln / WN, n = coln - gn * WN;
            if (sgn < SGn && n < N) {
                const int p = blk + (c0 + gn) * nblk;
                const uint32_t *rp = recs + q.ndev + (size_t)p * WN + n;
                uint32_t sv = 0u, sr_ = 0u;
#pragma unroll 8
                for (int slot = sgn; slot < nslots; slot += SGn) {
                    const int sr = src_s[slot];
                    const uint32_t v = __ldcg(rp + (size_t)slot * q.ncnt);
                    const uint32_t vm = sr >= 0 ? v : 0u;
                    sv += vm;
                    sr_ += (sr >= 0 && n != (sh.node[sr < 0 ? 0 : sr] & (WN - 1))) ? vm : 0u;
                }
                if (sv) atomicAdd(&sc_s[gn * 8 + 3], sv);
                if (sr_) atomicAdd(&sc_s[gn * 8 + 4], sr_);
            }
            // load_pairs[d] = sum of the counts of the experts placed on d
            for (int i = tid; i < ng * E; i += nthr) {
                const int g2 = i / E, e = i - g2 * E;
                const int p = blk + (c0 + g2) * nblk;
                const int dd = q.maps[((size_t)layer * P + p) * E + e];
                const uint32_t cv = cnt_s[e];
                if ((unsigned)dd < (unsigned)D && cv) atomicAdd(&lp_s[g2 * 64 + dd], cv);
            }
        }
        __syncthreads();
        if (warp < ng) {
            const int g = warp;
            const int p = blk + (c0 + g) * nblk;
            const size_t o = (size_t)layer * P + p;
            long long mx = 0, smm = 0, mxr = 0, smr = 0;
            for (int d = lane; d < D; d += 32) {
                const long long l = (long long)lp_s[g * 64 + d];
                const long long r = (long long)rv_s[g * 64 + d];
                if (q.out.load_pairs) q.out.load_pairs[o * D + d] = l;
                if (q.out.recv_tokens) q.out.recv_tokens[o * D + d] = r;
                mx = max(mx, l);
                smm += l;
                mxr = max(mxr, r);
                smr += r;
            }
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) {
                mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, off));
                mxr = max(mxr, __shfl_xor_sync(0xffffffffu, mxr, off));
                smm += __shfl_xor_sync(0xffffffffu, smm, off);
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
                if (q.out.imbalance) q.out.imbalance[o] = smm ? __ddiv_rn((double)(mx * D), (double)smm) : 0.0;
                if (q.out.imbalance_recv) q.out.imbalance_recv[o] = smr ? __ddiv_rn((double)(mxr * D), (double)smr) : 0.0;
            }
        }
        __syncthreads();
    }
    F2_TR(8);
}

template <int E>
__global__ void __launch_bounds__(F2_THREADS, 1) trace_fused2_kernel(const __grid_constant__ F2Params q)
{
    extern __shared__ __align__(1024) unsigned char f2_sm[];
    __shared__ F2Shared sh;
    using K = F2Const<E>;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    F2_TR(15);
    const int nthr = blockDim.x;
    const int ns3w = q.nwd + q.nwn;
    const F2Smem lay = f2_smem_layout(E, K::EP, q.Cd, q.Cn, q.nwd, q.nwn, q.nst);

    // ---- set-up: thread 0 derives the block's token range, arms the barriers and requests the first
    //      ring of logits tiles at once (same two splits of the tokens as cap_fused.cu) ----
    if (tid == 0) {
        const int blk = blockIdx.x, D = q.D;
        const long long T = q.T;
        long long t0, t1;
        if (q.cps > 0 && T * (D + 1) < 0x7fffffffll) {
            // the same split in 32-bit arithmetic (64-bit divisions are ~100 instructions each on one thread)
            const uint32_t cps = (uint32_t)q.cps, Tu = (uint32_t)T, Du = (uint32_t)D;
            const uint32_t srcd = (uint32_t)blk / cps, jj = (uint32_t)blk % cps;
            const uint32_t b0 = (srcd * Tu + Du - 1u) / Du, b1 = ((srcd + 1u) * Tu + Du - 1u) / Du;
            const uint32_t nts = (b1 - b0 + F2_TILE - 1u) / F2_TILE;
            const uint32_t base = nts / cps, rem = nts % cps;
            const uint32_t ts = jj * base + (jj < rem ? jj : rem), tn = base + (jj < rem ? 1u : 0u);
            t0 = min(b1, b0 + ts * F2_TILE);
            t1 = min((long long)b1, t0 + (long long)tn * F2_TILE);
        } else if (q.cps > 0) {
            const int srcd = blk / q.cps, jj = blk % q.cps;
            const long long b0 = ((long long)srcd * T + D - 1) / D, b1 = ((long long)(srcd + 1) * T + D - 1) / D;
            const long long nts = (b1 - b0 + F2_TILE - 1) / F2_TILE;
            const long long base = nts / q.cps, rem = nts % q.cps;
            const long long ts = jj * base + (jj < rem ? jj : rem), tn = base + (jj < rem ? 1 : 0);
            t0 = min(b1, b0 + ts * F2_TILE);
            t1 = min(b1, t0 + tn * F2_TILE);
        } else {
            t0 = min(T, (long long)blk * q.tiles_per_cta * F2_TILE);
            t1 = min(T, t0 + q.tiles_per_cta * F2_TILE);
        }
        const int nt = (int)((t1 - t0 + F2_TILE - 1) / F2_TILE);
        sh.t0 = t0;
        sh.t1 = t1;
        sh.nt = nt;
        sh.ntp = ((nt + F2_TPB - 1) / F2_TPB) * F2_TPB;      // with ghost tiles: whole 64-token blocks
        sh.nb = sh.ntp / F2_TPB;
        for (int s = 0; s < q.nst; ++s) {
            mbar_init(&sh.full_bar[s], 1);
            mbar_init(&sh.empty_bar[s], 1);
        }
        for (int s = 0; s < F2_OB; ++s) mbar_init(&sh.offs_full[s], F2_TPB);
        for (int s = 0; s < 2; ++s) {
            mbar_init(&sh.tile_full[s], F2_TPB);
            mbar_init(&sh.mma_done[s], 1);
        }
        for (int s = 0; s < 16; ++s) sh.s3_prog[s] = s < ns3w ? 0u : 0x7fffffffu;
        sh.recycled = 0u;
        sh.tile_ctr = 0u;
        mbar_init(&sh.acc_done, 1);
        mbar_init(&sh.tbl_bar, 1);
        mbar_fence_init();
        // the first ring of tiles: in flight while every warp builds the code tables
        const float *logits = q.logits + (size_t)blockIdx.y * T * E;
        unsigned char *ring = f2_sm + lay.ring;
        const int npre = min(nt, q.nst);
        for (int j = 0; j < npre; ++j) {
            const long long tok0 = t0 + (long long)j * F2_TILE;
            const int rows = (int)min((long long)F2_TILE, t1 - tok0);
            mbar_expect_tx(&sh.full_bar[j], (uint32_t)rows * E * 4);
            bulk_g2s(ring + (size_t)j * K::TILE_BYTES, logits + tok0 * E, (uint32_t)rows * E * 4, &sh.full_bar[j]);
        }
    }
    if (warp == 1) tmem_alloc(&sh.tmem, K::NCOLS);
    {
        uint4 *z = reinterpret_cast<uint4 *>(f2_sm + lay.tiles);
        for (int i = tid; i < 2 * K::EP * F2_BT / 16; i += nthr) z[i] = make_uint4(0u, 0u, 0u, 0u);
    }
    if (tid < 64) sh.node[tid] = tid < q.D ? (unsigned char)(q.dev_node[tid] & 63) : 0;
    if (tid >= 64 && tid < 64 + q.maxrec)
        q.rec_src[((size_t)blockIdx.y * gridDim.x + blockIdx.x) * q.maxrec + (tid - 64)] = -1;
    proxy_fence_async();
    tc_fence_before();
    F2_TR(13);
    __syncthreads();
    tc_fence_after();
    F2_TR(14);
    // the layer's one-hot code tables: every block builds its share in the workspace, one grid barrier, then
    // each block fetches the finished tables with one bulk copy that lands while S1 selects its first tiles
    {
        const uint32_t tab_bytes = (uint32_t)E * (uint32_t)(q.Cd + q.Cn) * 16u;
        unsigned char *gt = q.gtab + (size_t)blockIdx.y * tab_bytes;
        f2_build_tables(q.maps + (size_t)blockIdx.y * q.P * E, sh.node, E, q.P, q.D, q.WD, q.WN, q.Cd, q.Cn, gt,
                        gt + (size_t)E * q.Cd * 16, tid, nthr);
        {
            // the layer's co-activation matrix and counts are accumulated with reductions: cleared here, by slices
            const int nblk = gridDim.x, blk = blockIdx.x;
            const int total4 = E * E / 4, per = (total4 + nblk - 1) / nblk;
            int4 *c4 = reinterpret_cast<int4 *>(q.coact + (size_t)blockIdx.y * E * E);
            for (int v = blk * per + tid; v < min(total4, (blk + 1) * per); v += nthr) c4[v] = make_int4(0, 0, 0, 0);
            if (blk == 0)
                for (int e = tid; e < E; e += nthr) q.counts[(size_t)blockIdx.y * E + e] = 0ll;
        }
        asm volatile("fence.proxy.async;" ::: "memory");      // generic stores above, bulk-copy reads below
        __threadfence();
        cg::this_grid().sync();
        if (tid == 0) {
            mbar_expect_tx(&sh.tbl_bar, tab_bytes);
            bulk_g2s(f2_sm + lay.tabD, gt, tab_bytes, &sh.tbl_bar);
        }
    }
    F2_TR(0);

    if (warp == 0) {
        if (lane == 0) f2_role_producer<E>(q, sh, f2_sm, min(sh.nt, q.nst));
    } else if (warp == 1) {
        f2_role_mma<E>(q, sh, f2_sm);
    } else if (warp < (nthr >> 5) - ns3w) {
        f2_role_s1<E>(q, sh, f2_sm, warp - 2, (nthr >> 5) - 2 - ns3w);
    } else {
        // the scoring warps take the highest warp ids: the issue arbiter prefers them, so the consumer
        // side of the S1 -> S3 hand-over never starves behind the (much longer) selection code
        f2_role_s3<E>(q, sh, f2_sm, warp - ((nthr >> 5) - ns3w));
    }

    // ================= every partial result of the layer is in the workspace =================
    F2_TR(5);
    tc_fence_before();
    __threadfence();
    cg::this_grid().sync();
    F2_TR(6);
    if (warp == 1) tmem_dealloc(sh.tmem, K::NCOLS);
    f2_phase1<E>(q, sh, f2_sm);
}

// ---- host side ------------------------------------------------------------------------------------------
struct F2Geom {
    int WD, WN, Cd, Cn, nwd, nwn, nst, EP, cps, maxrec, ncnt, ndev, nblk, nthreads;
    int64_t tiles_per_cta, tpc;
    size_t smem;
    size_t rec_words, rec_slots, gtab_bytes;
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
    // Opt-in (CAP_FUSED2=1): on B200 this single-launch variant is slower than the four-kernel path of
    // cap_fused.cu at every BASELINE size (config 3: 55.5 vs 49.0 us per call, config 2: 388 vs 179 us; see
    // DESIGN.md 6.4 for the timeline that explains it), so the library does not select it by default.
    {
        const char *env = getenv("CAP_FUSED2");
        if (!env || env[0] != '1') F2_FAIL("not enabled");
    }
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
    const size_t budget = 194 * 1024;      // carve-out 196 KB: 32 KB stay L1 for the few register spills of the cold paths
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
    g->gtab_bytes = (size_t)L * E * (size_t)(g->Cd + g->Cn) * 16;
    // phase 1 reuses the front of the dynamic shared memory: counts, per-round sums, record sources
    if (4096 + F2_CG * (64 + 64 + 8) * 4 + (size_t)g->nblk * g->maxrec + 64 > g->smem) F2_FAIL("phase-1 smem");
    return true;
#undef F2_FAIL
}

size_t fused2_ws_bytes(int32_t L, int64_t T, int32_t k, int32_t E, int32_t D, int32_t P)
{
    size_t best = 0;
    for (int N = 2; N <= 8; N *= 2) {
        F2Geom g;
        if (!f2_geom(L, T, k, E, D, N, P, &g)) continue;
        const size_t b = g.rec_words * 4 + 256 + g.rec_slots * 4 + 256 + g.gtab_bytes + 256;
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
    prm.recs = reinterpret_cast<uint32_t *>(a);
    a = (a + g.rec_words * 4 + 255) & ~(uintptr_t)255;
    prm.rec_src = reinterpret_cast<int32_t *>(a);
    a = (a + g.rec_slots * 4 + 255) & ~(uintptr_t)255;
    prm.gtab = reinterpret_cast<unsigned char *>(a);
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

#ifdef CAP_F2_TRACE
extern "C" int cap_debug_f2_trace(unsigned long long *host_out, int n)
{
    if (n > 160 * 24 * 32) n = 160 * 24 * 32;
    return (int)cudaMemcpyFromSymbol(host_out, cap::g_f2_trace, sizeof(unsigned long long) * (size_t)n);
}
#endif

// S3 fast path -- bit-sliced scoring of P candidate placements (Eq. 3, Eq. 4, Fig. 6 axes,
// Tables II-IV).  Used when the token sources are the default contiguous blocks (token_src NULL,
// reading R5) and no per-token output is wanted; otherwise the generic kernel of cap_eval.cu runs.
// Method and data layout: cap_eval_fast.cuh and DESIGN.md section 6.
#include <cstdio>
#include <cstdlib>
#include <cstring>

#include "cap_eval_fast.cuh"

namespace cap {

// ---- host geometry ----------------------------------------------------------------------------------
static int ceil_log2(long long v)
{
    int b = 0;
    while ((1ll << b) < v) ++b;
    return b;
}

bool eval_fast_geom(int32_t L, int64_t T, int32_t k, int32_t E, int32_t D, int32_t N, int32_t P,
                    int target_ctas, size_t smem_budget, EvalFastGeom *g, bool explicit_src, int rs_limit)
{
    if (L < 1 || T < 1 || P < 1 || D < 1 || D > 64 || N < 1 || N > 8 || k < 1 || k > 16) return false;
    g->WD = D <= 8 ? 8 : D <= 16 ? 16 : D <= 32 ? 32 : 64;
    g->WN = N <= 2 ? 2 : N <= 4 ? 4 : 8;
    g->KP = (k + 3) & ~3;
    const int unit = 128 / g->WD;                 // candidates per 16-byte column of the device section
    const int Pfull = ((P + unit - 1) / unit) * unit;
    // largest chunk whose table fits: (E + 1) rows of RS * 16 bytes; the chunk shrinks in single-column steps and
    // the chunks are then equalised
    const bool alone = rs_limit == EF_RS_ALONE;
    auto fits = [&](int Pc, bool commit) {
        const int dcol = Pc * g->WD / 128;
        const int ncol = (Pc * g->WN + 127) / 128;
        const int R = dcol + ncol;
        // stand-alone kernel: a sub-slot takes whole groups of 8 lanes (see eval_fast_kernel), every group reads one
        // contiguous piece of one row, so the row stride needs no odd padding there
        const int RS = alone ? R : (R | 1);
        const int Rt = alone ? ((R + 7) & ~7) : R;
        int S = 1;
        while (S < 64 && Rt * (S * 2) <= rs_limit) S *= 2;
        const size_t tbl = (size_t)(E + 1) * RS * 16;
        const size_t offs = (size_t)2 * EF_PASSES * S * g->KP * 4;
        // exchange area of the flush tree: all planes in one round, or (stand-alone kernel) four planes per round
        // when that is what lets a larger chunk fit
        int xpl = EF_NPL;
        size_t xch = (size_t)(S / 2) * R * xpl * 16;
        if (alone && tbl + offs + xch + 128 > smem_budget) {
            xpl = 4;
            xch = (size_t)(S / 2) * R * xpl * 16;
        }
        const size_t smem = tbl + offs + xch + 128;
        if (smem > smem_budget || R > 320) return false;
        if (xpl < EF_NPL) {
            // rounds of the flush use the (idle) offsets ring as well: planes per round
            xpl = (int)((offs + xch) / ((size_t)(S / 2 > 0 ? S / 2 : 1) * R * 16));
            if (xpl >= EF_NPL) xpl = EF_NPL - 1;
        }
        if (commit) {
            g->xpl = xpl;
            g->Pc = Pc;
            g->DW = dcol * 4;
            g->NW = ncol * 4;
            g->R = R;
            g->RS = RS;
            g->W = R * 4;
            g->S = S;
            g->logS = ceil_log2(S);
            g->smem = smem;
        }
        return true;
    };
    int Pc = Pfull;
    while (!fits(Pc, false)) {
        if (Pc <= unit) return false;
        Pc -= unit;
    }
    {
        const int chunks = (Pfull + Pc - 1) / Pc;
        int eq = (((Pfull + chunks - 1) / chunks + unit - 1) / unit) * unit;
        if (eq > Pc || !fits(eq, false)) eq = Pc;
        fits(eq, true);
    }
    if (alone) {
        // The kernel is bound by the shared-memory wavefronts of its row loads -- chunks x ceil(R / 8) per (token,
        // expert) -- provided it has the warps to keep them in flight (measured on config 5: 37 chunks of R = 16 on
        // 8 warps 531 us, 29 chunks of R = 21 on 12 warps 455 us).  Among the chunk sizes that fit, keep those with
        // the most threads (at least 320 when some chunk size reaches that) and take the smallest product.
        auto probe = [&](int pc, EvalFastGeom *t) {
            *t = *g;
            EvalFastGeom *keep = g;
            g = t;
            const bool ok = fits(pc, true);
            g = keep;
            return ok;
        };
        int max_threads = 0;
        for (int pc = Pc; pc >= unit; pc -= unit) {
            EvalFastGeom t;
            if (probe(pc, &t) && ((t.R + 7) & ~7) * t.S > max_threads) max_threads = ((t.R + 7) & ~7) * t.S;
        }
        const int need_threads = max_threads < 320 ? max_threads : 320;
        long best = -1;
        int best_pc = g->Pc;
        for (int pc = Pc; pc >= unit; pc -= unit) {
            EvalFastGeom t;
            if (!probe(pc, &t) || ((t.R + 7) & ~7) * t.S < need_threads) continue;
            const long cost = (long)((Pfull + pc - 1) / pc) * ((t.R + 7) / 8);
            if (best < 0 || cost < best) {
                best = cost;
                best_pc = pc;
            }
        }
        fits(best_pc, true);
    }
    g->PC = (P + g->Pc - 1) / g->Pc;
    // enough threads to own every (sub-slot, column) pair and to prefetch a block's index entries
    // with at most EF_PRE registers each (threads beyond R * S only help with the staging)
    while (g->S > 1 && EF_PASSES * g->S * g->KP > EF_PRE * EF_MAXTHREADS) {
        g->S /= 2;
        g->logS -= 1;
    }
    const int need_pre = (EF_PASSES * g->S * g->KP + EF_PRE - 1) / EF_PRE;
    const int Rt = rs_limit == EF_RS_ALONE ? ((g->R + 7) & ~7) : g->R;
    const int need = Rt * g->S > need_pre ? Rt * g->S : need_pre;
    g->nthreads = ((need + 31) / 32) * 32;
    if (g->nthreads > EF_MAXTHREADS) return false;
    const int64_t blk = (int64_t)EF_PASSES * g->S;
    // Blocks along the token axis per (layer, chunk).  All blocks do the same work, so the kernel lasts
    // ceil(blocks / SMs) block-times of 1 / want of a unit each: pick the `want` that minimises
    // ceil(units * want / SMs) / want (ncu on config 5: 32 units x 5 = 160 blocks on 148 SMs was 1.08 waves, i.e.
    // two block-times with 12 blocks alone in the second; 32 x 9 = 288 blocks is 1.95 waves of blocks half the size),
    // among block sizes that still amortise the table copy (>= 16 scoring blocks of tokens each).
    const int64_t units = (int64_t)g->PC * L;
    int64_t want = 1;
    {
        const int64_t max_want = (T / (16 * blk)) > 1 ? (T / (16 * blk)) : 1;
        double best = 1e30;
        const int64_t cap_want = 64 > (target_ctas + units - 1) / units ? 64 : (target_ctas + units - 1) / units;
        for (int64_t wnt = 1; wnt <= cap_want && wnt <= max_want; ++wnt) {
            const int64_t waves = (units * wnt + target_ctas - 1) / target_ctas;
            const double cost = (double)waves / (double)wnt * (1.0 + 0.01 * (double)wnt);   // mild pull toward fewer blocks
            if (cost < best - 1e-12) {
                best = cost;
                want = wnt;
            }
        }
    }
    int64_t tpc = (T + want - 1) / want;
    tpc = ((tpc + blk - 1) / blk) * blk;
    g->tpc = tpc;
    g->ncta_t = (int)((T + tpc - 1) / tpc);
    if (g->ncta_t > 65535) return false;
    const int64_t cap_run = (int64_t)EF_MAXBLK * blk;
    // runs split at capacity and at source boundaries
    // source boundaries inside a block's range (an explicit token_src can put all of them into one block)
    const int64_t srcb = explicit_src ? D - 1 : ((tpc - 1) * D) / T + 1;
    g->maxrec = (int)((tpc + cap_run - 1) / cap_run + (srcb < D - 1 ? srcb : D - 1));
    if (g->maxrec < 1) g->maxrec = 1;
    g->NPR = EF_BT + g->logS;
    g->rec_slots = (size_t)L * g->PC * g->ncta_t * g->maxrec;
    g->rec_words = g->rec_slots * (size_t)EF_RECW * g->W;
    g->table_words = (size_t)L * g->PC * (E + 1) * g->RS * 4;
    return true;
}

static size_t ef_budget() { return 224 * 1024; }    // of the 227 KB a block may opt into (no static shared memory here)

size_t eval_fast_ws_bytes(int32_t L, int64_t T, int32_t k, int32_t E, int32_t D, int32_t P)
{
    size_t best = 0;
    for (int N = 2; N <= 8; N *= 2) {
        EvalFastGeom g;
        if (!eval_fast_geom(L, T, k, E, D, N, P, sm_count(), ef_budget(), &g, false, EF_RS_ALONE)) continue;
        const size_t b = g.rec_slots * 4 + 256 + g.rec_words * 4 + 256 + g.table_words * 4 + 256;
        if (b > best) best = b;
    }
    for (int N = 2; N <= 8; N *= 2) {      // explicit token_src: more record slots, the permutation and the sort
        EvalFastGeom g;
        if (!eval_fast_geom(L, T, k, E, D, N, P, sm_count(), ef_budget(), &g, true, EF_RS_ALONE)) continue;
        const size_t b = g.rec_slots * 4 + 256 + g.rec_words * 4 + 256 + g.table_words * 4 + 256 + (size_t)L * T * 4 + 256 +
                         (size_t)L * (D + 1) * 8 + 256 + (size_t)L * 64 * 4 + 256 + dispatch_ws_bytes_batched(L, T, 1, D) + 256;
        if (b > best) best = b;
    }
    const size_t fb = fused_ws_bytes(L, T, k, E, D, P);
    if (fb > best) best = fb;
    const size_t f2 = fused2_ws_bytes(L, T, k, E, D, P) + 256;
    return f2 > best ? f2 : best;
}

// start of the region behind the generic accumulators that the fast paths carve (one of them runs per call)
void *eval_fast_region(void *ws, int32_t L, int32_t E, int32_t D, int32_t P)
{
    EvalWs base = eval_ws_carve(ws, L, E, D, P);
    uintptr_t a = reinterpret_cast<uintptr_t>(base.ldirect + (size_t)L * 64);
    return reinterpret_cast<void *>((a + 255) & ~(uintptr_t)255);
}

EvalFastWs eval_fast_ws_carve(void *ws, int32_t L, int32_t E, int32_t D, int32_t P,
                              const EvalFastGeom &g, int64_t T)
{
    // the fast-path region follows the generic region (acc, recv, mcounts)
    EvalWs base = eval_ws_carve(ws, L, E, D, P);
    uintptr_t a = reinterpret_cast<uintptr_t>(base.ldirect + (size_t)L * 64);
    a = (a + 255) & ~(uintptr_t)255;
    EvalFastWs w;
    w.rec_src = reinterpret_cast<int32_t *>(a);
    a += g.rec_slots * 4;
    a = (a + 255) & ~(uintptr_t)255;
    w.rec_planes = reinterpret_cast<uint32_t *>(a);
    a += g.rec_words * 4;
    a = (a + 255) & ~(uintptr_t)255;
    w.table = reinterpret_cast<uint32_t *>(a);
    a += g.table_words * 4;
    a = (a + 255) & ~(uintptr_t)255;
    w.perm = reinterpret_cast<int32_t *>(a);
    a += (size_t)L * T * 4;
    a = (a + 255) & ~(uintptr_t)255;
    w.srcoff = reinterpret_cast<long long *>(a);
    a += (size_t)L * (D + 1) * 8;
    a = (a + 255) & ~(uintptr_t)255;
    w.ident = reinterpret_cast<int32_t *>(a);
    a += (size_t)L * 64 * 4;
    a = (a + 255) & ~(uintptr_t)255;
    w.sort_ws = reinterpret_cast<void *>(a);
    return w;
}

// identity maps [L][64] for the sort of the tokens by source device (entries >= D are never a valid key)
__global__ void eval_iota_kernel(int32_t *p)
{
    pdl_launch_dependents();
    pdl_wait();
    if (threadIdx.x < 64) p[blockIdx.x * 64 + threadIdx.x] = (int)threadIdx.x;
}

// ---- main kernel ---------------------------------------------------------------------------------------
struct EvalFastParams {
    const int32_t *idx;          // [L][T][k]
    const uint8_t *kept;         // [L][T][k] or NULL
    const int32_t *expert_dev;   // [L][P][E]
    const int32_t *dev_node;     // [D]
    int32_t *rec_src;
    uint32_t *rec_planes;
    const uint32_t *table;       // [L][PC][E + 1][RS * 4]
    // explicit token sources (reading R5): token ids grouped by source device by a stable counting sort, and the
    // start of every source's range in that order; NULL = contiguous blocks floor(t D / T), no indirection
    const int32_t *perm;         // [L][T]
    const long long *srcoff;     // [L][D + 1]
    int64_t T, tpc;
    int32_t k, E, P, D;
    int32_t WD, WN, Pc, PC, DW, NW, R, RS, S, logS, ncta_t, maxrec, NPR, XPL;
    // optional fills done by the table kernel (saves separate memset nodes): 32-bit words
    uint32_t *fill_ptr[4];
    unsigned long long fill_words[4];
    uint32_t fill_val[4];
};

// one thread per table word; grid (words of a table / 256, PC, L)
__global__ void __launch_bounds__(256) eval_table_kernel(EvalFastParams q)
{
    const int layer = blockIdx.z, pc = blockIdx.y;
    const int rowq = q.RS * 4;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    __shared__ unsigned char s_node[64];
    pdl_launch_dependents();
    pdl_wait();
    if (threadIdx.x < 64) s_node[threadIdx.x] = (int)threadIdx.x < q.D ? (unsigned char)q.dev_node[threadIdx.x] : 0;
    __syncthreads();
    {
        const unsigned long long nthr = (unsigned long long)gridDim.x * gridDim.y * gridDim.z * blockDim.x;
        const unsigned long long me = ((unsigned long long)(blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x) *
                                          blockDim.x + threadIdx.x;
#pragma unroll
        for (int j = 0; j < 4; ++j)
            for (unsigned long long x = me; x < q.fill_words[j]; x += nthr) q.fill_ptr[j][x] = q.fill_val[j];
    }
    if (i >= (q.E + 1) * rowq) return;
    const int e = i / rowq, w = i - e * rowq;
    uint32_t *t = const_cast<uint32_t *>(q.table) + ((size_t)layer * q.PC + pc) * (size_t)(q.E + 1) * rowq;
    t[i] = ef_table_word(q.expert_dev + ((size_t)layer * q.P) * q.E, s_node, q.E, q.P, q.D, pc * q.Pc,
                         q.WD, q.WN, q.DW, q.NW, e, w);
}

// KU <= KP: slots that can hold an expert (k rounded up to even); the offsets of slots KU.. point at the zero
// row and are not loaded (k = 10 in a KP = 12 kernel: 10 row loads per token instead of 12)
template <int KP, int KU>
__device__ __forceinline__ uint4 ef_token_mask(const unsigned char *tblc, const uint16_t *op)
{
    // the token's row offsets are 16-bit, in 16-byte units (a table has at most 14 336 of them): 8 / 16 / 24 / 32
    // bytes per token instead of twice that -- the offset loads were 12 % of the kernel's shared-memory wavefronts
    uint4 m = make_uint4(0u, 0u, 0u, 0u);
    const uint4 z = make_uint4(0u, 0u, 0u, 0u);
    uint32_t pk[KP / 2];
    if (KP % 8 == 0) {
#pragma unroll
        for (int q = 0; q < KP / 8; ++q) {
            const uint4 o = *reinterpret_cast<const uint4 *>(op + 8 * q);
            pk[4 * q] = o.x; pk[4 * q + 1] = o.y; pk[4 * q + 2] = o.z; pk[4 * q + 3] = o.w;
        }
    } else {
#pragma unroll
        for (int q = 0; q < KP / 4; ++q) {
            if (4 * q >= KU) { pk[2 * q] = pk[2 * q + 1] = 0u; continue; }
            const uint2 o = *reinterpret_cast<const uint2 *>(op + 4 * q);
            pk[2 * q] = o.x; pk[2 * q + 1] = o.y;
        }
    }
#pragma unroll
    for (int q = 0; q < KP / 4; ++q) {
        if (4 * q >= KU) break;
        const uint32_t o0 = (pk[2 * q] & 0xffffu) << 4, o1 = (pk[2 * q] >> 16) << 4;
        const uint32_t o2 = (pk[2 * q + 1] & 0xffffu) << 4, o3 = (pk[2 * q + 1] >> 16) << 4;
        const uint4 v0 = *reinterpret_cast<const uint4 *>(tblc + o0);
        const uint4 v1 = 4 * q + 1 < KU ? *reinterpret_cast<const uint4 *>(tblc + o1) : z;
        const uint4 v2 = 4 * q + 2 < KU ? *reinterpret_cast<const uint4 *>(tblc + o2) : z;
        const uint4 v3 = 4 * q + 3 < KU ? *reinterpret_cast<const uint4 *>(tblc + o3) : z;
        m.x = lop_or3(lop_or3(m.x, v0.x, v1.x), v2.x, v3.x);
        m.y = lop_or3(lop_or3(m.y, v0.y, v1.y), v2.y, v3.y);
        m.z = lop_or3(lop_or3(m.z, v0.z, v1.z), v2.z, v3.z);
        m.w = lop_or3(lop_or3(m.w, v0.w, v1.w), v2.w, v3.w);
    }
    return m;
}

// One block of EF_PASSES tokens per thread: Harley-Seal carry-save tree into planes 0..2, the
// "eights" carry rippled into planes 3..EF_BT-1.
#define CAP_EF_WORD(F)                                                                            \
    do {                                                                                          \
        uint32_t tA, tB, fA, fB, e8, s;                                                           \
        CAP_CSA(s, tA, pl[0].F, x[0].F, x[1].F);                                                  \
        CAP_CSA(s, tB, s, x[2].F, x[3].F);                                                        \
        CAP_CSA(pl[1].F, fA, pl[1].F, tA, tB);                                                    \
        CAP_CSA(s, tA, s, x[4].F, x[5].F);                                                        \
        CAP_CSA(s, tB, s, x[6].F, x[7].F);                                                        \
        pl[0].F = s;                                                                              \
        CAP_CSA(pl[1].F, fB, pl[1].F, tA, tB);                                                    \
        CAP_CSA(pl[2].F, e8, pl[2].F, fA, fB);                                                    \
        _Pragma("unroll") for (int p = 3; p < EF_BT; ++p) {                                       \
            const uint32_t c = pl[p].F & e8;                                                      \
            pl[p].F ^= e8;                                                                        \
            e8 = c;                                                                               \
        }                                                                                         \
    } while (0)

template <int KP, int KU>
__global__ void __launch_bounds__(EF_MAXTHREADS) eval_fast_kernel(EvalFastParams q)
{
    extern __shared__ __align__(16) unsigned char ef_sm[];
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int layer = blockIdx.z, pc = blockIdx.y;
    const int E = q.E, D = q.D, k = q.k, S = q.S, R = q.R;
    const int rowb = q.RS * 16;
    unsigned char *tbl = ef_sm;
    uint32_t *offs_region = reinterpret_cast<uint32_t *>(tbl + (size_t)(E + 1) * rowb);
    uint16_t *offs = reinterpret_cast<uint16_t *>(offs_region);       // 16-bit row offsets in 16-byte units (half the region)
    uint4 *xch = reinterpret_cast<uint4 *>(offs_region + 2 * EF_PASSES * S * KP);

    ef_copy_table(tbl, q.table + ((size_t)layer * q.PC + pc) * (size_t)(E + 1) * q.RS * 4, (E + 1) * q.RS,
                  tid, nthr);

    // (sub-slot, column) of a thread: a sub-slot takes ceil(R / 8) whole groups of 8 lanes.  A 128-bit shared-memory
    // load is served 8 lanes at a time; with R consecutive threads per sub-slot (R = 21 on config 5, 36 on config 4)
    // nearly every group of 8 held the tail of one table row and the head of another, i.e. two 16-byte-aligned
    // pieces whose banks overlap: ncu counted 4.95 wavefronts per row load against 3.82 ideal.  Whole groups read
    // one contiguous piece of one row: never a conflict, at the price of (8 - R % 8) % 8 idle lanes per sub-slot.
    const int Rq = (R + 7) & ~7;
    const int sub_t = tid / Rq, col_t = tid - sub_t * Rq;
    const bool active = sub_t < S && col_t < R;
    const int sub = active ? sub_t : 0;
    const int col = active ? col_t : 0;
    const unsigned char *tblc = tbl + col * 16;
    const int32_t *idx = q.idx + (size_t)layer * q.T * k;
    const uint8_t *kept = q.kept ? q.kept + (size_t)layer * q.T * k : nullptr;
    const uint32_t rowu = (uint32_t)q.RS;            // row stride in 16-byte units
    const uint32_t zero_row = (uint32_t)E * rowu;
    const int nent = EF_PASSES * S * KP;          // index entries per block of tokens
    const int64_t T = q.T;
    __shared__ long long s_srcoff[65];
    const int32_t *perm = q.perm ? q.perm + (size_t)layer * q.T : nullptr;
    if (perm) {
        if (tid <= D) s_srcoff[tid] = q.srcoff[(size_t)layer * (D + 1) + tid];
        __syncthreads();
    }
    const int64_t Tend = perm ? min(T, (int64_t)s_srcoff[D]) : T;     // tokens with an out-of-range source are left out
    const int64_t t0 = (int64_t)blockIdx.x * q.tpc;
    const int64_t t1 = min(Tend, t0 + q.tpc);
    const size_t slot0 = (((size_t)layer * q.PC + pc) * q.ncta_t + blockIdx.x) * q.maxrec;
    const int blk_tokens = EF_PASSES * S;

    int nrec = 0;
    int psrc = 0;                                   // sources only grow along the sorted order
    int64_t t = t0;
    while (t < t1) {
        // ---- one run: tokens [t, rend) share the source device and fit the thread counters ----
        int src;
        int64_t bnd;
        if (perm) {
            while (psrc < D - 1 && (int64_t)s_srcoff[psrc + 1] <= t) ++psrc;
            src = psrc;
            bnd = (int64_t)s_srcoff[src + 1];
        } else {
            src = (int)((t * D) / T);
            bnd = ((int64_t)(src + 1) * T + D - 1) / D;
        }
        int64_t rend = min(t1, bnd);
        rend = min(rend, t + (int64_t)EF_MAXBLK * blk_tokens);
        uint4 pl[EF_NPL];
#pragma unroll
        for (int p = 0; p < EF_NPL; ++p) pl[p] = make_uint4(0u, 0u, 0u, 0u);

        // prefetch registers: entry i of a block = (slot = i / KP, s = i % KP); token = base + slot
        uint32_t pre[EF_PRE];
        auto fetch = [&](int64_t base) {
#pragma unroll
            for (int j = 0; j < EF_PRE; ++j) {
                const int i = tid + j * nthr;
                uint32_t o = zero_row;
                if (i < nent) {
                    const int slot = i / KP, s = i - slot * KP;
                    const int64_t tok = base + slot;
                    if (tok < rend && s < k) {
                        const int64_t a = (perm ? (int64_t)perm[tok] : tok) * k + s;
                        const int e = idx[a];
                        if ((!kept || kept[a]) && (unsigned)e < (unsigned)E) o = (uint32_t)e * rowu;
                    }
                }
                pre[j] = o;
            }
        };
        auto stash = [&](int buf) {
#pragma unroll
            for (int j = 0; j < EF_PRE; ++j) {
                const int i = tid + j * nthr;
                if (i < nent) offs[buf * nent + i] = (uint16_t)pre[j];
            }
        };
        __syncthreads();     // the previous run's readers of offs are done
        fetch(t);
        stash(0);
        __syncthreads();
        int buf = 0;
        for (int64_t b = t; b < rend; b += blk_tokens) {
            const bool more = b + blk_tokens < rend;
            if (more) fetch(b + blk_tokens);
            if (active) {
                uint4 x[EF_PASSES];
                const uint16_t *ob = offs + buf * nent + sub * KP;
#pragma unroll
                for (int ps = 0; ps < EF_PASSES; ++ps) x[ps] = ef_token_mask<KP, KU>(tblc, ob + ps * S * KP);
                CAP_EF_WORD(x);
                CAP_EF_WORD(y);
                CAP_EF_WORD(z);
                CAP_EF_WORD(w);
            }
            if (more) stash(buf ^ 1);
            __syncthreads();
            buf ^= 1;
        }
        // ---- flush: add the S sub-slots in the bit-sliced domain, write the record ----
        if (q.XPL >= EF_NPL) {
            // the exchange area holds every plane of half the sub-slots: one round per level
            for (int lvl = 0; lvl < q.logS; ++lvl) {
                const int half = S >> (lvl + 1);
                const int stride = half * R;
                if (active && sub >= half && sub < 2 * half) {
#pragma unroll
                    for (int p = 0; p < EF_NPL; ++p) xch[(size_t)p * stride + (sub - half) * R + col] = pl[p];
                }
                __syncthreads();
                if (active && sub < half) {
                    const uint4 *b = xch + sub * R + col;
                    uint4 carry = make_uint4(0u, 0u, 0u, 0u);
#pragma unroll
                    for (int p = 0; p < EF_NPL; ++p) {
                        const uint4 x = b[(size_t)p * stride];
                        uint4 s_, c_;
                        CAP_CSA(s_.x, c_.x, pl[p].x, x.x, carry.x);
                        CAP_CSA(s_.y, c_.y, pl[p].y, x.y, carry.y);
                        CAP_CSA(s_.z, c_.z, pl[p].z, x.z, carry.z);
                        CAP_CSA(s_.w, c_.w, pl[p].w, x.w, carry.w);
                        pl[p] = s_;
                        carry = c_;
                    }
                }
                __syncthreads();
            }
        } else {
            // A small exchange area (the price of a larger candidate chunk): q.XPL planes per round, and only the
            // planes that can be non-zero (counts < 2^np before level lvl).  The offsets ring in front of the area is
            // idle during a flush (every thread has passed the barrier that ends the run's last block) and is
            // used as exchange space too.
            uint4 *xf = reinterpret_cast<uint4 *>(offs_region);
            for (int lvl = 0; lvl < q.logS; ++lvl) {
                const int half = S >> (lvl + 1);
                const int stride = half * R;
                const int np = EF_BT + lvl;
                const bool wr = active && sub >= half && sub < 2 * half, rd = active && sub < half;
                uint4 carry = make_uint4(0u, 0u, 0u, 0u);
                for (int p0 = 0; p0 < np; p0 += q.XPL) {
                    if (wr) {
#pragma unroll
                        for (int p = 0; p < EF_NPL; ++p)
                            if (p >= p0 && p < p0 + q.XPL && p < np)
                                xf[(size_t)(p - p0) * stride + (sub - half) * R + col] = pl[p];
                    }
                    __syncthreads();
                    if (rd) {
                        const uint4 *b = xf + sub * R + col;
#pragma unroll
                        for (int p = 0; p < EF_NPL; ++p) {
                            if (p >= p0 && p < p0 + q.XPL && p < np) {
                                const uint4 x = b[(size_t)(p - p0) * stride];
                                uint4 s_, c_;
                                CAP_CSA(s_.x, c_.x, pl[p].x, x.x, carry.x);
                                CAP_CSA(s_.y, c_.y, pl[p].y, x.y, carry.y);
                                CAP_CSA(s_.z, c_.z, pl[p].z, x.z, carry.z);
                                CAP_CSA(s_.w, c_.w, pl[p].w, x.w, carry.w);
                                pl[p] = s_;
                                carry = c_;
                            }
                        }
                    }
                    __syncthreads();
                }
                if (rd) {
#pragma unroll
                    for (int p = EF_BT; p < EF_NPL; ++p)
                        if (p == np) pl[p] = carry;      // plane np was zero on both sides
                }
            }
        }
        if (active && sub == 0) {
            uint32_t *rp = q.rec_planes + ((slot0 + nrec) * (size_t)(R * 4) + (size_t)col * 4) * EF_RECW;
            uint32_t v[EF_RECW];
#pragma unroll
            for (int p = 0; p < EF_RECW; ++p) v[p] = (p < EF_NPL && p < q.NPR) ? pl[p < EF_NPL ? p : 0].x : 0u;
            ef_store_word_planes(rp, v);
#pragma unroll
            for (int p = 0; p < EF_RECW; ++p) v[p] = (p < EF_NPL && p < q.NPR) ? pl[p < EF_NPL ? p : 0].y : 0u;
            ef_store_word_planes(rp + EF_RECW, v);
#pragma unroll
            for (int p = 0; p < EF_RECW; ++p) v[p] = (p < EF_NPL && p < q.NPR) ? pl[p < EF_NPL ? p : 0].z : 0u;
            ef_store_word_planes(rp + 2 * EF_RECW, v);
#pragma unroll
            for (int p = 0; p < EF_RECW; ++p) v[p] = (p < EF_NPL && p < q.NPR) ? pl[p < EF_NPL ? p : 0].w : 0u;
            ef_store_word_planes(rp + 3 * EF_RECW, v);
        }
        if (tid == 0) q.rec_src[slot0 + nrec] = src;
        ++nrec;
        t = rend;
    }
}

// ---- decode + finalize: add all records of one record word in the bit-sliced domain, extract the integers
// once and turn them straight into the caller's outputs (Eq. 3 costs, Eq. 4 imbalance).  A block
// owns one record word, i.e. a few whole candidates: a device word carries the received tokens per device and the
// local / same-node sums of its candidates (both 32-bit halves of a 64-bit field are done by the block of the even
// word), a node word the node sums -- no accumulator array, no atomics, no separate finalize launch.  load_pairs is
// gathered from counts x map at the start of the block, while the record loads are in flight.
struct DecodeParams {
    const int32_t *rec_src;
    const uint32_t *rec_planes;
    const int32_t *dev_node;
    const int32_t *expert_dev;  // [L][P][E]
    const long long *counts;    // [L][E]
    cap_eval_out out;
    long long bytes_per_token;
    int32_t P, D, N, E, WD, WN, Pc, PC, DW, W, NPR, nslots, na;
    int32_t cost_local, cost_intra, cost_inter;
};

#define CAP_DEC_ADD(ACC, MASK)                                        \
    do {                                                              \
        uint32_t cy = 0u;                                             \
        _Pragma("unroll") for (int p = 0; p < NA; ++p) {              \
            if (p < NA) {                                           \
                const uint32_t xx = p < EF_NPL ? (a[p < EF_NPL ? p : 0] & (MASK)) : 0u; \
                const uint32_t s = lop_xor3(ACC[p], xx, cy);          \
                cy = lop_maj(ACC[p], xx, cy);                         \
                ACC[p] = s;                                           \
            }                                                         \
        }                                                             \
    } while (0)

#define CAP_DEC_ADD32(ACC)                                            \
    do {                                                              \
        uint32_t cy = 0u;                                             \
        _Pragma("unroll") for (int p = 0; p < NA; ++p) {              \
            if (p < NA) {                                           \
                const uint32_t s = lop_xor3(ACC[p], a[p], cy);        \
                cy = lop_maj(ACC[p], a[p], cy);                       \
                ACC[p] = s;                                           \
            }                                                         \
        }                                                             \
    } while (0)

#define CAP_DEC_BFLY(ACC, OFF)                                        \
    do {                                                              \
        uint32_t cy = 0u;                                             \
        _Pragma("unroll") for (int p = 0; p < NA; ++p) {              \
            if (p < NA) {                                           \
                const uint32_t xx = __shfl_xor_sync(0xffffffffu, ACC[p], OFF); \
                const uint32_t s = lop_xor3(ACC[p], xx, cy);          \
                cy = lop_maj(ACC[p], xx, cy);                         \
                ACC[p] = s;                                           \
            }                                                         \
        }                                                             \
    } while (0)

constexpr int DEC_WARPS = 4;
// WPW = warps per table word.  4: one word per block, the four warps split its records and exchange their sums
// through shared memory (config 3: ~290 records per word).  1: every warp decodes a word of its own -- no block
// barrier after the prologue, four words per block (configs 2, 4, 5: 40-90 records per word, where the fixed
// part of a block, not the records, was the cost: 130 us on config 4, 60 us on config 5 with one word per block).
template <int NA, int WPW>
__global__ void __launch_bounds__(32 * DEC_WARPS) eval_decode_kernel(DecodeParams q)
{
    constexpr int NG = DEC_WARPS / WPW;                  // words per block
    __shared__ unsigned long long nodeset[8];
    __shared__ unsigned char s_dn[64];
    __shared__ uint32_t s_part[WPW > 1 ? WPW - 1 : 1][3][NA];
    __shared__ unsigned long long s_lp[NG][4][64];      // load_pairs of a word's candidates (<= 4 per device word)
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int grp = warp / WPW, wl = warp % WPW, gt = wl * 32 + lane;
    const int w0 = blockIdx.x * NG + grp, pc = blockIdx.y, layer = blockIdx.z;
    const bool devword = w0 < q.DW;
    const int fw = devword ? q.WD : q.WN;                 // field width of this word
    const int nwords = (devword && q.WD == 64) ? 2 : 1;   // both halves of a 64-bit device field
    pdl_launch_dependents();
    pdl_wait();
    if (threadIdx.x < 64) s_dn[threadIdx.x] = (int)threadIdx.x < q.D ? (unsigned char)q.dev_node[threadIdx.x] : 0;
    for (int i = threadIdx.x; i < NG * 4 * 64; i += blockDim.x) (&s_lp[0][0][0])[i] = 0ull;
    __syncthreads();
    if (threadIdx.x < 8) {
        const int n = threadIdx.x;              // from the shared copy: one round of global loads, not D
        unsigned long long m = 0ull;
        for (int d = 0; d < q.D; ++d)
            if (s_dn[d] == n) m |= 1ull << d;
        nodeset[n] = m;
    }
    // words past the table, and the odd half of a 64-bit device field (done with the even word): nothing to do.
    // WPW = 4: uniform over the block.  WPW = 1: per warp -- no block barrier may follow the next one.
    const bool idle = w0 >= q.W || (devword && q.WD == 64 && (w0 & 1));
    if (WPW > 1 && idle) return;
    // candidates of this word: device word -> 32 / WD of them (one for WD >= 32); their load_pairs
    const int ncand = devword ? (q.WD >= 32 ? 1 : 32 / q.WD) : 0;
    const int pl0 = devword ? (q.WD == 64 ? (w0 >> 1) : w0 * 32 / q.WD) : 0;
    if (!idle && devword && (q.out.load_pairs || q.out.imbalance)) {
        const long long *cnt = q.counts + (size_t)layer * q.E;
        for (int c = 0; c < ncand; ++c) {
            const int p = pc * q.Pc + pl0 + c;
            if (pl0 + c >= q.Pc || p >= q.P) continue;
            const int32_t *pi = q.expert_dev + ((size_t)layer * q.P + p) * q.E;
            for (int e = gt; e < q.E; e += 32 * WPW) {
                const int d = pi[e];
                const long long v = __ldcg(cnt + e);
                if ((unsigned)d < (unsigned)q.D && v) atomicAdd(&s_lp[grp][c][d], (unsigned long long)v);
            }
        }
    }
    __syncthreads();                                      // the last block barrier of the WPW = 1 variant
    if (idle) return;
    // running per-candidate results over the words of this block (meaningful on the field's leader lane)
    unsigned long long a_gt = 0ull, a_gl = 0ull, a_gs = 0ull;
    long long mx = 0, sm = 0, mxr = 0, smr = 0;
    const size_t sbase = ((size_t)layer * q.PC + pc) * q.nslots;
    for (int wi = 0; wi < nwords; ++wi) {
        const int w = w0 + wi;
        uint32_t tot[NA], loc[NA], sam[NA];
#pragma unroll
        for (int p = 0; p < NA; ++p) tot[p] = loc[p] = sam[p] = 0u;
        constexpr int DEC_SL = 2;     // record slots a thread has in flight
        for (int s0 = gt; s0 < q.nslots; s0 += 32 * WPW * DEC_SL) {
            int srcs[DEC_SL];
#pragma unroll
            for (int j = 0; j < DEC_SL; ++j) {
                const int s = s0 + j * 32 * WPW;
                srcs[j] = s < q.nslots ? q.rec_src[sbase + s] : -1;
            }
            uint32_t av[DEC_SL][EF_NPL];
#pragma unroll
            for (int j = 0; j < DEC_SL; ++j) {
                const int s = s0 + j * 32 * WPW;
                // one 64-byte run per (slot, word); not conditional on srcs[j]: the loads go out together with the
                // header loads (unused slots hold stale planes, skipped below)
                const uint4 *pp = reinterpret_cast<const uint4 *>(q.rec_planes + ((sbase + s) * (size_t)q.W + w) * EF_RECW);
                uint32_t t16[EF_RECW];
#pragma unroll
                for (int i = 0; i < EF_RECW / 4; ++i) {
                    const uint4 x = s < q.nslots ? pp[i] : make_uint4(0u, 0u, 0u, 0u);
                    t16[4 * i] = x.x;
                    t16[4 * i + 1] = x.y;
                    t16[4 * i + 2] = x.z;
                    t16[4 * i + 3] = x.w;
                }
#pragma unroll
                for (int p = 0; p < EF_NPL; ++p) av[j][p] = t16[p];
            }
#pragma unroll
            for (int j = 0; j < DEC_SL; ++j) {
                if (srcs[j] < 0) continue;
                const int src = srcs[j] & 63;
                const int node = s_dn[src] & 7;
                uint32_t mloc, msam;
                if (devword) {
                    mloc = ef_devmask_word(q.WD, w, 1ull << src);
                    msam = ef_devmask_word(q.WD, w, nodeset[node]);
                } else {
                    mloc = ef_nodemask_word(q.WN, node);
                    msam = 0u;
                }
                const uint32_t(&a)[EF_NPL] = av[j];
                CAP_DEC_ADD(tot, 0xffffffffu);
                CAP_DEC_ADD(loc, mloc);
                CAP_DEC_ADD(sam, msam);
            }
        }
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) {
            CAP_DEC_BFLY(tot, off);
            CAP_DEC_BFLY(loc, off);
            CAP_DEC_BFLY(sam, off);
        }
        // every lane of a warp now holds the warp's sums; with several warps per word, warps 1.. hand theirs to warp 0
        if (WPW > 1) {
            __syncthreads();                 // s_part of the previous word has been read
            if (wl > 0 && lane < 3) {
#pragma unroll
                for (int p = 0; p < NA; ++p) {
                    const uint32_t v = lane == 0 ? tot[p] : lane == 1 ? loc[p] : sam[p];
                    s_part[wl - 1][lane][p] = v;
                }
            }
            __syncthreads();
        }
        if (wl == 0) {
            for (int o = 0; o < WPW - 1; ++o) {
                uint32_t a[NA];
#pragma unroll
                for (int p = 0; p < NA; ++p) a[p] = s_part[o][0][p];
                CAP_DEC_ADD32(tot);
#pragma unroll
                for (int p = 0; p < NA; ++p) a[p] = s_part[o][1][p];
                CAP_DEC_ADD32(loc);
#pragma unroll
                for (int p = 0; p < NA; ++p) a[p] = s_part[o][2][p];
                CAP_DEC_ADD32(sam);
            }
            unsigned long long vt = 0ull, vl = 0ull, vs = 0ull;
#pragma unroll
            for (int p = 0; p < NA; ++p) {
                vt |= (unsigned long long)((tot[p] >> lane) & 1u) << p;
                vl |= (unsigned long long)((loc[p] >> lane) & 1u) << p;
                vs |= (unsigned long long)((sam[p] >> lane) & 1u) << p;
            }
            // lane = bit position of the word = (candidate, device or node) of this chunk
            const int bitpos = (devword ? w : w - q.DW) * 32 + lane;
            const int pl = bitpos / fw, f = bitpos - pl * fw;
            const int p = pc * q.Pc + pl;
            const bool pvalid = pl < q.Pc && p < q.P;
            const size_t o = (size_t)layer * q.P + p;
            const int gw = fw < 32 ? fw : 32;
            unsigned long long gt2 = vt, gl = vl, gs = vs;
            long long l = 0, r = 0;
            if (devword) {
                const int c = pl - pl0;
                if (pvalid && f < q.D) {
                    l = (long long)s_lp[grp][c & 3][f];
                    r = (long long)vt;
                    if (q.out.load_pairs) q.out.load_pairs[o * q.D + f] = l;
                    if (q.out.recv_tokens) q.out.recv_tokens[o * q.D + f] = r;
                }
            }
            long long wmx = l, wsm = l, wmxr = r, wsmr = r;
            for (int off = 1; off < gw; off <<= 1) {
                gt2 += __shfl_xor_sync(0xffffffffu, gt2, off);
                gl += __shfl_xor_sync(0xffffffffu, gl, off);
                gs += __shfl_xor_sync(0xffffffffu, gs, off);
                wmx = max(wmx, __shfl_xor_sync(0xffffffffu, wmx, off));
                wmxr = max(wmxr, __shfl_xor_sync(0xffffffffu, wmxr, off));
                wsm += __shfl_xor_sync(0xffffffffu, wsm, off);
                wsmr += __shfl_xor_sync(0xffffffffu, wsmr, off);
            }
            a_gt += gt2;
            a_gl += gl;
            a_gs += gs;
            mx = max(mx, wmx);
            mxr = max(mxr, wmxr);
            sm += wsm;
            smr += wsmr;
            if (wi == nwords - 1 && (lane & (gw - 1)) == 0 && pvalid) {
                if (devword) {
                    const long long dv = (long long)a_gt, lc = (long long)a_gl, same = (long long)a_gs;
                    const long long rdev = dv - lc, intra = same - lc, inter = dv - same;
                    if (q.out.dev_visits) q.out.dev_visits[o] = dv;
                    if (q.out.remote_dev) q.out.remote_dev[o] = rdev;
                    if (q.out.remote_intra) q.out.remote_intra[o] = intra;
                    if (q.out.remote_inter) q.out.remote_inter[o] = inter;
                    if (q.out.cost)
                        q.out.cost[o] = (long long)q.cost_local * lc + (long long)q.cost_intra * intra +
                                        (long long)q.cost_inter * inter;
                    if (q.out.bytes) q.out.bytes[o] = rdev * q.bytes_per_token;
                    if (q.out.imbalance) q.out.imbalance[o] = sm ? __ddiv_rn((double)(mx * q.D), (double)sm) : 0.0;
                    if (q.out.imbalance_recv)
                        q.out.imbalance_recv[o] = smr ? __ddiv_rn((double)(mxr * q.D), (double)smr) : 0.0;
                } else {
                    if (q.out.node_visits) q.out.node_visits[o] = (long long)a_gt;
                    if (q.out.remote_node) q.out.remote_node[o] = (long long)(a_gt - a_gl);
                }
            }
        }
    }
}

// ---- launcher ------------------------------------------------------------------------------------------
template <int KP, int KU>
static int launch_kp(const EvalFastParams &prm, const EvalFastGeom &g, int L, cudaStream_t st)
{
    // per device and cheap: set on every launch, to what this launch needs (the kernel also has 520 B of static
    // shared memory, so the full 227 KB would not be a legal dynamic size)
    if (cudaFuncSetAttribute(eval_fast_kernel<KP, KU>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)g.smem) != cudaSuccess)
        return check_launch("eval_fast_kernel attribute");
    dim3 grid((unsigned)g.ncta_t, (unsigned)g.PC, (unsigned)L);
    {
        KernelTimerScope ts("eval", st);
        eval_fast_kernel<KP, KU><<<grid, g.nthreads, g.smem, st>>>(prm);
    }
    note_launch();
    return check_launch("eval_fast_kernel");
}

// builds the one-hot code tables of all layers and candidate chunks (g.table_words words at fw.table)
int ef_launch_table(const EvalFastGeom &g, const EvalFastWs &fw, const int32_t *expert_dev, const int32_t *dev_node,
                    int32_t L, int32_t E, int32_t P, int32_t D, cudaStream_t st, const EfFill *fills, int nfill)
{
    EvalFastParams prm = {};
    for (int j = 0; j < 4; ++j) {
        prm.fill_ptr[j] = j < nfill ? reinterpret_cast<uint32_t *>(fills[j].ptr) : nullptr;
        prm.fill_words[j] = j < nfill ? fills[j].bytes / 4 : 0;
        prm.fill_val[j] = j < nfill ? fills[j].value : 0u;
    }
    prm.expert_dev = expert_dev;
    prm.dev_node = dev_node;
    prm.table = fw.table;
    prm.E = E;
    prm.P = P;
    prm.D = D;
    prm.WD = g.WD;
    prm.WN = g.WN;
    prm.Pc = g.Pc;
    prm.PC = g.PC;
    prm.DW = g.DW;
    prm.NW = g.NW;
    prm.RS = g.RS;
    const int nw = (E + 1) * g.RS * 4;
    {
        KernelTimerScope ts("eval_table", st);
        launch_pdl(eval_table_kernel, dim3((unsigned)((nw + 255) / 256), (unsigned)g.PC, (unsigned)L), dim3(256), 0, st, prm);
    }
    note_launch();
    return check_launch("eval_table_kernel");
}

static int decode_launch(const DecodeParams &dq, dim3 dgrid, cudaStream_t st)
{
    const int na = dq.na;
    {
        KernelTimerScope ts("eval_decode", st);
        if (dq.nslots <= 128) {
            // few records per word: a warp per word, four words per block
            const dim3 g1((dgrid.x + DEC_WARPS - 1) / DEC_WARPS, dgrid.y, dgrid.z);
            if (na <= 12) launch_pdl(eval_decode_kernel<12, 1>, g1, dim3(32 * DEC_WARPS), 0, st, dq);
            else if (na <= 16) launch_pdl(eval_decode_kernel<16, 1>, g1, dim3(32 * DEC_WARPS), 0, st, dq);
            else if (na <= 20) launch_pdl(eval_decode_kernel<20, 1>, g1, dim3(32 * DEC_WARPS), 0, st, dq);
            else if (na <= 24) launch_pdl(eval_decode_kernel<24, 1>, g1, dim3(32 * DEC_WARPS), 0, st, dq);
            else if (na <= 28) launch_pdl(eval_decode_kernel<28, 1>, g1, dim3(32 * DEC_WARPS), 0, st, dq);
            else launch_pdl(eval_decode_kernel<32, 1>, g1, dim3(32 * DEC_WARPS), 0, st, dq);
        } else {
            if (na <= 12) launch_pdl(eval_decode_kernel<12, DEC_WARPS>, dgrid, dim3(32 * DEC_WARPS), 0, st, dq);
            else if (na <= 16) launch_pdl(eval_decode_kernel<16, DEC_WARPS>, dgrid, dim3(32 * DEC_WARPS), 0, st, dq);
            else if (na <= 20) launch_pdl(eval_decode_kernel<20, DEC_WARPS>, dgrid, dim3(32 * DEC_WARPS), 0, st, dq);
            else if (na <= 24) launch_pdl(eval_decode_kernel<24, DEC_WARPS>, dgrid, dim3(32 * DEC_WARPS), 0, st, dq);
            else if (na <= 28) launch_pdl(eval_decode_kernel<28, DEC_WARPS>, dgrid, dim3(32 * DEC_WARPS), 0, st, dq);
            else launch_pdl(eval_decode_kernel<32, DEC_WARPS>, dgrid, dim3(32 * DEC_WARPS), 0, st, dq);
        }
    }
    note_launch();
    return check_launch("eval_decode_kernel");
}

// A decode launch parked on this host thread (cap_trace_fused_begin arms it, ef_launch_decode fills it,
// cap_trace_fused_begin takes it): plain data, copied into the caller's cap_pending.
struct ParkedDecode {
    DecodeParams dq;
    uint32_t gx, gy, gz;
};
static thread_local bool t_park_armed = false, t_park_full = false;
static thread_local ParkedDecode t_park;

// adds all records (g.ncta_t * g.maxrec slots per layer and chunk) and writes the caller's outputs (out: device
// pointers, members may be NULL; counts: [L][E] kept pairs per expert, complete before this launch)
int ef_launch_decode(const EvalFastGeom &g, const EvalFastWs &fw, int32_t L, int64_t T, int32_t E, int32_t P,
                     const cap_topology &topo, const int32_t *expert_dev, const int64_t *counts,
                     const cap_eval_out &out, cudaStream_t st)
{
    DecodeParams dq;
    dq.rec_src = fw.rec_src;
    dq.rec_planes = fw.rec_planes;
    dq.dev_node = topo.dev_node;
    dq.expert_dev = expert_dev;
    dq.counts = reinterpret_cast<const long long *>(counts);
    dq.out = out;
    dq.bytes_per_token = topo.bytes_per_token;
    dq.cost_local = topo.cost_local;
    dq.cost_intra = topo.cost_intra;
    dq.cost_inter = topo.cost_inter;
    dq.E = E;
    dq.P = P;
    dq.D = topo.D;
    dq.N = topo.N;
    dq.WD = g.WD;
    dq.WN = g.WN;
    dq.Pc = g.Pc;
    dq.PC = g.PC;
    dq.DW = g.DW;
    dq.W = g.W;
    dq.NPR = g.NPR;
    dq.nslots = g.ncta_t * g.maxrec;
    int na = 1;
    while (na < 32 && (1ll << na) <= T) ++na;
    dq.na = na;
    const dim3 dgrid((unsigned)g.W, (unsigned)g.PC, (unsigned)L);
    if (t_park_armed) {
        // cap_trace_fused_begin: the launch is handed back to the caller, who issues it with cap_trace_fused_finish
        t_park.dq = dq;
        t_park.gx = dgrid.x;
        t_park.gy = dgrid.y;
        t_park.gz = dgrid.z;
        t_park_full = true;
        return CAP_OK;
    }
    return decode_launch(dq, dgrid, st);
}

void ef_decode_park(bool on)
{
    t_park_armed = on;
    t_park_full = false;
}

bool ef_decode_take(void *blob, size_t cap)
{
    static_assert(sizeof(ParkedDecode) <= 496, "cap_pending.blob (include/cap.h) is too small for a parked decode launch");
    if (!t_park_full || cap < sizeof(ParkedDecode)) return false;
    memcpy(blob, &t_park, sizeof(ParkedDecode));
    t_park_full = false;
    return true;
}

int ef_decode_launch_parked(const void *blob, cudaStream_t st)
{
    ParkedDecode pd;
    memcpy(&pd, blob, sizeof(ParkedDecode));
    if (pd.gx == 0 || pd.gy == 0 || pd.gz == 0 || pd.gy > 65535u || pd.gz > 65535u) return CAP_EINVAL;
    return decode_launch(pd.dq, dim3(pd.gx, pd.gy, pd.gz), st);
}

int launch_eval_fast(const int32_t *idx, const uint8_t *kept, int32_t L, int64_t T, int32_t k,
                     int32_t E, const int32_t *expert_dev, int32_t P, const cap_topology &topo,
                     const int64_t *counts, const cap_eval_out &out, void *ws, cudaStream_t st, bool *used,
                     const int32_t *token_src)
{
    *used = false;
    EvalFastGeom g;
    if (!eval_fast_geom(L, T, k, E, topo.D, topo.N, P, sm_count(), ef_budget(), &g, token_src != nullptr, EF_RS_ALONE))
        return CAP_OK;
    EvalFastWs fw = eval_fast_ws_carve(ws, L, E, topo.D, P, g, T);
    if (token_src) {
        // explicit sources (reading R5): group the token ids by source device with the stable counting sort of S5
        // (pairs = tokens, k = 1, "expert" = the source, identity map); runs of one source follow from its offsets
        launch_pdl(eval_iota_kernel, dim3((unsigned)L), dim3(64), 0, st, fw.ident);
        note_launch();
        CAP_TRY(check_launch("eval_iota_kernel"));
        CAP_TRY(launch_dispatch_batched(token_src, nullptr, L, T, 1, 64, fw.ident, topo.D, fw.perm, nullptr,
                                        reinterpret_cast<int64_t *>(fw.srcoff), fw.sort_ws, st));
    }
    const EfFill fill = {fw.rec_src, g.rec_slots * 4, 0xffffffffu};
    CAP_TRY(ef_launch_table(g, fw, expert_dev, topo.dev_node, L, E, P, topo.D, st, &fill, 1));
    EvalFastParams prm = {};
    prm.idx = idx;
    prm.kept = kept;
    prm.expert_dev = expert_dev;
    prm.dev_node = topo.dev_node;
    prm.rec_src = fw.rec_src;
    prm.rec_planes = fw.rec_planes;
    prm.table = fw.table;
    prm.perm = token_src ? fw.perm : nullptr;
    prm.srcoff = token_src ? fw.srcoff : nullptr;
    prm.T = T;
    prm.tpc = g.tpc;
    prm.k = k;
    prm.E = E;
    prm.P = P;
    prm.D = topo.D;
    prm.WD = g.WD;
    prm.WN = g.WN;
    prm.Pc = g.Pc;
    prm.PC = g.PC;
    prm.DW = g.DW;
    prm.NW = g.NW;
    prm.R = g.R;
    prm.RS = g.RS;
    prm.S = g.S;
    prm.logS = g.logS;
    prm.XPL = g.xpl;
    prm.ncta_t = g.ncta_t;
    prm.maxrec = g.maxrec;
    prm.NPR = g.NPR;
    int rc;
    switch (g.KP) {
    case 4: rc = launch_kp<4, 4>(prm, g, L, st); break;
    case 8: rc = launch_kp<8, 8>(prm, g, L, st); break;
    case 12: rc = k <= 10 ? launch_kp<12, 10>(prm, g, L, st) : launch_kp<12, 12>(prm, g, L, st); break;
    default: rc = launch_kp<16, 16>(prm, g, L, st); break;
    }
    CAP_TRY(rc);
    CAP_TRY(ef_launch_decode(g, fw, L, T, E, P, topo, expert_dev, counts, out, st));
    *used = true;
    return CAP_OK;
}

}  // namespace cap

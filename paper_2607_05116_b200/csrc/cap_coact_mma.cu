// S2 fast path -- counts and the E x E co-activation matrix as an exact int8 -> int32 tensor-core
// contraction C = A^T A of the one-hot routing matrix A [tokens x E] (BASELINE.json
// north_star (2)).  A is never materialised in HBM: each block synthesises 128-token tiles of A^T
// ([E rows] x [128 tokens], int8, K-major canonical core-matrix layout) in shared memory straight
// from the index stream, and one thread issues tcgen05.mma.kind::i8 (M = 128, N = E, K = 32) with
// the SAME tile as both operands, accumulating in TMEM.  At the end the accumulator is read back
// with tcgen05.ld and added into the global matrix; symmetry (C[r][c] = C[c][r]) lets lane r write
// address [c][r], which makes the atomic adds coalesced.  diag(C) gives the counts.
// 256 < E <= 512 (config 5): the 512 x 512 accumulator is four times the TMEM of an SM, so blockIdx.z
// names the 128-row block a CTA accumulates (A = rows [128 z, 128 z + 128) of the tile, B = the whole
// 512-row tile as two N = 256 halves -> all 512 TMEM columns); every CTA builds the whole one-hot tile.
#include "cap_async.cuh"
#include "cap_internal.cuh"
#include "cap_tc.cuh"

namespace cap {

constexpr int CM_TK = 128;          // tokens per tile (4 MMAs of K = 32)
constexpr int CM_THREADS = 128;
constexpr int CM_NB = 2;            // tiles whose indices are fetched together (even: buffer = tile & 1)

struct CoactMmaParams {
    const int32_t *idx;        // [L][T][k]
    const uint8_t *kept;       // [L][T][k] or NULL
    unsigned long long *counts;   // [L][E]
    int *coact;                // [L][E][E]
    int64_t T, tpc;            // tokens per layer, tokens per block
    int32_t k, E, EP;          // EP = E padded to 128, 256 or 512 (rows of the tile)
    int32_t pack64;            // E even and coact 8-byte aligned: pairs of counters per 64-bit reduction
};

template <int EP, int KMAX>
__global__ void __launch_bounds__(CM_THREADS) coact_mma_kernel(CoactMmaParams q)
{
    extern __shared__ __align__(1024) unsigned char cm_sm[];   // two tiles [EP rows][CM_TK tokens] int8
    __shared__ uint64_t done_bar[2];
    __shared__ uint32_t s_tmem;
    constexpr int TILEB = EP * CM_TK;
    constexpr uint32_t LBO = 128u, SBO = (CM_TK / 16) * 128u;
    constexpr uint32_t NCOLS = EP == 128 ? 128u : 512u;
    constexpr int NMMA = EP == 128 ? 128 : 256;         // N of one MMA (256 is the instruction's maximum)
    constexpr uint32_t IDESC = (2u << 4) | ((uint32_t)(NMMA >> 3) << 17) | (8u << 24);   // S32 acc, u8 x u8, N, M = 128
    const int mb = EP == 512 ? (int)blockIdx.z : 0;     // accumulator row block of this CTA (EP = 512)
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int layer = blockIdx.y;
    const int E = q.E, k = q.k;

    if (warp == 0) tmem_alloc(&s_tmem, NCOLS);
    if (tid == 0) {
        mbar_init(&done_bar[0], 1);
        mbar_init(&done_bar[1], 1);
        mbar_fence_init();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = s_tmem;

    const int64_t t0 = (int64_t)blockIdx.x * q.tpc;
    const int64_t t1 = min(q.T, t0 + q.tpc);
    const int ntile = t1 > t0 && mb * 128 < E ? (int)((t1 - t0 + CM_TK - 1) / CM_TK) : 0;
    const int32_t *idx = q.idx + (size_t)layer * q.T * k;
    const uint8_t *kept = q.kept ? q.kept + (size_t)layer * q.T * k : nullptr;

    // The thread's token of each tile: its k expert rows as byte offsets into the tile (-1 = not
    // kept).  A thread only ever writes the bytes of its own token column, so a tile buffer is not
    // cleared between uses: both buffers are zeroed once, and when a buffer comes back (its MMAs
    // have completed) the thread takes back the ones it set two tiles ago and sets the new ones --
    // k byte stores each instead of a 32 / 64 KB clear and a block barrier.  Indices are fetched
    // one batch of CM_NB tiles ahead, so their global-load latency overlaps the tiles in work.
    {
        uint4 *t4 = reinterpret_cast<uint4 *>(cm_sm);
        for (int j = tid; j < 2 * TILEB / 16; j += CM_THREADS) t4[j] = make_uint4(0u, 0u, 0u, 0u);
    }
    const bool vec8 = KMAX == 8 && k == 8 && !kept && (reinterpret_cast<uintptr_t>(idx) & 15u) == 0;
    const bool vec2 = !vec8 && (k & 1) == 0 && !kept && (reinterpret_cast<uintptr_t>(idx) & 7u) == 0;
    int raw[CM_NB][KMAX];
    auto fetch = [&](int ib) {
#pragma unroll
        for (int u = 0; u < CM_NB; ++u) {
            const int64_t tok = t0 + (int64_t)(ib + u) * CM_TK + tid;
            const bool ok = tok < t1 && ib + u < ntile;
            if (vec8) {
                int4 lo = make_int4(-1, -1, -1, -1), hi = lo;
                if (ok) {
                    lo = __ldg(reinterpret_cast<const int4 *>(idx + tok * 8));
                    hi = __ldg(reinterpret_cast<const int4 *>(idx + tok * 8) + 1);
                }
                raw[u][0] = lo.x; raw[u][1] = lo.y; raw[u][2] = lo.z; raw[u][3] = lo.w;
                raw[u][4 % KMAX] = hi.x; raw[u][5 % KMAX] = hi.y; raw[u][6 % KMAX] = hi.z;
                raw[u][7 % KMAX] = hi.w;
            } else if (vec2) {
#pragma unroll
                for (int s = 0; s < KMAX; s += 2) {
                    int2 v = make_int2(-1, -1);
                    if (s < k && ok) v = __ldg(reinterpret_cast<const int2 *>(idx + tok * k + s));
                    raw[u][s] = v.x;
                    raw[u][(s + 1) % KMAX] = v.y;
                }
            } else {
#pragma unroll
                for (int s = 0; s < KMAX; ++s) {
                    int e = -1;
                    if (s < k && ok) {
                        const int64_t a = tok * k + s;
                        e = __ldg(idx + a);
                        if (kept && !__ldg(kept + a)) e = -1;
                    }
                    raw[u][s] = e;
                }
            }
        }
    };
    int prev[2][KMAX];          // what this thread set in each buffer (offsets, -1 = nothing)
#pragma unroll
    for (int s = 0; s < KMAX; ++s) prev[0][s] = prev[1][s] = -1;
    if (ntile > 0) fetch(0);
    __syncthreads();            // the buffers are zero
    for (int ib = 0; ib < ntile; ib += CM_NB) {
        int rowoff[CM_NB][KMAX];
#pragma unroll
        for (int u = 0; u < CM_NB; ++u) {
#pragma unroll
            for (int s = 0; s < KMAX; ++s) {
                const int e = raw[u][s];
                rowoff[u][s] = (unsigned)e < (unsigned)E ? (e >> 3) * (int)SBO + (e & 7) * 16 : -1;
            }
        }
        if (ib + CM_NB < ntile) fetch(ib + CM_NB);
#pragma unroll
        for (int u = 0; u < CM_NB; ++u) {
            const int i = ib + u;
            if (i >= ntile) break;
            const int buf = u & 1;                 // = i & 1 (CM_NB is even)
            unsigned char *tile = cm_sm + (size_t)buf * TILEB;
            if (i >= 2) mbar_wait(&done_bar[buf], (uint32_t)(((i >> 1) - 1) & 1));   // tile i-2 consumed
            {
                unsigned char *col = tile + (tid >> 4) * LBO + (tid & 15);
#pragma unroll
                for (int s = 0; s < KMAX; ++s)
                    if (prev[buf][s] >= 0) col[prev[buf][s]] = 0;
#pragma unroll
                for (int s = 0; s < KMAX; ++s) {
                    if (rowoff[u][s] >= 0) col[rowoff[u][s]] = 1;
                    prev[buf][s] = rowoff[u][s];
                }
            }
            proxy_fence_async();   // generic-proxy writes -> visible to the tensor core's async proxy
            __syncthreads();
            if (tid == 0) {
                tc_fence_after();
                const uint32_t base = smem_u32(tile);
#pragma unroll
                for (int j = 0; j < CM_TK / 32; ++j) {
                    const uint64_t bd = umma_desc(base + j * 2 * LBO, LBO, SBO);
                    if (EP == 512) {
                        const uint64_t ad = umma_desc(base + mb * 16 * SBO + j * 2 * LBO, LBO, SBO);
                        const uint64_t b1 = umma_desc(base + 32 * SBO + j * 2 * LBO, LBO, SBO);
                        umma_i8(tmem, ad, bd, IDESC, (uint32_t)((i | j) != 0));
                        umma_i8(tmem + 256u, ad, b1, IDESC, (uint32_t)((i | j) != 0));
                        continue;
                    }
                    umma_i8(tmem, bd, bd, IDESC, (uint32_t)((i | j) != 0));
                    if (EP == 256) {
                        const uint64_t a1 = umma_desc(base + 16 * SBO + j * 2 * LBO, LBO, SBO);
                        umma_i8(tmem + 256u, a1, bd, IDESC, (uint32_t)((i | j) != 0));
                    }
                }
                umma_commit(&done_bar[buf]);
            }
        }
    }
    if (ntile > 0) {
        const int last = ntile - 1;
        mbar_wait(&done_bar[last & 1], (uint32_t)((last >> 1) & 1));
        tc_fence_after();
        int *C = q.coact + (size_t)layer * E * E;
        unsigned long long *cnt = q.counts + (size_t)layer * E;
#pragma unroll 1
        for (int h = 0; h < (EP == 256 ? 2 : 1); ++h) {
            const int r = (mb + h) * 128 + warp * 32 + lane;   // accumulator row of this thread
#pragma unroll 1
            for (int cb0 = 0; cb0 < EP / 32; ++cb0) {
                // blocks start at different column groups so that they do not queue on the same L2 lines
                const int cb = (cb0 + (int)blockIdx.x) % (EP / 32);
                if (cb * 32 >= E) continue;                    // padding columns (warp-uniform)
                uint32_t v[32];
                tmem_ld32(tmem + ((uint32_t)(warp * 32) << 16) + (uint32_t)(h * 256 + cb * 32), v);
                // C symmetric: the value of (r, c) is added at [c][r], consecutive lanes -> consecutive
                // addresses.  Two neighbouring int32 counters are added with ONE 64-bit reduction
                // (counts are < 2^31, so the low word never carries into the high word): even lanes
                // take even columns, odd lanes odd columns, each packing its own and its neighbour's value.
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
                    for (int j = 0; j < 32; ++j) {
                        if (rok && cb * 32 + j < E)
                            asm volatile("red.global.add.s32 [%0], %1;" ::"l"(cp + (size_t)j * E), "r"(v[j]) : "memory");
                    }
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
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc(tmem, NCOLS);
}

template <int EP, int KMAX>
static int launch_ep(const CoactMmaParams &prm, int L, cudaStream_t st)
{
    // per device and cheap: set on every launch (a per-process flag would leave a second GPU without the opt-in)
    cudaFuncSetAttribute(coact_mma_kernel<EP, KMAX>, cudaFuncAttributeMaxDynamicSharedMemorySize,
    2 * EP * CM_TK);
    const int64_t nblk = (prm.T + prm.tpc - 1) / prm.tpc;
    const unsigned nz = EP == 512 ? (unsigned)((prm.E + 127) / 128) : 1u;
    {
        KernelTimerScope ts("coact", st);
        coact_mma_kernel<EP, KMAX><<<dim3((unsigned)nblk, (unsigned)L, nz), CM_THREADS, 2 * EP * CM_TK, st>>>(prm);
    }
    note_launch();
    return check_launch("coact_mma_kernel");
}

// counts / coact must already be zeroed.  *used = false when E > 512 (generic kernel instead).
int launch_coact_mma(const int32_t *idx, const uint8_t *kept, int32_t L, int64_t T, int32_t k, int32_t E,
                     int64_t *counts, int32_t *coact, cudaStream_t st, bool *used)
{
    *used = false;
    if (E > 512 || T < 1 || L < 1) return CAP_OK;
    CoactMmaParams prm;
    prm.idx = idx;
    prm.kept = kept;
    prm.counts = reinterpret_cast<unsigned long long *>(counts);
    prm.coact = coact;
    prm.T = T;
    prm.k = k;
    prm.E = E;
    prm.EP = E <= 128 ? 128 : E <= 256 ? 256 : 512;
    prm.pack64 = (E % 2 == 0) && (reinterpret_cast<uintptr_t>(coact) & 7u) == 0;
    // one block per SM is resident at EP = 256 (all 512 TMEM columns); every block ends with E^2 reductions into
    // the matrix, so a block should own at least ~1 000 tokens
    const int64_t nz = prm.EP == 512 ? (E + 127) / 128 : 1;
    int64_t want = balanced_blocks_per_unit(L * nz, sm_count(), T / 1024 > 1 ? T / 1024 : 1);
    int64_t tpc = (T + want - 1) / want;
    tpc = ((tpc + CM_TK - 1) / CM_TK) * CM_TK;
    prm.tpc = tpc;
    *used = true;
    if (prm.EP == 128) return k <= 8 ? launch_ep<128, 8>(prm, L, st) : launch_ep<128, 16>(prm, L, st);
    if (prm.EP == 256) return k <= 8 ? launch_ep<256, 8>(prm, L, st) : launch_ep<256, 16>(prm, L, st);
    return k <= 8 ? launch_ep<512, 8>(prm, L, st) : launch_ep<512, 16>(prm, L, st);
}

}  // namespace cap

// S1 fast path, standalone kernel (Eq. 1): persistent blocks, producer warps that
// stream 16-token tiles of logits into a shared-memory ring with TMA bulk copies (one copy per
// tile; rows are dense and the per-thread 128-bit row reads are XOR-swizzled so that they stay
// bank-conflict free), consumer warps that run the two-lanes-per-token selection network of
// cap_gate_fast.cuh.  Applies to softmax scoring with renormalised weights, no group limit,
// k <= 8, E in {64, 128, 256}; everything else takes the generic kernel of cap_gate.cu.
#include "cap_async.cuh"
#include "cap_gate_fast.cuh"

namespace cap {

constexpr int GF_NP = 2;                       // producer warps
constexpr int GF_NC = 12;                      // consumer warps; stages = a multiple of GF_NC (one consumer warp per stage:
                                               // with 14 warps on the 12 stages of E = 256 a warp's first tile could be the
                                               // SECOND use of a stage, whose parity wait passes before the first use landed)
constexpr int GF_THREADS = 32 * (GF_NC + GF_NP);
constexpr int GF_MAXST = 32;
constexpr int GF_TILE = 16;                    // tokens per tile (one warp, two lanes per token)

struct GateFastParams {
    const float *logits;
    int32_t *idx;
    float *w;
    int64_t LT;          // tokens
    int64_t tiles_per_cta;
    int32_t k, nst, vec_out;
    float scale;
};

template <int E>
__global__ void __launch_bounds__(GF_THREADS) gate_fast_kernel(GateFastParams q)
{
    extern __shared__ __align__(128) unsigned char gf_sm[];
    __shared__ uint64_t full_bar[GF_MAXST], empty_bar[GF_MAXST];
    constexpr int ROWB = E * 4;                  // dense rows; reads are XOR-swizzled per lane
    constexpr int STAGEB = GF_TILE * ROWB;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int nst = q.nst;
    if (threadIdx.x == 0) {
        for (int s = 0; s < nst; ++s) {
            mbar_init(&full_bar[s], 1);
            mbar_init(&empty_bar[s], 1);
        }
        mbar_fence_init();
    }
    __syncthreads();
    const int64_t ntiles = (q.LT + GF_TILE - 1) / GF_TILE;
    const int64_t tile0 = (int64_t)blockIdx.x * q.tiles_per_cta;
    int64_t nt = ntiles - tile0;
    if (nt > q.tiles_per_cta) nt = q.tiles_per_cta;
    if (nt <= 0) return;

    if (warp < GF_NP) {
        // ---- producers: warp p streams tiles p, p + NP, ...; one elected lane issues the row copies ----
        if (lane == 0) {
            for (int64_t j = warp; j < nt; j += GF_NP) {
                const int st = (int)(j % nst);
                if (j >= nst) mbar_wait(&empty_bar[st], (uint32_t)(((j / nst) - 1) & 1));
                const int64_t tok0 = (tile0 + j) * GF_TILE;
                const int rows = (int)min((int64_t)GF_TILE, q.LT - tok0);
                mbar_expect_tx(&full_bar[st], (uint32_t)rows * E * 4);
                bulk_g2s(gf_sm + (size_t)st * STAGEB, q.logits + tok0 * E, (uint32_t)rows * E * 4,
                         &full_bar[st]);           // the tile's rows are contiguous in global memory
            }
        }
    } else {
        // ---- consumers: warp c takes tiles c, c + NC, ...; lanes l and l ^ 16 share token l & 15 ----
        const int c = warp - GF_NP;
        const int k = q.k;
        const int h = lane >> 4, tl = lane & 15;
        for (int64_t j = c; j < nt; j += GF_NC) {
            const int st = (int)(j % nst);
            mbar_wait(&full_bar[st], (uint32_t)((j / nst) & 1));
            const int64_t tok = (tile0 + j) * GF_TILE + tl;
            const bool valid = tok < q.LT;
            // rows past the end of a ragged last tile were not written: those lanes redo row 0
            const float *row =
                reinterpret_cast<const float *>(gf_sm + (size_t)st * STAGEB + (valid ? tl : 0) * ROWB);
            int sel[8];
            float wv[4];
            gate_select_pair<E>(row, h, tl & 7, k, sel);
            gate_weights_softmax_pair(row, h, k, sel, q.scale, wv);
            if (valid) {
                if (q.vec_out) {
                    int4 *ip = reinterpret_cast<int4 *>(q.idx + tok * 8 + 4 * h);
                    float4 *wp = reinterpret_cast<float4 *>(q.w + tok * 8 + 4 * h);
                    *ip = h ? make_int4(sel[4], sel[5], sel[6], sel[7]) : make_int4(sel[0], sel[1], sel[2], sel[3]);
                    *wp = make_float4(wv[0], wv[1], wv[2], wv[3]);
                } else {
#pragma unroll
                    for (int jj = 0; jj < 4; ++jj) {
                        const int s = 4 * h + jj;
                        if (s < k) {
                            q.idx[tok * k + s] = h ? sel[4 + jj] : sel[jj];
                            q.w[tok * k + s] = wv[jj];
                        }
                    }
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty_bar[st]);
        }
    }
}

template <int E>
static int launch_e(GateFastParams prm, cudaStream_t st)
{
    constexpr int STAGEB = GF_TILE * (E * 4);
    int nst = (200 * 1024) / STAGEB;
    if (nst > GF_MAXST) nst = GF_MAXST;
    nst = (nst / GF_NC) * GF_NC;
    prm.nst = nst;
    // per device and cheap: set on every launch (a per-process flag would leave a second GPU without the opt-in)
    cudaFuncSetAttribute(gate_fast_kernel<E>, cudaFuncAttributeMaxDynamicSharedMemorySize, 210 * 1024);
    const int64_t ntiles = (prm.LT + GF_TILE - 1) / GF_TILE;
    int64_t grid = sm_count();
    if (grid > ntiles) grid = ntiles;
    prm.tiles_per_cta = (ntiles + grid - 1) / grid;
    grid = (ntiles + prm.tiles_per_cta - 1) / prm.tiles_per_cta;
    {
        KernelTimerScope ts("gate_topk", st);
        gate_fast_kernel<E><<<(unsigned)grid, GF_THREADS, (size_t)nst * STAGEB, st>>>(prm);
    }
    note_launch();
    return check_launch("gate_fast_kernel");
}

int launch_gate_fast(const float *logits, const float *bias, int32_t L, int64_t T,
                     const cap_gate_cfg &cfg, int32_t *idx, float *w, cudaStream_t st, bool *used)
{
    *used = false;
    if (cfg.scoring != 0 || cfg.renormalize != 1 || cfg.n_group != 1 || cfg.k > 8 || bias != nullptr)
        return CAP_OK;
    if (cfg.E != 64 && cfg.E != 128 && cfg.E != 256) return CAP_OK;
    if (reinterpret_cast<uintptr_t>(logits) & 15u) return CAP_OK;
    GateFastParams prm;
    prm.logits = logits;
    prm.idx = idx;
    prm.w = w;
    prm.LT = (int64_t)L * T;
    prm.k = cfg.k;
    prm.scale = cfg.scale;
    prm.vec_out = cfg.k == 8 && ((reinterpret_cast<uintptr_t>(idx) | reinterpret_cast<uintptr_t>(w)) & 15u) == 0;
    prm.nst = 0;
    prm.tiles_per_cta = 0;
    *used = true;
    if (prm.LT == 0) return CAP_OK;
    switch (cfg.E) {
    case 64: return launch_e<64>(prm, st);
    case 128: return launch_e<128>(prm, st);
    default: return launch_e<256>(prm, st);
    }
}

}  // namespace cap

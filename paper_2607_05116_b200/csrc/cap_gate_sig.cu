// S1 fast path for sigmoid scoring (+ selection bias, + group-limited routing over groups of 32 experts),
// standalone kernel (Eq. 1; BASELINE.json config 4, reading R14).  Same structure as
// cap_gate_fast.cu: persistent blocks, producer warps stream 16-token tiles of logits into a
// shared-memory ring with TMA bulk copies, consumer warps run the two-lanes-per-token selection of
// cap_gate_sig.cuh (cheap special-function sigmoid inside payload-carrying keys, sort-8 / merge-8
// networks per group, exact whole-warp redo of the tokens the keys cannot certify).  The selection bias
// of the tile's layer is read through L1 with the same swizzled 128-bit accesses as the row.
// Applies to scoring = sigmoid, renormalised weights, k <= 8, E in {64, 128, 256}, either no group limit
// or groups of exactly 32 experts, and T a multiple of the 16-token tile (a tile then lies inside one
// layer); everything else takes the generic kernel of cap_gate.cu.
#include "cap_async.cuh"
#include "cap_gate_sig.cuh"

namespace cap {

constexpr int GS_NP = 2;                       // producer warps
constexpr int GS_NC = 12;                      // consumer warps (24 measured slower: the 12 stages of E = 256 cannot feed them)
constexpr int GS_THREADS = 32 * (GS_NC + GS_NP);
constexpr int GS_MAXST = 32;
constexpr int GS_TILE = 16;                    // tokens per tile (one warp, two lanes per token)

struct GateSigParams {
    const float *logits;
    const float *bias;   // [L][E] or NULL
    int32_t *idx;
    float *w;
    int64_t LT, T;       // tokens in all layers / per layer
    int64_t tiles_per_cta;
    int32_t k, nst, vec_out, topk_group, group_score;
    float scale;
};

template <int E>
__global__ void __launch_bounds__(GS_THREADS) gate_sig_kernel(GateSigParams q)
{
    extern __shared__ __align__(1024) unsigned char gs_sm[];
    __shared__ uint64_t full_bar[GS_MAXST], empty_bar[GS_MAXST];
    // use number of every stage, set by the producer before it refills the stage.  There are more consumer warps
    // than stages, so consecutive uses of a stage belong to different warps, and a warp may reach use u of a
    // stage whose barrier is still two phases behind -- where `try_wait.parity` would report "done".  A consumer
    // therefore first waits until the stage is in ITS use, then on the barrier's parity.
    __shared__ uint32_t stage_use[GS_MAXST];
    constexpr int ROWB = E * 4;
    constexpr int STAGEB = GS_TILE * ROWB;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int nst = q.nst;
    if (threadIdx.x == 0) {
        for (int s = 0; s < nst; ++s) {
            mbar_init(&full_bar[s], 1);
            mbar_init(&empty_bar[s], 1);
            stage_use[s] = 0xffffffffu;
        }
        mbar_fence_init();
    }
    __syncthreads();
    const int64_t ntiles = (q.LT + GS_TILE - 1) / GS_TILE;
    const int64_t tile0 = (int64_t)blockIdx.x * q.tiles_per_cta;
    int64_t nt = ntiles - tile0;
    if (nt > q.tiles_per_cta) nt = q.tiles_per_cta;
    if (nt <= 0) return;

    if (warp < GS_NP) {
        if (lane == 0) {
            for (int64_t j = warp; j < nt; j += GS_NP) {
                const int st = (int)(j % nst);
                if (j >= nst) mbar_wait(&empty_bar[st], (uint32_t)(((j / nst) - 1) & 1));
                const int64_t tok0 = (tile0 + j) * GS_TILE;
                const int rows = (int)min((int64_t)GS_TILE, q.LT - tok0);
                st_release_shared(&stage_use[st], (uint32_t)(j / nst));
                mbar_expect_tx(&full_bar[st], (uint32_t)rows * E * 4);
                bulk_g2s(gs_sm + (size_t)st * STAGEB, q.logits + tok0 * E, (uint32_t)rows * E * 4, &full_bar[st]);
            }
        }
    } else {
        const int c = warp - GS_NP;
        const int k = q.k;
        const int h = lane >> 4, tl = lane & 15;
        for (int64_t j = c; j < nt; j += GS_NC) {
            const int st = (int)(j % nst);
            const uint32_t use = (uint32_t)(j / nst);
            while (ld_acquire_shared(&stage_use[st]) != use) __nanosleep(32);
            mbar_wait(&full_bar[st], use & 1u);
            const int64_t tok0 = (tile0 + j) * GS_TILE;
            const int64_t tok = tok0 + tl;
            const bool valid = tok < q.LT;
            const float *bias_g = q.bias ? q.bias + (tok0 / q.T) * E : nullptr;      // T % 16 == 0: one layer per tile
            const float *row =
                reinterpret_cast<const float *>(gs_sm + (size_t)st * STAGEB + (valid ? tl : 0) * ROWB);
            int sel[8];
            float wv[4];
            gate_select_sig_pair<E>(row, bias_g, h, tl & 7, k, q.topk_group, q.group_score, sel);
            gate_weights_sigmoid_pair(row, h, k, sel, q.scale, wv);
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
static int launch_sig_e(GateSigParams prm, cudaStream_t st)
{
    constexpr int STAGEB = GS_TILE * (E * 4);
    int nst = (200 * 1024) / STAGEB;
    if (nst > GS_MAXST) nst = GS_MAXST;
    prm.nst = nst;
    // set on every launch: the attribute is per device and cheap (cap.h: calls are re-entrant)
    cudaFuncSetAttribute(gate_sig_kernel<E>, cudaFuncAttributeMaxDynamicSharedMemorySize, 210 * 1024);
    const int64_t ntiles = (prm.LT + GS_TILE - 1) / GS_TILE;
    int64_t grid = sm_count();
    if (grid > ntiles) grid = ntiles;
    prm.tiles_per_cta = (ntiles + grid - 1) / grid;
    grid = (ntiles + prm.tiles_per_cta - 1) / prm.tiles_per_cta;
    {
        KernelTimerScope ts("gate_topk", st);
        gate_sig_kernel<E><<<(unsigned)grid, GS_THREADS, (size_t)nst * STAGEB, st>>>(prm);
    }
    note_launch();
    return check_launch("gate_sig_kernel");
}

int launch_gate_sig(const float *logits, const float *bias, int32_t L, int64_t T, const cap_gate_cfg &cfg,
                    int32_t *idx, float *w, cudaStream_t st, bool *used)
{
    *used = false;
    if (cfg.scoring != 1 || cfg.renormalize != 1 || cfg.k > 8) return CAP_OK;
    if (cfg.E != 64 && cfg.E != 128 && cfg.E != 256) return CAP_OK;
    const int ng = cfg.E / 32;
    if (cfg.n_group != 1 && cfg.n_group != ng) return CAP_OK;
    if (T % GS_TILE != 0) return CAP_OK;
    if ((reinterpret_cast<uintptr_t>(logits) | reinterpret_cast<uintptr_t>(bias)) & 15u) return CAP_OK;
    GateSigParams prm;
    prm.logits = logits;
    prm.bias = bias;
    prm.idx = idx;
    prm.w = w;
    prm.LT = (int64_t)L * T;
    prm.T = T;
    prm.k = cfg.k;
    prm.scale = cfg.scale;
    // no group limit = every group selected
    prm.topk_group = cfg.n_group == 1 ? ng : cfg.topk_group;
    prm.group_score = cfg.n_group == 1 ? 0 : cfg.group_score;
    prm.vec_out = cfg.k == 8 && ((reinterpret_cast<uintptr_t>(idx) | reinterpret_cast<uintptr_t>(w)) & 15u) == 0;
    prm.nst = 0;
    prm.tiles_per_cta = 0;
    *used = true;
    if (prm.LT == 0) return CAP_OK;
    switch (cfg.E) {
    case 64: return launch_sig_e<64>(prm, st);
    case 128: return launch_sig_e<128>(prm, st);
    default: return launch_sig_e<256>(prm, st);
    }
}

}  // namespace cap

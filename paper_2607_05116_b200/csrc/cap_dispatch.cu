// S5 -- dispatch layout (P:L58 device-centric routing; BASELINE.json stage 5): stable counting
// sort of the kept (token,slot) pairs by destination device.  The pair stream is cut into sub-chunks
// of DS_SUB consecutive pairs, one per WARP.  Three kernels: (1) every warp counts the keys of its
// sub-chunk (warp match, private counters: no block-level synchronisation, no atomics); (2) an
// ordered scan over (device, sub-chunk) fixes every sub-chunk's base per device -- this is what makes
// the sort stable across warps and blocks without global cursors; (3) every warp scatters its
// sub-chunk in pair order, ranking equal keys inside a 32-pair round with match/popc.
#include "cap_eval_final.cuh"
#include "cap_internal.cuh"

namespace cap {

constexpr int DS_SUB = 256;       // pairs per warp (8 rounds of 32)
constexpr int DS_THREADS = 256;   // 8 warps: 2048 pairs per block
constexpr int DS_NW = DS_THREADS / 32;
constexpr int DS_MAXD = 64;

// sub-chunks of n pairs, padded so that every lane of the scan owns whole 16-byte vectors
int64_t dispatch_stride_subs(int64_t nsub) { return ((nsub + 127) / 128) * 128; }
static int64_t ds_stride(int64_t n) { return dispatch_stride_subs((n + DS_SUB - 1) / DS_SUB); }

size_t dispatch_ws_bytes(int64_t T, int32_t k, int32_t D)
{
    const int64_t n = T * k;
    return (size_t)(2 * ds_stride(n) * D + 64) * sizeof(int) + 256;
}

// all layers of cap_dispatch_layout_batched: [L][hist | base | 64 device totals]
size_t dispatch_ws_bytes_batched(int32_t L, int64_t T, int32_t k, int32_t D)
{
    const int64_t n = T * k;
    return (size_t)(L < 1 ? 1 : L) * (size_t)(2 * ds_stride(n) * D + 64) * sizeof(int) + 256;
}

// layer strides of the batched call (blockIdx.y = layer; all zero-cost for a single layer)
struct DsBatch {
    int64_t pair_stride;    // T k: idx / kept / sorted_pairs / pair_pos
    int64_t ws_stride;      // 2 stride D + 64 ints: hist, base and the device totals of one layer
    int32_t map_stride;     // E
    int32_t off_stride;     // D + 1
};

// expert of pair i, -1 if the pair is pruned or past the end (both loads are issued unconditionally and
// before the placement map is staged: one memory round trip instead of three)
__device__ __forceinline__ int pair_expert(const int32_t *idx, const uint8_t *kept, int64_t i, int64_t n)
{
    if (i >= n) return -1;
    const int e = idx[i];
    const int kp = kept ? (int)kept[i] : 1;
    return kp ? e : -1;
}
// destination device of an expert, -1 for "no pair" or an out-of-range expert or device (memory-safe on
// garbage inputs: such pairs are left out of the layout)
__device__ __forceinline__ int expert_key(int e, const int *s_map, int E, int D)
{
    if ((unsigned)e >= (unsigned)E) return -1;
    const int d = s_map[e];
    return (unsigned)d < (unsigned)D ? d : -1;
}

// hist[d][sub] = kept pairs of sub-chunk `sub` going to device d (rows of `stride` entries, zero padded)
__global__ void __launch_bounds__(DS_THREADS)
dispatch_hist_kernel(const int32_t *__restrict__ idx, const uint8_t *__restrict__ kept, int64_t n,
                     int E, int D, const int32_t *__restrict__ expert_dev, int *__restrict__ hist,
                     int64_t stride, DsBatch lb)
{
    extern __shared__ int sm[];
    int *s_map = sm;                               // [E]
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int *cnt = sm + E + warp * DS_MAXD;            // [D] private to the warp
    idx += blockIdx.y * lb.pair_stride;
    if (kept) kept += blockIdx.y * lb.pair_stride;
    expert_dev += blockIdx.y * lb.map_stride;
    hist += blockIdx.y * lb.ws_stride;
    pdl_launch_dependents();
    pdl_wait();
    const int64_t sub = (int64_t)blockIdx.x * DS_NW + warp;
    const int64_t i0 = sub * DS_SUB;
    int key[DS_SUB / 32];
#pragma unroll
    for (int r = 0; r < DS_SUB / 32; ++r) key[r] = pair_expert(idx, kept, i0 + r * 32 + lane, n);
    for (int i = threadIdx.x; i < E; i += blockDim.x) s_map[i] = expert_dev[i];
    for (int d = lane; d < D; d += 32) cnt[d] = 0;
    __syncthreads();
    if (sub >= stride) return;
    if (i0 < n) {
#pragma unroll
        for (int r = 0; r < DS_SUB / 32; ++r) key[r] = expert_key(key[r], s_map, E, D);
#pragma unroll
        for (int r = 0; r < DS_SUB / 32; ++r) {
            const unsigned grp = __match_any_sync(0xffffffffu, key[r]);
            if (key[r] >= 0 && (grp & ((1u << lane) - 1u)) == 0u) cnt[key[r]] += __popc(grp);   // one lane per key
            __syncwarp();
        }
    }
    for (int d = lane; d < D; d += 32) hist[(int64_t)d * stride + sub] = cnt[d];
}

// One block per device row: warp w owns a contiguous span of the row's 128-entry chunks.  Pass 1 adds the span up,
// the span totals are scanned across the warps, pass 2 writes the exclusive prefixes (one int4 per lane, eight
// chunks in flight) starting from the span's base.  The row total goes to devtot[d]; the scatter kernel turns the
// D totals into the device offsets.  (Round 1 scanned all rows in ONE block: 893 of S5's 1 455 us at 2^22 tokens.)
// cap_prune_dispatch: block D of every layer adds up the per-block partial sums the S4 kernel left (PD_PART 32-bit
// columns per block: the evaluation accumulators, then the tokens received per device) into the 64-bit sums the
// finalize step reads.  Plain stores: nothing has to be zeroed beforehand.
__global__ void __launch_bounds__(512)
dispatch_scan_kernel(const int *__restrict__ hist, int *__restrict__ base, int D, int64_t stride, DsBatch lb, DsReduce rd)
{
    __shared__ int s_span[16];
    __shared__ unsigned long long s_red[7][PD_PART];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
    const int d = blockIdx.x;
    if (d >= D) {
        // reduce block j = d - D: S4 blocks [j per_rb, (j + 1) per_rb)
        pdl_launch_dependents();
        pdl_wait();
        const int j = d - D;
        const int ng = (int)blockDim.x / PD_PART;          // 7 groups of 72 threads in a 512-thread block, else 1
        const int g = (int)threadIdx.x / PD_PART, col = (int)threadIdx.x % PD_PART;
        const uint32_t *pp = rd.part + (size_t)blockIdx.y * rd.nblk * PD_PART;
        const int64_t b_lo = (int64_t)j * rd.per_rb, b_hi = min(rd.nblk, b_lo + rd.per_rb);
        unsigned long long sum = 0ull;
        if (g < ng)
            for (int64_t b = b_lo + g; b < b_hi; b += ng) sum += pp[b * PD_PART + col];
        if (g < ng) s_red[g][col] = sum;
        __syncthreads();
        if ((int)threadIdx.x < PD_PART) {
            unsigned long long tot = 0ull;
            for (int g2 = 0; g2 < ng; ++g2) tot += s_red[g2][threadIdx.x];
            rd.red[((size_t)blockIdx.y * rd.nrb + j) * PD_PART + threadIdx.x] = tot;
        }
        return;
    }
    hist += blockIdx.y * lb.ws_stride + (int64_t)d * stride;
    base += blockIdx.y * lb.ws_stride + (int64_t)d * stride;
    int *devtot = const_cast<int *>(hist) - (int64_t)d * stride + 2 * stride * D;     // behind hist and base of the layer
    const int64_t nch = stride / 128;
    const int64_t cpw = (nch + nw - 1) / nw;
    const int64_t c_lo = min(nch, (int64_t)warp * cpw), c_hi = min(nch, c_lo + cpw);
    pdl_launch_dependents();
    pdl_wait();
    const int4 *h = reinterpret_cast<const int4 *>(hist) + lane;
    int4 *bs = reinterpret_cast<int4 *>(base) + lane;
    int acc = 0;
    for (int64_t c0 = c_lo; c0 < c_hi; c0 += 8) {
        int4 v[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) v[j] = c0 + j < c_hi ? h[(c0 + j) * 32] : make_int4(0, 0, 0, 0);
#pragma unroll
        for (int j = 0; j < 8; ++j) acc += (v[j].x + v[j].y) + (v[j].z + v[j].w);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if (lane == 0) s_span[warp] = acc;
    __syncthreads();
    int run = 0, total = 0;                        // pairs of device d before this warp's span / in the row
    for (int w2 = 0; w2 < nw; ++w2) {
        const int v = s_span[w2];
        run += w2 < warp ? v : 0;
        total += v;
    }
    if (threadIdx.x == 0) devtot[d] = total;
    for (int64_t c0 = c_lo; c0 < c_hi; c0 += 8) {
        int4 v[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) v[j] = c0 + j < c_hi ? h[(c0 + j) * 32] : make_int4(0, 0, 0, 0);
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            const int sum = (v[j].x + v[j].y) + (v[j].z + v[j].w);
            int inc = sum;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int y = __shfl_up_sync(0xffffffffu, inc, o);
                if (lane >= o) inc += y;
            }
            int4 o;
            o.x = run + inc - sum;             // exclusive, within device d
            o.y = o.x + v[j].x;
            o.z = o.y + v[j].y;
            o.w = o.z + v[j].z;
            if (c0 + j < c_hi) bs[(c0 + j) * 32] = o;
            run += __shfl_sync(0xffffffffu, inc, 31);
        }
    }
}

// RMAX >= rounds: a warp's sub-chunk is `rounds` rounds of 32 consecutive pairs (8 for the stand-alone call; k for
// cap_prune_dispatch, whose S4 kernel counted 32 tokens per warp).  fin_block >= 0: that block of every layer does
// not scatter; it finishes the after-metrics of cap_prune_dispatch from the sums the scan kernel left (fin) and
// from the pairs per device (= the row totals of the scan).
template <int RMAX>
__global__ void __launch_bounds__(DS_THREADS)
dispatch_scatter_kernel(const int32_t *__restrict__ idx, const uint8_t *__restrict__ kept, int64_t n,
                        int E, int D, const int32_t *__restrict__ expert_dev,
                        const int *__restrict__ base, long long *__restrict__ offsets,
                        int32_t *__restrict__ sorted_pairs, int32_t *__restrict__ pair_pos, int64_t stride,
                        DsBatch lb, int rounds, int fin_block, FinalParams fin, DsReduce rd)
{
    extern __shared__ int sm[];
    __shared__ int s_off[65];                      // exclusive prefix of the device totals (T k < 2^31)
    __shared__ unsigned long long s_lp[64];
    int *s_map = sm;                               // [E]
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int *running = sm + E + warp * DS_MAXD;        // [D] next free position per device, private to the warp
    idx += blockIdx.y * lb.pair_stride;
    if (kept) kept += blockIdx.y * lb.pair_stride;
    expert_dev += blockIdx.y * lb.map_stride;
    base += blockIdx.y * lb.ws_stride;
    offsets += blockIdx.y * lb.off_stride;
    sorted_pairs += blockIdx.y * lb.pair_stride;
    if (pair_pos) pair_pos += blockIdx.y * lb.pair_stride;
    const int64_t sub = (int64_t)blockIdx.x * DS_NW + warp;
    pdl_launch_dependents();
    pdl_wait();
    if ((int)blockIdx.x == fin_block) {
        if ((int)threadIdx.x < PD_PART) {
            unsigned long long tot = 0ull;
            for (int j = 0; j < rd.nrb; ++j) tot += rd.red[((size_t)blockIdx.y * rd.nrb + j) * PD_PART + threadIdx.x];
            if (threadIdx.x < ACC_N) rd.acc[(size_t)blockIdx.y * ACC_N + threadIdx.x] = tot;
            else if ((int)threadIdx.x - ACC_N < D) rd.recv[(size_t)blockIdx.y * D + threadIdx.x - ACC_N] = tot;
        }
        __threadfence();
        __syncthreads();
        if (warp == 0) {
            const int *devtot = base + 2 * stride * D - stride * D;
            s_lp[lane] = lane < D ? (unsigned long long)devtot[lane] : 0ull;
            s_lp[lane + 32] = lane + 32 < D ? (unsigned long long)devtot[lane + 32] : 0ull;
            eval_finalize_one(fin, (int)blockIdx.y, lane, s_lp, true);
        }
        return;
    }
    const int64_t i0 = sub * 32 * rounds;
    int key[RMAX];
#pragma unroll
    for (int r = 0; r < RMAX; ++r) key[r] = r < rounds ? pair_expert(idx, kept, i0 + r * 32 + lane, n) : -1;
    for (int i = threadIdx.x; i < E; i += blockDim.x) s_map[i] = expert_dev[i];
    if (warp == 0) {
        // device offsets from the row totals the scan kernel left behind hist and base
        const int *devtot = base + 2 * stride * D - stride * D;
        int v0 = lane < D ? devtot[lane] : 0, v1 = lane + 32 < D ? devtot[lane + 32] : 0;
        int i0s = v0, i1s = v1;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int y0 = __shfl_up_sync(0xffffffffu, i0s, o), y1 = __shfl_up_sync(0xffffffffu, i1s, o);
            if (lane >= o) { i0s += y0; i1s += y1; }
        }
        const int t0 = __shfl_sync(0xffffffffu, i0s, 31);
        s_off[lane] = i0s - v0;
        s_off[lane + 32] = t0 + i1s - v1;
        if (lane == 31) s_off[64] = t0 + i1s;
    }
    __syncthreads();
    if (blockIdx.x == 0 && (int)threadIdx.x <= D)
        offsets[threadIdx.x] = (long long)((int)threadIdx.x < D ? s_off[threadIdx.x] : s_off[D < 64 ? D : 64]);
    if (i0 < n)
        for (int d = lane; d < D; d += 32) running[d] = s_off[d] + base[(int64_t)d * stride + sub];
    __syncwarp();
    if (i0 >= n) return;
#pragma unroll
    for (int r = 0; r < RMAX; ++r) key[r] = expert_key(key[r], s_map, E, D);
#pragma unroll
    for (int r = 0; r < RMAX; ++r) {
        if (r < rounds) {
            const int64_t i = i0 + r * 32 + lane;
            const int d = key[r];
            const unsigned grp = __match_any_sync(0xffffffffu, d);
            const int rank = __popc(grp & ((1u << lane) - 1u));
            int pos = -1;
            if (d >= 0) {
                pos = running[d] + rank;
                sorted_pairs[pos] = (int32_t)i;
            }
            if (pair_pos && i < n) pair_pos[i] = pos;
            __syncwarp();
            if (d >= 0 && rank == 0) running[d] += __popc(grp);
            __syncwarp();
        }
    }
}

// scan + scatter over a histogram that is already in place (hist rows of `stride` sub-chunks of 32 * rounds pairs).
// rd / fin: the extra blocks of cap_prune_dispatch (rd.part == NULL: none).
int launch_dispatch_tail(const int32_t *idx, const uint8_t *kept, int32_t L, int64_t n, int32_t E,
                         const int32_t *expert_dev, int32_t D, int32_t *sorted_pairs, int32_t *pair_pos,
                         int64_t *offsets, int *hist, int64_t stride, int rounds, const DsReduce &rd,
                         const FinalParams *fin, cudaStream_t st)
{
    const int64_t nsub = (n + 32 * rounds - 1) / (32 * rounds);
    const int64_t nb = (nsub + DS_NW - 1) / DS_NW;
    const size_t smem = sizeof(int) * (size_t)(E + DS_NW * DS_MAXD);
    int *base = hist + stride * D;
    DsBatch lb;
    lb.pair_stride = n;
    lb.ws_stride = 2 * stride * D + 64;
    lb.map_stride = E;
    lb.off_stride = D + 1;
    const bool extra = rd.part != nullptr;
    {
    KernelTimerScope ts("dispatch_scan", st);
    launch_pdl_edge(dispatch_scan_kernel, dim3((unsigned)(D + (extra ? rd.nrb : 0)), (unsigned)L), dim3(stride >= 128 * 16 ? 512 : 128), 0, st,
               (const int *)hist, base, D, stride, lb, rd);
    }
    note_launch();
    CAP_TRY(check_launch("dispatch_scan_kernel"));
    FinalParams f0 = {};
    const FinalParams &f = fin ? *fin : f0;
    const int fin_block = fin ? (int)nb : -1;
    const dim3 grid((unsigned)(nb + (fin ? 1 : 0)), (unsigned)L);
    {
    KernelTimerScope ts("dispatch_scatter", st);
#define CAP_SCATTER(R)                                                                                              \
    launch_pdl(dispatch_scatter_kernel<R>, grid, dim3(DS_THREADS), smem, st, idx, kept, n, E, D, expert_dev,          \
               (const int *)base, reinterpret_cast<long long *>(offsets), sorted_pairs, pair_pos, stride, lb, rounds, \
               fin_block, f, rd)
    if (rounds <= 4) CAP_SCATTER(4);
    else if (rounds <= 8) CAP_SCATTER(8);
    else if (rounds <= 12) CAP_SCATTER(12);
    else CAP_SCATTER(16);
#undef CAP_SCATTER
    }
    note_launch();
    return check_launch("dispatch_scatter_kernel");
}

// L layers in three launches (blockIdx.y = layer): idx / kept [L][T][k], expert_dev [L][E], sorted_pairs / pair_pos
// [L][T k], offsets [L][D + 1]; ws holds hist and base of every layer.
int launch_dispatch_batched(const int32_t *idx, const uint8_t *kept, int32_t L, int64_t T, int32_t k, int32_t E,
                            const int32_t *expert_dev, int32_t D, int32_t *sorted_pairs, int32_t *pair_pos,
                            int64_t *offsets, void *ws, cudaStream_t st)
{
    if (L == 0) return CAP_OK;
    const int64_t n = T * k;
    if (n == 0) {
        if (cudaMemsetAsync(offsets, 0, sizeof(int64_t) * (size_t)L * (size_t)(D + 1), st) != cudaSuccess)
            return check_launch("memset offsets");
        return CAP_OK;
    }
    const int64_t stride = ds_stride(n);
    const int64_t nbh = stride / DS_NW;
    const size_t smem = sizeof(int) * (size_t)(E + DS_NW * DS_MAXD);
    int *hist = reinterpret_cast<int *>((reinterpret_cast<uintptr_t>(ws) + 255) & ~(uintptr_t)255);
    DsBatch lb;
    lb.pair_stride = n;
    lb.ws_stride = 2 * stride * D + 64;
    lb.map_stride = E;
    lb.off_stride = D + 1;
    {
    KernelTimerScope ts("dispatch_hist", st);
    launch_pdl(dispatch_hist_kernel, dim3((unsigned)nbh, (unsigned)L), dim3(DS_THREADS), smem, st, idx, kept, n, E, D,
               expert_dev, hist, stride, lb);
    }
    note_launch();
    CAP_TRY(check_launch("dispatch_hist_kernel"));
    DsReduce rd = {};
    return launch_dispatch_tail(idx, kept, L, n, E, expert_dev, D, sorted_pairs, pair_pos, offsets, hist, stride,
                                DS_SUB / 32, rd, nullptr, st);
}

int launch_dispatch(const int32_t *idx, const uint8_t *kept, int64_t T, int32_t k, int32_t E,
                    const int32_t *expert_dev, int32_t D, int32_t *sorted_pairs, int32_t *pair_pos,
                    int64_t *offsets, void *ws, cudaStream_t st)
{
    return launch_dispatch_batched(idx, kept, 1, T, k, E, expert_dev, D, sorted_pairs, pair_pos, offsets, ws, st);
}

}  // namespace cap

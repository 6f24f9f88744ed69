// S5 -- dispatch layout (P:L58 device-centric routing; BASELINE.json stage 5): stable counting
// sort of the kept (token,slot) pairs by destination device.  Three kernels: per-chunk key
// histograms, an ordered scan over (device, chunk) that fixes every chunk's base per device
// (this is what makes the sort stable across blocks -- no global cursors), and a scatter that
// ranks pairs inside a chunk with warp match/ballot and per-warp prefixes.
#include "cap_internal.cuh"

namespace cap {

constexpr int DS_CHUNK = 2048;   // pairs per block
constexpr int DS_THREADS = 256;

size_t dispatch_ws_bytes(int64_t T, int32_t k, int32_t D)
{
    const int64_t n = T * k;
    const int64_t nb = (n + DS_CHUNK - 1) / DS_CHUNK;
    return (size_t)(2 * nb * D) * sizeof(int) + 256;
}

__device__ __forceinline__ int pair_key(const int32_t *idx, const uint8_t *kept, const int *s_map,
                                        int64_t i, int64_t n)
{
    if (i >= n) return -1;
    if (kept && !kept[i]) return -1;
    return s_map[idx[i]];
}

__global__ void __launch_bounds__(DS_THREADS)
dispatch_hist_kernel(const int32_t *__restrict__ idx, const uint8_t *__restrict__ kept, int64_t n,
                     int E, int D, const int32_t *__restrict__ expert_dev, int *__restrict__ hist,
                     int64_t nb)
{
    extern __shared__ int sm[];
    int *s_map = sm;          // [E]
    int *cnt = sm + E;        // [D]
    for (int i = threadIdx.x; i < E; i += blockDim.x) s_map[i] = expert_dev[i];
    for (int i = threadIdx.x; i < D; i += blockDim.x) cnt[i] = 0;
    __syncthreads();
    const int64_t i0 = (int64_t)blockIdx.x * DS_CHUNK;
    for (int j = threadIdx.x; j < DS_CHUNK; j += blockDim.x) {
        int d = pair_key(idx, kept, s_map, i0 + j, n);
        if (d >= 0) atomicAdd(&cnt[d], 1);
    }
    __syncthreads();
    for (int d = threadIdx.x; d < D; d += blockDim.x) hist[(int64_t)d * nb + blockIdx.x] = cnt[d];
}

// One block.  Warp w scans device d = w, w+nwarps, ... over all chunks (device-major layout).
__global__ void __launch_bounds__(1024)
dispatch_scan_kernel(const int *__restrict__ hist, int *__restrict__ base, long long *__restrict__ offsets,
                     int D, int64_t nb)
{
    __shared__ long long tot[64];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
    for (int d = warp; d < D; d += nw) {
        int run = 0;
        for (int64_t b0 = 0; b0 < nb; b0 += 32) {
            int64_t b = b0 + lane;
            int v = (b < nb) ? hist[(int64_t)d * nb + b] : 0;
            int inc = v;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                int y = __shfl_up_sync(0xffffffffu, inc, o);
                if (lane >= o) inc += y;
            }
            if (b < nb) base[(int64_t)d * nb + b] = run + inc - v;   // exclusive, within device d
            run += __shfl_sync(0xffffffffu, inc, 31);
        }
        if (lane == 0) tot[d] = run;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        long long acc = 0;
        for (int d = 0; d < D; ++d) { offsets[d] = acc; acc += tot[d]; }
        offsets[D] = acc;
    }
}

__global__ void __launch_bounds__(DS_THREADS)
dispatch_scatter_kernel(const int32_t *__restrict__ idx, const uint8_t *__restrict__ kept, int64_t n,
                        int E, int D, const int32_t *__restrict__ expert_dev,
                        const int *__restrict__ base, const long long *__restrict__ offsets,
                        int32_t *__restrict__ sorted_pairs, int32_t *__restrict__ pair_pos, int64_t nb)
{
    extern __shared__ int sm[];
    constexpr int NW = DS_THREADS / 32;
    int *s_map = sm;              // [E]
    int *running = sm + E;        // [D]   next free position of device d for this chunk
    int *wcnt = running + D;      // [NW][D]
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int i = threadIdx.x; i < E; i += blockDim.x) s_map[i] = expert_dev[i];
    for (int d = threadIdx.x; d < D; d += blockDim.x)
        running[d] = (int)offsets[d] + base[(int64_t)d * nb + blockIdx.x];
    __syncthreads();
    const int64_t i0 = (int64_t)blockIdx.x * DS_CHUNK;
    for (int r = 0; r < DS_CHUNK / DS_THREADS; ++r) {
        for (int i = threadIdx.x; i < NW * D; i += blockDim.x) wcnt[i] = 0;
        __syncthreads();
        const int64_t i = i0 + (int64_t)r * DS_THREADS + threadIdx.x;
        const int d = pair_key(idx, kept, s_map, i, n);
        const unsigned grp = __match_any_sync(0xffffffffu, d);
        const int rank = __popc(grp & ((1u << lane) - 1u));
        if (d >= 0 && rank == 0) wcnt[warp * D + d] = __popc(grp);
        __syncthreads();
        if (d >= 0) {
            int pos = running[d] + rank;
            for (int w = 0; w < warp; ++w) pos += wcnt[w * D + d];
            sorted_pairs[pos] = (int32_t)i;
            if (pair_pos) pair_pos[i] = pos;
        } else if (pair_pos && i < n) {
            pair_pos[i] = -1;
        }
        __syncthreads();
        for (int dd = threadIdx.x; dd < D; dd += blockDim.x) {
            int s = 0;
            for (int w = 0; w < NW; ++w) s += wcnt[w * D + dd];
            running[dd] += s;
        }
        __syncthreads();
    }
}

int launch_dispatch(const int32_t *idx, const uint8_t *kept, int64_t T, int32_t k, int32_t E,
                    const int32_t *expert_dev, int32_t D, int32_t *sorted_pairs, int32_t *pair_pos,
                    int64_t *offsets, void *ws, cudaStream_t st)
{
    const int64_t n = T * k;
    if (n == 0) {
        if (cudaMemsetAsync(offsets, 0, sizeof(int64_t) * (size_t)(D + 1), st) != cudaSuccess)
            return check_launch("memset offsets");
        return CAP_OK;
    }
    const int64_t nb = (n + DS_CHUNK - 1) / DS_CHUNK;
    int *hist = reinterpret_cast<int *>((reinterpret_cast<uintptr_t>(ws) + 255) & ~(uintptr_t)255);
    int *base = hist + nb * D;
    {
    KernelTimerScope ts("dispatch_hist", st);
    dispatch_hist_kernel<<<(unsigned)nb, DS_THREADS, sizeof(int) * (size_t)(E + D), st>>>(
        idx, kept, n, E, D, expert_dev, hist, nb);
    }
    note_launch();
    CAP_TRY(check_launch("dispatch_hist_kernel"));
    {
    KernelTimerScope ts("dispatch_scan", st);
    dispatch_scan_kernel<<<1, 1024, 0, st>>>(hist, base, reinterpret_cast<long long *>(offsets), D, nb);
    }
    note_launch();
    CAP_TRY(check_launch("dispatch_scan_kernel"));
    {
    KernelTimerScope ts("dispatch_scatter", st);
    dispatch_scatter_kernel<<<(unsigned)nb, DS_THREADS,
                              sizeof(int) * (size_t)(E + D + (DS_THREADS / 32) * D), st>>>(
        idx, kept, n, E, D, expert_dev, base, reinterpret_cast<const long long *>(offsets), sorted_pairs,
        pair_pos, nb);
    }
    note_launch();
    return check_launch("dispatch_scatter_kernel");
}

}  // namespace cap

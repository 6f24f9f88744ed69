// cap_dispatch_rows: the device-centric dispatch layout of P:L58 (sec. II-C, Fig. 2) -- one row per
// (token, destination device), grouped by device, ascending token inside a device, plus for every kept
// (token, slot) pair the row that carries its token to its expert's device.
//
// HBM-bound streaming work like S5: read 4k (+k) bytes per token twice, write <= 4 min(k, D) + 4k.
// Three kernels: (1) per block of 256 tokens the number of distinct (token, device) rows per device
// (thread per token builds a 64-bit device mask; a warp counts a device with one ballot), (2) one block
// per device scans those counts over the token blocks, (3) the same ballots give every row its stable
// position: device base + block prefix + warp prefix + rank among the lower lanes.
#include "cap_internal.cuh"

namespace cap {
namespace {

constexpr int RT = 256;   // tokens (threads) per block
constexpr int RW = RT / 32;

// vec: k % 4 == 0 and 16-byte aligned index / 4-byte aligned mask streams -> 128-bit index loads (a warp's
// scalar loads of a [T][k] row-major stream touch 32 sectors per request; measured 30 sectors / request)
__device__ __forceinline__ unsigned long long token_mask(const int32_t *__restrict__ idx, const uint8_t *__restrict__ kept,
                                                         const uint8_t *sdev, int64_t t, int64_t T, int k, int E,
                                                         int8_t *dv, bool vec)
{
    int ev[16];
    unsigned kp[4] = {0x01010101u, 0x01010101u, 0x01010101u, 0x01010101u};
    if (vec) {
        const int4 *p4 = reinterpret_cast<const int4 *>(idx + t * k);
        const unsigned *k4 = reinterpret_cast<const unsigned *>(kept + t * k);
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            int4 v = make_int4(0, 0, 0, 0);
            if (q * 4 < k && t < T) {
                v = p4[q];
                if (kept) kp[q] = k4[q];
            }
            ev[4 * q] = v.x;
            ev[4 * q + 1] = v.y;
            ev[4 * q + 2] = v.z;
            ev[4 * q + 3] = v.w;
        }
    } else {
#pragma unroll
        for (int s = 0; s < 16; ++s) {
            ev[s] = 0;
            if (s < k && t < T) {
                ev[s] = idx[t * k + s];
                if (kept) {
                    unsigned b = kept[t * k + s];
                    kp[s >> 2] = (kp[s >> 2] & ~(0xffu << ((s & 3) * 8))) | (b << ((s & 3) * 8));
                }
            }
        }
    }
    unsigned long long m = 0;
#pragma unroll
    for (int s = 0; s < 16; ++s) {
        dv[s] = -1;
        if (s < k && t < T && ((kp[s >> 2] >> ((s & 3) * 8)) & 0xffu)) {
            int e = min(max(ev[s], 0), E - 1);          // memory-safe on garbage indices
            int d = sdev[e];
            dv[s] = (int8_t)d;
            m |= 1ull << d;
        }
    }
    return m;
}

__device__ __forceinline__ unsigned long long warp_or(unsigned long long m)
{
    unsigned lo = __reduce_or_sync(0xffffffffu, (unsigned)m);
    unsigned hi = __reduce_or_sync(0xffffffffu, (unsigned)(m >> 32));
    return ((unsigned long long)hi << 32) | lo;
}

__device__ __forceinline__ void stage_map(uint8_t *sdev, const int32_t *__restrict__ expert_dev, int E, int D)
{
    for (int e = threadIdx.x; e < E; e += blockDim.x) sdev[e] = (uint8_t)min(max(expert_dev[e], 0), D - 1);
}

__global__ void __launch_bounds__(RT)
rows_hist_kernel(const int32_t *__restrict__ idx, const uint8_t *__restrict__ kept, int64_t T, int k, int E,
                 const int32_t *__restrict__ expert_dev, int D, int32_t *bc /*[nb][D]*/, bool vec)
{
    __shared__ uint8_t sdev[1024];
    __shared__ int sh[64];
    stage_map(sdev, expert_dev, E, D);
    if (threadIdx.x < 64) sh[threadIdx.x] = 0;
    __syncthreads();
    int8_t dv[16];
    int64_t t = (int64_t)blockIdx.x * RT + threadIdx.x;
    unsigned long long m = token_mask(idx, kept, sdev, t, T, k, E, dv, vec);
    unsigned long long u = warp_or(m);
    const int lane = threadIdx.x & 31;
    while (u) {
        int d = __ffsll((long long)u) - 1;
        u &= u - 1;
        unsigned bal = __ballot_sync(0xffffffffu, (m >> d) & 1ull);
        if (lane == 0) atomicAdd(&sh[d], __popc(bal));
    }
    __syncthreads();
    if (threadIdx.x < D) bc[(size_t)blockIdx.x * D + threadIdx.x] = sh[threadIdx.x];
}

// block d: exclusive scan of bc[.][d] over the token blocks (in place), total[d]
__global__ void __launch_bounds__(256)
rows_scan_kernel(int32_t *bc, int nb, int D, int32_t *total)
{
    __shared__ int wsum[8];
    __shared__ int carry;
    const int d = blockIdx.x, tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    if (tid == 0) carry = 0;
    __syncthreads();
    for (int base = 0; base < nb; base += 256) {
        int b = base + tid;
        int v = b < nb ? bc[(size_t)b * D + d] : 0;
        int x = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int y = __shfl_up_sync(0xffffffffu, x, o);
            if (lane >= o) x += y;
        }
        if (lane == 31) wsum[wid] = x;
        __syncthreads();
        int wb = 0;
        for (int w = 0; w < wid; ++w) wb += wsum[w];
        int c = carry;
        if (b < nb) bc[(size_t)b * D + d] = c + wb + x - v;
        __syncthreads();
        if (tid == 255) carry = c + wb + x;
        __syncthreads();
    }
    if (tid == 0) total[d] = carry;
}

__global__ void __launch_bounds__(RT)
rows_scatter_kernel(const int32_t *__restrict__ idx, const uint8_t *__restrict__ kept, int64_t T, int k, int E,
                    const int32_t *__restrict__ expert_dev, int D, const int32_t *__restrict__ bc,
                    const int32_t *__restrict__ total, int32_t *rows_token, int32_t *pair_row, int64_t *row_offsets,
                    bool vec)
{
    __shared__ uint8_t sdev[1024];
    __shared__ int wc[RW][64];
    __shared__ int base[64], tot[64];
    stage_map(sdev, expert_dev, E, D);
    for (int q = threadIdx.x; q < RW * 64; q += RT) (&wc[0][0])[q] = 0;
    if (threadIdx.x < D) {
        tot[threadIdx.x] = total[threadIdx.x];
        base[threadIdx.x] = bc[(size_t)blockIdx.x * D + threadIdx.x];
    }
    __syncthreads();
    if (threadIdx.x == 0) {                 // device bases: prefix of the totals (D <= 64)
        long long run = 0;
        for (int d = 0; d < D; ++d) {
            base[d] += (int)run;
            if (blockIdx.x == 0) row_offsets[d] = run;
            run += tot[d];
        }
        if (blockIdx.x == 0) row_offsets[D] = run;
    }
    __syncthreads();
    int8_t dv[16];
    int64_t t = (int64_t)blockIdx.x * RT + threadIdx.x;
    unsigned long long m = token_mask(idx, kept, sdev, t, T, k, E, dv, vec);
    const unsigned long long uw = warp_or(m);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    unsigned long long u = uw;
    while (u) {
        int d = __ffsll((long long)u) - 1;
        u &= u - 1;
        unsigned bal = __ballot_sync(0xffffffffu, (m >> d) & 1ull);
        if (lane == 0) wc[wid][d] = __popc(bal);
    }
    __syncthreads();
    if (threadIdx.x < D) {                  // exclusive prefix over the warps of this block
        int run = 0;
        for (int w = 0; w < RW; ++w) {
            int c = wc[w][threadIdx.x];
            wc[w][threadIdx.x] = run;
            run += c;
        }
    }
    __syncthreads();
    int rowof[16];
#pragma unroll
    for (int s = 0; s < 16; ++s) rowof[s] = -1;
    u = uw;
    while (u) {
        int d = __ffsll((long long)u) - 1;
        u &= u - 1;
        unsigned bal = __ballot_sync(0xffffffffu, (m >> d) & 1ull);
        if ((m >> d) & 1ull) {
            int row = base[d] + wc[wid][d] + __popc(bal & ((1u << lane) - 1u));
            rows_token[row] = (int32_t)t;
#pragma unroll
            for (int s = 0; s < 16; ++s)
                if (dv[s] == d) rowof[s] = row;
        }
    }
    if (pair_row && t < T) {
        if (vec && (reinterpret_cast<uintptr_t>(pair_row) & 15) == 0) {
            int4 *o4 = reinterpret_cast<int4 *>(pair_row + t * k);
#pragma unroll
            for (int q = 0; q < 4; ++q)
                if (q * 4 < k) o4[q] = make_int4(rowof[4 * q], rowof[4 * q + 1], rowof[4 * q + 2], rowof[4 * q + 3]);
        } else {
#pragma unroll
            for (int s = 0; s < 16; ++s)
                if (s < k) pair_row[t * k + s] = rowof[s];
        }
    }
}

}  // namespace

size_t dispatch_rows_ws_bytes(int64_t T, int32_t D)
{
    size_t nb = (size_t)((T + RT - 1) / RT);
    return (nb * D + 64) * sizeof(int32_t) + 256;
}

}  // namespace cap

extern "C" int cap_dispatch_rows(const int32_t *topk_idx, const uint8_t *kept, int64_t T, int32_t k, int32_t E,
                                 const int32_t *expert_dev, int32_t D, int32_t *rows_token, int32_t *pair_row,
                                 int64_t *row_offsets, void *ws, size_t ws_bytes, void *stream)
{
    using namespace cap;
    if (T < 0 || E < 1 || E > 1024 || k < 1 || k > 16 || k > E || D < 1 || D > 64) return CAP_EINVAL;
    if (T * k >= ((int64_t)1 << 31)) return CAP_EINVAL;
    if (!expert_dev || !row_offsets) return CAP_EINVAL;
    if (T > 0 && (!topk_idx || !rows_token)) return CAP_EINVAL;
    if (!ws || ws_bytes < dispatch_rows_ws_bytes(T, D)) return CAP_EWORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    int nb = (int)((T + RT - 1) / RT);
    const bool vec = (k & 3) == 0 && ((uintptr_t)topk_idx & 15) == 0 && ((uintptr_t)kept & 3) == 0;
    int32_t *bc = (int32_t *)(((uintptr_t)ws + 255) & ~(uintptr_t)255);
    int32_t *total = bc + (size_t)nb * D;
    if (nb > 0) {
        KernelTimerScope kt("rows_hist", st);
        rows_hist_kernel<<<nb, RT, 0, st>>>(topk_idx, kept, T, k, E, expert_dev, D, bc, vec);
        note_launch();
        CAP_TRY(check_launch("rows_hist_kernel"));
    }
    {
        KernelTimerScope kt("rows_scan", st);
        rows_scan_kernel<<<D, 256, 0, st>>>(bc, nb, D, total);
        note_launch();
        CAP_TRY(check_launch("rows_scan_kernel"));
    }
    {
        KernelTimerScope kt("rows_scatter", st);
        // one block at least, so that the offsets are written for T = 0
        rows_scatter_kernel<<<nb > 0 ? nb : 1, RT, 0, st>>>(topk_idx, kept, T, k, E, expert_dev, D, bc, total,
                                                          rows_token, pair_row, row_offsets, vec);
        note_launch();
        CAP_TRY(check_launch("rows_scatter_kernel"));
    }
    return CAP_OK;
}

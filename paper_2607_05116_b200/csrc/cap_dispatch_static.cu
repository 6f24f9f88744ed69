// cap_dispatch_layout_static: S5 (dispatch layout; BASELINE.json stage 5) for callers that cannot
// allocate -- code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  Same
// three kernels as cap_dispatch_layout (cap_dispatch.cu: warp-private histogram, ordered scan, stable
// scatter); the only difference is where their scratch lives: not in a caller workspace but in ONE
// file-scope device array of CAP_STATIC_SCRATCH_BYTES, which every GPU that loads the library holds
// until the process exits.
//
// The array's name is a host-side stand-in in host code, not a device address: its address on the
// current device is resolved once per device with cudaGetSymbolAddress (checked) and that pointer is
// what the kernels receive.  This entry point calls no cudaMalloc / cudaFree and no allocating routine.
//
// Sharing: every call on a device uses the same array, and the array keeps the last call's contents.
// Nothing has to start at zero -- each call writes every hist / base entry it later reads (sub-chunks
// past the end of the pair stream write zeros; dispatch_hist_kernel, dispatch_scan_kernel) -- but two
// calls that OVERLAP on one GPU (different streams, or concurrent graph branches) race on it: callers
// must order them (same stream, or an event between them).
#include <mutex>

#include "cap_internal.cuh"

namespace cap {

static __device__ __align__(256) unsigned char g_dispatch_scratch[CAP_STATIC_SCRATCH_BYTES];

constexpr int SS_MAXDEV = 64;
static void *g_scratch_ptr[SS_MAXDEV];      // device address of g_dispatch_scratch, per device ordinal
static std::mutex g_scratch_mu;

// address of the scratch array on the CURRENT device (resolved on first use, with that device current)
static int static_scratch(void **out)
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) return check_launch("cudaGetDevice");
    if (dev < 0 || dev >= SS_MAXDEV) return CAP_EINVAL;
    std::lock_guard<std::mutex> lock(g_scratch_mu);
    if (!g_scratch_ptr[dev]) {
        void *p = nullptr;
        if (cudaGetSymbolAddress(&p, g_dispatch_scratch) != cudaSuccess || !p) return check_launch("cudaGetSymbolAddress");
        g_scratch_ptr[dev] = p;
    }
    *out = g_scratch_ptr[dev];
    return CAP_OK;
}

}  // namespace cap

using namespace cap;

extern "C" {

size_t cap_static_scratch_bytes(void) { return (size_t)CAP_STATIC_SCRATCH_BYTES; }

int cap_dispatch_layout_static(const int32_t *topk_idx, const uint8_t *kept, int64_t T, int32_t k, int32_t E,
                               const int32_t *expert_dev, int32_t D, int32_t *sorted_pairs, int32_t *pair_pos,
                               int64_t *offsets, void *stream)
{
    // the argument rules of cap_dispatch_layout (cap_api.cu)
    if (T < 0 || E < 1 || E > 1024 || k < 1 || k > 16 || k > E || D < 1 || D > 64 || !offsets || !expert_dev)
        return CAP_EINVAL;
    if (T * k >= ((int64_t)1 << 31)) return CAP_EINVAL;
    if (T > 0 && (!topk_idx || !sorted_pairs)) return CAP_EINVAL;
    // sizes beyond the static array are refused, never truncated
    if (T > 0 && dispatch_ws_bytes(T, k, D) > (size_t)CAP_STATIC_SCRATCH_BYTES) return CAP_EWORKSPACE;
    void *ws = nullptr;
    CAP_TRY(static_scratch(&ws));
    return launch_dispatch(topk_idx, kept, T, k, E, expert_dev, D, sorted_pairs, pair_pos, offsets, ws,
                           (cudaStream_t)stream);
}

}  // extern "C"

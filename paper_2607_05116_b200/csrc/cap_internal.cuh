// Internal declarations shared by the CUDA translation units of libcap_b200.so.
// Nothing here is shared with oracle/ (the CPU oracle is an independent restatement).
#pragma once
#include <cstdlib>
#include <cuda_runtime.h>
#include <stdint.h>

#include "cap.h"

namespace cap {

// ---- host-side launch bookkeeping -------------------------------------------------------
void note_launch(int n = 1);            // counts kernels launched (cap_launch_count)
int check_launch(const char *what);     // cudaGetLastError -> CAP_OK / CAP_ECUDA (records it)
int sm_count();                         // SMs of the current device (cached)

// Optional profiling aid (cap_kernel_timer_arm): records a cudaEvent pair around the next launch
// of the kernel with the armed tag.  Costs one table scan per launch when nothing is armed.
struct KernelTimerScope {
    KernelTimerScope(const char *tag, cudaStream_t st);
    ~KernelTimerScope();
    int slot_;
    cudaStream_t st_;
};

// ---- programmatic dependent launch (PDL) ---------------------------------------------------
// The stages of a step are short kernels that follow each other on one stream; launched with the
// programmatic-serialization attribute, kernel n+1 is scheduled while kernel n still runs and blocks
// in pdl_wait() until kernel n has completed and flushed its memory (so the dependency is exactly the
// stream order; only launch latency, block scheduling and the smem-only prologue overlap).  EVERY
// kernel launched through launch_pdl() must execute pdl_wait() before its first global access.
// Inside a stream capture the attribute is left out: measured on B200, programmatic edges made the
// graph replay of a step slower (dispatch 18.5 -> 25.5 us), while directly launched kernels gain
// (fused kernel back to back 33.2 -> 30.0 us).
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st,
                              Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    cudaStreamIsCapturing(st, &cs);
    cfg.attrs = at;
    cfg.numAttrs = cs == cudaStreamCaptureStatusNone ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}

// Blocks per unit (layer, candidate chunk) of a grid whose blocks all do the same work on `slots` concurrently
// resident blocks: the kernel lasts ceil(units * w / slots) block-times of 1 / w of a unit each, so minimise
// ceil(units * w / slots) / w (58 layers x 3 = 174 blocks on 148 SMs is two block-times; x 5 = 290 is two block-times
// of blocks 3/5 the size).  A small per-block term keeps the count low where it does not matter.
inline int64_t balanced_blocks_per_unit(int64_t units, int64_t slots, int64_t max_w)
{
    if (units < 1) units = 1;
    if (max_w > slots) max_w = slots;
    int64_t best_w = 1;
    double best = 1e300;
    for (int64_t w = 1; w <= max_w; ++w) {
        const int64_t waves = (units * w + slots - 1) / slots;
        const double cost = (double)waves / (double)w * (1.0 + 0.002 * (double)w);
        if (cost < best - 1e-12) {
            best = cost;
            best_w = w;
        }
    }
    return best_w;
}

// The same launch with the programmatic edge kept INSIDE a stream capture as well.  Only for a kernel whose early
// part is independent of its predecessor's output and that calls pdl_wait() exactly where it first consumes it
// (trace_fused_kernel after eval_table_kernel): there the overlap pays; on the chains of short kernels it did not.
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl_edge(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st,
                                   Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}

#define CAP_TRY(expr)                      \
    do {                                   \
        int _rc = (expr);                  \
        if (_rc != CAP_OK) return _rc;     \
    } while (0)

// ---- accumulator slots of the evaluation (ws, int64 per (layer, candidate)) --------------
enum { ACC_DEV = 0, ACC_LOCAL = 1, ACC_SAMENODE = 2, ACC_NODE = 3, ACC_RNODE = 4, ACC_NEAR = 5, ACC_TICKET = 6, ACC_N = 8 };

struct EvalWs {
    unsigned long long *acc;      // [L][P][ACC_N]
    unsigned long long *recv;     // [L][P][D]
    unsigned long long *mcounts;  // [L][E] kept pairs per expert (when the caller gave none)
    unsigned long long *ldirect;  // [L][64] kept pairs per device, counted directly (cap_prune, P = 1)
};

size_t eval_ws_bytes(int32_t L, int64_t T, int32_t E, int32_t k, int32_t D, int32_t P);
EvalWs eval_ws_carve(void *ws, int32_t L, int32_t E, int32_t D, int32_t P);

// ---- stage launchers (arguments already validated) ---------------------------------------
int launch_gate_topk(const float *logits, const float *bias, int32_t L, int64_t T,
                     const cap_gate_cfg &cfg, int32_t *idx, float *w, cudaStream_t st);
// S1 fast path (cap_gate_fast.cu): *used = false when the configuration does not fit it
int launch_gate_fast(const float *logits, const float *bias, int32_t L, int64_t T,
                     const cap_gate_cfg &cfg, int32_t *idx, float *w, cudaStream_t st, bool *used);
// S1 fast path for sigmoid (+ bias, + groups of 32) scoring (cap_gate_sig.cu): *used = false when it does not apply
int launch_gate_sig(const float *logits, const float *bias, int32_t L, int64_t T, const cap_gate_cfg &cfg,
                    int32_t *idx, float *w, cudaStream_t st, bool *used);
// S1 fast path for E = 512, k <= 10, softmax + renormalisation (cap_gate_wide.cu): *used = false when it does not apply
int launch_gate_wide(const float *logits, const float *bias, int32_t L, int64_t T, const cap_gate_cfg &cfg,
                     int32_t *idx, float *w, cudaStream_t st, bool *used);
// S2 fast path (cap_coact_mma.cu): tcgen05 int8 A^T A; outputs must be zeroed by the caller
int launch_coact_mma(const int32_t *idx, const uint8_t *kept, int32_t L, int64_t T, int32_t k, int32_t E,
                     int64_t *counts, int32_t *coact, cudaStream_t st, bool *used);
int launch_coactivation(const int32_t *idx, const uint8_t *kept, int32_t L, int64_t T, int32_t k,
                        int32_t E, int64_t *counts, int32_t *coact, cudaStream_t st);
int launch_eval(const int32_t *idx, const uint8_t *kept, const int32_t *token_src, int32_t L,
                int64_t T, int32_t k, int32_t E, const int32_t *expert_dev, int32_t P,
                int64_t layer_stride_maps, const cap_topology &topo, const int64_t *counts,
                const cap_eval_out &out, void *ws, cudaStream_t st);
int launch_eval_finalize(int32_t L, int32_t E, int32_t P, const int32_t *expert_dev, const cap_topology &topo,
                         const int64_t *counts, const cap_eval_out &out, void *ws, cudaStream_t st,
                         int64_t *near_out = nullptr);
int eval_zero_ws(int32_t L, int32_t E, int32_t D, int32_t P, bool with_mcounts, void *ws, cudaStream_t st);
// fused S1+S2+S3 kernel (cap_fused.cu): *used = false when the configuration does not fit it
int launch_trace_fused_fast(const float *logits, const float *bias, int32_t L, int64_t T, const cap_gate_cfg &cfg,
                            int32_t *idx, float *w, int64_t *counts, int32_t *coact, const int32_t *token_src,
                            const int32_t *expert_dev, int32_t P, const cap_topology &topo,
                            const cap_eval_out &out, void *ws, cudaStream_t st, bool *used);
int profile_trace_fused_kernel(const float *const *logits_list, int nlist, int nrep, float *avg_ms, int32_t L,
                               int64_t T, const cap_gate_cfg &cfg, int32_t *idx, float *w, int64_t *counts,
                               int32_t *coact, const int32_t *expert_dev, int32_t P, const cap_topology &topo,
                               const cap_eval_out &out, void *ws, cudaStream_t st, bool *used);
size_t fused_ws_bytes(int32_t L, int64_t T, int32_t k, int32_t E, int32_t D, int32_t P);
// single-launch fused kernel (cap_fused2.cu): *used = false when the configuration does not fit it;
// ws_f2 = the fast-path region of the evaluation workspace (eval_fast_region)
int launch_trace_fused2(const float *logits, const float *bias, int32_t L, int64_t T, const cap_gate_cfg &cfg,
                        int32_t *idx, float *w, int64_t *counts, int32_t *coact, const int32_t *token_src,
                        const int32_t *expert_dev, int32_t P, const cap_topology &topo, const cap_eval_out &out,
                        void *ws_f2, cudaStream_t st, bool *used);
size_t fused2_ws_bytes(int32_t L, int64_t T, int32_t k, int32_t E, int32_t D, int32_t P);
bool fused2_plan(int32_t L, int64_t T, const cap_gate_cfg &cfg, int32_t D, int32_t N, int32_t P, int64_t *plan);
void *eval_fast_region(void *ws, int32_t L, int32_t E, int32_t D, int32_t P);
bool fused_plan(int32_t L, int64_t T, const cap_gate_cfg &cfg, int32_t D, int32_t N, int32_t P, int64_t *plan);
int launch_prune(const int32_t *idx, const float *w, const int32_t *token_src, int32_t L,
                 int64_t T, int32_t k, int32_t E, const int32_t *expert_dev,
                 const cap_topology &topo, float p, uint8_t *kept, int64_t *near_margin,
                 const cap_eval_out *after, void *ws, cudaStream_t st);
// S3 fast path (cap_eval_fast.cu): *used = false when the sizes do not fit it
// (decodes and finishes the outputs itself: no launch_eval_finalize after it)
// cap_prune_dispatch (S4 + S5 in three launches): the S4 kernel leaves, per block, PD_PART 32-bit partial sums
// (ACC_N evaluation accumulators, then tokens received per device) and, per warp of 32 tokens, the kept pairs per
// device in the histogram rows of S5; the S5 scan / scatter kernels carry one extra block each that adds the
// partials up and writes the after-metrics.
constexpr int PD_PART = ACC_N + 64;
constexpr int PD_MAXRB = 64;
struct DsReduce {
    const uint32_t *part;            // [L][nblk][PD_PART] or NULL
    unsigned long long *red;         // [L][nrb][PD_PART]: sums of nrb slices of the blocks (scan kernel -> scatter kernel)
    unsigned long long *acc, *recv;  // [L][ACC_N], [L][D]: the totals (written and read by the finishing block)
    int64_t nblk;
    int32_t nrb, per_rb;             // reduce blocks per layer, S4 blocks per reduce block
};
struct FinalParams;
int64_t dispatch_stride_subs(int64_t nsub);
int launch_dispatch_tail(const int32_t *idx, const uint8_t *kept, int32_t L, int64_t n, int32_t E,
                         const int32_t *expert_dev, int32_t D, int32_t *sorted_pairs, int32_t *pair_pos,
                         int64_t *offsets, int *hist, int64_t stride, int rounds, const DsReduce &rd,
                         const FinalParams *fin, cudaStream_t st);
size_t prune_dispatch_ws_bytes(int32_t L, int64_t T, int32_t k, int32_t E, int32_t D);
int launch_prune_dispatch(const int32_t *idx, const float *w, const int32_t *token_src, int32_t L, int64_t T,
                          int32_t k, int32_t E, const int32_t *expert_dev, const cap_topology &topo, float p,
                          uint8_t *kept, int64_t *near_margin, const cap_eval_out *after, int32_t *sorted_pairs,
                          int32_t *pair_pos, int64_t *offsets, void *ws, cudaStream_t st);
// deferred decode of the bit-sliced S3 path (cap_trace_fused_begin / _finish; cap_eval_fast.cu): while parking is on
// for this host thread, the decode launch is stored instead of issued
void ef_decode_park(bool on);
bool ef_decode_take(void *blob, size_t cap);
int ef_decode_launch_parked(const void *blob, cudaStream_t st);
int launch_eval_fast(const int32_t *idx, const uint8_t *kept, int32_t L, int64_t T, int32_t k,
                     int32_t E, const int32_t *expert_dev, int32_t P, const cap_topology &topo,
                     const int64_t *counts, const cap_eval_out &out, void *ws, cudaStream_t st, bool *used,
                     const int32_t *token_src = nullptr);
size_t eval_fast_ws_bytes(int32_t L, int64_t T, int32_t k, int32_t E, int32_t D, int32_t P);
size_t dispatch_ws_bytes(int64_t T, int32_t k, int32_t D);
size_t dispatch_ws_bytes_batched(int32_t L, int64_t T, int32_t k, int32_t D);
int launch_dispatch_batched(const int32_t *idx, const uint8_t *kept, int32_t L, int64_t T, int32_t k, int32_t E,
                            const int32_t *expert_dev, int32_t D, int32_t *sorted_pairs, int32_t *pair_pos,
                            int64_t *offsets, void *ws, cudaStream_t st);
size_t place_ws_bytes(int32_t L, int32_t E, int32_t D);   // cap_place.cu
size_t dispatch_rows_ws_bytes(int64_t T, int32_t D);        // cap_dispatch_rows.cu
int launch_dispatch(const int32_t *idx, const uint8_t *kept, int64_t T, int32_t k, int32_t E,
                    const int32_t *expert_dev, int32_t D, int32_t *sorted_pairs, int32_t *pair_pos,
                    int64_t *offsets, void *ws, cudaStream_t st);

// ---- device helpers ------------------------------------------------------------------------
// Reproducible fp32 exponential (DESIGN.md R-S1.3): IEEE-exact operations only.
__device__ __forceinline__ float exp_s(float x)
{
    float t = fminf(fmaxf(x, -87.0f), 87.0f);
    float n = rintf(__fmul_rn(t, 0x1.715476p+0f));
    float r = __fmaf_rn(n, -0x1.62ep-1f, t);
    r = __fmaf_rn(n, -0x1.0bfbe8p-15f, r);
    float p = 0x1.a01a02p-13f;
    p = __fmaf_rn(p, r, 0x1.6c16c2p-10f);
    p = __fmaf_rn(p, r, 0x1.111112p-7f);
    p = __fmaf_rn(p, r, 0x1.555556p-5f);
    p = __fmaf_rn(p, r, 0x1.555556p-3f);
    p = __fmaf_rn(p, r, 0x1p-1f);
    p = __fmaf_rn(p, r, 1.0f);
    p = __fmaf_rn(p, r, 1.0f);
    int ni = __float2int_rn(n);
    return __fmul_rn(p, __int_as_float((ni + 127) << 23));
}

__device__ __forceinline__ float sig_s(float x)
{
    return __fdiv_rn(1.0f, __fadd_rn(1.0f, exp_s(-x)));
}

// Order-preserving map fp32 -> u32 (larger float <=> larger key); -0 is folded onto +0 so that
// the two compare equal as IEEE says.  Every finite float gets a key > 0: key 0 means "absent".
__device__ __forceinline__ uint32_t okey(float x)
{
    uint32_t b = __float_as_uint(x);
    if (b == 0x80000000u) b = 0u;
    return b ^ ((uint32_t)((int32_t)b >> 31) | 0x80000000u);
}

__device__ __forceinline__ float unkey(uint32_t key)
{
    uint32_t b = (key & 0x80000000u) ? (key ^ 0x80000000u) : ~key;
    return __uint_as_float(b);
}

}  // namespace cap

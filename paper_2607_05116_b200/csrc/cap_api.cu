// C ABI of libcap_b200.so (declared in include/cap.h): host-side argument checks, workspace
// carving and kernel launches.  No allocation, no synchronisation (cap_validate_placements
// excepted), no global state beyond the launch counter and the per-thread last CUDA error.
#include <atomic>
#include <cstdio>
#include <cstdlib>
#include <cstring>

#include "cap_internal.cuh"

namespace cap {

static std::atomic<long long> g_launches{0};
static thread_local int tl_last_err = 0;

void note_launch(int n) { g_launches.fetch_add(n, std::memory_order_relaxed); }

int check_launch(const char *what)
{
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        if (getenv("CAP_DEBUG")) fprintf(stderr, "cap: %s: %s\n", what ? what : "?", cudaGetErrorString(e));
        tl_last_err = (int)e;
        return CAP_ECUDA;
    }
    return CAP_OK;
}

int sm_count()
{
    // SMs of the CURRENT device, cached per device ordinal (grid and workspace geometry depend on it)
    static std::atomic<int> cache[64];
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return 148;
    int n = cache[dev].load(std::memory_order_relaxed);
    if (n == 0) {
        if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) n = 148;
        cache[dev].store(n, std::memory_order_relaxed);
    }
    return n;
}

// ---- kernel timer table -------------------------------------------------------------------
constexpr int KT_SLOTS = 4096;
constexpr int KT_ARMED = 128;
struct KtSlot { cudaEvent_t a = nullptr, b = nullptr; int state = 0; };   // state 2 = both recorded
struct KtArm { char tag[32]; int slot; bool on; };
static KtSlot g_kt[KT_SLOTS];
static KtArm g_arm[KT_ARMED];
static std::atomic<int> g_armed{0};

KernelTimerScope::KernelTimerScope(const char *tag, cudaStream_t st) : slot_(-1), st_(st)
{
    if (g_armed.load(std::memory_order_relaxed) == 0) return;
    for (int i = 0; i < KT_ARMED; ++i) {
        if (g_arm[i].on && strcmp(g_arm[i].tag, tag) == 0) {
            slot_ = g_arm[i].slot;
            g_arm[i].on = false;
            g_armed.fetch_sub(1);
            cudaEventRecord(g_kt[slot_].a, st_);
            g_kt[slot_].state = 1;
            return;
        }
    }
}

KernelTimerScope::~KernelTimerScope()
{
    if (slot_ >= 0) {
        cudaEventRecord(g_kt[slot_].b, st_);
        g_kt[slot_].state = 2;
    }
}

static bool sizes_ok(int32_t L, int64_t T, int32_t E, int32_t k)
{
    if (L < 0 || T < 0 || E < 1 || E > 1024 || k < 1 || k > 16 || k > E) return false;
    if (T * k >= ((int64_t)1 << 31)) return false;
    if (L > 65535) return false;
    if ((double)L * (double)T * (double)k >= 1099511627776.0) return false;
    return true;
}

static bool topo_ok(const cap_topology *t)
{
    return t && t->D >= 1 && t->D <= 64 && t->N >= 1 && t->N <= 64 && t->dev_node != nullptr &&
           t->cost_local >= 0 && t->cost_intra >= 0 && t->cost_inter >= 0 && t->bytes_per_token >= 0;
}

static bool gate_ok(const cap_gate_cfg *c)
{
    if (!c) return false;
    if (c->E < 1 || c->E > 1024 || c->k < 1 || c->k > 16 || c->k > c->E) return false;
    if (c->scoring != 0 && c->scoring != 1) return false;
    if (c->n_group < 1 || c->n_group > 32 || c->E % c->n_group != 0) return false;
    if (c->n_group > 1) {
        if (c->topk_group < 1 || c->topk_group > c->n_group) return false;
        if ((int64_t)c->k > (int64_t)c->topk_group * (c->E / c->n_group)) return false;
        if (c->group_score != 0 && c->group_score != 1) return false;
        if (c->group_score == 1 && c->E / c->n_group < 2) return false;
    }
    return true;
}

__global__ void validate_maps_kernel(const int32_t *maps, long long n, int D, int *bad)
{
    long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long stride = (long long)gridDim.x * blockDim.x;
    int b = 0;
    for (; i < n; i += stride) b |= (maps[i] < 0 || maps[i] >= D);
    if (b) atomicOr(bad, 1);
}

}  // namespace cap

using namespace cap;

extern "C" {

int cap_kernel_timer_arm(const char *tag, int slot)
{
    if (!tag || slot < 0 || slot >= KT_SLOTS || strlen(tag) >= sizeof(g_arm[0].tag)) return CAP_EINVAL;
    if (!g_kt[slot].a) {
        if (cudaEventCreate(&g_kt[slot].a) != cudaSuccess || cudaEventCreate(&g_kt[slot].b) != cudaSuccess)
            return check_launch("event create");
    }
    g_kt[slot].state = 0;
    for (int i = 0; i < KT_ARMED; ++i)
        if (g_arm[i].on && g_arm[i].slot == slot && strcmp(g_arm[i].tag, tag) == 0) return CAP_OK;
    for (int i = 0; i < KT_ARMED; ++i) {
        if (!g_arm[i].on) {
            strcpy(g_arm[i].tag, tag);
            g_arm[i].slot = slot;
            g_arm[i].on = true;
            g_armed.fetch_add(1);
            return CAP_OK;
        }
    }
    return CAP_EINVAL;
}

float cap_kernel_timer_ms(int slot)
{
    if (slot < 0 || slot >= KT_SLOTS || g_kt[slot].state != 2) return -1.0f;
    float ms = -1.0f;
    if (cudaEventElapsedTime(&ms, g_kt[slot].a, g_kt[slot].b) != cudaSuccess) {
        cudaGetLastError();
        return -1.0f;
    }
    return ms;
}

const char *cap_version(void) { return "cap-b200 0.1 (sm_100a)"; }
int cap_last_cuda_error(void) { return tl_last_err; }
int64_t cap_launch_count(void) { return (int64_t)g_launches.load(); }

size_t cap_workspace_bytes(int which_call, int32_t L, int64_t T, int32_t E, int32_t k, int32_t D,
                           int32_t P)
{
    if (L < 0 || T < 0 || E < 1 || k < 1) return 0;
    switch (which_call) {
    case CAP_CALL_GATE_TOPK:
    case CAP_CALL_COACTIVATION:
        return 256;
    case CAP_CALL_EVAL_PLACEMENTS:
    case CAP_CALL_TRACE_FUSED:
        if (D < 1 || P < 0) return 0;
        return eval_ws_bytes(L, T, E, k, D, P);
    case CAP_CALL_PRUNE:
        if (D < 1) return 0;
        return eval_ws_bytes(L, T, E, k, D, 1);
    case CAP_CALL_DISPATCH_LAYOUT:
        if (D < 1) return 0;
        return L > 1 ? dispatch_ws_bytes_batched(L, T, k, D) : dispatch_ws_bytes(T, k, D);   // L > 1: the batched call
    case CAP_CALL_DISPATCH_ROWS:
        if (D < 1) return 0;
        return dispatch_rows_ws_bytes(T, D);
    case CAP_CALL_PRUNE_DISPATCH:
        if (D < 1) return 0;
        return prune_dispatch_ws_bytes(L, T, k, E, D);
    case CAP_CALL_COACT_PLACEMENT:
        if (D < 1) return 0;
        return place_ws_bytes(L, E, D);
    default:
        return 0;
    }
}

int cap_gate_topk(const float *logits, const float *bias, int32_t L, int64_t T,
                  const cap_gate_cfg *cfg, int32_t *topk_idx, float *topk_w, void *, size_t,
                  void *stream)
{
    if (!gate_ok(cfg) || !sizes_ok(L, T, cfg->E, cfg->k)) return CAP_EINVAL;
    if (cfg->scoring == 0 && bias != nullptr) return CAP_EINVAL;
    if ((int64_t)L * T > 0 && (!logits || !topk_idx || !topk_w)) return CAP_EINVAL;
    return launch_gate_topk(logits, bias, L, T, *cfg, topk_idx, topk_w, (cudaStream_t)stream);
}

int cap_coactivation(const int32_t *topk_idx, const uint8_t *kept, int32_t L, int64_t T, int32_t k,
                     int32_t E, int64_t *counts, int32_t *coact, void *, size_t, void *stream)
{
    if (!sizes_ok(L, T, E, k)) return CAP_EINVAL;
    if (L > 0 && (!counts || !coact)) return CAP_EINVAL;
    if ((int64_t)L * T > 0 && !topk_idx) return CAP_EINVAL;
    return launch_coactivation(topk_idx, kept, L, T, k, E, counts, coact, (cudaStream_t)stream);
}

int cap_eval_placements(const int32_t *topk_idx, const uint8_t *kept, const int32_t *token_src,
                        int32_t L, int64_t T, int32_t k, int32_t E, const int32_t *expert_dev,
                        int32_t P, const cap_topology *topo, const int64_t *counts,
                        const cap_eval_out *out, void *ws, size_t ws_bytes, void *stream)
{
    if (!sizes_ok(L, T, E, k) || !topo_ok(topo) || P < 0 || !out) return CAP_EINVAL;
    if ((int64_t)L * P > 0 && !expert_dev) return CAP_EINVAL;
    if ((int64_t)L * T > 0 && !topk_idx) return CAP_EINVAL;
    if ((int64_t)L * P >= ((int64_t)1 << 31)) return CAP_EINVAL;
    if (!ws || ws_bytes < eval_ws_bytes(L, T, E, k, topo->D, P)) return CAP_EWORKSPACE;
    return launch_eval(topk_idx, kept, token_src, L, T, k, E, expert_dev, P, (int64_t)P * E, *topo,
                       counts, *out, ws, (cudaStream_t)stream);
}

int cap_prune(const int32_t *topk_idx, const float *topk_w, const int32_t *token_src, int32_t L,
              int64_t T, int32_t k, int32_t E, const int32_t *expert_dev, const cap_topology *topo,
              float p, uint8_t *kept, const cap_eval_out *after, int64_t *near_margin, void *ws,
              size_t ws_bytes, void *stream)
{
    if (!sizes_ok(L, T, E, k) || !topo_ok(topo)) return CAP_EINVAL;
    if (!(p < 1.0f)) return CAP_EINVAL;   // also rejects NaN
    if (L > 0 && !expert_dev) return CAP_EINVAL;
    if ((int64_t)L * T > 0 && (!topk_idx || !topk_w || !kept)) return CAP_EINVAL;
    if (after && (!ws || ws_bytes < eval_ws_bytes(L, T, E, k, topo->D, 1))) return CAP_EWORKSPACE;
    return launch_prune(topk_idx, topk_w, token_src, L, T, k, E, expert_dev, *topo, p, kept, near_margin, after,
                        ws, (cudaStream_t)stream);
}

int cap_prune_dispatch(const int32_t *topk_idx, const float *topk_w, const int32_t *token_src, int32_t L,
                       int64_t T, int32_t k, int32_t E, const int32_t *expert_dev, const cap_topology *topo,
                       float p, uint8_t *kept, const cap_eval_out *after, int64_t *near_margin,
                       int32_t *sorted_pairs, int32_t *pair_pos, int64_t *offsets, void *ws, size_t ws_bytes,
                       void *stream)
{
    if (!sizes_ok(L, T, E, k) || !topo_ok(topo)) return CAP_EINVAL;
    if (!(p < 1.0f)) return CAP_EINVAL;   // also rejects NaN
    if (L > 0 && (!expert_dev || !offsets)) return CAP_EINVAL;
    if ((int64_t)L * T > 0 && (!topk_idx || !topk_w || !kept || !sorted_pairs)) return CAP_EINVAL;
    if (L > 0 && (!ws || ws_bytes < prune_dispatch_ws_bytes(L, T, k, E, topo->D))) return CAP_EWORKSPACE;
    return launch_prune_dispatch(topk_idx, topk_w, token_src, L, T, k, E, expert_dev, *topo, p, kept, near_margin,
                                 after, sorted_pairs, pair_pos, offsets, ws, (cudaStream_t)stream);
}

int cap_dispatch_layout(const int32_t *topk_idx, const uint8_t *kept, int64_t T, int32_t k,
                        int32_t E, const int32_t *expert_dev, int32_t D, int32_t *sorted_pairs,
                        int32_t *pair_pos, int64_t *offsets, void *ws, size_t ws_bytes, void *stream)
{
    if (!sizes_ok(1, T, E, k) || D < 1 || D > 64 || !offsets || !expert_dev) return CAP_EINVAL;
    if (T > 0 && (!topk_idx || !sorted_pairs)) return CAP_EINVAL;
    if (T > 0 && (!ws || ws_bytes < dispatch_ws_bytes(T, k, D))) return CAP_EWORKSPACE;
    return launch_dispatch(topk_idx, kept, T, k, E, expert_dev, D, sorted_pairs, pair_pos, offsets, ws,
                           (cudaStream_t)stream);
}

int cap_dispatch_layout_batched(const int32_t *topk_idx, const uint8_t *kept, int32_t L, int64_t T, int32_t k,
                                int32_t E, const int32_t *expert_dev, int32_t D, int32_t *sorted_pairs,
                                int32_t *pair_pos, int64_t *offsets, void *ws, size_t ws_bytes, void *stream)
{
    if (!sizes_ok(L, T, E, k) || D < 1 || D > 64) return CAP_EINVAL;
    if (L > 0 && (!offsets || !expert_dev)) return CAP_EINVAL;
    if ((int64_t)L * T > 0 && (!topk_idx || !sorted_pairs)) return CAP_EINVAL;
    if ((int64_t)L * T > 0 && (!ws || ws_bytes < dispatch_ws_bytes_batched(L, T, k, D))) return CAP_EWORKSPACE;
    return launch_dispatch_batched(topk_idx, kept, L, T, k, E, expert_dev, D, sorted_pairs, pair_pos, offsets, ws,
                                   (cudaStream_t)stream);
}

int cap_trace_fused(const float *logits, const float *bias, int32_t L, int64_t T,
                    const cap_gate_cfg *cfg, int32_t *topk_idx, float *topk_w, int64_t *counts,
                    int32_t *coact, const int32_t *token_src, const int32_t *expert_dev, int32_t P,
                    const cap_topology *topo, const cap_eval_out *out, void *ws, size_t ws_bytes,
                    void *stream)
{
    if (!gate_ok(cfg) || !sizes_ok(L, T, cfg->E, cfg->k) || !topo_ok(topo) || P < 0 || !out)
        return CAP_EINVAL;
    if (cfg->scoring == 0 && bias != nullptr) return CAP_EINVAL;
    if ((int64_t)L * T > 0 && (!logits || !topk_idx || !topk_w)) return CAP_EINVAL;
    if (L > 0 && (!counts || !coact)) return CAP_EINVAL;
    if ((int64_t)L * P > 0 && !expert_dev) return CAP_EINVAL;
    if ((int64_t)L * P >= ((int64_t)1 << 31)) return CAP_EINVAL;
    if (!ws || ws_bytes < eval_ws_bytes(L, T, cfg->E, cfg->k, topo->D, P)) return CAP_EWORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    if (L == 0) return CAP_OK;
    bool fused = false;
    CAP_TRY(launch_trace_fused_fast(logits, bias, L, T, *cfg, topk_idx, topk_w, counts, coact, token_src,
                                    expert_dev, P, *topo, *out, ws, st, &fused));
    if (fused) return CAP_OK;
    CAP_TRY(launch_gate_topk(logits, bias, L, T, *cfg, topk_idx, topk_w, st));
    CAP_TRY(launch_coactivation(topk_idx, nullptr, L, T, cfg->k, cfg->E, counts, coact, st));
    return launch_eval(topk_idx, nullptr, token_src, L, T, cfg->k, cfg->E, expert_dev, P,
                       (int64_t)P * cfg->E, *topo, counts, *out, ws, st);
}

int cap_trace_fused_begin(const float *logits, const float *bias, int32_t L, int64_t T,
                          const cap_gate_cfg *cfg, int32_t *topk_idx, float *topk_w, int64_t *counts,
                          int32_t *coact, const int32_t *token_src, const int32_t *expert_dev, int32_t P,
                          const cap_topology *topo, const cap_eval_out *out, void *ws, size_t ws_bytes,
                          cap_pending *pend, void *stream)
{
    if (!pend) return CAP_EINVAL;
    memset(pend, 0, sizeof(*pend));
    ef_decode_park(true);
    const int rc = cap_trace_fused(logits, bias, L, T, cfg, topk_idx, topk_w, counts, coact, token_src, expert_dev, P,
                                   topo, out, ws, ws_bytes, stream);
    if (rc == CAP_OK && ef_decode_take(pend->blob, sizeof(pend->blob))) pend->kind = 1;
    ef_decode_park(false);
    return rc;
}

int cap_trace_fused_finish(const cap_pending *pend, void *stream)
{
    if (!pend) return CAP_EINVAL;
    if (pend->kind == 0) return CAP_OK;
    if (pend->kind != 1) return CAP_EINVAL;
    return ef_decode_launch_parked(pend->blob, (cudaStream_t)stream);
}

int cap_trace_fused_plan(int32_t L, int64_t T, const cap_gate_cfg *cfg, int32_t D, int32_t N, int32_t P,
                         int64_t plan[8])
{
    if (!plan || !gate_ok(cfg) || !sizes_ok(L, T, cfg->E, cfg->k) || D < 1 || D > 64 || N < 1 || N > 64 || P < 0)
        return CAP_EINVAL;
    fused_plan(L, T, *cfg, D, N, P, plan);
    return CAP_OK;
}

int cap_profile_fused_kernel(const float *const *logits_list, int32_t n_list, int32_t n_rep, int32_t L,
                             int64_t T, const cap_gate_cfg *cfg, int32_t *topk_idx, float *topk_w,
                             int64_t *counts, int32_t *coact, const int32_t *expert_dev, int32_t P,
                             const cap_topology *topo, const cap_eval_out *out, void *ws, size_t ws_bytes,
                             void *stream, float *avg_ms)
{
    if (!logits_list || n_list < 1 || n_rep < 1 || !avg_ms) return CAP_EINVAL;
    if (!gate_ok(cfg) || !sizes_ok(L, T, cfg->E, cfg->k) || !topo_ok(topo) || P < 1 || !out || L < 1 || T < 1)
        return CAP_EINVAL;
    if (!topk_idx || !topk_w || !counts || !coact || !expert_dev) return CAP_EINVAL;
    if (!ws || ws_bytes < eval_ws_bytes(L, T, cfg->E, cfg->k, topo->D, P)) return CAP_EWORKSPACE;
    bool used = false;
    CAP_TRY(profile_trace_fused_kernel(logits_list, n_list, n_rep, avg_ms, L, T, *cfg, topk_idx, topk_w, counts,
                                       coact, expert_dev, P, *topo, *out, ws, (cudaStream_t)stream, &used));
    return used ? CAP_OK : CAP_EINVAL;
}

int cap_validate_placements(const int32_t *expert_dev, int32_t L, int32_t P, int32_t E, int32_t D,
                            void *stream)
{
    if (L < 0 || P < 0 || E < 1 || D < 1 || D > 64) return CAP_EINVAL;
    const long long n = (long long)L * P * E;
    if (n == 0) return CAP_OK;
    if (!expert_dev) return CAP_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    int *bad = nullptr;
    // synchronous by contract: a 4-byte flag in mapped pinned host memory, no device allocation
    if (cudaHostAlloc(&bad, sizeof(int), cudaHostAllocMapped) != cudaSuccess) return check_launch("hostalloc");
    *bad = 0;
    int *dbad = nullptr;
    cudaHostGetDevicePointer(&dbad, bad, 0);
    long long blocks = (n + 255) / 256;
    if (blocks > 1024) blocks = 1024;
    validate_maps_kernel<<<(unsigned)blocks, 256, 0, st>>>(expert_dev, n, D, dbad);
    note_launch();
    int rc = check_launch("validate_maps_kernel");
    if (rc == CAP_OK && cudaStreamSynchronize(st) != cudaSuccess) rc = check_launch("sync");
    const int isbad = *bad;
    cudaFreeHost(bad);
    if (rc != CAP_OK) return rc;
    return isbad ? CAP_EINVAL : CAP_OK;
}

}  // extern "C"

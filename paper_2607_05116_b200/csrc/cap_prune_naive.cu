// Remaining pieces of SURVEY.md 8(f) rank 4:
//   cap_prune_naive         naive expert-level top-p pruning (the baseline of Fig. 14): per token the
//                           experts in descending routing weight (ties -> lower expert id), kept while the kept
//                           weight is < 1 - p -- Eq. 6's greedy with one expert per device and c_d = 1.
//   cap_dispatch_row_weights  combine weight a_d of every (token, device) row of cap_dispatch_rows (expert
//                           outputs are "locally aggregated via a weighted summation"): fp32 sum, in slot order, of
//                           the routing weights of the token's kept experts on that device.
// Both are one thread per token, everything in registers (k <= 16); HBM-bound streaming (8k + k and 8k + 4 rows
// bytes per token), launch-latency-bound at the BASELINE sizes.
#include "cap_internal.cuh"

namespace cap {

template <int K>
__global__ void __launch_bounds__(256) prune_naive_kernel(const int32_t *__restrict__ idx, const float *__restrict__ w,
                                                          long long T, int k, float p, uint8_t *__restrict__ kept,
                                                          unsigned long long *__restrict__ near_margin)
{
    const int layer = blockIdx.y;
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    pdl_launch_dependents();
    pdl_wait();
    int near = 0;
    if (t < T) {
        const size_t base = ((size_t)layer * T + t) * k;
        if (p <= 0.0f) {
            for (int s = 0; s < k; ++s) kept[base + s] = 1;
        } else {
            float ws[K];
            int es[K], rank[K];
#pragma unroll
            for (int s = 0; s < K; ++s) {
                ws[s] = s < k ? w[base + s] : 0.0f;
                es[s] = s < k ? idx[base + s] : 0x7fffffff;
            }
            // rank = position in the order (weight desc, ties -> lower expert id, then lower slot)
#pragma unroll
            for (int s = 0; s < K; ++s) {
                int r = 0;
#pragma unroll
                for (int s2 = 0; s2 < K; ++s2)
                    if (s2 < k && s2 != s)
                        r += (ws[s2] > ws[s] || (ws[s2] == ws[s] && (es[s2] < es[s] || (es[s2] == es[s] && s2 < s)))) ? 1 : 0;
                rank[s] = s < k ? r : K;
            }
            const float target = __fsub_rn(1.0f, p);
            float cum = 0.0f, last_kept = 0.0f, first_dropped = 0.0f;
            int nk = 0;
            unsigned keep = 0u;
            bool stopped = false;
            for (int i = 0; i < k; ++i) {
                float wi = 0.0f;
                int si = 0;
#pragma unroll
                for (int s = 0; s < K; ++s)
                    if (rank[s] == i) { wi = ws[s]; si = s; }
                if (!stopped) {
                    if (fabsf(__fsub_rn(cum, target)) < 1e-6f) near = 1;
                    if (cum >= target) {
                        stopped = true;
                        first_dropped = wi;
                    } else {
                        keep |= 1u << si;
                        cum = __fadd_rn(cum, wi);
                        last_kept = wi;
                        nk = i + 1;
                    }
                }
            }
            if (nk < k && __fsub_rn(last_kept, first_dropped) < 1e-6f) near = 1;
            for (int s = 0; s < k; ++s) kept[base + s] = (uint8_t)((keep >> s) & 1u);
        }
    }
    if (near_margin) {
        const unsigned n = __reduce_add_sync(0xffffffffu, (unsigned)near);
        if ((threadIdx.x & 31) == 0 && n) atomicAdd(&near_margin[layer], (unsigned long long)n);
    }
}

template <int K>
__global__ void __launch_bounds__(256) row_weights_kernel(const float *__restrict__ w, const int32_t *__restrict__ pair_row,
                                                          long long T, int k, long long n_rows, float *__restrict__ row_w)
{
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    pdl_launch_dependents();
    pdl_wait();
    if (t >= T) return;
    const size_t base = (size_t)t * k;
    float ws[K];
    int rs[K];
#pragma unroll
    for (int s = 0; s < K; ++s) {
        ws[s] = s < k ? w[base + s] : 0.0f;
        rs[s] = s < k ? pair_row[base + s] : -1;
    }
    // the first slot of every row adds the later slots of the same row in slot order and writes the sum: every row
    // belongs to exactly one token, so no two threads write the same element
#pragma unroll
    for (int s = 0; s < K; ++s) {
        if (s >= k || rs[s] < 0 || (long long)rs[s] >= n_rows) continue;
        bool first = true;
#pragma unroll
        for (int s2 = 0; s2 < K; ++s2)
            if (s2 < s && rs[s2] == rs[s]) first = false;
        if (!first) continue;
        float a = ws[s];
#pragma unroll
        for (int s2 = 0; s2 < K; ++s2)
            if (s2 > s && s2 < k && rs[s2] == rs[s]) a = __fadd_rn(a, ws[s2]);
        row_w[rs[s]] = a;
    }
}

}  // namespace cap

using namespace cap;

extern "C" {

int cap_prune_naive(const int32_t *topk_idx, const float *topk_w, int32_t L, int64_t T, int32_t k, float p,
                    uint8_t *kept, int64_t *near_margin, void *stream)
{
    if (L < 0 || T < 0 || k < 1 || k > 16 || L > 65535) return CAP_EINVAL;
    if (!(p < 1.0f)) return CAP_EINVAL;                          // also rejects NaN
    if ((int64_t)L * T > 0 && (!topk_idx || !topk_w || !kept)) return CAP_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    if (near_margin && L > 0 && cudaMemsetAsync(near_margin, 0, sizeof(int64_t) * (size_t)L, st) != cudaSuccess)
        return check_launch("memset near_margin");
    if ((int64_t)L * T == 0) return CAP_OK;
    const dim3 grid((unsigned)((T + 255) / 256), (unsigned)L);
    unsigned long long *nm = reinterpret_cast<unsigned long long *>(near_margin);
    {
        KernelTimerScope ts("prune_naive", st);
        if (k <= 8) launch_pdl(prune_naive_kernel<8>, grid, dim3(256), 0, st, topk_idx, topk_w, (long long)T, k, p, kept, nm);
        else launch_pdl(prune_naive_kernel<16>, grid, dim3(256), 0, st, topk_idx, topk_w, (long long)T, k, p, kept, nm);
    }
    note_launch();
    return check_launch("prune_naive_kernel");
}

int cap_dispatch_row_weights(const float *topk_w, const int32_t *pair_row, int64_t T, int32_t k, int64_t n_rows,
                             float *row_w, void *stream)
{
    if (T < 0 || k < 1 || k > 16 || n_rows < 0) return CAP_EINVAL;
    if (T > 0 && (!topk_w || !pair_row)) return CAP_EINVAL;
    if (n_rows > 0 && !row_w) return CAP_EINVAL;
    if (T == 0 || n_rows == 0) return CAP_OK;
    cudaStream_t st = (cudaStream_t)stream;
    const dim3 grid((unsigned)((T + 255) / 256));
    {
        KernelTimerScope ts("row_weights", st);
        if (k <= 8) launch_pdl(row_weights_kernel<8>, grid, dim3(256), 0, st, topk_w, pair_row, (long long)T, k, (long long)n_rows, row_w);
        else launch_pdl(row_weights_kernel<16>, grid, dim3(256), 0, st, topk_w, pair_row, (long long)T, k, (long long)n_rows, row_w);
    }
    note_launch();
    return check_launch("row_weights_kernel");
}

}  // extern "C"

// S4 -- communication-aware pruning (Eq. 6 and its greedy solver).  One thread per
// token: aggregate the slot weights per destination device in slot order (fp32), price each
// device by topology relative to the token's source, keep devices by descending a_d/c_d until
// the kept weight reaches 1-p.  Every fp32 step is a single IEEE operation (readings R7-R10).
#include <math_constants.h>

#include "cap_internal.cuh"

namespace cap {

struct PruneParams {
    const int32_t *idx;
    const float *w;
    const int32_t *token_src;
    const int32_t *expert_dev;   // [L][E]
    const int32_t *dev_node;
    uint8_t *kept;
    unsigned long long *near_margin;   // [L] or NULL
    int64_t T;
    int32_t k, E, D, cost_local, cost_intra, cost_inter;
    float p;
};

template <int KMAX>
__global__ void __launch_bounds__(256) prune_kernel(PruneParams prm)
{
    extern __shared__ int s_map[];     // [E] expert -> device of this layer, then [D] dev -> node
    const int layer = blockIdx.y;
    const int E = prm.E, D = prm.D, k = prm.k;
    int *s_dn = s_map + E;
    for (int i = threadIdx.x; i < E; i += blockDim.x) s_map[i] = prm.expert_dev[(size_t)layer * E + i];
    for (int i = threadIdx.x; i < D; i += blockDim.x) s_dn[i] = prm.dev_node[i];
    __syncthreads();

    const int64_t T = prm.T;
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    int near = 0;
    if (t < T) {
        const int64_t base = ((int64_t)layer * T + t) * k;
        if (prm.p <= 0.0f) {
            for (int s = 0; s < k; ++s) prm.kept[base + s] = 1;
        } else {
            const int src = prm.token_src ? prm.token_src[(int64_t)layer * T + t] : (int)((t * D) / T);
            const int srcn = s_dn[src];
            int dev[KMAX], sdev[KMAX];
            float a[KMAX], ratio[KMAX];
            int m = 0;
#pragma unroll
            for (int s = 0; s < KMAX; ++s) {
                if (s < k) {
                    const int d = s_map[prm.idx[base + s]];
                    sdev[s] = d;
                    const float ws = prm.w[base + s];
                    int j = 0;
                    while (j < m && dev[j] != d) ++j;
                    if (j == m) { dev[m] = d; a[m] = ws; ++m; }
                    else a[j] = __fadd_rn(a[j], ws);
                }
            }
            for (int j = 0; j < m; ++j) {
                const int d = dev[j];
                const int c = (d == src) ? prm.cost_local : (s_dn[d] == srcn) ? prm.cost_intra : prm.cost_inter;
                ratio[j] = (c == 0) ? CUDART_INF_F : __fdiv_rn(a[j], (float)c);
            }
            // order by ratio descending, ties -> lower device id (insertion sort, m <= k)
            for (int i = 1; i < m; ++i) {
                const int d = dev[i];
                const float r = ratio[i], av = a[i];
                int j = i - 1;
                while (j >= 0 && (ratio[j] < r || (ratio[j] == r && dev[j] > d))) {
                    dev[j + 1] = dev[j]; ratio[j + 1] = ratio[j]; a[j + 1] = a[j];
                    --j;
                }
                dev[j + 1] = d; ratio[j + 1] = r; a[j + 1] = av;
            }
            const float target = __fsub_rn(1.0f, prm.p);
            float cum = 0.0f;
            int nk = 0;
            unsigned long long keepmask = 0ull;
            for (int i = 0; i < m; ++i) {
                if (fabsf(__fsub_rn(cum, target)) < 1e-6f) near = 1;
                if (cum >= target) break;
                keepmask |= 1ull << dev[i];
                cum = __fadd_rn(cum, a[i]);
                nk = i + 1;
            }
            if (nk < m) {
                const float r1 = ratio[nk - 1], r2 = ratio[nk];
                if (r1 != CUDART_INF_F && r2 != CUDART_INF_F && __fsub_rn(r1, r2) < 1e-6f) near = 1;
            }
#pragma unroll
            for (int s = 0; s < KMAX; ++s)
                if (s < k) prm.kept[base + s] = (uint8_t)((keepmask >> sdev[s]) & 1ull);
        }
    }
    if (prm.near_margin) {
        const unsigned b = __ballot_sync(0xffffffffu, near != 0);
        if ((threadIdx.x & 31) == 0 && b) atomicAdd(&prm.near_margin[layer], (unsigned long long)__popc(b));
    }
}

int launch_prune(const int32_t *idx, const float *w, const int32_t *token_src, int32_t L,
                 int64_t T, int32_t k, int32_t E, const int32_t *expert_dev,
                 const cap_topology &topo, float p, uint8_t *kept, int64_t *near_margin,
                 cudaStream_t st)
{
    if (L == 0) return CAP_OK;
    if (near_margin &&
        cudaMemsetAsync(near_margin, 0, sizeof(int64_t) * (size_t)L, st) != cudaSuccess)
        return check_launch("memset near_margin");
    if (T == 0) return CAP_OK;
    PruneParams prm;
    prm.idx = idx;
    prm.w = w;
    prm.token_src = token_src;
    prm.expert_dev = expert_dev;
    prm.dev_node = topo.dev_node;
    prm.kept = kept;
    prm.near_margin = reinterpret_cast<unsigned long long *>(near_margin);
    prm.T = T;
    prm.k = k;
    prm.E = E;
    prm.D = topo.D;
    prm.cost_local = topo.cost_local;
    prm.cost_intra = topo.cost_intra;
    prm.cost_inter = topo.cost_inter;
    prm.p = p;
    dim3 grid((unsigned)((T + 255) / 256), (unsigned)L);
    const size_t smem = sizeof(int) * ((size_t)E + topo.D);
    {
        KernelTimerScope ts("prune", st);
        if (k <= 8) prune_kernel<8><<<grid, 256, smem, st>>>(prm);
        else prune_kernel<16><<<grid, 256, smem, st>>>(prm);
    }
    note_launch();
    return check_launch("prune_kernel");
}

}  // namespace cap

// S2 -- per-expert activation counts and the E x E co-activation matrix.
// Generic kernel: one thread per (token, slot) pair adds its row of pair increments, into a
// block-private shared-memory matrix when E*E int32 fits, else straight into global memory.
#include "cap_internal.cuh"

namespace cap {

__global__ void __launch_bounds__(256)
coact_kernel(const int32_t *__restrict__ idx, const uint8_t *__restrict__ kept, int64_t T, int k,
             int E, unsigned long long *__restrict__ counts, int *__restrict__ coact,
             int64_t tok_per_block, int use_smem)
{
    extern __shared__ int sm[];
    int *hist = sm;                                  // [E*E] (use_smem) then [E]
    int *cnt = use_smem ? sm + (size_t)E * E : sm;
    const int layer = blockIdx.y;
    idx += (int64_t)layer * T * k;
    if (kept) kept += (int64_t)layer * T * k;
    counts += (int64_t)layer * E;
    coact += (int64_t)layer * E * E;

    const int nsm = (use_smem ? E * E : 0) + E;
    for (int i = threadIdx.x; i < nsm; i += blockDim.x) sm[i] = 0;
    __syncthreads();

    const int64_t t0 = (int64_t)blockIdx.x * tok_per_block;
    const int64_t t1 = min(T, t0 + tok_per_block);
    const int64_t items = (t1 > t0 ? (t1 - t0) : 0) * k;
    for (int64_t it = threadIdx.x; it < items; it += blockDim.x) {
        const int64_t t = t0 + it / k;
        const int a = (int)(it % k);
        const int64_t base = t * k;
        if (kept && !kept[base + a]) continue;
        const int i = idx[base + a];
        if ((unsigned)i >= (unsigned)E) continue;    // out-of-range ids: undefined result, memory-safe (cap.h)
        atomicAdd(&cnt[i], 1);
        if (!use_smem) {
            // straight into global memory: only the pairs with a larger partner id, i.e. the upper triangle (half the
            // reductions); coact_mirror_kernel copies it below the diagonal and writes the diagonal from the counts
            // (a token's expert ids are distinct: include/cap.h)
            for (int b = 0; b < k; ++b) {
                if (b == a || (kept && !kept[base + b])) continue;
                const int j = idx[base + b];
                if ((unsigned)j < (unsigned)E && j > i) atomicAdd(&coact[(size_t)i * E + j], 1);
            }
            continue;
        }
        int *rowp = hist + (size_t)i * E;
        for (int b = 0; b < k; ++b) {
            if (b != a && kept && !kept[base + b]) continue;
            const int j = idx[base + b];
            if ((unsigned)j < (unsigned)E) atomicAdd(&rowp[j], 1);      // b == a gives the diagonal
        }
    }
    __syncthreads();
    if (use_smem) {
        for (int i = threadIdx.x; i < E * E; i += blockDim.x) {
            int v = hist[i];
            if (v) atomicAdd(&coact[i], v);
        }
    }
    for (int i = threadIdx.x; i < E; i += blockDim.x) {
        int v = cnt[i];
        if (v) atomicAdd(&counts[i], (unsigned long long)v);
    }
}

// the lower triangle and the diagonal of every layer's matrix after the upper-triangle pass of coact_kernel
__global__ void __launch_bounds__(256)
coact_mirror_kernel(const unsigned long long *__restrict__ counts, int *__restrict__ coact, int E)
{
    coact += (size_t)blockIdx.y * E * E;
    counts += (size_t)blockIdx.y * E;
    __shared__ int tile[32][33];
    // 32 x 32 tiles of the upper triangle (tile row <= tile column), transposed through shared memory
    const int nt = (E + 31) / 32;
    int tr = 0, rem = blockIdx.x;
    while (rem >= nt - tr) {
        rem -= nt - tr;
        ++tr;
    }
    const int tc = tr + rem;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    for (int r = ty; r < 32; r += 8) {
        const int i = tr * 32 + r, j = tc * 32 + tx;
        tile[r][tx] = (i < E && j < E && j > i) ? coact[(size_t)i * E + j] : 0;
    }
    __syncthreads();
    for (int r = ty; r < 32; r += 8) {
        const int i = tc * 32 + r, j = tr * 32 + tx;          // element (i, j) below the diagonal <- (j, i)
        if (i < E && j < E && j < i) coact[(size_t)i * E + j] = tile[tx][r];
        if (i < E && tr == tc && j == i) coact[(size_t)i * E + i] = (int)counts[i];
    }
}

int launch_coactivation(const int32_t *idx, const uint8_t *kept, int32_t L, int64_t T, int32_t k,
                        int32_t E, int64_t *counts, int32_t *coact, cudaStream_t st)
{
    if (L == 0) return CAP_OK;
    if (cudaMemsetAsync(counts, 0, sizeof(int64_t) * (size_t)L * E, st) != cudaSuccess)
        return check_launch("memset counts");
    if (cudaMemsetAsync(coact, 0, sizeof(int32_t) * (size_t)L * E * E, st) != cudaSuccess)
        return check_launch("memset coact");
    if (T == 0) return CAP_OK;
    bool mma = false;
    CAP_TRY(launch_coact_mma(idx, kept, L, T, k, E, counts, coact, st, &mma));
    if (mma) return CAP_OK;
    const size_t smem_full = sizeof(int) * ((size_t)E * E + E);
    const int use_smem = smem_full <= 160 * 1024;
    const size_t smem = use_smem ? smem_full : sizeof(int) * (size_t)E;
    // per device and cheap: set on every launch (a per-process flag would leave a second GPU without the opt-in)
    cudaFuncSetAttribute(coact_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 164 * 1024);
    // enough blocks per layer to fill the machine, but each block's flush costs E*E atomics
    int64_t want = (2 * (int64_t)sm_count() + L - 1) / L;
    if (want < 1) want = 1;
    int64_t tpb = (T + want - 1) / want;
    if (tpb < 256) tpb = 256;
    const int64_t nblk = (T + tpb - 1) / tpb;
    dim3 grid((unsigned)nblk, (unsigned)L);
    KernelTimerScope ts("coact", st);
    coact_kernel<<<grid, 256, smem, st>>>(idx, kept, T, k, E, reinterpret_cast<unsigned long long *>(counts), coact, tpb,
                                          use_smem);
    note_launch();
    CAP_TRY(check_launch("coact_kernel"));
    if (!use_smem) {
        const int nt = (E + 31) / 32;
        coact_mirror_kernel<<<dim3((unsigned)(nt * (nt + 1) / 2), (unsigned)L), 256, 0, st>>>(
            reinterpret_cast<const unsigned long long *>(counts), coact, E);
        note_launch();
        return check_launch("coact_mirror_kernel");
    }
    return CAP_OK;
}

}  // namespace cap

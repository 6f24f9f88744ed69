// Bit-sliced candidate scoring (S3 fast path): declarations shared by the standalone evaluation
// kernel (cap_eval_fast.cu) and the fused trace kernel (cap_fused.cu).  See DESIGN.md section 6.
//
// Idea.  For every expert e a shared-memory table row holds, for each candidate p of the block's
// candidate chunk, the one-hot code 1 << pi_p(e) in a WD-bit field (WD = 8/16/32/64 >= D) and the
// one-hot node code 1 << node(pi_p(e)) in a WN-bit field (WN = 2/4/8 >= N).  A token's device sets
// under all candidates are the bitwise OR of its k rows; a thread owns one 16-byte column of the
// rows (4 words) and keeps, per bit position, a bit-sliced counter of how many tokens had the bit
// set (carry-save adders on whole words: ~3 LOP3 per token per word instead of one add per
// (token, candidate, device)).  Tokens are processed in runs that share one source device, so the
// "local" and "same node" totals are recovered later by masking the per-run counters with the
// source's device / node bits.  A run's counters leave the block as bit planes (a "record"); a
// small decode kernel adds all records in the bit-sliced domain and extracts the integers once.
#pragma once
#include "cap_internal.cuh"

namespace cap {

constexpr int EF_BT = 8;        // planes a thread accumulates between flushes (counts < 256)
constexpr int EF_NPL = 14;      // planes after the sub-slot tree (S <= 64)
constexpr int EF_RECW = 16;     // record layout [word][EF_RECW planes]: a word's planes are one 64-byte run
constexpr int EF_PASSES = 8;    // tokens per thread per block of the CSA tree
constexpr int EF_MAXBLK = 31;   // blocks per run: 248 inputs per thread < 2^EF_BT
constexpr int EF_PRE = 16;      // prefetched index entries per thread
constexpr int EF_MAXTHREADS = 384;
constexpr int EF_RS_FUSED = 320;        // (column, sub-slot) threads of the scoring warps inside the fused kernel
constexpr int EF_RS_ALONE = 384;        // of the stand-alone scoring kernel: a whole SM's registers at 168 per thread

struct EvalFastGeom {
    int WD, WN;          // field widths (bits) of the device / node codes
    int Pc, PC;          // candidates per chunk (padded to whole 16-byte columns), chunks
    int DW, NW;          // words per row: device section (multiple of 4), node section (multiple of 4)
    int R, RS;           // 16-byte columns per row used / row stride in columns (odd)
    int W;               // words per record plane = 4 R
    int S, logS;         // token sub-slots processed concurrently (power of two)
    int xpl;             // planes per exchange round of the flush tree (stand-alone kernel; EF_NPL = one round)
    int KP;              // k padded to a multiple of 4
    int nthreads;
    int ncta_t;          // blocks along the token axis (per layer and candidate chunk)
    int64_t tpc;         // tokens per block (multiple of EF_PASSES * S)
    int maxrec;          // records a block can emit
    int NPR;             // planes per record = EF_BT + logS
    size_t smem;         // dynamic shared memory of the standalone kernel
    size_t rec_words;    // uint32 words of all records
    size_t rec_slots;    // record headers
    size_t table_words;  // uint32 words of the code tables of all layers and chunks
};

// false when the fast path does not apply to these sizes (the generic kernel is used instead)
// explicit_src: the tokens come grouped by an arbitrary token_src (any number of source boundaries per block)
bool eval_fast_geom(int32_t L, int64_t T, int32_t k, int32_t E, int32_t D, int32_t N, int32_t P,
                    int target_ctas, size_t smem_budget, EvalFastGeom *g, bool explicit_src = false,
                    int rs_limit = EF_RS_FUSED);
size_t eval_fast_ws_bytes(int32_t L, int64_t T, int32_t k, int32_t E, int32_t D, int32_t P);

struct EvalFastWs {
    int32_t *rec_src;       // [L][PC][ncta_t][maxrec], -1 = unused
    uint32_t *rec_planes;   // [L][PC][ncta_t][maxrec][W][EF_RECW] (word-major: the decode reads 64-byte runs)
    uint32_t *table;        // [L][PC][E + 1][RS * 4] one-hot code table
    // explicit token_src only: tokens sorted by source device
    int32_t *perm;          // [L][T]
    long long *srcoff;      // [L][D + 1]
    int32_t *ident;         // [L][64] identity maps of the sort
    void *sort_ws;          // workspace of the batched counting sort (k = 1)
};
EvalFastWs eval_fast_ws_carve(void *ws, int32_t L, int32_t E, int32_t D, int32_t P,
                              const EvalFastGeom &g, int64_t T = 0);

// a buffer the table kernel fills with a 32-bit value on the side (bytes must be a multiple of 4)
struct EfFill {
    void *ptr;
    size_t bytes;
    uint32_t value;
};
int ef_launch_table(const EvalFastGeom &g, const EvalFastWs &fw, const int32_t *expert_dev, const int32_t *dev_node,
                    int32_t L, int32_t E, int32_t P, int32_t D, cudaStream_t st, const EfFill *fills, int nfill);
int ef_launch_decode(const EvalFastGeom &g, const EvalFastWs &fw, int32_t L, int64_t T, int32_t E, int32_t P,
                     const cap_topology &topo, const int32_t *expert_dev, const int64_t *counts,
                     const cap_eval_out &out, cudaStream_t st);

// ---- device helpers ------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t lop_xor3(uint32_t a, uint32_t b, uint32_t c)
{
    uint32_t r;
    asm("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(r) : "r"(a), "r"(b), "r"(c));
    return r;
}
__device__ __forceinline__ uint32_t lop_maj(uint32_t a, uint32_t b, uint32_t c)
{
    uint32_t r;
    asm("lop3.b32 %0, %1, %2, %3, 0xE8;" : "=r"(r) : "r"(a), "r"(b), "r"(c));
    return r;
}
__device__ __forceinline__ uint32_t lop_or3(uint32_t a, uint32_t b, uint32_t c)
{
    uint32_t r;
    asm("lop3.b32 %0, %1, %2, %3, 0xFE;" : "=r"(r) : "r"(a), "r"(b), "r"(c));
    return r;
}
// carry-save adder on whole words: (s, c) with s + 2c = a + b + x per bit position
#define CAP_CSA(s, c, a, b, x)                \
    do {                                      \
        const uint32_t _a = (a), _b = (b), _x = (x); \
        (c) = lop_maj(_a, _b, _x);            \
        (s) = lop_xor3(_a, _b, _x);           \
    } while (0)

// planes of one record word (EF_NPL values, the rest of the EF_RECW-word run zero) as four 16-byte stores
__device__ __forceinline__ void ef_store_word_planes(uint32_t *dst, const uint32_t (&v)[EF_RECW])
{
    uint4 *d4 = reinterpret_cast<uint4 *>(dst);
#pragma unroll
    for (int i = 0; i < EF_RECW / 4; ++i) d4[i] = make_uint4(v[4 * i], v[4 * i + 1], v[4 * i + 2], v[4 * i + 3]);
}

// Word mask of the bit positions of record word w whose device belongs to `set` (bit d = device d).
__device__ __forceinline__ uint32_t ef_devmask_word(int WD, int w, unsigned long long set)
{
    if (WD == 64) return (uint32_t)(set >> ((w & 1) * 32));
    if (WD == 32) return (uint32_t)set;
    if (WD == 16) return ((uint32_t)set & 0xffffu) * 0x00010001u;
    return ((uint32_t)set & 0xffu) * 0x01010101u;
}
__device__ __forceinline__ uint32_t ef_nodemask_word(int WN, int node)
{
    const uint32_t rep = WN == 2 ? 0x55555555u : WN == 4 ? 0x11111111u : 0x01010101u;
    return rep << node;
}

// One word of the code table: row e (e == E is the all-zero row), word w of candidate chunk
// [p0, p0 + Pc).  Words [0, DW) hold device codes, [DW, DW + NW) node codes.  node_of: node code of
// every device (a shared-memory copy).  The map entries of a word (up to 16 candidates) are fetched
// with independent loads first -- the [P][E] maps are read with a stride of E, one L2 round trip each.
__device__ __forceinline__ uint32_t ef_table_word(const int32_t *__restrict__ maps /*[P][E]*/,
                                                  const unsigned char *node_of, int E, int P,
                                                  int D, int p0, int WD, int WN, int DW, int NW, int e,
                                                  int w)
{
    if (e >= E || w >= DW + NW) return 0u;
    const bool devw = w < DW;
    uint32_t word = 0u;
    if (devw) {
        // 1 (WD = 64: half a field per word, or WD = 32), 2 or 4 candidates per word: at most four independent loads
        const int fpw = WD >= 32 ? 1 : 32 / WD;
        const int pb = p0 + (WD == 64 ? (w >> 1) : w * fpw);
        int dv[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int p = pb + j;
            dv[j] = (j < fpw && p < P) ? maps[(size_t)p * E + e] : -1;
        }
        if (WD == 64) {
            const int d = dv[0];
            if ((unsigned)d < (unsigned)D && (d >> 5) == (w & 1)) word = 1u << (d & 31);
        } else {
#pragma unroll
            for (int j = 0; j < 4; ++j)
                if ((unsigned)dv[j] < (unsigned)D) word |= 1u << (j * WD + dv[j]);
        }
    } else {
        // 4, 8 or 16 candidates per node word, four loads in flight
        const int fpw = 32 / WN;
        const int pb = p0 + (w - DW) * fpw;
        for (int j0 = 0; j0 < fpw; j0 += 4) {
            int dv[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int p = pb + j0 + j;
                dv[j] = p < P ? maps[(size_t)p * E + e] : -1;
            }
#pragma unroll
            for (int j = 0; j < 4; ++j)
                if ((unsigned)dv[j] < (unsigned)D) word |= 1u << ((j0 + j) * WN + (node_of[dv[j]] & (WN - 1)));
        }
    }
    return word;
}

// Copy a prebuilt table ((E + 1) rows of RS * 16 bytes) from global to shared memory.
__device__ __forceinline__ void ef_copy_table(unsigned char *tbl, const uint32_t *__restrict__ gtbl,
                                              int n16, int tid, int nthr)
{
    const uint4 *g4 = reinterpret_cast<const uint4 *>(gtbl);
    uint4 *t4 = reinterpret_cast<uint4 *>(tbl);
#pragma unroll 4
    for (int i = tid; i < n16; i += nthr) t4[i] = __ldg(g4 + i);
}

}  // namespace cap

// topk.cu -- exact K-nearest-neighbour lookup in the embedding space (PAPER.md:225 sec. 3.5; :289:
// "top K nearest neighbors ... from a sample of 5 million test pins", K = 500): the exact form of
// what the paper serves approximately with LSH + Weak-AND.  Reading C1: nearest = largest inner
// product z_q . z_i (the score of Eq. 1), ties to the smaller id.
//
// The scores of a block of candidates come from the tcgen05 GEMM.  This file keeps, per query, a
// running list of the k best (score, id) pairs as 64-bit keys
//     key = orderable(score) << 32 | (0xFFFFFFFF - id)        (larger key = better)
// plus a 1024-key candidate buffer.  Two ways in:
//  * two-pass (the first block(s), option topk_fused = 0, redone blocks): the GEMM stores fp32 scores,
//    topk_scan_kernel (one CTA per query) scans them coalesced and appends what beats the current k-th
//    key to the buffer; only when the buffer could overflow does it merge (sort buffer, bitonic-merge
//    with the list, keep k);
//  * fused (every later block): the GEMM's selection epilogue (gemm_tcgen05.cu) appends the keepers
//    itself -- no score matrix in HBM -- and topk_maintain_kernel merges buffers that are filling up
//    and flags the (block, query) pairs whose buffer overflowed, which the caller redoes two-pass.
// The result is the exact top k under a total order, so it does not depend on the order in which
// candidates were buffered, merged or redone.
#include "internal.h"

namespace pinsage {
namespace {

constexpr int TK_THREADS = 256;
static_assert(TK_THREADS == 256 && TK_LIST == 1024, "cta_sort_desc maps 8 warps onto 1024 + 2048 keys");

// s[0 .. TK_LIST) is the running list, sorted descending (zeros at its end); s[TK_LIST .. TK_TOTAL) is the
// buffer in any order.  Sorts the buffer ascending (bitonic network on 1024 keys) -- list + buffer is
// then one bitonic sequence -- and finishes with a bitonic merge of all 2048 keys, descending: 38
// stage-equivalents instead of the 66 of a full sort.  Each warp owns a contiguous run of keys, so
// every stage whose partner distance stays inside the run needs a __syncwarp only (10 CTA-wide
// barriers in all instead of 66).
__device__ void cta_sort_desc(unsigned long long *s)
{
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    unsigned long long *b = s + TK_LIST;
    for (int k = 2; k <= TK_LIST; k <<= 1)
        for (int j = k >> 1; j > 0; j >>= 1) {
            if (j >= 128) __syncthreads();
#pragma unroll
            for (int r = 0; r < 2; ++r) {                      // warp w: pairs inside b[128 w, 128 w + 128) for j <= 64
                const int p = warp * 64 + r * 32 + lane;
                const int i = ((p & ~(j - 1)) << 1) | (p & (j - 1)), l = i | j;
                const unsigned long long a = b[i], c = b[l];
                if ((a > c) == ((i & k) == 0)) {
                    b[i] = c;
                    b[l] = a;
                }
            }
            if (j >= 128) __syncthreads();
            else __syncwarp();
        }
    __syncthreads();
    for (int j = TK_LIST; j > 0; j >>= 1) {
        if (j >= 256) __syncthreads();
#pragma unroll
        for (int r = 0; r < 4; ++r) {                          // warp w: pairs inside s[256 w, 256 w + 256) for j <= 128
            const int p = warp * 128 + r * 32 + lane;
            const int i = ((p & ~(j - 1)) << 1) | (p & (j - 1)), l = i | j;
            const unsigned long long a = s[i], c = s[l];
            if (a < c) {
                s[i] = c;
                s[l] = a;
            }
        }
        if (j >= 256) __syncthreads();
        else __syncwarp();
    }
    __syncthreads();
}

// sort list + buffer, keep the best k, empty the buffer; returns the new k-th best key
__device__ __noinline__ unsigned long long merge_buffer(unsigned long long *s, int *cnt, int k)
{
    __syncthreads();
    cta_sort_desc(s);
    for (int i = k + threadIdx.x; i < TK_TOTAL; i += TK_THREADS) s[i] = 0ull;
    if (threadIdx.x == 0) *cnt = 0;
    __syncthreads();
    return s[k - 1];
}

// Per-query state in global memory: state[q] = TK_TOTAL keys (running list, sorted descending, in
// [0, k); zeros up to TK_LIST; candidate buffer in [TK_LIST, TK_LIST + cnt[q])), cnt[q] buffered keys.
// scores [nq x ld] fp32 (ld % 4 == 0, rows 16-byte aligned), columns [0, nb) valid = candidates id0 ...
// One CTA per query scans its row, TK_BLOCK scores per iteration (four float4 per thread up front),
// and appends what beats the current k-th key straight to the global buffer -- in steady state a
// handful of keys per block of scores.  Only when the buffer could overflow (the first blocks of a
// fresh list) does the CTA pull the state into shared memory, merge (bitonic sort of 2048 keys, keep
// k) and continue there in 256-key steps.  No sort and no state traffic otherwise.
constexpr int TK_BLOCK = 16 * TK_THREADS;
__global__ void __launch_bounds__(TK_THREADS)
topk_scan_kernel(const float *__restrict__ scores, long long ld, int nb, long long id0, int k,
                 unsigned long long *__restrict__ state, int *__restrict__ cnts,
                 const unsigned char *__restrict__ only)
{
    __shared__ unsigned long long s[TK_TOTAL];
    __shared__ int cnt, blk;
    const long long q = blockIdx.x;
    if (only != nullptr && only[q] == 0) return;
    const float *row = scores + q * ld;
    unsigned long long *st = state + q * TK_TOTAL;
    int have = cnts[q];
    unsigned long long tau = st[k - 1];                        // current k-th best (0 while not full)
    if (threadIdx.x == 0) blk = 0;
    __syncthreads();
    // software pipeline: the loads of block b+1 are in flight while block b is tested
    auto load_block = [&](int base, float4 (&dst)[4]) {
#pragma unroll
        for (int i = 0; i < 4; ++i) {                          // columns base + (i*256 + t)*4 .. +3
            const int j = base + (i * TK_THREADS + threadIdx.x) * 4;
            dst[i] = j < nb ? __ldcs(reinterpret_cast<const float4 *>(row + j))   // (ld is padded past nb)
                            : make_float4(0.f, 0.f, 0.f, 0.f);
        }
    };
    float4 nxt[4];
    load_block(0, nxt);
    for (int base = 0; base < nb; base += TK_BLOCK) {
        float4 v[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) v[i] = nxt[i];
        load_block(base + TK_BLOCK, nxt);                      // (past the end: zeros, no loads)
        // cheap float pre-filter (a score below the k-th best score can never enter); keys are built
        // only for the few survivors -- an un-built key is 0 and loses every comparison
        const float tau_f = tau ? unord_f32((unsigned)(tau >> 32)) : -INFINITY;
        unsigned long long key[16];
        int mine = 0;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int j = base + (i * TK_THREADS + threadIdx.x) * 4;
            const float x[4] = {v[i].x, v[i].y, v[i].z, v[i].w};
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                key[4 * i + e] = 0ull;
                if (x[e] >= tau_f && j + e < nb) {
                    key[4 * i + e] = make_key(x[e], id0 + j + e);
                    mine += key[4 * i + e] > tau;
                }
            }
        }
        if (!__syncthreads_or(mine)) continue;                 // steady state: nothing beats the k-th key
        int at = 0;
        if (mine) at = atomicAdd(&blk, mine);                  // my offset among this block's keepers
        __syncthreads();
        const int total = blk;
        __syncthreads();
        if (threadIdx.x == 0) blk = 0;
        if (have + total <= TK_LIST) {                         // fits: append to the global buffer
            if (mine) {
                at += TK_LIST + have;
#pragma unroll
                for (int e = 0; e < 16; ++e)
                    if (key[e] > tau) st[at++] = key[e];
            }
            have += total;
        } else {                                               // could overflow: merge in shared memory
            __syncthreads();
            for (int i = threadIdx.x; i < TK_TOTAL; i += TK_THREADS)
                s[i] = (i < TK_LIST || i < TK_LIST + have) ? st[i] : 0ull;
            if (threadIdx.x == 0) cnt = have;
            __syncthreads();
#pragma unroll                                             // (a rolled loop would index key[] dynamically
            for (int e = 0; e < 16; ++e) {                      //  and push the whole array to local memory)
                if (cnt + TK_THREADS > TK_LIST) tau = merge_buffer(s, &cnt, k);
                if (key[e] > tau) s[TK_LIST + atomicAdd(&cnt, 1)] = key[e];
                __syncthreads();
            }
            tau = merge_buffer(s, &cnt, k);
            for (int i = threadIdx.x; i < TK_LIST; i += TK_THREADS) st[i] = s[i];
            have = 0;
            __syncthreads();
        }
    }
    if (threadIdx.x == 0) cnts[q] = have;
}

// bookkeeping after a block that went through the GEMM's selection epilogue (see internal.h)
__global__ void __launch_bounds__(TK_THREADS)
topk_maintain_kernel(unsigned long long *__restrict__ state, int *__restrict__ cnts, int k, int merge_at,
                     int *__restrict__ cnt_prev, unsigned char *__restrict__ ovf, int *__restrict__ any)
{
    __shared__ unsigned long long s[TK_TOTAL];
    const long long q = blockIdx.x;
    const int have = cnts[q];
    if (have > TK_LIST) {                                      // some of this block's keepers were dropped
        if (threadIdx.x == 0) {
            cnts[q] = cnt_prev[q];
            ovf[q] = 1;
            *any = 1;
        }
        return;
    }
    if (threadIdx.x == 0) ovf[q] = 0;
    if (have < merge_at) {
        if (threadIdx.x == 0) cnt_prev[q] = have;
        return;
    }
    unsigned long long *st = state + q * TK_TOTAL;
    for (int i = threadIdx.x; i < TK_TOTAL; i += TK_THREADS) s[i] = i < TK_LIST + have ? st[i] : 0ull;
    __syncthreads();
    cta_sort_desc(s);
    for (int i = threadIdx.x; i < TK_LIST; i += TK_THREADS) st[i] = i < k ? s[i] : 0ull;
    if (threadIdx.x == 0) cnts[q] = cnt_prev[q] = 0;
}

// final merge of list + buffer and decoding: idx / score [nq x k]
__global__ void __launch_bounds__(TK_THREADS)
topk_finish_kernel(const unsigned long long *__restrict__ state, const int *__restrict__ cnts, int k,
                   int *__restrict__ idx, float *__restrict__ score)
{
    __shared__ unsigned long long s[TK_TOTAL];
    const long long q = blockIdx.x;
    const unsigned long long *st = state + q * TK_TOTAL;
    const int have = cnts[q];
    for (int i = threadIdx.x; i < TK_TOTAL; i += TK_THREADS)
        s[i] = (i < TK_LIST || i < TK_LIST + have) ? st[i] : 0ull;
    __syncthreads();
    cta_sort_desc(s);
    for (int i = threadIdx.x; i < k; i += TK_THREADS) {
        const unsigned long long key = s[i];
        idx[q * k + i] = key ? (int)(0xFFFFFFFFu - (unsigned)(key & 0xFFFFFFFFull)) : -1;
        score[q * k + i] = key ? unord_f32((unsigned)(key >> 32)) : -INFINITY;
    }
}

}  // namespace

size_t topk_state_bytes(int64_t nq) { return (size_t)nq * TK_TOTAL * 8 + (size_t)nq * 4; }

// state: topk_state_bytes(nq) zeroed bytes (keys, then the counters) before the first block of scores
cudaError_t launch_topk_merge(const float *scores, int64_t nq, int64_t ld, int32_t nb, int64_t id0,
                              int32_t k, void *state, const unsigned char *only, cudaStream_t s,
                              int *launches)
{
    if (k < 1 || k > TK_LIST) return cudaErrorNotSupported;
    unsigned long long *keys = static_cast<unsigned long long *>(state);
    int *cnts = reinterpret_cast<int *>(keys + (size_t)nq * TK_TOTAL);
    topk_scan_kernel<<<(unsigned)nq, TK_THREADS, 0, s>>>(scores, ld, nb, id0, k, keys, cnts, only);
    if (launches) ++*launches;
    return cudaGetLastError();
}

cudaError_t launch_topk_maintain(void *state, int64_t nq, int32_t k, int32_t merge_at, int *cnt_prev,
                                 unsigned char *ovf, int *any, cudaStream_t s, int *launches)
{
    unsigned long long *keys = static_cast<unsigned long long *>(state);
    int *cnts = reinterpret_cast<int *>(keys + (size_t)nq * TK_TOTAL);
    topk_maintain_kernel<<<(unsigned)nq, TK_THREADS, 0, s>>>(keys, cnts, k, merge_at, cnt_prev, ovf, any);
    if (launches) ++*launches;
    return cudaGetLastError();
}

cudaError_t launch_topk_finish(const void *state, int64_t nq, int32_t k, int32_t *idx, float *score,
                               cudaStream_t s, int *launches)
{
    const unsigned long long *keys = static_cast<const unsigned long long *>(state);
    const int *cnts = reinterpret_cast<const int *>(keys + (size_t)nq * TK_TOTAL);
    topk_finish_kernel<<<(unsigned)nq, TK_THREADS, 0, s>>>(keys, cnts, k, idx, score);
    if (launches) ++*launches;
    return cudaGetLastError();
}

}  // namespace pinsage

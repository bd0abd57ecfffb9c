// subset.cu -- Algorithm 2 lines 1-7: the K-hop sets of a minibatch M,
//   S^(K) = M,   S^(k-1) = S^(k) U N(u) for u in S^(k),
// and the re-indexing of the sub-tables ("re-indexing ... to create a sub-graph")
// that lets the full-graph kernels run on the closure only (targeted / incremental inference).
//
// A set is kept three ways: a byte flag per node, its sorted member list, and pos[v] = rank of v in
// the list.  Flags -> list is a three-kernel compaction (per-block counts, scan of the counts,
// scatter), so lists come out in ascending id order without a sort.  Integer work throughout.
#include "internal.h"

#include <algorithm>

namespace pinsage {
namespace {

constexpr int CB = 1024;   // nodes per compaction block

__global__ void mark_targets_kernel(const int *__restrict__ targets, long long M, long long N,
                                    unsigned char *__restrict__ mark, long long *__restrict__ first_bad)
{
    const long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= M) return;
    const int v = targets[j];
    if (v < 0 || v >= N) {
        atomicMin(first_bad, j);
        return;
    }
    mark[v] = 1;
}

// mark_prev[v] = 1 for every member v of the list and for each of its T neighbours (one warp per member)
__global__ void __launch_bounds__(256)
expand_marks_kernel(const int *__restrict__ list, long long n, const int *__restrict__ idx, int T,
                    unsigned char *__restrict__ mark_prev)
{
    const long long i = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (i >= n) return;
    const int lane = threadIdx.x & 31;
    const long long v = list[i];
    if (lane == 0) mark_prev[v] = 1;
    for (int t = lane; t < T; t += 32) mark_prev[idx[v * T + t]] = 1;
}

__global__ void __launch_bounds__(256)
block_count_kernel(const unsigned char *__restrict__ mark, long long N, long long *__restrict__ counts)
{
    __shared__ int wsum[8];
    const long long base = (long long)blockIdx.x * CB;
    int c = 0;
    for (int i = threadIdx.x; i < CB; i += 256) c += (base + i < N && mark[base + i]) ? 1 : 0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
    if ((threadIdx.x & 31) == 0) wsum[threadIdx.x >> 5] = c;
    __syncthreads();
    if (threadIdx.x == 0) {
        int t = 0;
        for (int w = 0; w < 8; ++w) t += wsum[w];
        counts[blockIdx.x] = t;
    }
}

// exclusive scan of counts[0 .. nb) in place, total to counts[nb]; one CTA of 1024 threads
__global__ void __launch_bounds__(1024) scan_counts_kernel(long long *__restrict__ counts, long long nb)
{
    __shared__ long long part[1024];
    const long long per = (nb + 1023) / 1024;
    const long long b0 = (long long)threadIdx.x * per, b1 = min(nb, b0 + per);
    long long s = 0;
    for (long long b = b0; b < b1; ++b) s += counts[b];
    part[threadIdx.x] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        long long run = 0;
        for (int i = 0; i < 1024; ++i) {
            const long long t = part[i];
            part[i] = run;
            run += t;
        }
        counts[nb] = run;
    }
    __syncthreads();
    long long run = part[threadIdx.x];
    for (long long b = b0; b < b1; ++b) {
        const long long t = counts[b];
        counts[b] = run;
        run += t;
    }
}

// list[offset[b] + rank within block] = v and pos[v] = that index, for every flagged v (ascending)
__global__ void __launch_bounds__(256)
scatter_kernel(const unsigned char *__restrict__ mark, long long N, const long long *__restrict__ offsets,
               int *__restrict__ list, int *__restrict__ pos)
{
    __shared__ int wbase[8];
    const long long base = (long long)blockIdx.x * CB;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    long long run = offsets[blockIdx.x];
    for (int chunk = 0; chunk < CB; chunk += 256) {      // 256 consecutive nodes per pass, in id order
        const long long v = base + chunk + threadIdx.x;
        const bool f = v < N && mark[v];
        const unsigned b = __ballot_sync(0xffffffffu, f);
        if (lane == 0) wbase[wid] = __popc(b);
        __syncthreads();
        int before = 0, total = 0;
        for (int w = 0; w < 8; ++w) {
            before += w < wid ? wbase[w] : 0;
            total += wbase[w];
        }
        if (f) {
            const long long p = run + before + __popc(b & ((1u << lane) - 1u));
            list[p] = (int)v;
            pos[v] = (int)p;
        }
        run += total;
        __syncthreads();
    }
}

// dst[i, :] = src[row(i), :],  row(i) = map ? map[ids[i]] : ids[i];  rows of chunks16 16-byte words
__global__ void __launch_bounds__(256)
gather_rows_kernel(const uint4 *__restrict__ src, const int *__restrict__ ids, const int *__restrict__ map,
                   long long n, int chunks16, uint4 *__restrict__ dst)
{
    const long long total = n * chunks16;
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < total;
         e += (long long)gridDim.x * blockDim.x) {
        const long long i = e / chunks16;
        const int c = (int)(e - i * chunks16);
        int r = ids[i];
        if (map) r = map[r];
        dst[e] = src[(size_t)r * chunks16 + c];
    }
}

// idx_loc[i, t] = pos_prev[idx[list[i], t]],  w_loc[i, t] = w[list[i], t]
__global__ void __launch_bounds__(256)
remap_tables_kernel(const int *__restrict__ list, long long n, const int *__restrict__ idx,
                    const float *__restrict__ w, int T, const int *__restrict__ pos_prev,
                    int *__restrict__ idx_loc, float *__restrict__ w_loc)
{
    const long long total = n * T;
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < total;
         e += (long long)gridDim.x * blockDim.x) {
        const long long i = e / T;
        const int t = (int)(e - i * T);
        const long long g = (long long)list[i] * T + t;
        idx_loc[e] = pos_prev[idx[g]];
        w_loc[e] = w[g];
    }
}

__global__ void set_ll_kernel(long long *p, long long v) { *p = v; }

inline unsigned grid_for(long long total)
{
    long long b = (total + 255) / 256;
    return (unsigned)std::max<long long>(1, std::min<long long>(b, 148LL * 32));
}

}  // namespace

long long subset_blocks(int64_t N) { return (N + CB - 1) / CB; }

cudaError_t subset_mark_targets(const int32_t *targets, int64_t M, int64_t N, unsigned char *mark,
                                long long *first_bad, cudaStream_t s, int *launches)
{
    set_ll_kernel<<<1, 1, 0, s>>>(first_bad, 0x7fffffffffffffffLL);
    mark_targets_kernel<<<(unsigned)((M + 255) / 256), 256, 0, s>>>(targets, M, N, mark, first_bad);
    if (launches) *launches += 2;
    return cudaGetLastError();
}

cudaError_t subset_expand(const int32_t *list, int64_t n, const int32_t *idx, int32_t T,
                          unsigned char *mark_prev, cudaStream_t s, int *launches)
{
    if (n <= 0) return cudaSuccess;
    expand_marks_kernel<<<(unsigned)((n + 7) / 8), 256, 0, s>>>(list, n, idx, T, mark_prev);
    if (launches) ++*launches;
    return cudaGetLastError();
}

// counts: device scratch of subset_blocks(N) + 1 int64; after the call counts[nb] holds |set| (device)
cudaError_t subset_compact(const unsigned char *mark, int64_t N, long long *counts, int32_t *list,
                           int32_t *pos, bool scatter, cudaStream_t s, int *launches)
{
    const long long nb = subset_blocks(N);
    if (!scatter) {
        block_count_kernel<<<(unsigned)nb, 256, 0, s>>>(mark, N, counts);
        scan_counts_kernel<<<1, 1024, 0, s>>>(counts, nb);
        if (launches) *launches += 2;
    } else {
        scatter_kernel<<<(unsigned)nb, 256, 0, s>>>(mark, N, counts, list, pos);
        if (launches) ++*launches;
    }
    return cudaGetLastError();
}

cudaError_t subset_gather_rows(const void *src, const int32_t *ids, const int32_t *map, int64_t n,
                               size_t row_bytes, void *dst, cudaStream_t s, int *launches)
{
    if (n <= 0) return cudaSuccess;
    const int chunks16 = (int)(row_bytes / 16);
    gather_rows_kernel<<<grid_for(n * chunks16), 256, 0, s>>>(static_cast<const uint4 *>(src), ids, map, n,
                                                              chunks16, static_cast<uint4 *>(dst));
    if (launches) ++*launches;
    return cudaGetLastError();
}

cudaError_t subset_remap_tables(const int32_t *list, int64_t n, const int32_t *idx, const float *w,
                                int32_t T, const int32_t *pos_prev, int32_t *idx_loc, float *w_loc,
                                cudaStream_t s, int *launches)
{
    if (n <= 0) return cudaSuccess;
    remap_tables_kernel<<<grid_for(n * T), 256, 0, s>>>(list, n, idx, w, T, pos_prev, idx_loc, w_loc);
    if (launches) ++*launches;
    return cudaGetLastError();
}

}  // namespace pinsage

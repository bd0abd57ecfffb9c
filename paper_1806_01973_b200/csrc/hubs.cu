// hubs.cu -- the hub part of the S2 pool on skewed graphs as a dense contraction.
//
// N(u) = the T nodes with the highest visit counts of random walks from u.  On a
// graph with a power-law degree distribution (BASELINE config 4) a few hundred "hub" nodes sit in
// almost every neighbourhood: the pool n_u = sum_t alpha_ut P[idx_ut] (Alg. 1 l.1) then spends most of
// its gathers on the same few rows, and is bound by the SM's L1 / issue rate instead of by HBM
// (profiles/r01_pool_cfg4.md).  Splitting the sum over the neighbour's kind,
//     n_u = sum_{t: idx_ut not a hub} alpha_ut P[idx_ut]  +  sum_h A[u, h] P[hub_h],
//     A[u, h] = sum_{t: idx_ut = hub_h} alpha_ut,
// the first term is a gather over what is left of the lists and the second a dense contraction.  It is
// not even formed: S3 multiplies n by W2 (Alg. 1 l.2), and  (A P_hub) W2^T = A (P_hub W2^T), so the hub
// term enters S3 as a THIRD K segment -- A [n x H] against the small matrix G = P_hub W2^T [H x d],
// computed once per layer on the tensor cores in fp32.  A and G are rounded to bf16 (K3 = H), their
// products are exact and the sum is fp32: the hub term carries two independent 2^-9 roundings per
// product, averaged over the node's hub entries, where the plain path rounds all of n to bf16 (2^-9
// per element, not averaged) before S3 -- the same error level, a different rounding.  Which nodes are
// hubs is a choice, not part of the result: any set gives the same z in real arithmetic.
//
// Kernels: sampled visit histogram -> candidates -> top-H selection (one CTA) and rank table ->
// remapped index table (hub entries become -(rank + 1), which the pool kernel skips) -> per layer the
// hub rows of P and the extended weight matrix [W1 | W2 | G^T], per chunk the matrix A.
#include "internal.h"

#include <algorithm>

namespace pinsage {
namespace {

constexpr int HUB_CAND = 2048;   // candidate ids whose sampled count can reach the threshold (see hub_cmin)

__global__ void __launch_bounds__(256)
hub_count_kernel(const int *__restrict__ idx, long long rows, long long row_stride, int T, int *__restrict__ counts)
{
    const long long total = rows * T;
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < total;
         e += (long long)gridDim.x * blockDim.x) {
        const long long r = e / T;
        const int t = (int)(e - r * T);
        atomicAdd(counts + idx[r * row_stride * T + t], 1);
    }
}

// ids with counts[i] >= cmin: at most sum(counts) / cmin of them, HUB_CAND by the choice of cmin
__global__ void __launch_bounds__(256)
hub_candidates_kernel(const int *__restrict__ counts, long long n, int cmin, unsigned long long *__restrict__ cand,
                      int *__restrict__ n_cand)
{
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n;
         i += (long long)gridDim.x * blockDim.x) {
        const int c = counts[i];
        if (c >= cmin) {
            const int slot = atomicAdd(n_cand, 1);
            if (slot < HUB_CAND) cand[slot] = ((unsigned long long)(unsigned)c << 32) | (0xFFFFFFFFu - (unsigned)i);
        }
    }
}

// one CTA: sort the candidates (count descending, id ascending), keep H, write hub_ids [H] (-1 beyond
// the number found), rank[id] = position, info = {hubs found, sampled entries they cover}
__global__ void __launch_bounds__(1024)
hub_select_kernel(const unsigned long long *__restrict__ cand, const int *__restrict__ n_cand, int H,
                  int *__restrict__ hub_ids, int *__restrict__ rank, long long *__restrict__ info)
{
    __shared__ unsigned long long s[HUB_CAND];
    __shared__ long long cover;
    const int nc = min(*n_cand, HUB_CAND);
    for (int i = threadIdx.x; i < HUB_CAND; i += blockDim.x) s[i] = i < nc ? cand[i] : 0ull;
    if (threadIdx.x == 0) cover = 0;
    __syncthreads();
    for (int k = 2; k <= HUB_CAND; k <<= 1)
        for (int j = k >> 1; j > 0; j >>= 1) {
            for (int i = threadIdx.x; i < HUB_CAND; i += blockDim.x) {
                const int l = i ^ j;
                if (l > i) {
                    const unsigned long long a = s[i], b = s[l];
                    if ((a < b) == ((i & k) == 0)) {
                        s[i] = b;
                        s[l] = a;
                    }
                }
            }
            __syncthreads();
        }
    const int found = min(H, nc);
    long long mine = 0;
    for (int r = threadIdx.x; r < H; r += blockDim.x) {
        int id = -1;
        if (r < found) {
            id = (int)(0xFFFFFFFFu - (unsigned)(s[r] & 0xFFFFFFFFull));
            rank[id] = r;
            mine += (long long)(s[r] >> 32);
        }
        hub_ids[r] = id;
    }
    atomicAdd(reinterpret_cast<unsigned long long *>(&cover), (unsigned long long)mine);
    __syncthreads();
    if (threadIdx.x == 0) {
        info[0] = found;
        info[1] = cover;
    }
}

__global__ void __launch_bounds__(256)
hub_remap_kernel(const int *__restrict__ idx, const int *__restrict__ rank, long long total, int *__restrict__ out)
{
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < total;
         e += (long long)gridDim.x * blockDim.x) {
        const int id = idx[e];
        const int r = rank[id];
        out[e] = r >= 0 ? -(r + 1) : id;
    }
}

// Targeted inference (pinsage_embed_nodes): the sub-table idx_loc [n x T] of the members list[0..n) holds
// positions inside the previous set; entries whose WHOLE-GRAPH id is a hub become -(rank + 1) instead, as
// in the remapped whole-graph table, so that the closure runs the same split as the whole graph.
__global__ void __launch_bounds__(256)
hub_remap_sub_kernel(const int *__restrict__ list, long long n, const int *__restrict__ idx, int T,
                     const int *__restrict__ rank, int *__restrict__ idx_loc)
{
    const long long total = n * T;
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < total;
         e += (long long)gridDim.x * blockDim.x) {
        const long long i = e / T;
        const int t = (int)(e - i * T);
        const int r = rank[idx[(long long)list[i] * T + t]];
        if (r >= 0) idx_loc[e] = -(r + 1);
    }
}

// hub_loc[h] = position of hub h inside the previous set (its row of the compact P), or -1 when no member
// lists it (its column of A is then zero, and so is the row of P_hub that stands for it)
__global__ void hub_localize_kernel(const int *__restrict__ hub_ids, int H, const unsigned char *__restrict__ mark,
                                    const int *__restrict__ pos, int *__restrict__ hub_loc)
{
    const int h = blockIdx.x * blockDim.x + threadIdx.x;
    if (h >= H) return;
    const int id = hub_ids[h];
    hub_loc[h] = (id >= 0 && mark[id]) ? pos[id] : -1;
}

// A [rows x H] bf16, A[u, h] = sum of the weights of u's entries that point at hub h (mean aggregator:
// 1/T each), summed in table order without atomics (the same scheme as pool.cu's hub_accumulate, so the
// stand-alone kernel and the gather kernel's fused form give the same bits).  One warp per node.
__global__ void __launch_bounds__(256)
hub_matrix_kernel(const int *__restrict__ idxm, const float *__restrict__ w, long long rows, int T, int H, int mean,
                  __nv_bfloat16 *__restrict__ A)
{
    extern __shared__ float hub_smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    float *buf = hub_smem + (size_t)warp * H;
    const long long v = (long long)blockIdx.x * 8 + warp;
    if (v >= rows) return;
    for (int h = lane; h < H; h += 32) buf[h] = 0.f;
    __syncwarp();
    const float wmean = 1.0f / (float)T;
    for (int tb = 0; tb < T; tb += 32) {
        const int t = tb + lane;
        const int i = t < T ? idxm[v * T + t] : 0;
        const bool is_hub = t < T && i < 0;
        const float wt = is_hub ? (mean ? wmean : w[v * T + t]) : 0.f;
        const unsigned hm = __ballot_sync(0xffffffffu, is_hub);
        if (hm == 0) continue;
        if (is_hub) {
            const int r = -(i + 1);
            const unsigned peers = __match_any_sync(hm, r);
            const int leader = __ffs(peers) - 1;
            float sum = lane == leader ? buf[r] : 0.f;
            for (unsigned rem = peers; rem; rem &= rem - 1) sum += __shfl_sync(peers, wt, __ffs(rem) - 1);
            if (lane == leader) buf[r] = sum;
        }
        __syncwarp();
    }
    __nv_bfloat16 *row = A + v * H;
    for (int h = lane; h < H; h += 32) row[h] = __float2bfloat16_rn(buf[h]);
}

// Ph [H x pw] = the hub rows of P (zero rows for unused hub slots)
__global__ void __launch_bounds__(256)
hub_gather_kernel(const __nv_bfloat16 *__restrict__ P, const int *__restrict__ hub_ids, int H, int pw,
                  __nv_bfloat16 *__restrict__ Ph)
{
    const int total = H * pw;
    for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < total; e += gridDim.x * blockDim.x) {
        const int h = e / pw, c = e - h * pw;
        const int id = hub_ids[h];
        Ph[e] = id >= 0 ? P[(size_t)id * pw + c] : __float2bfloat16_rn(0.f);
    }
}

// Wext [d x (kw + H)] bf16: columns [0, kw) = W (row stride kw), then G^T with G [H x d] fp32 (G[h, j]
// multiplies A[u, h] in output column j): Wext[j, kw + h] = bf16(G[h, j])
__global__ void __launch_bounds__(256)
hub_weights_kernel(const __nv_bfloat16 *__restrict__ W, int kw, const float *__restrict__ G, int H, int d,
                   __nv_bfloat16 *__restrict__ Wext)
{
    const int ld = kw + H;
    const long long total = (long long)d * ld;
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < total;
         e += (long long)gridDim.x * blockDim.x) {
        const int j = (int)(e / ld), c = (int)(e - (long long)j * ld);
        if (c < kw) {
            Wext[e] = W[(size_t)j * kw + c];
        } else {
            Wext[e] = __float2bfloat16_rn(G[(size_t)(c - kw) * d + j]);
        }
    }
}

inline unsigned grid_for(long long total)
{
    return (unsigned)std::max<long long>(1, std::min<long long>((total + 255) / 256, 148LL * 16));
}

}  // namespace

// Sampled histogram of the neighbour ids (every row_stride-th row of idx [N x T]), the H most frequent
// ids and their rank table.  counts / rank: device int32 [n_src] (rank is filled with -1 here); cand:
// device scratch of 2048 keys + one int; hub_ids: device int32 [H]; info: device int64 [2] = {hubs
// found, sampled entries they cover}.  Returns the number of sampled entries in *sampled.
cudaError_t launch_hub_select(const int32_t *idx, int64_t N, int32_t T, int64_t n_src, int32_t H,
                              int32_t *counts, int32_t *rank, void *cand, int32_t *hub_ids, long long *info,
                              int64_t *sampled, cudaStream_t s, int *launches)
{
    const int64_t rows = std::min<int64_t>(N, 16384), stride = N / rows;
    const int64_t entries = rows * T;
    *sampled = entries;
    unsigned long long *keys = static_cast<unsigned long long *>(cand);
    int *n_cand = reinterpret_cast<int *>(keys + HUB_CAND);
    cudaError_t e = cudaMemsetAsync(counts, 0, (size_t)n_src * 4, s);
    if (e == cudaSuccess) e = cudaMemsetAsync(rank, 0xFF, (size_t)n_src * 4, s);
    if (e == cudaSuccess) e = cudaMemsetAsync(n_cand, 0, 4, s);
    if (e != cudaSuccess) return e;
    hub_count_kernel<<<grid_for(entries), 256, 0, s>>>(idx, rows, stride, T, counts);
    // an id needs cmin hits to be a candidate; at most entries / cmin <= HUB_CAND ids can have them
    const int cmin = (int)std::max<int64_t>(2, (entries + HUB_CAND - 1) / HUB_CAND);
    hub_candidates_kernel<<<grid_for(n_src), 256, 0, s>>>(counts, n_src, cmin, keys, n_cand);
    hub_select_kernel<<<1, 1024, 0, s>>>(keys, n_cand, H, hub_ids, rank, info);
    if (launches) *launches += 3;
    return cudaGetLastError();
}

size_t hub_cand_bytes() { return (size_t)HUB_CAND * 8 + 256; }

cudaError_t launch_hub_remap(const int32_t *idx, const int32_t *rank, int64_t total, int32_t *out,
                             cudaStream_t s, int *launches)
{
    hub_remap_kernel<<<grid_for(total), 256, 0, s>>>(idx, rank, total, out);
    if (launches) ++*launches;
    return cudaGetLastError();
}

cudaError_t launch_hub_remap_sub(const int32_t *list, int64_t n, const int32_t *idx, int32_t T, const int32_t *rank,
                                 int32_t *idx_loc, cudaStream_t s, int *launches)
{
    if (n <= 0) return cudaSuccess;
    hub_remap_sub_kernel<<<grid_for(n * (long long)T), 256, 0, s>>>(list, n, idx, T, rank, idx_loc);
    if (launches) ++*launches;
    return cudaGetLastError();
}

cudaError_t launch_hub_localize(const int32_t *hub_ids, int32_t H, const unsigned char *mark, const int32_t *pos,
                                int32_t *hub_loc, cudaStream_t s, int *launches)
{
    hub_localize_kernel<<<(H + 255) / 256, 256, 0, s>>>(hub_ids, H, mark, pos, hub_loc);
    if (launches) ++*launches;
    return cudaGetLastError();
}

cudaError_t launch_hub_matrix(const int32_t *idxm, const float *w, int64_t rows, int32_t T, int32_t H,
                              int mean, void *A, cudaStream_t s, int *launches)
{
    if (rows <= 0) return cudaSuccess;
    hub_matrix_kernel<<<(unsigned)((rows + 7) / 8), 256, (size_t)8 * H * 4, s>>>(
        idxm, w, rows, T, H, mean, static_cast<__nv_bfloat16 *>(A));
    if (launches) ++*launches;
    return cudaGetLastError();
}

cudaError_t launch_hub_gather(const void *P, const int32_t *hub_ids, int32_t H, int32_t pw, void *Ph,
                              cudaStream_t s, int *launches)
{
    hub_gather_kernel<<<grid_for((long long)H * pw), 256, 0, s>>>(static_cast<const __nv_bfloat16 *>(P), hub_ids, H,
                                                                  pw, static_cast<__nv_bfloat16 *>(Ph));
    if (launches) ++*launches;
    return cudaGetLastError();
}

cudaError_t launch_hub_weights(const void *W, int32_t kw, const float *G, int32_t H, int32_t d, void *Wext,
                               cudaStream_t s, int *launches)
{
    hub_weights_kernel<<<grid_for((long long)d * (kw + H)), 256, 0, s>>>(
        static_cast<const __nv_bfloat16 *>(W), kw, G, H, d, static_cast<__nv_bfloat16 *>(Wext));
    if (launches) ++*launches;
    return cudaGetLastError();
}

}  // namespace pinsage

// pool.cu -- S2, the importance pool (PAPER.md:114 gamma, :124 "importance pooling";
// sec. 3.4 job 2 :219):   n[v] = sum_{t<T} w[v,t] * P[idx[v,t], :]
//
// HBM-bound gather-weighted-sum.  A group of LPN lanes owns one destination node; every lane
// owns CPL 16-byte chunks of the feature row and keeps their fp32 partial sums in registers.
// The node's (id, weight) pairs are read once with a coalesced load and broadcast with warp
// shuffles; U neighbour rows are requested before the first FMA so that U*CPL 16-byte loads
// per lane are in flight.  The sum over t runs in table order per lane: no atomics, no
// cross-lane reduction, bit-reproducible.  Row offsets are 64-bit.
//
// Also here: the L1-normalisation of visit counts and table validation.
#include "internal.h"

#include <algorithm>
#include <climits>

namespace pinsage {
namespace {

__device__ __forceinline__ int ld_stream_i32(const int *p)
{
    int v;
    asm("ld.global.nc.L1::no_allocate.s32 %0, [%1];" : "=r"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ float ld_stream_f32(const float *p)
{
    float v;
    asm("ld.global.nc.L1::no_allocate.f32 %0, [%1];" : "=f"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ uint4 ld_row16(const uint4 *p)
{
    uint4 v;
    asm volatile("ld.global.nc.v4.u32 {%0, %1, %2, %3}, [%4];"
                 : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w)
                 : "l"(p));
    return v;
}
// L2 cache-policy variants: gathered rows are worth keeping (evict_last), tables are read once
__device__ __forceinline__ uint4 ld_row16_keep(const uint4 *p, uint64_t pol)
{
    uint4 v;
    asm volatile("ld.global.nc.L2::cache_hint.v4.u32 {%0, %1, %2, %3}, [%4], %5;"
                 : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w)
                 : "l"(p), "l"(pol));
    return v;
}
__device__ __forceinline__ int ld_once_i32(const int *p, uint64_t pol)
{
    int v;
    asm("ld.global.nc.L1::no_allocate.L2::cache_hint.s32 %0, [%1], %2;" : "=r"(v) : "l"(p), "l"(pol));
    return v;
}
__device__ __forceinline__ float ld_once_f32(const float *p, uint64_t pol)
{
    float v;
    asm("ld.global.nc.L1::no_allocate.L2::cache_hint.f32 %0, [%1], %2;" : "=f"(v) : "l"(p), "l"(pol));
    return v;
}
__device__ __forceinline__ void st_stream16(uint4 *p, const uint4 &v)
{
    asm volatile("st.global.cs.v4.u32 [%0], {%1, %2, %3, %4};" ::"l"(p), "r"(v.x), "r"(v.y),
                 "r"(v.z), "r"(v.w)
                 : "memory");
}

template <bool BF16>
struct Chunk;

template <>
struct Chunk<true> {  // 8 bf16 per 16 bytes
    static constexpr int E = 8;
    static __device__ __forceinline__ void fma(const uint4 &r, float wt, float (&acc)[8])
    {
        const uint32_t u[4] = {r.x, r.y, r.z, r.w};
#pragma unroll
        for (int i = 0; i < 4; ++i) {                      // packed fp32x2 FMA (sm_100): same two IEEE fmas, one issue slot
            const float2 z = __ffma2_rn(make_float2(wt, wt),
                                        make_float2(__uint_as_float(u[i] << 16), __uint_as_float(u[i] & 0xffff0000u)),
                                        make_float2(acc[2 * i], acc[2 * i + 1]));
            acc[2 * i] = z.x;
            acc[2 * i + 1] = z.y;
        }
    }
    static __device__ __forceinline__ void vmax(const uint4 &r, float (&acc)[8])
    {
        const uint32_t u[4] = {r.x, r.y, r.z, r.w};
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            acc[2 * i] = fmaxf(acc[2 * i], __uint_as_float(u[i] << 16));
            acc[2 * i + 1] = fmaxf(acc[2 * i + 1], __uint_as_float(u[i] & 0xffff0000u));
        }
    }
    static __device__ __forceinline__ uint4 pack(const float (&acc)[8])
    {
        uint32_t u[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            __nv_bfloat162 b = __floats2bfloat162_rn(acc[2 * i], acc[2 * i + 1]);
            u[i] = *reinterpret_cast<uint32_t *>(&b);
        }
        return make_uint4(u[0], u[1], u[2], u[3]);
    }
};

template <>
struct Chunk<false> {  // 4 fp32 per 16 bytes
    static constexpr int E = 4;
    static __device__ __forceinline__ void fma(const uint4 &r, float wt, float (&acc)[4])
    {
        acc[0] = fmaf(wt, __uint_as_float(r.x), acc[0]);
        acc[1] = fmaf(wt, __uint_as_float(r.y), acc[1]);
        acc[2] = fmaf(wt, __uint_as_float(r.z), acc[2]);
        acc[3] = fmaf(wt, __uint_as_float(r.w), acc[3]);
    }
    static __device__ __forceinline__ void vmax(const uint4 &r, float (&acc)[4])
    {
        acc[0] = fmaxf(acc[0], __uint_as_float(r.x));
        acc[1] = fmaxf(acc[1], __uint_as_float(r.y));
        acc[2] = fmaxf(acc[2], __uint_as_float(r.z));
        acc[3] = fmaxf(acc[3], __uint_as_float(r.w));
    }
    static __device__ __forceinline__ uint4 pack(const float (&acc)[4])
    {
        return make_uint4(__float_as_uint(acc[0]), __float_as_uint(acc[1]),
                          __float_as_uint(acc[2]), __float_as_uint(acc[3]));
    }
};

// A[v, r] += w for the lanes of one 32-entry batch whose entry names hub r (idx = -(r + 1)), in TABLE
// ORDER and without atomics: the lanes that name the same hub find each other with a match, the lowest
// one adds their weights lane by lane to the running sum in shared memory.  Batches follow each other
// in table order, so A[v, r] is the sum a sequential loop over t = 0..T-1 would form, bit for bit
// (a list may legally name a hub several times: reading A7).  Called by all 32 lanes of the warp.
__device__ __forceinline__ void hub_accumulate(float *hbuf, int *claim, bool is_hub, int my_i, float my_w, int lane)
{
    const unsigned hm = __ballot_sync(0xffffffffu, is_hub);
    if (hm == 0) return;                                   // (warp-uniform)
    // Is any hub named twice in this batch?  Every hub lane signs claim[r]; a hub named by two lanes leaves at
    // least one of them reading the other's signature.  (A shared-memory round trip instead of a MATCH.ANY,
    // whose result was the largest single stall of the kernel; lists rarely repeat an id.)
    const int r = is_hub ? -(my_i + 1) : 0;
    if (is_hub) claim[r] = lane;
    __syncwarp();
    const unsigned dup = __ballot_sync(0xffffffffu, is_hub && claim[r] != lane);
    if (dup == 0) {                                        // the usual case: every hub named once
        if (is_hub) hbuf[r] += my_w;
    } else if (is_hub) {
        const unsigned peers = __match_any_sync(hm, r);
        const int leader = __ffs(peers) - 1;
        float sum = lane == leader ? hbuf[r] : 0.f;
        for (unsigned rem = peers; rem; rem &= rem - 1) {
            const float wv = __shfl_sync(peers, my_w, __ffs(rem) - 1);
            sum += wv;                                     // (only the leader's sum is used)
        }
        if (lane == leader) hbuf[r] = sum;
    }
    __syncwarp();                                          // the next batch may update the same sums from other lanes
}

// UU neighbour rows (slots j0 .. j0+UU-1 of the current batch) for one lane: every one of the
// UU*CPL 16-byte loads is issued before the first FMA (memory-level parallelism).
// MODE: 0 importance pooling (weighted sum), 1 element-wise mean (my_w holds 1/T in every lane),
// 2 element-wise max -- the aggregator variants of PAPER.md:118, :262-263.
template <bool BF16, int LPN, int CPL, int UU, bool EXACT, int MODE>
__device__ __forceinline__ void gather_fma(const uint4 *__restrict__ P, int my_i, float my_w, int j0,
                                           int sl, int chunks,
                                           float (&acc)[CPL][Chunk<BF16>::E])
{
    using C = Chunk<BF16>;
    uint4 r[UU][CPL];
    float wt[UU];
    const uint4 *row[UU];
#pragma unroll
    for (int u = 0; u < UU; ++u) {
        const int id = __shfl_sync(0xffffffffu, my_i, j0 + u, LPN);
        wt[u] = MODE == 0 ? __shfl_sync(0xffffffffu, my_w, j0 + u, LPN) : my_w;
        row[u] = P + (size_t)id * (size_t)chunks + sl;
    }
#pragma unroll
    for (int u = 0; u < UU; ++u)
#pragma unroll
        for (int c = 0; c < CPL; ++c) {
            if (EXACT) r[u][c] = ld_row16(row[u] + c * LPN);
            else r[u][c] = (sl + c * LPN < chunks) ? ld_row16(row[u] + c * LPN) : make_uint4(0, 0, 0, 0);
        }
#pragma unroll
    for (int u = 0; u < UU; ++u)
#pragma unroll
        for (int c = 0; c < CPL; ++c) {
            if (MODE == 2) C::vmax(r[u][c], acc[c]);
            else C::fma(r[u][c], wt[u], acc[c]);
        }
}

// LPN lanes per node (4..32), CPL chunks per lane, U neighbour rows in flight,
// EXACT: the row is exactly LPN*CPL chunks wide (no per-chunk guard).
// An explicit minBlocksPerSM matters: without it ptxas (-O3) re-serialises the load batch to
// minimise registers (32 regs, 2 loads in flight); with it the U*CPL loads stay batched.
template <bool BF16, int LPN, int CPL, int U, bool EXACT, int MODE>
__global__ void __launch_bounds__(256, (CPL <= 2) ? (U == 1 ? 5 : 4) : 2)
pool_kernel(const uint4 *__restrict__ P, const int *__restrict__ idx, const float *__restrict__ w,
            uint4 *__restrict__ out, long long n_dst, int T, int chunks, int skip_neg,
            __nv_bfloat16 *__restrict__ hubA, int H)
{
    extern __shared__ __align__(16) float hub_acc[];       // hub mode (LPN == 32): H sums per warp
    __shared__ int2 squeeze[8][32];                        // skip_neg: the (id, weight) pairs that remain, per warp
    using C = Chunk<BF16>;
    constexpr int NPW = 32 / LPN;
    static_assert(LPN % U == 0, "U must divide LPN");
    const int lane = threadIdx.x & 31;
    const int sl = lane % LPN;
    // LOOP (the hub-split instantiations, one node per warp at a time): a warp walks nodes warp, warp + stride,
    // ... and requests the first table batch of its next node during the last batch of the current one, so that
    // no node starts with an exposed table latency.  Elsewhere: one pass, one node (group) per lane group.
    constexpr bool LOOP = U == 1 && CPL <= 2 && LPN == 32;
    const long long warp = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const long long wstride = (long long)gridDim.x * (blockDim.x >> 5);
    if (warp * NPW >= n_dst) return;                       // whole warp out of range
    const long long v_raw = warp * NPW + lane / LPN;
    const bool active = v_raw < n_dst;
    long long v = active ? v_raw : n_dst - 1;              // idle groups shadow the last node
    int nx_i = 0;
    float nx_w = 0.f;
    bool first = true;
  for (;;) {
    float acc[CPL][C::E];
#pragma unroll
    for (int c = 0; c < CPL; ++c)
#pragma unroll
        for (int e = 0; e < C::E; ++e) acc[c][e] = MODE == 2 ? -INFINITY : 0.f;

    const int *irow = idx + v * T;
    const float *wrow = w + v * T;
    float *hbuf = hub_acc + (size_t)(threadIdx.x >> 5) * H;
    int *claim = reinterpret_cast<int *>(hub_acc + (size_t)8 * H) + (size_t)(threadIdx.x >> 5) * H;   // (see hub_accumulate)
    if (hubA != nullptr) {                                 // (one node per warp: LPN == 32; H % 64 == 0)
        for (int h = lane * 4; h < H; h += 128) *reinterpret_cast<float4 *>(hbuf + h) = make_float4(0.f, 0.f, 0.f, 0.f);
        __syncwarp();
    }
    // the (id, weight) pairs of the NEXT batch are requested before the current batch's rows are gathered,
    // so that the table load is off the node's chain of dependent memory latencies
    if ((!LOOP || first) && sl < T) {
        nx_i = ld_stream_i32(irow + sl);
        if (MODE == 0) nx_w = ld_stream_f32(wrow + sl);
    }
    first = false;
    const long long v_next = v + wstride;                  // (LOOP only)
    for (int tb = 0; tb < T; tb += LPN) {
        const int t = tb + sl;
        int my_i = t < T ? nx_i : 0;
        float my_w = MODE == 1 ? 1.0f / (float)T : (t < T ? nx_w : 0.f);
        if (t + LPN < T) {
            nx_i = ld_stream_i32(irow + t + LPN);
            if (MODE == 0) nx_w = ld_stream_f32(wrow + t + LPN);
        }
        if (LOOP && tb + LPN >= T && v_next < n_dst && sl < T) {      // last batch: the next node's first one
            nx_i = ld_stream_i32(idx + v_next * T + sl);
            if (MODE == 0) nx_w = ld_stream_f32(w + v_next * T + sl);
        }
        int cnt = min(LPN, T - tb);
        if (hubA != nullptr)                               // hub entry -(rank + 1): its weight goes to A[v, rank]
            hub_accumulate(hbuf, claim, t < T && my_i < 0, my_i, my_w, lane);
        if (skip_neg) {
            // entries with a negative id (hub neighbours, summed by the hub GEMM: hubs.cu) are squeezed
            // out of this batch: lane k of a node's group takes the k-th remaining entry.  Groups of
            // one warp run the same number of steps (the shuffles below are warp-wide); a group that
            // has fewer entries pads with weight 0 on row 0.
            // (through shared memory: a live entry knows its rank among the live ones, i.e. where it goes;
            // __fns, which finds where an entry comes from, is a software loop of ~60 instructions)
            const bool lv = t < T && my_i >= 0;
            const unsigned live = __ballot_sync(0xffffffffu, lv);
            const int g0 = lane / LPN * LPN;
            const unsigned gm = LPN == 32 ? live : (live >> g0) & ((1u << (LPN & 31)) - 1u);
            int2 *sq = squeeze[threadIdx.x >> 5];
            __syncwarp();                                          // the previous batch has been read
            if (lv) sq[g0 + __popc(gm & ((1u << sl) - 1u))] = make_int2(my_i, __float_as_int(my_w));
            __syncwarp();
            const int n_live = __popc(gm);
            const int2 e = sq[g0 + sl];
            my_i = sl < n_live ? e.x : 0;
            my_w = sl < n_live ? __int_as_float(e.y) : 0.f;
            cnt = LPN == 32 ? n_live : __reduce_max_sync(0xffffffffu, n_live);
        }
        int j0 = 0;
        for (; j0 + U <= cnt; j0 += U)
            gather_fma<BF16, LPN, CPL, U, EXACT, MODE>(P, my_i, my_w, j0, sl, chunks, acc);
        // the remainder (< U rows) in at most three rounds of 4, 2 and 1 rows in flight, still in table
        // order (one row at a time would cost a memory latency each: T = 100 leaves 4 rows, T = 50 two)
        if (U > 4 && j0 + 4 <= cnt) {
            gather_fma<BF16, LPN, CPL, 4, EXACT, MODE>(P, my_i, my_w, j0, sl, chunks, acc);
            j0 += 4;
        }
        if (U > 2 && j0 + 2 <= cnt) {
            gather_fma<BF16, LPN, CPL, 2, EXACT, MODE>(P, my_i, my_w, j0, sl, chunks, acc);
            j0 += 2;
        }
        for (; j0 < cnt; ++j0)
            gather_fma<BF16, LPN, CPL, 1, EXACT, MODE>(P, my_i, my_w, j0, sl, chunks, acc);
    }
    if (hubA != nullptr) {                                 // A[v, :] = bf16 of the sums (hubs.cu)
        __syncwarp();
        __nv_bfloat16 *arow = hubA + (size_t)v * H;
        for (int h = lane * 8; h < H; h += 256) {          // eight sums per lane: one 16-byte store
            const float4 a = *reinterpret_cast<const float4 *>(hbuf + h);
            const float4 b = *reinterpret_cast<const float4 *>(hbuf + h + 4);
            const __nv_bfloat162 p0 = __floats2bfloat162_rn(a.x, a.y), p1 = __floats2bfloat162_rn(a.z, a.w);
            const __nv_bfloat162 p2 = __floats2bfloat162_rn(b.x, b.y), p3 = __floats2bfloat162_rn(b.z, b.w);
            *reinterpret_cast<uint4 *>(arow + h) =
                make_uint4(*reinterpret_cast<const uint32_t *>(&p0), *reinterpret_cast<const uint32_t *>(&p1),
                           *reinterpret_cast<const uint32_t *>(&p2), *reinterpret_cast<const uint32_t *>(&p3));
        }
    }
    if (active) {
        uint4 *orow = out + (size_t)v * (size_t)chunks;
#pragma unroll
        for (int c = 0; c < CPL; ++c) {
            const int ch = sl + c * LPN;
            if (EXACT || ch < chunks) st_stream16(orow + ch, C::pack(acc[c]));
        }
    }
    if (!LOOP || v_next >= n_dst) break;
    v = v_next;
    __syncwarp();                                          // hbuf / squeeze of this node have been read
  }
}

template <bool BF16, int LPN, int CPL, int U, int MODE>
cudaError_t run_pool(const void *P, const int *idx, const float *w, void *out, long long n_dst,
                     int T, int chunks, cudaStream_t s, int skip_neg = 0, void *hubA = nullptr, int H = 0)
{
    if (hubA != nullptr && LPN != 32) return cudaErrorNotSupported;
    const size_t smem = hubA != nullptr ? (size_t)8 * H * 8 : 0;      // per warp: H sums and H signatures
    __nv_bfloat16 *hA = static_cast<__nv_bfloat16 *>(hubA);
    constexpr int NPW = 32 / LPN;
    const long long warps = (n_dst + NPW - 1) / NPW;
    long long blocks = (warps + 7) / 8;
    // the looping (hub-split) instantiations: enough blocks to fill every SM a few times over, each warp
    // then walks ~16 nodes or more
    if (U == 1 && CPL <= 2 && LPN == 32) blocks = std::min<long long>(blocks, (long long)TUNED_SMS * 5 * 8);
    if (blocks > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    if (chunks == LPN * CPL)
        pool_kernel<BF16, LPN, CPL, U, true, MODE><<<(unsigned)blocks, 256, smem, s>>>(
            static_cast<const uint4 *>(P), idx, w, static_cast<uint4 *>(out), n_dst, T, chunks, skip_neg, hA, H);
    else
        pool_kernel<BF16, LPN, CPL, U, false, MODE><<<(unsigned)blocks, 256, smem, s>>>(
            static_cast<const uint4 *>(P), idx, w, static_cast<uint4 *>(out), n_dst, T, chunks, skip_neg, hA, H);
    return cudaGetLastError();
}

// ---- column-slab variant: keep the gathered table L2-resident -------------------------------------
// When P is larger than L2 but n_src * SLAB bytes fits in it, the pool runs slab by slab over the
// feature columns: pass s gathers only bytes [s*SLAB, (s+1)*SLAB) of every row, a strided sub-table
// of n_src * SLAB bytes that stays in L2 after its first touch, so P crosses HBM about once instead
// of ~T times.  The price is that the (id, weight) tables are re-read once per slab (they are
// streamed through shared memory, coalesced).  Slabs are the slow grid dimension: all CTAs of slab
// s are scheduled before those of slab s+1.  A group of LPN = SLAB/16 lanes owns one node, a warp
// owns 32/LPN consecutive nodes whose table entries are contiguous in memory.  Per element the
// sum still runs t = 0..T-1 in fp32: results are bit-identical to pool_kernel.
template <bool BF16, int LPN, int U>
__global__ void __launch_bounds__(256, 4)
pool_slab_kernel(const uint4 *__restrict__ P, const int *__restrict__ idx, const float *__restrict__ w,
                 uint4 *__restrict__ out, long long n_dst, int T, int chunks, unsigned blocks_per_slab)
{
    using C = Chunk<BF16>;
    constexpr int NPW = 32 / LPN;
    extern __shared__ __align__(16) unsigned char pool_smem[];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int sl = lane % LPN, grp = lane / LPN;
    const unsigned slab = blockIdx.x / blocks_per_slab, dblk = blockIdx.x % blocks_per_slab;
    const long long v0 = ((long long)dblk * 8 + wid) * NPW;     // first node of this warp
    if (v0 >= n_dst) return;
    const int nv = (int)min((long long)NPW, n_dst - v0);
    int *sidx = reinterpret_cast<int *>(pool_smem) + (size_t)wid * NPW * T * 2;
    float *sw = reinterpret_cast<float *>(sidx + NPW * T);
    const int *irow = idx + v0 * T;
    const float *wrow = w + v0 * T;
    uint64_t pol_keep, pol_once;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol_keep));
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol_once));
    for (int i = lane; i < nv * T; i += 32) {
        sidx[i] = ld_once_i32(irow + i, pol_once);
        sw[i] = ld_once_f32(wrow + i, pol_once);
    }
    __syncwarp();
    const bool active = grp < nv;
    const int g = active ? grp : nv - 1;
    const uint4 *base = P + (size_t)slab * LPN + sl;
    float acc[C::E];
#pragma unroll
    for (int e = 0; e < C::E; ++e) acc[e] = 0.f;
    const int *gi = sidx + g * T;
    const float *gw = sw + g * T;
    int t = 0;
    for (; t + U <= T; t += U) {
        uint4 r[U];
        float wt[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            r[u] = ld_row16_keep(base + (size_t)gi[t + u] * (size_t)chunks, pol_keep);
            wt[u] = gw[t + u];
        }
#pragma unroll
        for (int u = 0; u < U; ++u) C::fma(r[u], wt[u], acc);
    }
    for (; t < T; ++t) C::fma(ld_row16_keep(base + (size_t)gi[t] * (size_t)chunks, pol_keep), gw[t], acc);
    if (active)
        st_stream16(out + (size_t)(v0 + grp) * (size_t)chunks + (size_t)slab * LPN + sl, C::pack(acc));
}

template <bool BF16, int LPN>
cudaError_t run_pool_slab(const void *P, const int *idx, const float *w, void *out, long long n_dst,
                          int T, int chunks, cudaStream_t s)
{
    constexpr int NPW = 32 / LPN;
    constexpr int U = 10;
    const long long bps = (n_dst + 8 * NPW - 1) / (8 * NPW);
    const long long nslabs = chunks / LPN;
    if (bps * nslabs > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    const size_t smem = (size_t)8 * NPW * T * 8;
    auto kern = pool_slab_kernel<BF16, LPN, U>;
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    kern<<<(unsigned)(bps * nslabs), 256, smem, s>>>(static_cast<const uint4 *>(P), idx, w,
                                                      static_cast<uint4 *>(out), n_dst, T, chunks,
                                                      (unsigned)bps);
    return cudaGetLastError();
}

// slab_bytes in {32, 64, 128}; requires row bytes % slab_bytes == 0 and the staging to fit smem.
template <bool BF16>
cudaError_t dispatch_pool_slab(int slab_bytes, const void *P, const int *idx, const float *w, void *out,
                               long long n_dst, int T, int chunks, cudaStream_t s)
{
    switch (slab_bytes) {
    case 32: return run_pool_slab<BF16, 2>(P, idx, w, out, n_dst, T, chunks, s);
    case 64: return run_pool_slab<BF16, 4>(P, idx, w, out, n_dst, T, chunks, s);
    case 128: return run_pool_slab<BF16, 8>(P, idx, w, out, n_dst, T, chunks, s);
    }
    return cudaErrorNotSupported;
}

template <bool BF16, int MODE>
cudaError_t dispatch_pool(const void *P, const int *idx, const float *w, void *out,
                          long long n_dst, int T, int chunks, cudaStream_t s, int skip_neg = 0,
                          void *hubA = nullptr, int H = 0)
{
    // what is left of the lists after the hub entries is a handful of rows per node: the kernel is then
    // bound by the chain table load -> gather -> store, and more resident warps (U = 1: fewer
    // registers) beat deeper load batches (re-measured in round 2 at config 4, pool per step: U = 1 42.2 ms,
    // U = 2 42.8 ms, U = 4 43.8 ms)
    if (skip_neg && chunks > 32 && chunks <= 64)
        return run_pool<BF16, 32, 2, 1, MODE>(P, idx, w, out, n_dst, T, chunks, s, skip_neg, hubA, H);
    if (skip_neg && chunks > 16 && chunks <= 32)
        return run_pool<BF16, 32, 1, 1, MODE>(P, idx, w, out, n_dst, T, chunks, s, skip_neg, hubA, H);
    if (chunks <= 4) return run_pool<BF16, 4, 1, 4, MODE>(P, idx, w, out, n_dst, T, chunks, s, skip_neg, hubA, H);
    if (chunks <= 8) return run_pool<BF16, 8, 1, 8, MODE>(P, idx, w, out, n_dst, T, chunks, s, skip_neg, hubA, H);
    if (chunks <= 16) return run_pool<BF16, 16, 1, 8, MODE>(P, idx, w, out, n_dst, T, chunks, s, skip_neg, hubA, H);
    if (chunks <= 32) return run_pool<BF16, 32, 1, 8, MODE>(P, idx, w, out, n_dst, T, chunks, s, skip_neg, hubA, H);
    if (chunks <= 64) return run_pool<BF16, 32, 2, 4, MODE>(P, idx, w, out, n_dst, T, chunks, s, skip_neg, hubA, H);
    if (chunks <= 128) return run_pool<BF16, 32, 4, 4, MODE>(P, idx, w, out, n_dst, T, chunks, s, skip_neg, hubA, H);
    if (chunks <= 256) return run_pool<BF16, 32, 8, 1, MODE>(P, idx, w, out, n_dst, T, chunks, s, skip_neg, hubA, H);
    return cudaErrorNotSupported;
}

template <bool BF16>
cudaError_t dispatch_pool_mode(int mode, const void *P, const int *idx, const float *w, void *out,
                               long long n_dst, int T, int chunks, cudaStream_t s)
{
    if (mode == 1) return dispatch_pool<BF16, 1>(P, idx, w, out, n_dst, T, chunks, s);
    if (mode == 2) return dispatch_pool<BF16, 2>(P, idx, w, out, n_dst, T, chunks, s);
    return dispatch_pool<BF16, 0>(P, idx, w, out, n_dst, T, chunks, s);
}

// One warp per row: alpha = (float)c / (float)sum(c), IEEE binary32 division.
__global__ void __launch_bounds__(256)
normalize_counts_kernel(const int *__restrict__ counts, float *__restrict__ w, long long N, int T)
{
    const long long row = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (row >= N) return;
    const int lane = threadIdx.x & 31;
    const int *c = counts + row * T;
    long long tot = 0;
    for (int t = lane; t < T; t += 32) tot += c[t];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) tot += __shfl_xor_sync(0xffffffffu, tot, o);
    const float ftot = (float)tot;
    // a row without any visit (an isolated node of the neighbourhood builder) gets all-zero weights
    for (int t = lane; t < T; t += 32) w[row * T + t] = tot > 0 ? __fdiv_rn((float)c[t], ftot) : 0.f;
}

__global__ void __launch_bounds__(256)
validate_kernel(const int *__restrict__ idx, const float *__restrict__ w, long long total,
                long long n_src, long long *first_bad)
{
    long long best = LLONG_MAX;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < total;
         i += (long long)gridDim.x * blockDim.x) {
        const int id = idx[i];
        const float x = w[i];
        if (id < 0 || id >= n_src || !isfinite(x)) {
            best = i;
            break;
        }
    }
    if (best != LLONG_MAX) atomicMin(first_bad, best);
}

__global__ void set_ll(long long *p, long long v) { *p = v; }
__global__ void fix_first_bad(long long *p)
{
    if (*p == LLONG_MAX) *p = -1;
}

}  // namespace

bool pool_slab_ok(DType dt, int32_t T, int32_t m, int slab_bytes)
{
    if (slab_bytes != 32 && slab_bytes != 64 && slab_bytes != 128) return false;
    const size_t row = (size_t)m * elem_size(dt);
    const size_t smem = (size_t)8 * (32 / (slab_bytes / 16)) * T * 8;
    return row % slab_bytes == 0 && row > (size_t)slab_bytes && smem <= 200 * 1024;
}

bool pool_hub_fused_ok(DType dt, int32_t m)
{
    const size_t chunks = (size_t)m * elem_size(dt) / 16;
    return chunks > 16 && chunks <= 256;       // one node per warp (LPN == 32)
}

cudaError_t launch_pool(DType dt, int mode, int64_t n_dst, int32_t T, int32_t m, const void *P,
                        const int32_t *idx, const float *w, void *out, int slab_bytes, cudaStream_t s,
                        int *launches, int skip_neg, void *hubA, int H)
{
    if (n_dst <= 0) return cudaSuccess;
    const int chunks = (int)((size_t)m * elem_size(dt) / 16);
    if (launches) ++*launches;
    if (skip_neg) {                            // hub-split pool: importance pooling, whole rows
        if (mode != 0) return cudaErrorNotSupported;
        return dt == DType::BF16 ? dispatch_pool<true, 0>(P, idx, w, out, n_dst, T, chunks, s, 1, hubA, H)
                                 : dispatch_pool<false, 0>(P, idx, w, out, n_dst, T, chunks, s, 1, hubA, H);
    }
    if (mode != 0)
        return dt == DType::BF16 ? dispatch_pool_mode<true>(mode, P, idx, w, out, n_dst, T, chunks, s)
                                 : dispatch_pool_mode<false>(mode, P, idx, w, out, n_dst, T, chunks, s);
    if (slab_bytes > 0 && pool_slab_ok(dt, T, m, slab_bytes))
        return dt == DType::BF16
                   ? dispatch_pool_slab<true>(slab_bytes, P, idx, w, out, n_dst, T, chunks, s)
                   : dispatch_pool_slab<false>(slab_bytes, P, idx, w, out, n_dst, T, chunks, s);
    return dt == DType::BF16 ? dispatch_pool<true, 0>(P, idx, w, out, n_dst, T, chunks, s)
                             : dispatch_pool<false, 0>(P, idx, w, out, n_dst, T, chunks, s);
}

cudaError_t launch_normalize_counts(int64_t N, int32_t T, const int32_t *counts, float *w,
                                    cudaStream_t s, int *launches)
{
    const long long blocks = (N + 7) / 8;
    if (blocks > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    normalize_counts_kernel<<<(unsigned)blocks, 256, 0, s>>>(counts, w, N, T);
    if (launches) ++*launches;
    return cudaGetLastError();
}

cudaError_t launch_validate(int64_t n_dst, int64_t n_src, int32_t T, const int32_t *idx,
                            const float *w, long long *first_bad, cudaStream_t s, int *launches)
{
    const long long total = n_dst * (long long)T;
    set_ll<<<1, 1, 0, s>>>(first_bad, LLONG_MAX);
    long long blocks = (total + 255) / 256;
    if (blocks > TUNED_SMS * 16) blocks = TUNED_SMS * 16;
    if (blocks < 1) blocks = 1;
    validate_kernel<<<(unsigned)blocks, 256, 0, s>>>(idx, w, total, n_src, first_bad);
    fix_first_bad<<<1, 1, 0, s>>>(first_bad);
    if (launches) *launches += 3;
    return cudaGetLastError();
}

}  // namespace pinsage

// calib.cu -- calibration kernels for the roofline report (SURVEY.md sec. 8(d) "How to report the pool
// honestly"): what this very device delivers, on the day, to the access patterns of the S2 pool.
//
//   m1  read-only streaming reduction over a large buffer      -> the READ ceiling (the figure in
//       MEASURED_PEAKS.json is a copy: half reads, half writes)
//   m2  un-weighted random-row gather-sum, T rows of row_bytes each per destination, from a table far
//       larger than L2                                         -> the random-row gather ceiling from HBM
//   m3  the same from a table that fits L2                     -> the L2 / LSU ceiling (what bounds the
//       pool on the power-law config, where ~90 % of the gathers hit hub rows)
//
// They do strictly less than the pool: no (id, weight) table is read (ids come from a counter-based hash
// in registers), there is no multiply by a weight, and the sum is an integer XOR.  None of the method's arithmetic
// lives here and nothing on the product path calls these kernels; bench.py reports the pool against them.
#include "internal.h"

namespace pinsage {
namespace {

__device__ __forceinline__ uint4 ldg16_stream(const uint4 *p)
{
    uint4 v;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];"
                 : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w)
                 : "l"(p));
    return v;
}
__device__ __forceinline__ uint4 ldg16(const uint4 *p)
{
    uint4 v;
    asm volatile("ld.global.nc.v4.u32 {%0, %1, %2, %3}, [%4];"
                 : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w)
                 : "l"(p));
    return v;
}
__device__ __forceinline__ void xor16(uint4 &a, const uint4 &b)
{
    a.x ^= b.x; a.y ^= b.y; a.z ^= b.z; a.w ^= b.w;
}
// row id of (destination v, slot t): a 32-bit finaliser of the pair, scaled to [0, n_src) by a multiply-high
// (a dozen integer instructions per row; a 64-bit modulo would make the kernel ALU-bound)
__device__ __forceinline__ unsigned row_id(unsigned key, int t, unsigned n_src)
{
    unsigned x = (key + (unsigned)t) * 0x9E3779B1u;
    x ^= x >> 15; x *= 0x85EBCA77u;
    x ^= x >> 13; x *= 0xC2B2AE3Du;
    x ^= x >> 16;
    return __umulhi(x, n_src);
}

// m1: every warp streams contiguous 4 KB blocks (8 x 512-byte warp loads in flight per lane), block after
// block in grid order, so that the front the grid reads at any time is one contiguous range of memory;
// one word per thread is written at the end.
__global__ void __launch_bounds__(256, 8)
calib_stream_kernel(const uint4 *__restrict__ buf, long long words, uint4 *__restrict__ sink)
{
    uint4 acc = make_uint4(0, 0, 0, 0);
    const int lane = threadIdx.x & 31;
    const long long warps = (long long)gridDim.x * (blockDim.x >> 5);
    const long long gwarp = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const long long blocks = words / 256;                  // whole 4 KB blocks (256 words)
    for (long long b = gwarp; b < blocks; b += warps) {
        const uint4 *p = buf + b * 256 + lane;
        uint4 r[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) r[u] = ldg16_stream(p + u * 32);
#pragma unroll
        for (int u = 0; u < 8; ++u) xor16(acc, r[u]);
    }
    for (long long i = blocks * 256 + gwarp * 32 + lane; i < words; i += warps * 32) xor16(acc, ldg16_stream(buf + i));
    sink[(long long)blockIdx.x * blockDim.x + threadIdx.x] = acc;
}

// m2 / m3: LPN lanes own one destination; each lane owns CPL 16-byte chunks of the row; U rows are
// requested before the first XOR (the pool kernel's load batching).  Row ids: hash(v, t) mod n_src.
template <int LPN, int CPL, int U>
__global__ void __launch_bounds__(256, (CPL <= 2) ? 4 : 2)
calib_gather_kernel(const uint4 *__restrict__ table, long long n_src, long long n_dst, int T,
                    uint4 *__restrict__ out)
{
    constexpr int NPW = 32 / LPN;
    const int lane = threadIdx.x & 31, sl = lane % LPN;
    const long long warp = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const long long v = warp * NPW + lane / LPN;
    if (v >= n_dst) return;
    constexpr int chunks = LPN * CPL;
    uint4 acc[CPL];
#pragma unroll
    for (int c = 0; c < CPL; ++c) acc[c] = make_uint4(0, 0, 0, 0);
    const unsigned key = (unsigned)v * (unsigned)T * 0x01000193u + 0x811C9DC5u;
    int t = 0;
    for (; t + U <= T; t += U) {
        uint4 r[U][CPL];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const uint4 *row = table + (size_t)row_id(key, t + u, (unsigned)n_src) * chunks + sl;
#pragma unroll
            for (int c = 0; c < CPL; ++c) r[u][c] = ldg16(row + c * LPN);
        }
#pragma unroll
        for (int u = 0; u < U; ++u)
#pragma unroll
            for (int c = 0; c < CPL; ++c) xor16(acc[c], r[u][c]);
    }
    for (; t < T; ++t) {
        const uint4 *row = table + (size_t)row_id(key, t, (unsigned)n_src) * chunks + sl;
#pragma unroll
        for (int c = 0; c < CPL; ++c) xor16(acc[c], ldg16(row + c * LPN));
    }
    uint4 *orow = out + v * chunks + sl;
#pragma unroll
    for (int c = 0; c < CPL; ++c) orow[c * LPN] = acc[c];
}

template <int LPN, int CPL, int U>
cudaError_t run_gather(const void *table, long long n_src, long long n_dst, int T, void *out, cudaStream_t s)
{
    constexpr int NPW = 32 / LPN;
    const long long blocks = ((n_dst + NPW - 1) / NPW + 7) / 8;
    if (blocks > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    calib_gather_kernel<LPN, CPL, U><<<(unsigned)blocks, 256, 0, s>>>(static_cast<const uint4 *>(table), n_src, n_dst,
                                                                      T, static_cast<uint4 *>(out));
    return cudaGetLastError();
}

}  // namespace

// kind 0: stream `bytes` of buf (sink: num_sms * 8 * 256 16-byte words).  kind 1: gather, row_bytes in
// {256, 512, 1024, 2048}, table of n_src rows, out [n_dst x row_bytes].
cudaError_t launch_calib(int kind, const void *buf, size_t bytes, int row_bytes, long long n_src, long long n_dst,
                         int T, void *out, int num_sms, cudaStream_t s, int *launches)
{
    if (launches) ++*launches;
    if (kind == 0) {
        calib_stream_kernel<<<(unsigned)(num_sms * 8), 256, 0, s>>>(static_cast<const uint4 *>(buf),
                                                                    (long long)(bytes / 16), static_cast<uint4 *>(out));
        return cudaGetLastError();
    }
    switch (row_bytes) {
    case 256: return run_gather<16, 1, 8>(buf, n_src, n_dst, T, out, s);
    case 512: return run_gather<32, 1, 8>(buf, n_src, n_dst, T, out, s);
    case 1024: return run_gather<32, 2, 4>(buf, n_src, n_dst, T, out, s);
    case 2048: return run_gather<32, 4, 4>(buf, n_src, n_dst, T, out, s);
    }
    return cudaErrorNotSupported;
}

}  // namespace pinsage

// walks.cu -- importance-based neighbourhoods by simulated random walks:
// "we simulate random walks starting from node u and compute the L1-normalized visit count of
// nodes visited by the random walk ... the top T nodes with the highest normalized visit counts".
// This is the step that PRODUCES the (nbr_idx, counts) tables the pool consumes.
//
// The paper gives no walk parameters; readings B1-B5: CSR graph; n_walks walks per node,
// each restarting at u and taking walk_len uniform out-neighbour steps (a dead end stops the walk);
// every arrival at v != u is a visit; keep the T most visited (ties to the smaller id), pad with
// (u, 0); draws are a counter-based function of (seed, u, walk, step) -- splitmix64 finaliser.
//
// One warp per node.  Lane l simulates walks l, l+32, ... (a latency-bound pointer chase, hidden by
// many resident warps) and drops every arrival into slot walk*walk_len + step of a shared-memory
// array of 64-bit keys (empty = all ones).  The warp then (1) bitonic-sorts the ids in registers (32-bit
// keys), (2) run-length encodes them in place (shared memory) into (~count << 32 | id) entries ordered by
// id, (3) bitonic-sorts 32-bit rank keys (2048 - count) << 11 | position in registers -- ascending order
// is (count descending, id ascending) -- and (4) writes the first T.  Integer work only: bit-exact and
// independent of scheduling.
#include "internal.h"

namespace pinsage {
namespace {

constexpr int WARPS_PER_CTA = 4;
constexpr unsigned long long EMPTY = ~0ull;

__device__ __forceinline__ unsigned long long mix64(unsigned long long z)
{
    z += 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

// ---- register-resident bitonic sort ------------------------------------------------------------------
// A warp sorts 32 * R keys held R per lane: key i lives in register i / 32 of lane i % 32.  Partners at
// distance j < 32 are in another lane (one shuffle), at distance j >= 32 in another register of the same
// lane (register indices are compile-time through the JR template).  No shared-memory traffic: the
// shared-memory version of these sorts ran at 78 % of the shared pipe and bounded the kernel.
template <typename K, int R, int JR>
__device__ __forceinline__ void cmpex_regs(K (&v)[R], int k, int lane)
{
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int rr = r ^ JR;
        if (rr > r) {
            const bool up = (((r << 5) | lane) & k) == 0;
            const K a = v[r], b = v[rr];
            const bool sw = (a > b) == up;
            v[r] = sw ? b : a;
            v[rr] = sw ? a : b;
        }
    }
}
template <typename K, int R>
__device__ __forceinline__ void stage_regs(K (&v)[R], int jr, int k, int lane)
{
    switch (jr) {
    case 1: if constexpr (R > 1) cmpex_regs<K, R, 1>(v, k, lane); break;
    case 2: if constexpr (R > 2) cmpex_regs<K, R, 2>(v, k, lane); break;
    case 4: if constexpr (R > 4) cmpex_regs<K, R, 4>(v, k, lane); break;
    case 8: if constexpr (R > 8) cmpex_regs<K, R, 8>(v, k, lane); break;
    case 16: if constexpr (R > 16) cmpex_regs<K, R, 16>(v, k, lane); break;
    case 32: if constexpr (R > 32) cmpex_regs<K, R, 32>(v, k, lane); break;
    }
}
template <typename K, int R>
__device__ __forceinline__ void stage_shfl(K (&v)[R], int j, int k, int lane)
{
    const bool lower = (lane & j) == 0;
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const bool up = (((r << 5) | lane) & k) == 0;
        const K a = v[r], b = __shfl_xor_sync(0xffffffffu, a, j);
        v[r] = (lower == up) ? (a < b ? a : b) : (a > b ? a : b);
    }
}
// ascending sort of the first n keys' worth of stages (n a power of two, 32 <= n <= 32 * R; keys at
// index >= n must be EMPTY so that they stay in place)
template <typename K, int R>
__device__ __forceinline__ void warp_sort_regs(K (&v)[R], int n, int lane)
{
    for (int k = 2; k <= n; k <<= 1)
        for (int j = k >> 1; j > 0; j >>= 1) {
            if (j >= 32) stage_regs<K, R>(v, j >> 5, k, lane);
            else stage_shfl<K, R>(v, j, k, lane);
        }
}

template <int R>
__global__ void __launch_bounds__(WARPS_PER_CTA * 32)
walk_neighbourhoods_kernel(const long long *__restrict__ row_ptr, const int *__restrict__ col_idx,
                           long long N, int n_walks, int walk_len, int T, unsigned long long seed,
                           int *__restrict__ nbr_idx, int *__restrict__ counts)
{
    constexpr int slots = 32 * R;            // power of two >= max(32, n_walks * walk_len)
    extern __shared__ __align__(16) unsigned long long walk_smem[];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const long long u = (long long)blockIdx.x * WARPS_PER_CTA + wid;
    if (u >= N) return;
    unsigned long long *s = walk_smem + (size_t)wid * slots;
    for (int i = lane; i < slots; i += 32) s[i] = EMPTY;
    __syncwarp();

    // ---- the walks (B2, B3, B5) -----------------------------------------------------------------
    const unsigned long long key = mix64(seed + 0x100000001B3ull * (unsigned long long)u);
    // A walk is a chain of dependent loads (row_ptr, then col_idx, per step): a lane advances all of its
    // walks (up to WPL = 8, i.e. n_walks <= 256) one step at a time, so that their loads are in flight
    // together.  Same draws, same arrivals, same slots as walking them one after the other.
    constexpr int WPL = 8;
    if (n_walks <= 32 * WPL) {
        long long cur[WPL];
        bool alive[WPL];
#pragma unroll
        for (int w = 0; w < WPL; ++w) {
            cur[w] = u;
            alive[w] = lane + 32 * w < n_walks;
        }
        for (int st = 0; st < walk_len; ++st) {
            long long beg[WPL], end[WPL];
#pragma unroll
            for (int w = 0; w < WPL; ++w)
                if (alive[w]) {
                    beg[w] = __ldg(row_ptr + cur[w]);
                    end[w] = __ldg(row_ptr + cur[w] + 1);
                }
#pragma unroll
            for (int w = 0; w < WPL; ++w)
                if (alive[w]) {
                    const long long deg = end[w] - beg[w];
                    if (deg <= 0) {
                        alive[w] = false;                     // dead end: the walk stops (B3)
                    } else {
                        const unsigned long long r = (unsigned long long)(lane + 32 * w);
                        const unsigned long long x = mix64(key ^ ((r << 32) | (unsigned long long)st));
                        const unsigned long long pick = ((x >> 32) * (unsigned long long)deg) >> 32;
                        cur[w] = __ldg(col_idx + beg[w] + (long long)pick);
                    }
                }
#pragma unroll
            for (int w = 0; w < WPL; ++w)
                if (alive[w] && cur[w] != u) s[(lane + 32 * w) * walk_len + st] = (unsigned long long)(unsigned)cur[w];
        }
    } else {
        for (int r = lane; r < n_walks; r += 32) {
            long long cur = u;
            for (int st = 0; st < walk_len; ++st) {
                const long long beg = __ldg(row_ptr + cur);
                const long long deg = __ldg(row_ptr + cur + 1) - beg;
                if (deg <= 0) break;
                const unsigned long long x = mix64(key ^ (((unsigned long long)r << 32) | (unsigned long long)st));
                const unsigned long long pick = ((x >> 32) * (unsigned long long)deg) >> 32;
                cur = __ldg(col_idx + beg + (long long)pick);
                if (cur != u) s[r * walk_len + st] = (unsigned long long)(unsigned)cur;
            }
        }
    }
    __syncwarp();

    // ---- (1) sort the arrivals (in registers); (2) run-length encode in place ----------------------
    {   // ids fit 31 bits: the first sort runs on 32-bit keys (half the registers, shuffles and ALU work)
        unsigned v1[R];
#pragma unroll
        for (int r = 0; r < R; ++r) v1[r] = (unsigned)s[r * 32 + lane];          // EMPTY -> 0xFFFFFFFF
        warp_sort_regs<unsigned, R>(v1, slots, lane);
#pragma unroll
        for (int r = 0; r < R; ++r) s[r * 32 + lane] = v1[r] == 0xFFFFFFFFu ? EMPTY : (unsigned long long)v1[r];
    }
    __syncwarp();
    int ns = 0;
    for (int base = 0; base < slots; base += 32)
        ns += __popc(__ballot_sync(0xffffffffu, s[base + lane] != EMPTY));
    int nv = 0;                              // distinct ids written so far
    unsigned long long carry_prev = EMPTY;   // last id of the previous chunk
    int carry_start = 0;                     // start index of the run that enters this chunk
    for (int base = 0; base < ns; base += 32) {
        const int i = base + lane;
        const bool valid = i < ns;
        const unsigned long long a = valid ? s[i] : EMPTY;
        const unsigned long long nxt = (i + 1 < ns) ? s[i + 1] : EMPTY;
        unsigned long long prev = __shfl_up_sync(0xffffffffu, a, 1);
        if (lane == 0) prev = carry_prev;
        const bool is_start = valid && (i == 0 || a != prev);
        const bool is_end = valid && a != nxt;
        int start = is_start ? i : -1;       // inclusive max-scan: start index of my run
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, start, o);
            if (lane >= o) start = max(start, t);
        }
        if (start < 0) start = carry_start;
        const unsigned ends = __ballot_sync(0xffffffffu, is_end);
        const int pos = nv + __popc(ends & ((1u << lane) - 1u));
        const unsigned count = (unsigned)(i - start + 1);
        __syncwarp();                        // every read of this chunk is done before any write
        if (is_end) s[pos] = ((unsigned long long)(0xFFFFFFFFu - count) << 32) | a;
        carry_prev = __shfl_sync(0xffffffffu, a, 31);
        carry_start = __shfl_sync(0xffffffffu, start, 31);
        nv += __popc(ends);
        __syncwarp();
    }

    // ---- (3) rank (B4).  The run-length output s[0 .. nv) is ordered by id, so a 32-bit key
    // (2048 - count) << 11 | position sorts ascending into (count descending, id ascending) --------
    unsigned v2[R];
    __shared__ unsigned sel_keys[WARPS_PER_CTA][128];
    if (R > 4 && T <= 128 && nv > 128) {
        // Only the top T <= 128 of (typically ~1000) distinct ids are wanted: instead of sorting them all,
        // find the count c* of the T-th best (binary search on the count, entries in registers), take
        // every id with a larger count and, of those with exactly c*, the smallest ids -- which are the
        // first in s, already ordered by id -- and sort just these T keys.
        unsigned cnt[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int i = r * 32 + lane;
            cnt[r] = i < nv ? 0xFFFFFFFFu - (unsigned)(s[i] >> 32) : 0u;
        }
        auto count_ge = [&](unsigned c) {
            int n = 0;
#pragma unroll
            for (int r = 0; r < R; ++r) n += cnt[r] >= c ? 1 : 0;
            return __reduce_add_sync(0xffffffffu, n);
        };
        int lo = 1, hi = 2048;                   // invariant: #(count >= lo) >= T  (nv > 128 >= T)
        while (lo < hi) {
            const int mid = (lo + hi + 1) >> 1;
            if (count_ge((unsigned)mid) >= T) lo = mid;
            else hi = mid - 1;
        }
        const unsigned cstar = (unsigned)lo;
        const int quota = T - count_ge(cstar + 1);
        const unsigned lt = (1u << lane) - 1u;
        int taken_eq = 0, npos = 0;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const bool eq = cnt[r] == cstar;
            const unsigned beq = __ballot_sync(0xffffffffu, eq);
            const bool take = cnt[r] > cstar || (eq && taken_eq + __popc(beq & lt) < quota);
            const unsigned bt = __ballot_sync(0xffffffffu, take);
            if (take) sel_keys[wid][npos + __popc(bt & lt)] = ((2048u - cnt[r]) << 11) | (unsigned)(r * 32 + lane);
            taken_eq += __popc(beq);
            npos += __popc(bt);
        }
        __syncwarp();
        unsigned w2[4];
#pragma unroll
        for (int r = 0; r < 4; ++r) w2[r] = r * 32 + lane < npos ? sel_keys[wid][r * 32 + lane] : 0xFFFFFFFFu;
        if (npos <= 64) {                        // (warp-uniform) two registers per lane are enough
            unsigned w1[2] = {w2[0], w2[1]};
            warp_sort_regs<unsigned, 2>(w1, 64, lane);
            w2[0] = w1[0];
            w2[1] = w1[1];
        } else {
            warp_sort_regs<unsigned, 4>(w2, 128, lane);
        }
#pragma unroll
        for (int r = 0; r < R; ++r) v2[r] = r < 4 ? w2[r < 4 ? r : 0] : 0xFFFFFFFFu;
    } else {
        int n2 = 32;
        while (n2 < nv) n2 <<= 1;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int i = r * 32 + lane;
            v2[r] = 0xFFFFFFFFu;
            if (i < nv) {
                const unsigned count = 0xFFFFFFFFu - (unsigned)(s[i] >> 32);
                v2[r] = ((2048u - count) << 11) | (unsigned)i;
            }
        }
        warp_sort_regs<unsigned, R>(v2, n2, lane);   // only the stages the nv distinct keys need
    }

    // ---- (4) the top T, padded with (u, 0): rank t sits in register t / 32 of lane t % 32 -------------
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int t = r * 32 + lane;
        if (t < T && t < slots) {
            int id = (int)u, c = 0;
            if (t < nv) {
                const unsigned long long e = s[v2[r] & 0x7FFu];
                id = (int)(unsigned)(e & 0xFFFFFFFFull);
                c = (int)(0xFFFFFFFFu - (unsigned)(e >> 32));
            }
            nbr_idx[u * T + t] = id;
            counts[u * T + t] = c;
        }
    }
    for (int t = slots + lane; t < T; t += 32) {         // T beyond the slot count: padding only
        nbr_idx[u * T + t] = (int)u;
        counts[u * T + t] = 0;
    }
}

}  // namespace

int walk_slots(int32_t n_walks, int32_t walk_len)
{
    const long long need = (long long)n_walks * walk_len;
    if (n_walks < 1 || walk_len < 1 || need > 2048) return 0;
    int s = 32;
    while (s < need) s <<= 1;
    return s;
}

cudaError_t launch_walk_neighbourhoods(int64_t N, const int64_t *row_ptr, const int32_t *col_idx,
                                       int32_t n_walks, int32_t walk_len, int32_t T, uint64_t seed,
                                       int32_t *nbr_idx, int32_t *counts, cudaStream_t s, int *launches)
{
    const int slots = walk_slots(n_walks, walk_len);
    if (slots == 0) return cudaErrorNotSupported;
    const long long blocks = (N + WARPS_PER_CTA - 1) / WARPS_PER_CTA;
    if (blocks > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    const size_t smem = (size_t)WARPS_PER_CTA * slots * sizeof(unsigned long long);
    auto go = [&](auto kern) -> cudaError_t {
        if (smem > 48 * 1024) {
            cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (e != cudaSuccess) return e;
        }
        kern<<<(unsigned)blocks, WARPS_PER_CTA * 32, smem, s>>>(
            reinterpret_cast<const long long *>(row_ptr), col_idx, N, n_walks, walk_len, T,
            (unsigned long long)seed, nbr_idx, counts);
        return cudaSuccess;
    };
    cudaError_t e = cudaErrorNotSupported;
    switch (slots / 32) {
    case 1: e = go(walk_neighbourhoods_kernel<1>); break;
    case 2: e = go(walk_neighbourhoods_kernel<2>); break;
    case 4: e = go(walk_neighbourhoods_kernel<4>); break;
    case 8: e = go(walk_neighbourhoods_kernel<8>); break;
    case 16: e = go(walk_neighbourhoods_kernel<16>); break;
    case 32: e = go(walk_neighbourhoods_kernel<32>); break;
    case 64: e = go(walk_neighbourhoods_kernel<64>); break;
    }
    if (e != cudaSuccess) return e;
    if (launches) ++*launches;
    return cudaGetLastError();
}

}  // namespace pinsage

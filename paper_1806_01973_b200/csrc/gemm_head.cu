// gemm_head.cu -- S4 -> S5 in one launch: out = ReLU(H G1^T + g) G2^T   (Alg. 2 l.16)
//
// The head's intermediate a = ReLU(H G1^T + g) [rows x g1] never reaches HBM: every CTA owns two 128-row
// slots of a small scratch array (grid x 2 x 128 rows: ~19 MB, rewritten every few microseconds, so it
// lives in L2), stores the a tile of a row tile there (bf16, the SAME rounding as the two-launch form) and
// reads it back as the A operand of the second GEMM.  Row tiles are taken two at a time and their four
// GEMM phases are software-pipelined over the two TMEM accumulators,
//
//      A(t0) -> acc0 | A(t1) -> acc1 | B(t0) -> acc0 | B(t1) -> acc1 |  A(t2) ...      (A: H G1^T, B: a G2^T)
//
// so that the only new dependency -- B(t) must not load a(t) before the epilogue of A(t) has stored it --
// always has a whole MMA phase of slack, and every epilogue runs under the next phase's MMAs.
// Result: bit-identical to pinsage_dense(G1, relu) followed by pinsage_dense(G2) (same K order, same
// roundings), with H read and out written once and nothing else crossing HBM.
//
// Single-CTA tiles (these shapes -- g1, d_out <= 256 -- are HBM-bound); warp roles as in gemm_tcgen05.cu:
// warp 0 TMA producer, warp 1 MMA issuer, warp 2 TMEM allocator, warps 4-7 epilogue.
#include "internal.h"

#include <algorithm>
#include <mutex>

#include <cuda.h>

#include "tc_ptx.cuh"

namespace pinsage {
namespace {

constexpr int HEAD_THREADS = 256;
constexpr int HEAD_PAIR_THREADS = 384;          // the pair kernel runs eight epilogue warps
constexpr int HEAD_LAG = 2;                     // ... and issues a G2^T of tile t after H G1^T of tile t + HEAD_LAG
constexpr int HEAD_SLOTS = HEAD_LAG + 1;        // a tiles a CTA has in the scratch at one time
constexpr int HEAD_MAX_STAGES = 8;
constexpr int HEAD_BIAS_FLOATS = 320;          // g1 <= 256, read in 64-column chunks
constexpr int HEAD_BAR_BYTES = 256;

struct HeadTcParams {
    long long M, m_blocks;
    int kb1, kb2;          // 64-wide K blocks of GEMM 1 (over d) and GEMM 2 (over g1)
    int N1, N2;            // g1, d_out
    int CN1, CN2;          // MMA N of the two GEMMs (N rounded up to 16)
    int stages, stage_bytes;
    const float *bias;     // g [g1]
    uint32_t idesc1, idesc2;
};

__device__ __forceinline__ void fence_proxy_async_global()
{
    asm volatile("fence.proxy.async.global;" ::: "memory");
}

__global__ void __launch_bounds__(HEAD_THREADS, 1)
head_tc_kernel(const __grid_constant__ CUtensorMap tmH, const __grid_constant__ CUtensorMap tmG1,
               const __grid_constant__ CUtensorMap tmScrOut, const __grid_constant__ CUtensorMap tmScrIn,
               const __grid_constant__ CUtensorMap tmG2, const __grid_constant__ CUtensorMap tmOut,
               const HeadTcParams p)
{
    extern __shared__ __align__(1024) uint8_t smem[];
    const uint32_t sbase = smem_u32(smem);
    if ((sbase & 1023u) != 0) __trap();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t stg_off = (uint32_t)p.stages * p.stage_bytes;
    const uint32_t bias_off = stg_off + 4 * 2 * STG_WARP_BYTES;
    const uint32_t bar_off = bias_off + HEAD_BIAS_FLOATS * 4;
    float *sbias = reinterpret_cast<float *>(smem + bias_off);
    const uint32_t bar_full = sbase + bar_off;                     // [8]
    const uint32_t bar_empty = bar_full + 8 * HEAD_MAX_STAGES;     // [8]
    const uint32_t bar_tfull = bar_empty + 8 * HEAD_MAX_STAGES;    // [2]
    const uint32_t bar_tempty = bar_tfull + 16;                    // [2]
    const uint32_t bar_aready = bar_tempty + 16;                   // [2]: a(t) of slot j is in the scratch
    volatile uint32_t *tmem_slot = reinterpret_cast<volatile uint32_t *>(smem + bar_off + 8 * (2 * HEAD_MAX_STAGES + 6));

    // this CTA's row tiles: blockIdx.x, + gridDim.x, ...; `cnt` of them
    const long long cnt = p.m_blocks > blockIdx.x ? (p.m_blocks - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
    const int scr_row0 = (int)blockIdx.x * 2 * BM;                 // this CTA's two slots of the scratch

    if (warp == 0 && lane == 0) {
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmH) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmG1) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmScrOut) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmScrIn) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmG2) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmOut) : "memory");
    }
    if (warp == 1 && lane == 0) {
        for (int s = 0; s < p.stages; ++s) {
            mbar_init(bar_full + 8 * s, 1);
            mbar_init(bar_empty + 8 * s, 1);
        }
        for (int a = 0; a < 2; ++a) {
            mbar_init(bar_tfull + 8 * a, 1);
            mbar_init(bar_tempty + 8 * a, 4);      // the four epilogue warps
            mbar_init(bar_aready + 8 * a, 4);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 2) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(
                         smem_u32(const_cast<uint32_t *>(tmem_slot))),
                     "r"(512u)
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    if (warp >= 4) {
        for (int c = threadIdx.x - 128; c < HEAD_BIAS_FLOATS; c += 128)
            sbias[c] = (p.bias != nullptr && c < p.N1) ? __ldg(p.bias + c) : 0.f;
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    // phase ph of pair pr: kind = ph >> 1 (0: H G1^T, 1: a G2^T), j = ph & 1 (tile of the pair = accumulator
    // = scratch slot); a pair's second tile may not exist
    if (warp == 0) {
        // ===== TMA producer ===================================================================
        uint64_t pol_stream, pol_keep;
        asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol_stream));
        asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol_keep));
        int stage = 0;
        uint32_t phase = 0;
        for (long long pr = 0; 2 * pr < cnt; ++pr) {
            for (int ph = 0; ph < 4; ++ph) {
                const int kind = ph >> 1, j = ph & 1;
                if (2 * pr + j >= cnt) continue;
                const long long mb = blockIdx.x + (2 * pr + j) * (long long)gridDim.x;
                const int m0 = (int)(mb * BM);
                const int KB = kind ? p.kb2 : p.kb1, CN = kind ? p.CN2 : p.CN1;
                if (kind) {                              // a(t) must have been stored by the epilogue
                    mbar_wait(bar_aready + 8 * j, (uint32_t)(pr & 1));
                    fence_proxy_async_global();
                }
                for (int kb = 0; kb < KB; ++kb) {
                    mbar_wait(bar_empty + 8 * stage, phase ^ 1);
                    if (elect_one()) {
                        const uint32_t full = bar_full + 8 * stage;
                        const uint32_t sA = sbase + (uint32_t)stage * p.stage_bytes;
                        mbar_expect_tx(full, (uint32_t)(A_BYTES + CN * 128));
                        if (kind) {
                            tma_load_2d(sA, &tmScrIn, kb * BK, scr_row0 + j * BM, full, pol_keep);
                            tma_load_2d(sA + A_BYTES, &tmG2, kb * BK, 0, full, pol_keep);
                        } else {
                            tma_load_2d(sA, &tmH, kb * BK, m0, full, pol_stream);
                            tma_load_2d(sA + A_BYTES, &tmG1, kb * BK, 0, full, pol_keep);
                        }
                    }
                    __syncwarp();
                    if (++stage == p.stages) {
                        stage = 0;
                        phase ^= 1;
                    }
                }
            }
        }
    } else if (warp == 1) {
        // ===== MMA issuer =====================================================================
        int stage = 0;
        uint32_t phase = 0, use[2] = {0, 0};
        for (long long pr = 0; 2 * pr < cnt; ++pr) {
            for (int ph = 0; ph < 4; ++ph) {
                const int kind = ph >> 1, j = ph & 1;
                if (2 * pr + j >= cnt) continue;
                const int KB = kind ? p.kb2 : p.kb1;
                const uint32_t idesc = kind ? p.idesc2 : p.idesc1;
                mbar_wait(bar_tempty + 8 * j, (use[j] & 1u) ^ 1u);    // the epilogue drained this accumulator
                tc_fence_after();
                const uint32_t d0 = tmem_base + (uint32_t)j * 256u;
                for (int kb = 0; kb < KB; ++kb) {
                    mbar_wait(bar_full + 8 * stage, phase);
                    tc_fence_after();
                    if (elect_one()) {
                        const uint32_t sA = sbase + (uint32_t)stage * p.stage_bytes;
                        const uint64_t ad = make_desc(sA), bd = make_desc(sA + A_BYTES);
#pragma unroll
                        for (int k = 0; k < BK / 16; ++k)
                            tc_mma(d0, ad + 2 * k, bd + 2 * k, idesc, k == 0 ? (uint32_t)kb : 1u);
                        tc_commit(bar_empty + 8 * stage);
                        if (kb == KB - 1) tc_commit(bar_tfull + 8 * j);
                    }
                    __syncwarp();
                    if (++stage == p.stages) {
                        stage = 0;
                        phase ^= 1;
                    }
                }
                ++use[j];
            }
        }
    } else if (warp >= 4) {
        // ===== epilogue: thread (ew, lane) owns row 32 * ew + lane of the tile ==================
        const int ew = warp & 3;
        uint8_t *stg = smem + stg_off + ew * 2 * STG_WARP_BYTES;
        int sbuf = 0;
        uint32_t use[2] = {0, 0};
        for (long long pr = 0; 2 * pr < cnt; ++pr) {
            for (int ph = 0; ph < 4; ++ph) {
                const int kind = ph >> 1, j = ph & 1;
                if (2 * pr + j >= cnt) continue;
                const long long mb = blockIdx.x + (2 * pr + j) * (long long)gridDim.x;
                const long long m0 = mb * BM;
                const int ncols = kind ? p.N2 : p.N1;
                mbar_wait(bar_tfull + 8 * j, use[j] & 1u);
                tc_fence_after();
                const uint32_t t0 = tmem_base + ((uint32_t)(ew * 32) << 16) + (uint32_t)j * 256u;
                for (int c0 = 0; c0 < ncols; c0 += OUT_CHUNK) {
                    uint32_t v[2][32];
                    tc_ld32(t0 + c0, v[0]);
                    tc_ld32(t0 + c0 + 32, v[1]);
                    tc_wait_ld();
                    uint32_t pk[32];
#pragma unroll
                    for (int h = 0; h < 2; ++h)
#pragma unroll
                        for (int i = 0; i < 32; i += 2) {
                            float2 z2 = make_float2(__uint_as_float(v[h][i]), __uint_as_float(v[h][i + 1]));
                            if (!kind) {                 // a = ReLU(acc + g)
                                z2 = __fadd2_rn(z2, *reinterpret_cast<const float2 *>(sbias + c0 + 32 * h + i));
                                z2.x = fmaxf(z2.x, 0.f);
                                z2.y = fmaxf(z2.y, 0.f);
                            }
                            __nv_bfloat162 b = __floats2bfloat162_rn(z2.x, z2.y);
                            pk[16 * h + i / 2] = *reinterpret_cast<uint32_t *>(&b);
                        }
                    if (lane == 0) tma_store_wait_read<1>();      // the buffer used two stores ago is free
                    __syncwarp();
                    uint8_t *buf = stg + sbuf * STG_WARP_BYTES;
                    uint8_t *rowp = buf + lane * 128;
#pragma unroll
                    for (int q = 0; q < 8; ++q)                   // 16-byte chunk q of the row, XOR-swizzled
                        *reinterpret_cast<uint4 *>(rowp + ((q ^ (lane & 7)) << 4)) =
                            make_uint4(pk[4 * q], pk[4 * q + 1], pk[4 * q + 2], pk[4 * q + 3]);
                    fence_proxy_async();
                    __syncwarp();
                    if (lane == 0) {
                        if (!kind) {
                            tma_store_2d(&tmScrOut, c0, scr_row0 + j * BM + ew * 32, smem_u32(buf));
                            tma_store_commit();
                        } else if (m0 + ew * 32 < p.M) {
                            tma_store_2d(&tmOut, c0, (int)(m0 + ew * 32), smem_u32(buf));
                            tma_store_commit();
                        }
                    }
                    sbuf ^= 1;
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) {
                    mbar_arrive(bar_tempty + 8 * j);
                    if (!kind) {
                        // the a tile is in the scratch (complete, not just read out of shared memory)
                        // before the producer may load it
                        tma_store_wait_all();
                        fence_proxy_async_global();
                        mbar_arrive(bar_aready + 8 * j);
                    }
                }
                ++use[j];
            }
        }
        if (lane == 0) tma_store_wait_all();
    }

    __syncwarp();
    tc_fence_before();
    __syncthreads();
    if (warp == 2) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(512u) : "memory");
    }
}


// ---- CTA-pair form with stationary weights ------------------------------------------------------------
// The single-CTA kernel above re-reads both weight matrices for every 128-row tile: 2 x 128 KB of the
// 450 KB that cross L2 -> shared memory per tile at 256 -> 256 -> 256, and at ~10 TB/s of L2 throughput
// that traffic, not HBM, is what bounds it (measured: 6.4 us per tile).
// Here the two SMs of a TPC own a 256-row tile (cta_group::2): each CTA keeps HALF of G1 and of G2 (its
// share of the N rows, all K blocks: 2 x 64 KB) in shared memory for the whole launch, so only the H rows
// and the a tile's round trip through the L2-resident scratch move per tile (192 KB per 128 rows).  Same
// phase pipeline over the two TMEM accumulators, same K order and roundings: bit-identical results.
struct HeadPairParams {
    long long M, m_blocks;     // m_blocks: 256-row tiles
    int kb1, kb2, N1, N2, CN1, CN2;
    int w1_blk, w2_blk;        // bytes of one K block of this CTA's half of G1 / G2
    int stages;
    const float *bias;
    uint32_t idesc1, idesc2;
};

__global__ void __launch_bounds__(HEAD_PAIR_THREADS, 1)
head_tc_pair_kernel(const __grid_constant__ CUtensorMap tmH, const __grid_constant__ CUtensorMap tmG1,
                    const __grid_constant__ CUtensorMap tmScrOut, const __grid_constant__ CUtensorMap tmScrIn,
                    const __grid_constant__ CUtensorMap tmG2, const __grid_constant__ CUtensorMap tmOut,
                    const HeadPairParams p)
{
    extern __shared__ __align__(1024) uint8_t smem[];
    const uint32_t sbase = smem_u32(smem);
    if ((sbase & 1023u) != 0) __trap();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t w2_off = (uint32_t)p.kb1 * p.w1_blk;
    const uint32_t ring_off = w2_off + (uint32_t)p.kb2 * p.w2_blk;
    const uint32_t stg_off = ring_off + (uint32_t)p.stages * A_BYTES;
    const uint32_t bias_off = stg_off + 4 * 2 * STG_WARP_BYTES;
    const uint32_t bar_off = bias_off + HEAD_BIAS_FLOATS * 4;
    float *sbias = reinterpret_cast<float *>(smem + bias_off);
    const uint32_t bar_full = sbase + bar_off;                     // [8]  the leader's are used
    const uint32_t bar_empty = bar_full + 8 * HEAD_MAX_STAGES;     // [8]
    const uint32_t bar_tfull = bar_empty + 8 * HEAD_MAX_STAGES;    // [2]
    const uint32_t bar_tempty = bar_tfull + 16;                    // [2]  the leader's are used
    const uint32_t bar_aready = bar_tempty + 16;                   // [HEAD_SLOTS]: a(t) of that slot is in the scratch
    const uint32_t bar_w = bar_aready + 8 * HEAD_SLOTS;            // weights have landed (the leader's)
    volatile uint32_t *tmem_slot =
        reinterpret_cast<volatile uint32_t *>(smem + bar_off + 8 * (2 * HEAD_MAX_STAGES + 4 + HEAD_SLOTS + 1));

    const uint32_t half = cluster_ctarank();                       // which 128 rows of the 256-row tile
    const long long unit = blockIdx.x >> 1, units = gridDim.x >> 1;
    const long long cnt = p.m_blocks > unit ? (p.m_blocks - unit + units - 1) / units : 0;
    const int scr_row0 = (int)blockIdx.x * HEAD_SLOTS * BM;        // this CTA's slots of the scratch

    if (warp == 0 && lane == 0) {
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmH) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmG1) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmScrOut) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmScrIn) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmG2) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmOut) : "memory");
    }
    if (warp == 1 && lane == 0) {
        for (int s = 0; s < p.stages; ++s) {
            mbar_init(bar_full + 8 * s, 1);
            mbar_init(bar_empty + 8 * s, 1);
        }
        for (int a = 0; a < 2; ++a) {
            mbar_init(bar_tfull + 8 * a, 1);
            mbar_init(bar_tempty + 8 * a, 16);     // the eight epilogue warps of both CTAs
        }
        for (int a = 0; a < HEAD_SLOTS; ++a) mbar_init(bar_aready + 8 * a, 8);   // this CTA's own epilogue warps
        mbar_init(bar_w, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 2) {
        asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(
                         smem_u32(const_cast<uint32_t *>(tmem_slot))),
                     "r"(512u)
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
    }
    if (warp >= 4) {
        for (int c = threadIdx.x - 128; c < HEAD_BIAS_FLOATS; c += HEAD_PAIR_THREADS - 128)
            sbias[c] = (p.bias != nullptr && c < p.N1) ? __ldg(p.bias + c) : 0.f;
    }
    tc_fence_before();
    cluster_sync_all();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    if (warp == 0) {
        // ===== TMA producer (both CTAs: their own rows of H / a, their halves of the weights) ==========
        uint64_t pol_stream, pol_keep;
        asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol_stream));
        asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol_keep));
        const uint32_t leader_full = map_to_cta(bar_full, 0);
        if (cnt > 0 && elect_one()) {
            const uint32_t lw = map_to_cta(bar_w, 0);
            if (half == 0) mbar_expect_tx(bar_w, 2u * (uint32_t)(p.kb1 * p.w1_blk + p.kb2 * p.w2_blk));
            for (int kb = 0; kb < p.kb1; ++kb)
                tma_load_2d_pair(sbase + (uint32_t)kb * p.w1_blk, &tmG1, kb * BK, (int)half * (p.CN1 / 2), lw, pol_keep);
            for (int kb = 0; kb < p.kb2; ++kb)
                tma_load_2d_pair(sbase + w2_off + (uint32_t)kb * p.w2_blk, &tmG2, kb * BK, (int)half * (p.CN2 / 2), lw,
                                 pol_keep);
        }
        __syncwarp();
        int stage = 0;
        uint32_t phase = 0;
        for (long long st = 0; st < cnt + HEAD_LAG; ++st) {
            for (int kind = 0; kind < 2; ++kind) {
                const long long t = kind ? st - HEAD_LAG : st;       // this CTA pair's t-th tile
                if (t < 0 || t >= cnt) continue;
                const long long mb = unit + t * units;
                const int m0 = (int)(mb * (2 * BM)) + (int)half * BM;
                const int KB = kind ? p.kb2 : p.kb1;
                const int slot = (int)(t % HEAD_SLOTS);
                if (kind) {                              // this CTA's rows of a(t) are in the scratch
                    mbar_wait(bar_aready + 8 * slot, (uint32_t)((t / HEAD_SLOTS) & 1));
                    fence_proxy_async_global();
                }
                for (int kb = 0; kb < KB; ++kb) {
                    mbar_wait(bar_empty + 8 * stage, phase ^ 1);
                    if (elect_one()) {
                        if (half == 0) mbar_expect_tx(bar_full + 8 * stage, 2u * A_BYTES);   // both CTAs' bytes
                        const uint32_t sA = sbase + ring_off + (uint32_t)stage * A_BYTES;
                        if (kind) tma_load_2d_pair(sA, &tmScrIn, kb * BK, scr_row0 + slot * BM, leader_full + 8 * stage, pol_keep);
                        else tma_load_2d_pair(sA, &tmH, kb * BK, m0, leader_full + 8 * stage, pol_stream);
                    }
                    __syncwarp();
                    if (++stage == p.stages) {
                        stage = 0;
                        phase ^= 1;
                    }
                }
            }
        }
    } else if (warp == 1) {
        // ===== MMA issuer: the pair's even CTA ==========================================================
        if (half == 0 && cnt > 0) {
            int stage = 0;
            uint32_t phase = 0, use[2] = {0, 0};
            int j = 0;                                   // accumulators alternate from phase to phase
            mbar_wait(bar_w, 0);
            tc_fence_after();
            for (long long st = 0; st < cnt + HEAD_LAG; ++st) {
                for (int kind = 0; kind < 2; ++kind) {
                    const long long t = kind ? st - HEAD_LAG : st;
                    if (t < 0 || t >= cnt) continue;
                    const int KB = kind ? p.kb2 : p.kb1;
                    const uint32_t idesc = kind ? p.idesc2 : p.idesc1;
                    const uint32_t wbase = sbase + (kind ? w2_off : 0u), wblk = (uint32_t)(kind ? p.w2_blk : p.w1_blk);
                    mbar_wait(bar_tempty + 8 * j, (use[j] & 1u) ^ 1u);    // both epilogues drained this accumulator
                    tc_fence_after();
                    const uint32_t d0 = tmem_base + (uint32_t)j * 256u;
                    for (int kb = 0; kb < KB; ++kb) {
                        mbar_wait(bar_full + 8 * stage, phase);
                        tc_fence_after();
                        if (elect_one()) {
                            const uint64_t ad = make_desc(sbase + ring_off + (uint32_t)stage * A_BYTES);
                            const uint64_t bd = make_desc(wbase + (uint32_t)kb * wblk);
#pragma unroll
                            for (int k = 0; k < BK / 16; ++k)
                                tc_mma_pair(d0, ad + 2 * k, bd + 2 * k, idesc, k == 0 ? (uint32_t)kb : 1u);
                            tc_commit_pair(bar_empty + 8 * stage, (uint16_t)3);
                            if (kb == KB - 1) tc_commit_pair(bar_tfull + 8 * j, (uint16_t)3);
                        }
                        __syncwarp();
                        if (++stage == p.stages) {
                            stage = 0;
                            phase ^= 1;
                        }
                    }
                    ++use[j];
                    j ^= 1;
                }
            }
        }
    } else if (warp >= 4) {
        // ===== epilogue: eight warps, two per row quarter (TMEM lanes 32 * ew ..), each one half of the
        // columns: with two epilogues per row tile (a, then out) four warps were the bottleneck of the launch
        const int ew = warp & 3, eh = (warp - 4) >> 2;
        uint8_t *buf = smem + stg_off + (eh * 4 + ew) * STG_WARP_BYTES;     // one staging buffer per warp
        const uint32_t tempty_leader = map_to_cta(bar_tempty, 0);
        uint32_t use[2] = {0, 0};
        int j = 0;
        for (long long st = 0; st < cnt + HEAD_LAG; ++st) {
            for (int kind = 0; kind < 2; ++kind) {
                const long long t = kind ? st - HEAD_LAG : st;
                if (t < 0 || t >= cnt) continue;
                const long long mb = unit + t * units;
                const long long m0 = mb * (2 * BM) + (long long)half * BM;
                const int ncols = kind ? p.N2 : p.N1;
                const int slot = (int)(t % HEAD_SLOTS);
                const int c_split = ((ncols + 1) / 2 + OUT_CHUNK - 1) / OUT_CHUNK * OUT_CHUNK;
                const int c_lo = eh ? c_split : 0, c_hi = eh ? ncols : min(c_split, ncols);
                mbar_wait(bar_tfull + 8 * j, use[j] & 1u);
                tc_fence_after();
                const uint32_t t0 = tmem_base + ((uint32_t)(ew * 32) << 16) + (uint32_t)j * 256u;
                for (int c0 = c_lo; c0 < c_hi; c0 += OUT_CHUNK) {
                    uint32_t v[2][32];
                    tc_ld32(t0 + c0, v[0]);
                    tc_ld32(t0 + c0 + 32, v[1]);
                    tc_wait_ld();
                    uint32_t pk[32];
#pragma unroll
                    for (int h = 0; h < 2; ++h)
#pragma unroll
                        for (int i = 0; i < 32; i += 2) {
                            float2 z2 = make_float2(__uint_as_float(v[h][i]), __uint_as_float(v[h][i + 1]));
                            if (!kind) {                 // a = ReLU(acc + g)
                                z2 = __fadd2_rn(z2, *reinterpret_cast<const float2 *>(sbias + c0 + 32 * h + i));
                                z2.x = fmaxf(z2.x, 0.f);
                                z2.y = fmaxf(z2.y, 0.f);
                            }
                            __nv_bfloat162 b = __floats2bfloat162_rn(z2.x, z2.y);
                            pk[16 * h + i / 2] = *reinterpret_cast<uint32_t *>(&b);
                        }
                    if (lane == 0) tma_store_wait_read<0>();      // the previous store has read the buffer
                    __syncwarp();
                    uint8_t *rowp = buf + lane * 128;
#pragma unroll
                    for (int q = 0; q < 8; ++q)
                        *reinterpret_cast<uint4 *>(rowp + ((q ^ (lane & 7)) << 4)) =
                            make_uint4(pk[4 * q], pk[4 * q + 1], pk[4 * q + 2], pk[4 * q + 3]);
                    fence_proxy_async();
                    __syncwarp();
                    if (lane == 0) {
                        if (!kind) {
                            tma_store_2d(&tmScrOut, c0, scr_row0 + slot * BM + ew * 32, smem_u32(buf));
                            tma_store_commit();
                        } else if (m0 + ew * 32 < p.M) {
                            tma_store_2d(&tmOut, c0, (int)(m0 + ew * 32), smem_u32(buf));
                            tma_store_commit();
                        }
                    }
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) {
                    mbar_arrive_remote_relaxed(tempty_leader + 8 * j);
                    if (!kind) {
                        tma_store_wait_all();
                        fence_proxy_async_global();
                        mbar_arrive(bar_aready + 8 * slot);
                    }
                }
                ++use[j];
                j ^= 1;
            }
        }
        if (lane == 0) tma_store_wait_all();
    }

    __syncwarp();
    tc_fence_before();
    cluster_sync_all();
    if (warp == 2) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(512u) : "memory");
    }
}

inline int round_up_i(int x, int a) { return (x + a - 1) / a * a; }

}  // namespace

bool head_tc_supported(int32_t d, int32_t g1, int32_t d_out)
{
    return d >= 8 && d % 8 == 0 && g1 >= 8 && g1 % 8 == 0 && g1 <= 256 && d_out >= 8 && d_out % 8 == 0 && d_out <= 256;
}

size_t head_tc_scratch_bytes(int32_t g1, int num_sms) { return (size_t)num_sms * HEAD_SLOTS * BM * g1 * 2; }

namespace {

// The CTA-pair kernel with stationary weights: taken when both halves of the weights fit beside an operand
// ring of at least three stages and every pair gets a tile.  *taken = false: the caller uses the single-CTA kernel.
cudaError_t launch_head_pair(GemmTcState *st, int64_t M, int32_t d, int32_t g1, int32_t d_out, const void *H,
                             const void *G1, const float *g, const void *G2, void *out, void *scratch, int num_sms,
                             cudaStream_t s, int *launches, bool *taken)
{
    *taken = false;
    HeadPairParams p{};
    p.M = M;
    p.m_blocks = (M + 2 * BM - 1) / (2 * BM);
    p.kb1 = (d + BK - 1) / BK;
    p.kb2 = (g1 + BK - 1) / BK;
    p.N1 = g1;
    p.N2 = d_out;
    p.CN1 = round_up_i(g1, 16);
    p.CN2 = round_up_i(d_out, 16);
    p.w1_blk = p.CN1 / 2 * 128;
    p.w2_blk = p.CN2 / 2 * 128;
    const int pairs = num_sms / 2;
    const int fixed = 4 * 2 * STG_WARP_BYTES + HEAD_BIAS_FLOATS * 4 + HEAD_BAR_BYTES;
    const int wbytes = p.kb1 * p.w1_blk + p.kb2 * p.w2_blk;
    p.stages = std::min((SMEM_LIMIT - fixed - wbytes) / A_BYTES, HEAD_MAX_STAGES);
    if (p.stages < 3 || pairs < 1 || p.m_blocks < pairs) return cudaSuccess;
    p.bias = g;
    p.idesc1 = (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(p.CN1 >> 3) << 17) | ((uint32_t)((2 * BM) >> 4) << 24);
    p.idesc2 = (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(p.CN2 >> 3) << 17) | ((uint32_t)((2 * BM) >> 4) << 24);
    const int grid = 2 * pairs;
    const long long scr_rows = (long long)grid * HEAD_SLOTS * BM;
    const CUtensorMap *m;
    if (!(m = gemm_tc_map(st, H, M, d, BM, 0, false))) return cudaErrorInvalidValue;
    const CUtensorMap tmH = *m;
    if (!(m = gemm_tc_map(st, G1, g1, d, p.CN1 / 2, 0, false))) return cudaErrorInvalidValue;
    const CUtensorMap tmG1 = *m;
    if (!(m = gemm_tc_map(st, scratch, scr_rows, g1, 32, 0, false))) return cudaErrorInvalidValue;
    const CUtensorMap tmScrOut = *m;
    if (!(m = gemm_tc_map(st, scratch, scr_rows, g1, BM, 0, false))) return cudaErrorInvalidValue;
    const CUtensorMap tmScrIn = *m;
    if (!(m = gemm_tc_map(st, G2, d_out, g1, p.CN2 / 2, 0, false))) return cudaErrorInvalidValue;
    const CUtensorMap tmG2 = *m;
    if (!(m = gemm_tc_map(st, out, M, d_out, 32, 0, false))) return cudaErrorInvalidValue;
    const CUtensorMap tmOut = *m;
    cudaError_t e = cudaFuncSetAttribute(head_tc_pair_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_LIMIT);
    if (e != cudaSuccess) return e;
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3(HEAD_PAIR_THREADS);
    cfg.dynamicSmemBytes = (size_t)(wbytes + p.stages * A_BYTES + fixed);
    cfg.stream = s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = 2;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    if (launches) ++*launches;
    *taken = true;
    return cudaLaunchKernelEx(&cfg, head_tc_pair_kernel, tmH, tmG1, tmScrOut, tmScrIn, tmG2, tmOut, p);
}

}  // namespace

cudaError_t launch_head_tc(GemmTcState *st, int64_t M, int32_t d, int32_t g1, int32_t d_out, const void *H,
                           const void *G1, const float *g, const void *G2, void *out, void *scratch, int num_sms,
                           cudaStream_t s, int *launches, bool pairs)
{
    if (!head_tc_supported(d, g1, d_out) || M < 1 || M >= (1LL << 31)) return cudaErrorNotSupported;
    if (pairs) {
        bool taken = false;
        cudaError_t e = launch_head_pair(st, M, d, g1, d_out, H, G1, g, G2, out, scratch, num_sms, s, launches, &taken);
        if (e != cudaSuccess || taken) return e;
    }
    HeadTcParams p{};
    p.M = M;
    p.m_blocks = (M + BM - 1) / BM;
    p.kb1 = (d + BK - 1) / BK;
    p.kb2 = (g1 + BK - 1) / BK;
    p.N1 = g1;
    p.N2 = d_out;
    p.CN1 = round_up_i(g1, 16);
    p.CN2 = round_up_i(d_out, 16);
    p.stage_bytes = A_BYTES + std::max(p.CN1, p.CN2) * 128;
    const int fixed = 4 * 2 * STG_WARP_BYTES + HEAD_BIAS_FLOATS * 4 + HEAD_BAR_BYTES;
    p.stages = std::min((SMEM_LIMIT - fixed) / p.stage_bytes, HEAD_MAX_STAGES);
    if (p.stages < 2) return cudaErrorNotSupported;
    p.bias = g;
    p.idesc1 = (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(p.CN1 >> 3) << 17) | ((uint32_t)(BM >> 4) << 24);
    p.idesc2 = (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(p.CN2 >> 3) << 17) | ((uint32_t)(BM >> 4) << 24);
    const int grid = (int)std::min<long long>(num_sms, p.m_blocks);
    const long long scr_rows = (long long)grid * 2 * BM;
    const CUtensorMap *m;
    if (!(m = gemm_tc_map(st, H, M, d, BM, 0, false))) return cudaErrorInvalidValue;
    const CUtensorMap tmH = *m;
    if (!(m = gemm_tc_map(st, G1, g1, d, p.CN1, 0, false))) return cudaErrorInvalidValue;
    const CUtensorMap tmG1 = *m;
    if (!(m = gemm_tc_map(st, scratch, scr_rows, g1, 32, 0, false))) return cudaErrorInvalidValue;
    const CUtensorMap tmScrOut = *m;
    if (!(m = gemm_tc_map(st, scratch, scr_rows, g1, BM, 0, false))) return cudaErrorInvalidValue;
    const CUtensorMap tmScrIn = *m;
    if (!(m = gemm_tc_map(st, G2, d_out, g1, p.CN2, 0, false))) return cudaErrorInvalidValue;
    const CUtensorMap tmG2 = *m;
    if (!(m = gemm_tc_map(st, out, M, d_out, 32, 0, false))) return cudaErrorInvalidValue;
    const CUtensorMap tmOut = *m;
    static_assert(sizeof(CUtensorMap) == 128, "tensor map size");
    cudaError_t e = cudaFuncSetAttribute(head_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_LIMIT);
    if (e != cudaSuccess) return e;
    const int smem = p.stages * p.stage_bytes + fixed;
    if (launches) ++*launches;
    head_tc_kernel<<<grid, HEAD_THREADS, smem, s>>>(tmH, tmG1, tmScrOut, tmScrIn, tmG2, tmOut, p);
    return cudaGetLastError();
}

// ---- the head without any allocation (pinsage_head_static) --------------------------------------------
// Callers that may not allocate (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc) get
// the same kernels with the a-tile scratch in a file-scope array instead of the context's cudaMalloc'ed
// buffer.  Its size is the most the kernels above ask for on the part this library is written for: 148 SMs x
// HEAD_SLOTS (3) tiles x 128 rows x g1 <= 256 bf16 values = 29 097 984 bytes, held by every GPU that loads
// the library until the process exits.  In host code `g_head_scratch` is only a stand-in for the symbol --
// not a device address -- so the address is asked for once per device with cudaGetSymbolAddress.
// The array keeps the previous call's contents; nothing has to start at zero (every a tile is written
// before the mbarrier that lets the second GEMM read it), but every call uses the same array, so two calls
// that overlap on the GPU (different streams, different contexts) race.
constexpr size_t HEAD_STATIC_BYTES = (size_t)TUNED_SMS * HEAD_SLOTS * BM * 256 * 2;
static __device__ __align__(256) unsigned char g_head_scratch[HEAD_STATIC_BYTES];

size_t head_static_scratch_bytes() { return HEAD_STATIC_BYTES; }

namespace {
constexpr int HEAD_STATIC_MAX_DEVICES = 64;
std::mutex g_head_static_mu;
void *g_head_static_ptr[HEAD_STATIC_MAX_DEVICES] = {};    // device address of g_head_scratch, per device
}  // namespace

// The calling thread's current device must be the one the launch goes to.  *too_big: the shape needs more
// scratch than the array holds (nothing is launched then).
cudaError_t launch_head_tc_static(GemmTcState *st, int64_t M, int32_t d, int32_t g1, int32_t d_out, const void *H,
                                  const void *G1, const float *g, const void *G2, void *out, int num_sms,
                                  cudaStream_t s, int *launches, bool *too_big)
{
    *too_big = head_tc_scratch_bytes(g1, num_sms) > HEAD_STATIC_BYTES;
    if (*too_big) return cudaSuccess;
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= HEAD_STATIC_MAX_DEVICES) return cudaErrorInvalidDevice;
    void *ptr = nullptr;
    {
        std::lock_guard<std::mutex> lock(g_head_static_mu);
        if (!g_head_static_ptr[dev]) {          // set-up, once per device, with that device current
            void *q = nullptr;
            e = cudaGetSymbolAddress(&q, g_head_scratch);
            if (e != cudaSuccess) return e;
            if (!q || (reinterpret_cast<uintptr_t>(q) & 255u)) return cudaErrorInvalidSymbol;
            g_head_static_ptr[dev] = q;
        }
        ptr = g_head_static_ptr[dev];
    }
    return launch_head_tc(st, M, d, g1, d_out, H, G1, g, G2, out, ptr, num_sms, s, launches, true);
}

}  // namespace pinsage

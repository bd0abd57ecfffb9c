// gemm_tcgen05.cu -- S1 / S3 / S4 / S5 on the 5th-generation tensor cores (sm_100a).
//
//   out[M x N] = epi( A1[M x K1] * B[:, 0:K1]^T  +  A2[M x K2] * B[:, K1:K1+K2]^T  [+ A3[M x K3] * B[:, K1+K2:]^T] + bias )
//
// bf16 operands, fp32 accumulation in TMEM.  B is the paper's "out x in" weight matrix
// (Q, W, G1, G2 -- PAPER.md:114-115, :166) = a K-major operand as it lies in memory; the
// concat [h ; n] of Alg. 1 l.2 (:115) is never materialised: its two halves are two K segments
// that accumulate into the same TMEM tile.  Epilogue, fused, all in fp32 before the single
// rounding to bf16: + bias -> ReLU -> (S3) row L2 normalisation (Alg. 1 l.3, :116).
//
// Two instantiations: CG = 1 (one CTA per 128-row tile) and CG = 2 (a CTA PAIR, the two SMs of a
// TPC, per 256-row tile: tcgen05.mma.cta_group::2 issued by the even CTA, each CTA stages its own
// 128 rows of A and HALF of the B tile, so shared-memory and L2 operand traffic per flop drop by a
// third to a half).  CG = 2 is used whenever M >= 256 and the tile shape allows it.
//
// Structure (one persistent CTA per SM, 256 threads, warp-specialised):
//   warp 0      TMA producer: 128x64 A tile + (NS x 64) B tile per stage, SWIZZLE_128B, mbarrier ring
//   warp 1      MMA issuer: one elected thread issues tcgen05.mma (M=128, N=CN<=256, K=16)
//   warp 2      TMEM allocator
//   warps 4-7   epilogue: tcgen05.ld (each thread owns one output row) -> bias/ReLU/norm ->
//               bf16 -> swizzled smem staging -> TMA store (clips the ragged M / N tails)
// Accumulators are double-buffered in TMEM when a row tile needs <= 256 columns, so the
// epilogue of tile i overlaps the MMAs of tile i+1.  A thread owns a whole output row, so the
// row norm needs no cross-thread reduction as long as one CTA holds all N columns (N <= 512);
// wider rows (N <= 4096) are split over a thread-block cluster along N whose CTAs exchange
// per-row partial sums of squares through distributed shared memory.
#include "internal.h"

#include <algorithm>
#include <new>
#include <vector>

#include <cuda.h>  // CUtensorMap and enums only; cuTensorMapEncodeTiled is fetched at run time

#include "tc_ptx.cuh"

namespace pinsage {
namespace {

constexpr int NUM_THREADS = 384;        // 4 role warps + up to 8 epilogue warps
constexpr int MAX_STAGES = 8;
constexpr int MAX_CLUSTER = 8;

struct TcParams {
    long long M;
    long long m_blocks;
    int kb1, kb2, kb3; // 64-wide K blocks in segment 1 / 2 / 3
    int K12;           // column of B where segment 3 starts
    int K1;            // column of B where segment 2 starts
    int N;             // output columns in total
    int NS;            // output columns owned by one CTA (a slab)
    int CN;            // N of one tcgen05.mma (multiple of 16, <= 256)
    int nchunks;       // MMAs side by side per K step: nchunks * CN >= NS
    int nacc;          // accumulators in TMEM (2 = epilogue overlaps the next tile's MMAs)
    int acc_cols;      // TMEM columns between accumulators = nchunks * CN rounded up to 64
    int tmem_cols;     // allocation (power of two >= 32)
    int stages;
    int stage_bytes;   // A_BYTES + nchunks * CN * 128 (A_BYTES alone when B is stationary)
    int bres_bytes;    // > 0: this CTA's share of its B slab stays in shared memory for the whole launch
                       // ([KB][nchunks * CN / cg rows x 128 B] ahead of the operand ring) and only A streams
    int b_kb_bytes;    // bytes of one K block of that share
    int epi_halves;    // 1: four epilogue warps own all columns; 2: eight warps, two per row quarter,
                       // each owning half of the slab's columns
    int c_split;       // first column of the second half (multiple of 64)
    int stg_bytes;     // output staging: epi_halves * 4 warps * 2 buffers * 4 KB
    int n_slabs;       // slabs along N (= units per cluster when l2norm spans several CTAs)
    int cg;            // CTAs per tile: 1, or 2 = CTA pair (tcgen05 cta_group::2, 256-row tiles)
    int cluster;       // CTAs per cluster: cg, or cg * n_slabs when the row norm is exchanged (DSMEM)
    const float *bias;
    const uint4 *addend;   // optional [M x N] bf16 added to the accumulator (row stride N), or null
    int relu, l2norm;
    int out_f32;           // store fp32 (32-column TMA boxes) instead of bf16 (64-column boxes)
    // top-K selection epilogue (internal.h): no output matrix; scores that beat row q's k-th key are
    // appended to q's candidate buffer.  sel_nb = valid columns (candidates sel_id0 + column).
    unsigned long long *sel_state;
    int *sel_cnt;
    int tile_major;        // see the unit decode in the kernel
    // row-norm exchange through global memory between the CTA pairs that hold the slabs of one row
    // tile (gx = 1; they are co-resident: the grid is persistent, one CTA per SM): no cluster needed
    int gx;
    float *gx_buf;         // [2 parities][lanes][n_slabs][BM * cg] partial sums of squares
    unsigned *gx_cnt;      // [2 parities][lanes][cg][4 row quarters] arrivals (zeroed before the launch)
    int sel_k, sel_nb;
    long long sel_id0;
    uint32_t idesc;
};

// Shared-memory plan (offsets from the 1024-byte aligned dynamic base):
//   [0, stages*stage_bytes)   operand ring: per stage A (16 KB) then B (nchunks*CN rows x 128 B)
//   + 32 / 64 KB              output staging: 4 / 8 epilogue warps x 2 buffers x (32 rows x 128 B)
//   + 2 KB                    bias of this CTA's slab (fp32, zero beyond N)
//   + 256 B                   mbarriers, TMEM base address
//   + 2 KB                    row sum-of-squares exchange between the two column halves [2][2][128] fp32
//   + 8 KB (cluster > 1)      row-norm exchange [2][MAX_CLUSTER][128] fp32
constexpr int SEL_Q = 8;                 // selection epilogue: queue slots per row and warp (2 KB per warp)
constexpr int BIAS_BYTES = 512 * 4;
constexpr int BAR_BYTES = 256;
constexpr int HALF_BYTES = 2 * 2 * BM * 4;
constexpr int XCHG_BYTES = 2 * MAX_CLUSTER * BM * 4;

// CG: CTAs per tile (1, or 2 = pair).  NCH: tcgen05.mma instructions side by side per K step (1 or 2;
// compile-time so that the issue loop unrolls into straight-line UTCHMMAs).
template <int CG, int NCH>
__global__ void __launch_bounds__(NUM_THREADS, 1)
gemm_tc_kernel(const __grid_constant__ CUtensorMap tmA1, const __grid_constant__ CUtensorMap tmA2,
               const __grid_constant__ CUtensorMap tmA3,
               const __grid_constant__ CUtensorMap tmB, const __grid_constant__ CUtensorMap tmOut,
               const TcParams p)
{
    extern __shared__ __align__(1024) uint8_t smem[];
    const uint32_t sbase = smem_u32(smem);
    if ((sbase & 1023u) != 0) __trap();  // SWIZZLE_128B tiles need 1024-byte alignment

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t ring_off = (uint32_t)p.bres_bytes;          // the operand ring follows the stationary B
    const uint32_t stg_off = ring_off + (uint32_t)p.stages * p.stage_bytes;
    const uint32_t bias_off = stg_off + (uint32_t)p.stg_bytes;
    const uint32_t bar_off = bias_off + BIAS_BYTES;
    const uint32_t half_off = bar_off + BAR_BYTES;
    const uint32_t xchg_off = half_off + (p.epi_halves == 2 ? HALF_BYTES : 0);
    float *sbias = reinterpret_cast<float *>(smem + bias_off);
    const uint32_t bar_full = sbase + bar_off;                 // [MAX_STAGES]  (CG 2: the leader's are used)
    const uint32_t bar_empty = bar_full + 8 * MAX_STAGES;      // [MAX_STAGES]
    const uint32_t bar_tfull = bar_empty + 8 * MAX_STAGES;     // [2]
    const uint32_t bar_tempty = bar_tfull + 16;                // [2]           (CG 2: the leader's are used)
    const uint32_t bar_xchg = bar_tempty + 16;                 // [2]
    const uint32_t bar_bres = bar_full + 184;                  // stationary B has landed (CG 2: the leader's)
    volatile uint32_t *tmem_slot = reinterpret_cast<volatile uint32_t *>(smem + bar_off + 8 * (2 * MAX_STAGES + 6));

    // A "unit" is the CTA (CG 1) or CTA pair (CG 2) that owns one (row tile, slab) at a time.
    const uint32_t crank = p.cluster > 1 ? cluster_ctarank() : 0;
    const uint32_t half = CG == 2 ? (crank & 1u) : 0u;         // which 128 rows of the 256-row tile
    const uint32_t leader = crank & ~1u;                       // cluster rank of this pair's even CTA
    const long long unit = blockIdx.x / CG, units = gridDim.x / CG;
    // Persistent schedule: a unit keeps its slab and walks the row tiles lane0, lane0 + lanes, ...
    // Tile-major schedule (p.tile_major; one tile per unit, row tile fastest): the units resident at
    // one time then share a few slabs of B instead of holding one each -- for long K with many slabs,
    // where the slabs in flight would not fit L2 and each would be re-read from HBM per row tile.
    const int slab = p.tile_major ? (int)(unit / p.m_blocks) : (int)(unit % p.n_slabs);
    const long long lane0 = p.tile_major ? unit % p.m_blocks : unit / p.n_slabs;
    const long long lanes = p.tile_major ? p.m_blocks : units / p.n_slabs;
    const int n0 = slab * p.NS;
    const int ncols = min(p.NS, p.N - n0);  // valid output columns of this slab
    const int KB = p.kb1 + p.kb2 + p.kb3;
    const int b_rows = p.CN / CG;           // rows of B this CTA stages per MMA chunk

    // ---- one-time setup ---------------------------------------------------------------------
    if (warp == 0 && lane == 0) {
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmA1) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmA2) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmA3) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmB) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmOut) : "memory");
    }
    if (warp == 1 && lane == 0) {
        for (int s = 0; s < p.stages; ++s) {
            mbar_init(bar_full + 8 * s, 1);
            mbar_init(bar_empty + 8 * s, 1);
        }
        for (int a = 0; a < 2; ++a) {
            mbar_init(bar_tfull + 8 * a, 1);
            mbar_init(bar_tempty + 8 * a, 4 * CG * p.epi_halves);  // every epilogue warp of the unit
            mbar_init(bar_xchg + 8 * a, 1);                         // armed per tile with the expected bytes
        }
        mbar_init(bar_bres, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 2) {
        if (CG == 2) {
            asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(
                             smem_u32(const_cast<uint32_t *>(tmem_slot))),
                         "r"((uint32_t)p.tmem_cols)
                         : "memory");
            asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
        } else {
            asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(
                             smem_u32(const_cast<uint32_t *>(tmem_slot))),
                         "r"((uint32_t)p.tmem_cols)
                         : "memory");
            asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
        }
    }
    if (warp >= 4 && warp < 8) {
        for (int c = threadIdx.x - 128; c < 512; c += 128)
            sbias[c] = (p.bias != nullptr && c < ncols) ? __ldg(p.bias + n0 + c) : 0.f;
    }
    tc_fence_before();
    if (p.cluster > 1) cluster_sync_all();
    else __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    if (warp == 0) {
        // ===== TMA producer (every CTA: its own 128 rows of A and its share of B) =================
        // the whole warp runs the loop; one elected lane issues
        uint64_t pol_stream, pol_keep;
        asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol_stream));
        asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol_keep));
        // A is read once per slab: keep it in L2 while the other slabs of the same rows still need it
        const uint64_t pol_a = p.n_slabs > 1 ? pol_keep : pol_stream;
        const uint32_t leader_full = CG == 2 ? map_to_cta(bar_full, leader) : bar_full;
        if (p.bres_bytes && lane0 < p.m_blocks) {
            // this CTA's share of the slab of B, once: every K block into its place ahead of the ring
            if (elect_one()) {
                const uint32_t lbar = CG == 2 ? map_to_cta(bar_bres, leader) : bar_bres;
                if (half == 0) mbar_expect_tx(bar_bres, (uint32_t)(CG * p.bres_bytes));
                for (int kb = 0; kb < KB; ++kb) {
                    const int seg = kb < p.kb1 ? 0 : kb < p.kb1 + p.kb2 ? 1 : 2;
                    const int ka = (seg == 0 ? kb : seg == 1 ? kb - p.kb1 : kb - p.kb1 - p.kb2) * BK;
                    const int kcol = (seg == 0 ? 0 : seg == 1 ? p.K1 : p.K12) + ka;
                    const uint32_t sB = sbase + (uint32_t)kb * p.b_kb_bytes;
#pragma unroll
                    for (int j = 0; j < NCH; ++j) {
                        if (CG == 2)
                            tma_load_2d_pair(sB + (uint32_t)j * b_rows * 128, &tmB, kcol,
                                             n0 + j * p.CN + (int)half * b_rows, lbar, pol_keep);
                        else
                            tma_load_2d(sB + (uint32_t)j * b_rows * 128, &tmB, kcol, n0 + j * p.CN, lbar, pol_keep);
                    }
                }
            }
            __syncwarp();
        }
        int stage = 0;
        uint32_t phase = 0;
        for (long long mb = lane0; mb < p.m_blocks; mb += lanes) {
            const int m0 = (int)(mb * (BM * CG)) + (int)half * BM;
            for (int kb = 0; kb < KB; ++kb) {
                mbar_wait(bar_empty + 8 * stage, phase ^ 1);
                if (elect_one()) {
                    const uint32_t full = bar_full + 8 * stage;
                    const int seg = kb < p.kb1 ? 0 : kb < p.kb1 + p.kb2 ? 1 : 2;
                    const int ka = (seg == 0 ? kb : seg == 1 ? kb - p.kb1 : kb - p.kb1 - p.kb2) * BK;
                    const uint32_t sA = sbase + ring_off + (uint32_t)stage * p.stage_bytes;
                    const int kcol = (seg == 0 ? 0 : seg == 1 ? p.K1 : p.K12) + ka;
                    const CUtensorMap *tmA = seg == 0 ? &tmA1 : seg == 1 ? &tmA2 : &tmA3;
                    if (CG == 2) {
                        // both CTAs' bytes complete on the leader's barrier
                        if (half == 0) mbar_expect_tx(full, 2u * (uint32_t)p.stage_bytes);
                        const uint32_t lfull = leader_full + 8 * stage;
                        tma_load_2d_pair(sA, tmA, ka, m0, lfull, pol_a);
                        if (!p.bres_bytes) {
#pragma unroll
                            for (int j = 0; j < NCH; ++j)
                                tma_load_2d_pair(sA + A_BYTES + (uint32_t)j * b_rows * 128, &tmB, kcol,
                                                 n0 + j * p.CN + (int)half * b_rows, lfull, pol_keep);
                        }
                    } else {
                        mbar_expect_tx(full, (uint32_t)p.stage_bytes);
                        tma_load_2d(sA, tmA, ka, m0, full, pol_a);
                        if (!p.bres_bytes) {
#pragma unroll
                            for (int j = 0; j < NCH; ++j)
                                tma_load_2d(sA + A_BYTES + (uint32_t)j * p.CN * 128, &tmB, kcol,
                                            n0 + j * p.CN, full, pol_keep);
                        }
                    }
                }
                __syncwarp();
                if (++stage == p.stages) {
                    stage = 0;
                    phase ^= 1;
                }
            }
        }
    } else if (warp == 1) {
        // ===== MMA issuer (CG 2: the pair's even CTA only) ========================================
        // the whole warp runs the loop (all lanes wait on the barriers); one elected lane issues
        if (half == 0) {
            const uint16_t pair_mask = (uint16_t)(3u << leader);
            const uint32_t b_step = (uint32_t)((b_rows * 128) >> 4);  // descriptor units between chunks
            int stage = 0, acc = 0;
            uint32_t phase = 0, accphase = 0;
            if (p.bres_bytes && lane0 < p.m_blocks) {            // stationary B (both CTAs' shares) has landed
                mbar_wait(bar_bres, 0);
                tc_fence_after();
            }
            for (long long mb = lane0; mb < p.m_blocks; mb += lanes) {
                mbar_wait(bar_tempty + 8 * acc, accphase ^ 1);   // epilogue(s) drained this accumulator
                tc_fence_after();
                const uint32_t d0 = tmem_base + (uint32_t)acc * p.acc_cols;
                for (int kb = 0; kb < KB; ++kb) {
                    mbar_wait(bar_full + 8 * stage, phase);      // TMA bytes have landed (both CTAs)
                    tc_fence_after();
                    if (elect_one()) {
                        const uint32_t sA = sbase + ring_off + (uint32_t)stage * p.stage_bytes;
                        const uint64_t ad = make_desc(sA);
                        const uint64_t bd = make_desc(p.bres_bytes ? sbase + (uint32_t)kb * p.b_kb_bytes : sA + A_BYTES);
#pragma unroll
                        for (int k = 0; k < BK / 16; ++k)        // 32 bytes along K per UMMA_K = 16
#pragma unroll
                            for (int j = 0; j < NCH; ++j) {
                                const uint32_t accum = k == 0 ? (uint32_t)kb : 1u;
                                if (CG == 2)
                                    tc_mma_pair(d0 + (uint32_t)j * p.CN, ad + 2 * k, bd + j * b_step + 2 * k,
                                                p.idesc, accum);
                                else
                                    tc_mma(d0 + (uint32_t)j * p.CN, ad + 2 * k, bd + j * b_step + 2 * k,
                                           p.idesc, accum);
                            }
                        // frees the stage (in both CTAs) when the MMAs retire
                        if (CG == 2) tc_commit_pair(bar_empty + 8 * stage, pair_mask);
                        else tc_commit(bar_empty + 8 * stage);
                        if (kb == KB - 1) {                      // accumulator complete
                            if (CG == 2) tc_commit_pair(bar_tfull + 8 * acc, pair_mask);
                            else tc_commit(bar_tfull + 8 * acc);
                        }
                    }
                    __syncwarp();
                    if (++stage == p.stages) {
                        stage = 0;
                        phase ^= 1;
                    }
                }
                if (++acc == p.nacc) {
                    acc = 0;
                    accphase ^= 1;
                }
            }
        }
    } else if (warp >= 4 && ((warp - 4) >> 2) < p.epi_halves) {
        // ===== epilogue: thread (ew, lane) owns output row m0 + 32*ew + lane; with eight warps the two
        // warps of a row quarter each own one half of the slab's columns =============================
        const int ew = warp & 3;                                  // == warp % 4: TMEM lanes 32*ew..
        const int eh = (warp - 4) >> 2;                           // column half
        const int row = ew * 32 + lane;
        const int c_lo = eh == 0 ? 0 : p.c_split;
        const int c_hi = (p.epi_halves == 2 && eh == 0) ? min(p.c_split, ncols) : ncols;
        uint8_t *stg = smem + stg_off + (eh * 4 + ew) * 2 * STG_WARP_BYTES;
        const int units_per_cluster = p.cluster / CG;
        const uint32_t my_unit = crank / CG;
        float *xbuf = reinterpret_cast<float *>(smem + xchg_off);  // [2][MAX_CLUSTER][BM]
        float *hbuf = reinterpret_cast<float *>(smem + half_off);  // [2][2][BM]
        const uint32_t tempty_leader = CG == 2 ? map_to_cta(bar_tempty, leader) : 0u;
        int acc = 0, sbuf = 0;
        uint32_t accphase = 0;
        long long it = 0;
        for (long long mb = lane0; mb < p.m_blocks; mb += lanes, ++it) {
            const long long m0 = mb * (BM * CG) + (long long)half * BM;
            mbar_wait(bar_tfull + 8 * acc, accphase);
            tc_fence_after();
            const uint32_t t0 = tmem_base + ((uint32_t)(ew * 32) << 16) + (uint32_t)acc * p.acc_cols;
            // this row's slice of the addend (slab column 0), null if there is none or the row is past M
            const uint4 *arow = (p.addend != nullptr && m0 + row < p.M)
                                    ? p.addend + (((size_t)(m0 + row) * (size_t)p.N + (size_t)n0) >> 3)
                                    : nullptr;
            float scale = 1.f;
            if (p.l2norm) {
                // pass 1: sum of squares of this row's z = act(acc + addend + bias) over my columns
                const int par = (int)(it & 1);
                float2 ss2 = make_float2(0.f, 0.f);       // sums of squares of the even / odd columns
                for (int c0 = c_lo; c0 < c_hi; c0 += 32) {
                    uint32_t v[32];
                    tc_ld32(t0 + c0, v);
                    tc_wait_ld();
                    if (p.addend != nullptr) add_addend32(arow, c0, c_hi, v);   // uniform branch
                    // packed fp32x2 adds / fmas (sm_100): half the issue slots of the scalar forms; z is
                    // parked back in TMEM so that the store pass only scales and rounds
#pragma unroll
                    for (int i = 0; i < 32; i += 2) {
                        const float2 b2 = *reinterpret_cast<const float2 *>(sbias + c0 + i);
                        float2 z2 = __fadd2_rn(make_float2(__uint_as_float(v[i]), __uint_as_float(v[i + 1])), b2);
                        if (p.relu) {
                            z2.x = fmaxf(z2.x, 0.f);
                            z2.y = fmaxf(z2.y, 0.f);
                        }
                        if (c0 + i < c_hi) ss2 = __ffma2_rn(z2, z2, ss2);   // N % 8 == 0: pairs never straddle
                        v[i] = __float_as_uint(z2.x);
                        v[i + 1] = __float_as_uint(z2.y);
                    }
                    tc_st32(t0 + c0, v);
                }
                tc_wait_st();
                float ss = ss2.x + ss2.y;
                if (p.epi_halves == 2) {
                    // the two warps of this row quarter add their halves (fixed order: low + high)
                    hbuf[(par * 2 + eh) * BM + row] = ss;
                    asm volatile("bar.sync %0, 64;" ::"r"(1 + ew) : "memory");
                    ss = hbuf[(par * 2 + 0) * BM + row] + hbuf[(par * 2 + 1) * BM + row];
                }
                if (units_per_cluster > 1) {
                    // push my slab's partial to the CTAs that hold the other slabs of the same rows
                    // (low-half warps only; st.async: DSMEM store + transaction count of the peer's
                    // barrier in one operation), then wait for theirs
                    if (eh == 0) {
                        // one thread arms this tile's phase: 128 rows x 4 bytes from each other slab
                        if (ew == 0 && lane == 0)
                            mbar_expect_tx(bar_xchg + 8 * par, (uint32_t)(BM * 4 * (units_per_cluster - 1)));
                        const uint32_t my_slot = sbase + xchg_off + ((par * MAX_CLUSTER + my_unit) * BM + row) * 4;
                        for (uint32_t u = 0; u < (uint32_t)units_per_cluster; ++u) {
                            if (u == my_unit) continue;
                            const uint32_t r = u * CG + half;
                            st_async_f32(map_to_cta(my_slot, r), ss, map_to_cta(bar_xchg + 8 * par, r));
                        }
                    }
                    mbar_wait_cluster(bar_xchg + 8 * par, (uint32_t)((it >> 1) & 1));
                    float tot = 0.f;
                    for (uint32_t u = 0; u < (uint32_t)units_per_cluster; ++u)   // same order in every CTA
                        tot += (u == my_unit) ? ss : xbuf[(par * MAX_CLUSTER + u) * BM + row];
                    ss = tot;
                }
                if (p.gx) {
                    // same exchange through global memory: publish my slab's partial, count the
                    // arrival of my 32 rows, wait until all slabs of this row quarter have arrived
                    const int rows_u = BM * CG;
                    float *slot = p.gx_buf + ((size_t)par * lanes + lane0) * p.n_slabs * rows_u + half * BM + row;
                    unsigned *cnt = p.gx_cnt + (((size_t)par * lanes + lane0) * CG + half) * 4 + ew;
                    if (eh == 0) {
                        __stcg(slot + (size_t)slab * rows_u, ss);
                        __threadfence();
                        __syncwarp();
                        if (lane == 0) atomicAdd(cnt, 1u);
                    }
                    const unsigned target = (unsigned)((it >> 1) + 1) * (unsigned)p.n_slabs;
                    if (lane == 0) {
                        // plain launch (gx 2): nothing but the idle device makes the peers co-resident,
                        // so a wait that outlasts ~2^32 cycles traps (a loud error, not a hang)
                        const long long t_start = p.gx == 2 ? clock64() : 0;
                        unsigned seen, polls = 0;
                        do {
                            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(cnt) : "memory");
                            if (p.gx == 2 && (++polls & 0xfffu) == 0 && clock64() - t_start > (1LL << 32)) __trap();
                        } while (seen < target);
                    }
                    __syncwarp();
                    __threadfence();
                    float tot = 0.f;
                    for (int u = 0; u < p.n_slabs; ++u)           // same order in every CTA
                        tot += (u == slab) ? ss : __ldcg(slot + (size_t)u * rows_u);
                    ss = tot;
                }
                scale = ss > 0.f ? rsqrtf(ss) : 0.f;             // zero row stays zero (reading A3)
            }
            if (p.sel_state != nullptr) {
                // selection epilogue of the top-K lookup: one max per score against the row's current
                // k-th score; the (rare) survivors become keys in the row's candidate buffer
                const long long q = m0 + row;
                const bool live = q < p.M;
                unsigned long long *st = p.sel_state + (size_t)(live ? q : 0) * TK_TOTAL;
                const unsigned long long tau = live ? st[p.sel_k - 1] : ~0ull;
                const float tau_f = !live ? INFINITY : tau ? unord_f32((unsigned)(tau >> 32)) : -INFINITY;
                // A score is kept when it reaches the k-th score (ties with it included: a key that
                // does not beat tau is dropped by the next merge, so a superset is harmless).  One pass
                // over the accumulator; the rare keepers become keys in this row's queue in the warp's
                // staging memory.  The accumulator is released before the queue goes to global memory,
                // so the one atomicAdd per row that reserves the slots is off the MMA's critical path.
                const int lim = min(c_hi, p.sel_nb - n0);         // valid columns of this slab
                unsigned long long *sq = reinterpret_cast<unsigned long long *>(
                    smem + stg_off + (eh * 4 + ew) * (SEL_Q * 32 * 8));                  // [SEL_Q][32 lanes]
                int nl = 0;
                for (int c0 = c_lo; c0 < c_hi; c0 += OUT_CHUNK) {
                    uint32_t v[2][32];
                    tc_ld32(t0 + c0, v[0]);                       // (warp-collective: never under a lane's branch)
                    tc_ld32(t0 + c0 + 32, v[1]);
                    tc_wait_ld();
                    if (c0 + OUT_CHUNK > lim) {                   // ragged end (uniform): columns past it lose
#pragma unroll
                        for (int i = 0; i < 64; ++i)
                            if (c0 + i >= lim) v[i >> 5][i & 31] = 0xff800000u;   // -inf
                    }
                    // eight columns at a time: one max tree and one warp vote; only a group in which some
                    // row has a keeper is looked at column by column, again under warp-uniform branches
#pragma unroll
                    for (int g8 = 0; g8 < 8; ++g8) {
                        const uint32_t *w = &v[g8 >> 2][(g8 & 3) * 8];
                        const float mx = fmaxf(
                            fmaxf(fmaxf(__uint_as_float(w[0]), __uint_as_float(w[1])),
                                  fmaxf(__uint_as_float(w[2]), __uint_as_float(w[3]))),
                            fmaxf(fmaxf(__uint_as_float(w[4]), __uint_as_float(w[5])),
                                  fmaxf(__uint_as_float(w[6]), __uint_as_float(w[7]))));
                        if (!__any_sync(0xffffffffu, mx >= tau_f)) continue;
#pragma unroll
                        for (int j = 0; j < 8; ++j) {
                            const float x = __uint_as_float(w[j]);
                            const bool hit = x >= tau_f;
                            if (!__any_sync(0xffffffffu, hit)) continue;
                            if (hit) {
                                const unsigned long long key = make_key(x, p.sel_id0 + n0 + c0 + g8 * 8 + j);
                                if (nl < SEL_Q) {
                                    sq[nl * 32 + lane] = key;
                                } else {                          // queue full (a very loose tau): one by one
                                    const int slot = atomicAdd(p.sel_cnt + q, 1);
                                    if (slot < TK_LIST) st[TK_LIST + slot] = key;
                                }
                                ++nl;
                            }
                        }
                    }
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) {
                    if (CG == 2) mbar_arrive_remote_relaxed(tempty_leader + 8 * acc);
                    else mbar_arrive(bar_tempty + 8 * acc);
                }
                nl = min(nl, SEL_Q);
                if (nl) {
                    const int at = atomicAdd(p.sel_cnt + q, nl);
                    for (int j = 0; j < nl && at + j < TK_LIST; ++j) st[TK_LIST + at + j] = sq[j * 32 + lane];
                }
                __syncwarp();
                if (++acc == p.nacc) {
                    acc = 0;
                    accphase ^= 1;
                }
                continue;
            } else
            // pass 2: 64 columns at a time -> bf16 -> swizzled staging -> TMA store
            for (int c0 = c_lo; c0 < c_hi; c0 += OUT_CHUNK) {
                uint32_t v[2][32];
                tc_ld32(t0 + c0, v[0]);
                tc_ld32(t0 + c0 + 32, v[1]);
                tc_wait_ld();
                uint32_t pk[32];
                if (p.l2norm) {                                   // TMEM already holds z: scale and round
                    const float2 sc2 = make_float2(scale, scale);
#pragma unroll
                    for (int h = 0; h < 2; ++h)
#pragma unroll
                        for (int i = 0; i < 32; i += 2) {
                            const float2 z2 = __fmul2_rn(
                                make_float2(__uint_as_float(v[h][i]), __uint_as_float(v[h][i + 1])), sc2);
                            __nv_bfloat162 b = __floats2bfloat162_rn(z2.x, z2.y);
                            pk[16 * h + i / 2] = *reinterpret_cast<uint32_t *>(&b);
                        }
                } else {
                    if (p.addend != nullptr) {                    // uniform branch
                        add_addend32(arow, c0, c_hi, v[0]);
                        add_addend32(arow, c0 + 32, c_hi, v[1]);
                    }
#pragma unroll
                    for (int h = 0; h < 2; ++h)
#pragma unroll
                        for (int i = 0; i < 32; i += 2) {
                            const float2 b2 = *reinterpret_cast<const float2 *>(sbias + c0 + 32 * h + i);
                            float2 z2 = __fadd2_rn(
                                make_float2(__uint_as_float(v[h][i]), __uint_as_float(v[h][i + 1])), b2);
                            if (p.relu) {
                                z2.x = fmaxf(z2.x, 0.f);
                                z2.y = fmaxf(z2.y, 0.f);
                            }
                            __nv_bfloat162 b = __floats2bfloat162_rn(z2.x, z2.y);
                            pk[16 * h + i / 2] = *reinterpret_cast<uint32_t *>(&b);
                        }
                }
                if (p.out_f32) {
                    // fp32 result: each 32-column half is one 32 x 128-byte box of raw accumulator values
                    // (after bias / ReLU), same XOR swizzle, one TMA store per half
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        if (c0 + 32 * h >= c_hi) break;
                        uint32_t z[32];
#pragma unroll
                        for (int i = 0; i < 32; ++i) {
                            float x = __uint_as_float(v[h][i]);
                            if (p.l2norm) {                       // TMEM already holds z
                                x *= scale;
                            } else {
                                x += sbias[c0 + 32 * h + i];
                                x = p.relu ? fmaxf(x, 0.f) : x;
                            }
                            z[i] = __float_as_uint(x);
                        }
                        if (lane == 0) tma_store_wait_read<1>();
                        __syncwarp();
                        uint8_t *fbuf = stg + sbuf * STG_WARP_BYTES;
                        uint8_t *frow = fbuf + lane * 128;
#pragma unroll
                        for (int q = 0; q < 8; ++q)
                            *reinterpret_cast<uint4 *>(frow + ((q ^ (lane & 7)) << 4)) =
                                make_uint4(z[4 * q], z[4 * q + 1], z[4 * q + 2], z[4 * q + 3]);
                        fence_proxy_async();
                        __syncwarp();
                        if (lane == 0 && m0 + ew * 32 < p.M) {
                            tma_store_2d(&tmOut, n0 + c0 + 32 * h, (int)(m0 + ew * 32), smem_u32(fbuf));
                            tma_store_commit();
                        }
                        sbuf ^= 1;
                    }
                    continue;
                }
                if (lane == 0) tma_store_wait_read<1>();          // the buffer used two stores ago is free
                __syncwarp();
                uint8_t *buf = stg + sbuf * STG_WARP_BYTES;
                uint8_t *rowp = buf + lane * 128;
#pragma unroll
                for (int q = 0; q < 8; ++q)                       // 16-byte chunk q of the row, XOR-swizzled
                    *reinterpret_cast<uint4 *>(rowp + ((q ^ (lane & 7)) << 4)) =
                        make_uint4(pk[4 * q], pk[4 * q + 1], pk[4 * q + 2], pk[4 * q + 3]);
                fence_proxy_async();
                __syncwarp();
                if (lane == 0 && m0 + ew * 32 < p.M) {
                    tma_store_2d(&tmOut, n0 + c0, (int)(m0 + ew * 32), smem_u32(buf));
                    tma_store_commit();
                }
                sbuf ^= 1;
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) {
                if (CG == 2) mbar_arrive_remote_relaxed(tempty_leader + 8 * acc);
                else mbar_arrive(bar_tempty + 8 * acc);
            }
            if (++acc == p.nacc) {
                acc = 0;
                accphase ^= 1;
            }
        }
        if (lane == 0) tma_store_wait_all();
    }

    // ---- teardown ---------------------------------------------------------------------------
    __syncwarp();
    tc_fence_before();
    if (p.cluster > 1) cluster_sync_all();
    else __syncthreads();
    if (warp == 2) {
        tc_fence_after();
        if (CG == 2)
            asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem_base),
                         "r"((uint32_t)p.tmem_cols)
                         : "memory");
        else
            asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base),
                         "r"((uint32_t)p.tmem_cols)
                         : "memory");
    }
}

// ---- host side ----------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *,
                                  const cuuint64_t *, const cuuint64_t *, const cuuint32_t *,
                                  const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn()
{
    static EncodeTiledFn fn = [] {          // (thread-safe: a C++11 function-local static)
        void *sym = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &sym, cudaEnableDefault, &q) != cudaSuccess ||
            q != cudaDriverEntryPointSuccess)
            sym = nullptr;
        return reinterpret_cast<EncodeTiledFn>(sym);
    }();
    return fn;
}

inline int round_up(int x, int a) { return (x + a - 1) / a * a; }

}  // namespace

// Everything the launcher remembers between calls lives here, one per context (internal.h).
struct GemmTcState {
    int num_sms = 0;
    bool attr_set[2][2] = {{false, false}, {false, false}};            // [CG - 1][NCH - 1]
    int clusters[2][2][MAX_CLUSTER + 1] = {};                          // co-resident clusters, 0 = not asked yet
    struct GxSlot { cudaStream_t s; void *mem; };
    std::vector<GxSlot> gx;                                            // exchange buffers, one per stream used
    size_t gx_buf_bytes = 0, gx_cnt_bytes = 0;
    // tensor maps by (pointer, shape): encoding one is a driver call, and a chunked layer reuses the
    // same few dozen descriptors call after call
    struct MapKey {
        const void *ptr; long long rows; int cols, box_rows, ld, f32;
        bool operator==(const MapKey &o) const
        {
            return ptr == o.ptr && rows == o.rows && cols == o.cols && box_rows == o.box_rows && ld == o.ld &&
                   f32 == o.f32;
        }
    };
    static constexpr int MAP_SLOTS = 512, MAP_WAYS = 4;
    struct MapEntry { MapKey key; CUtensorMap map; bool used; };
    std::vector<MapEntry> maps;
    unsigned map_clock = 0;
    long long map_hits = 0, map_misses = 0;
};

GemmTcState *gemm_tc_state_create(int num_sms)
{
    GemmTcState *st = new (std::nothrow) GemmTcState;
    if (!st) return nullptr;
    st->num_sms = num_sms;
    // [2 parities][lanes][n_slabs][BM * cg] floats with lanes * n_slabs * cg <= num_sms CTAs, and
    // [2][lanes][cg][4] arrival counters
    st->gx_buf_bytes = (size_t)2 * num_sms * BM * sizeof(float);
    st->gx_cnt_bytes = (size_t)2 * num_sms * 4 * sizeof(unsigned);
    st->maps.resize(GemmTcState::MAP_SLOTS);
    for (auto &m : st->maps) m.used = false;
    return st;
}

void gemm_tc_state_destroy(GemmTcState *st)
{
    if (!st) return;
    for (const auto &g : st->gx) cudaFree(g.mem);
    delete st;
}

namespace {

// Row-major matrix [rows x cols] (cols contiguous, bf16 or fp32), box = box_rows x 128 bytes,
// SWIZZLE_128B.  Out-of-bounds parts of a box read as zero and are not written.
const CUtensorMap *get_map(GemmTcState *st, const void *ptr, long long rows, int cols, int box_rows, int ld = 0,
                           bool f32 = false)
{
    EncodeTiledFn fn = encode_fn();
    if (!fn) return nullptr;
    const GemmTcState::MapKey key{ptr, rows, cols, box_rows, ld, f32 ? 1 : 0};
    size_t h = reinterpret_cast<uintptr_t>(ptr) >> 4;
    h = (h ^ (h >> 17) ^ (size_t)rows * 0x9E3779B1u ^ (size_t)cols * 0x85EBCA77u ^ (size_t)box_rows * 0xC2B2AE3Du ^
         (size_t)ld * 0x27D4EB2Fu ^ (size_t)key.f32) & (GemmTcState::MAP_SLOTS / GemmTcState::MAP_WAYS - 1);
    GemmTcState::MapEntry *set = st->maps.data() + h * GemmTcState::MAP_WAYS;
    for (int w = 0; w < GemmTcState::MAP_WAYS; ++w)
        if (set[w].used && set[w].key == key) {
            ++st->map_hits;
            return &set[w].map;
        }
    ++st->map_misses;
    GemmTcState::MapEntry *e = &set[st->map_clock++ % GemmTcState::MAP_WAYS];
    for (int w = 0; w < GemmTcState::MAP_WAYS; ++w)
        if (!set[w].used) {
            e = &set[w];
            break;
        }
    const int es = f32 ? 4 : 2;
    const cuuint64_t dims[2] = {(cuuint64_t)cols, (cuuint64_t)rows};
    const cuuint64_t strides[1] = {(cuuint64_t)(ld > 0 ? ld : cols) * es};
    const cuuint32_t box[2] = {(cuuint32_t)(128 / es), (cuuint32_t)box_rows};   // 128-byte rows
    const cuuint32_t estr[2] = {1, 1};
    e->used = false;
    if (fn(&e->map, f32 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2,
           const_cast<void *>(ptr), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
           CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return nullptr;
    e->key = key;
    e->used = true;
    return &e->map;
}

// cg: CTAs per tile (1 or 2).  Slabs without a row norm are 256 columns wide (double-buffered
// accumulators: the epilogue of tile i overlaps the MMAs of tile i+1).
bool plan(const GemmArgs &a, int cg, int gx_pref, int bres_pref, TcParams &p, int &smem_bytes, const char **why)
{
    auto no = [&](const char *msg) {
        if (why) *why = msg;
        return false;
    };
    if (a.M < 1 || a.M >= (1LL << 31)) return no("M outside [1, 2^31)");
    if (a.K1 < 8 || a.K1 % 8 || a.K2 < 0 || a.K2 % 8 || a.K3 < 0 || a.K3 % 8)
        return no("K1, K2, K3 must be multiples of 8");
    if (a.K3 > 0 && a.K2 == 0) return no("a third K segment needs the second");
    if (a.N < 8 || a.N % 8) return no("N must be a multiple of 8");
    if (a.ldb % 8 || (a.ldb > 0 && a.ldb < a.K1 + a.K2 + a.K3))
        return no("ldb must be a multiple of 8, >= K1 + K2 + K3");
    if (cg == 2 && (a.M <= BM || a.N % 16)) return no("CTA pairs need M > 128 and N % 16 == 0");
    if (a.out_f32 && a.addend) return no("fp32 output takes no addend");
    if (a.sel_state && (a.l2norm || a.addend || a.bias || a.relu || a.sel_k < 1 || a.sel_k > TK_LIST))
        return no("the selection epilogue takes plain products and 1 <= k <= 1024");
    p = TcParams{};
    p.cg = cg;
    p.M = a.M;
    p.m_blocks = (a.M + BM * cg - 1) / (BM * cg);
    p.kb1 = (a.K1 + BK - 1) / BK;
    p.kb2 = (a.K2 + BK - 1) / BK;
    p.kb3 = (a.K3 + BK - 1) / BK;
    p.K12 = a.K1 + a.K2;
    p.K1 = a.K1;
    p.N = a.N;
    // a normalised row of up to 512 columns sits in the TMEM of one CTA (one accumulator); a wider one
    // is cut into 256-column slabs (two accumulators each) whose partial norms are exchanged through
    // global memory, or -- gx 0, and rows beyond 2048 columns -- into 512-column slabs inside a cluster
    const bool gx = a.l2norm && gx_pref && a.N > 512 && a.N <= 2048;
    const int slab_max = a.l2norm ? (gx ? 256 : 512) : 256;
    p.n_slabs = (a.N + slab_max - 1) / slab_max;
    p.NS = p.n_slabs == 1 ? round_up(a.N, 16) : round_up((a.N + p.n_slabs - 1) / p.n_slabs, 64);
    p.n_slabs = (a.N + p.NS - 1) / p.NS;
    const int units_per_cluster = (a.l2norm && p.n_slabs > 1 && !gx) ? p.n_slabs : 1;
    p.cluster = cg * units_per_cluster;
    p.gx = (gx && p.n_slabs > 1) ? (gx_pref == 2 ? 2 : 1) : 0;
    if (p.cluster > MAX_CLUSTER) return no("row norm spans more CTAs than a portable cluster holds");
    p.nchunks = (p.NS + 255) / 256;
    p.CN = round_up((p.NS + p.nchunks - 1) / p.nchunks, 16);
    p.acc_cols = round_up(p.nchunks * p.CN, 64);
    p.nacc = p.acc_cols <= 256 ? 2 : 1;
    int cols = p.nacc * p.acc_cols;
    p.tmem_cols = 32;
    while (p.tmem_cols < cols) p.tmem_cols *= 2;
    p.b_kb_bytes = p.nchunks * (p.CN / cg) * 128;
    p.stage_bytes = A_BYTES + p.b_kb_bytes;
    // Eight epilogue warps (two per row quarter, half of the columns each) halve the two-pass row-norm
    // epilogue, which is exposed when the accumulator is single-buffered (measured: S3 +3 % at config 3,
    // +8 % at config 4; the one-pass epilogues lose more from the 32 KB of extra staging than they
    // gain, and with double-buffered accumulators the epilogue is hidden anyway).  Used for row-norm
    // GEMMs with a single accumulator when at least three operand stages still fit, and for the
    // selection epilogue (ALU work per score, not stores).
    int fixed = 0;
    const bool want8 = (a.sel_state && p.NS > 64) || (a.l2norm && p.nacc != 2);
    for (p.epi_halves = want8 ? 2 : 1; p.epi_halves >= 1; --p.epi_halves) {
        p.stg_bytes = a.sel_state ? p.epi_halves * 4 * (SEL_Q * 32 * 8) : p.epi_halves * 4 * 2 * STG_WARP_BYTES;
        fixed = p.stg_bytes + BIAS_BYTES + BAR_BYTES + (p.epi_halves == 2 ? HALF_BYTES : 0) +
                (units_per_cluster > 1 ? XCHG_BYTES : 0);
        p.stages = (SMEM_LIMIT - fixed) / p.stage_bytes;
        if (p.stages > MAX_STAGES) p.stages = MAX_STAGES;
        if (p.stages >= 3 || p.epi_halves == 1) break;
    }
    if (p.stages < 2) return no("tile does not fit shared memory");
    // Stationary B: a persistent unit keeps its slab of B for all of its row tiles, so when the CTA's
    // share of the slab (all K blocks) fits beside an A ring of at least four stages it is loaded once
    // and only A streams -- half of the L2 -> shared memory traffic of a 256 x 256 tile (short K: S1 / S4 /
    // S5 at K <= 512).  Not with the tile-major schedule (a unit's slab changes) or the selection epilogue.
    {
        const int kbt = p.kb1 + p.kb2 + p.kb3;
        const long long bres = (long long)kbt * p.b_kb_bytes;
        const long long room = (long long)SMEM_LIMIT - fixed - bres;
        const bool tile_major = !a.l2norm && !a.bias && p.n_slabs > TUNED_SMS / cg && p.m_blocks > 1 &&
                                (long long)(TUNED_SMS / cg) * p.NS * (a.K1 + a.K2 + a.K3) * 2 > (48LL << 20);
        // Measured on B200 (profiles/r02_gemm_bres.md): +4 % on the HBM-bound single-CTA shapes (K = 256,
        // N = 256: config 2 / 5's S1, S4, S5); with CTA pairs at K = 512 the four A stages that are left do
        // not cover the HBM latency of a tensor-bound tile stream (config 4 S1 -8 %, S3 at K = 512 -4 %).
        if (bres_pref && cg == 1 && !a.l2norm && !a.sel_state && !tile_major && room >= 4 * A_BYTES &&
            p.m_blocks * p.n_slabs > TUNED_SMS) {
            p.bres_bytes = (int)bres;
            p.stage_bytes = A_BYTES;
            p.stages = (int)std::min<long long>(room / A_BYTES, MAX_STAGES);
        }
    }
    p.c_split = round_up((p.NS + 1) / 2, 64);
    smem_bytes = p.bres_bytes + p.stages * p.stage_bytes + fixed;
    p.bias = a.bias;
    p.addend = static_cast<const uint4 *>(a.addend);
    p.out_f32 = a.out_f32;
    p.sel_state = a.sel_state;
    p.sel_cnt = a.sel_cnt;
    p.sel_k = a.sel_k;
    p.sel_nb = (int)(a.b_rows ? a.b_rows : a.N);
    p.sel_id0 = a.sel_id0;
    // slabs in flight (one per resident unit) against half of L2; only without per-slab state (bias,
    // row-norm exchange), i.e. the top-K lookup's products
    p.tile_major = !a.l2norm && !a.bias && p.n_slabs > TUNED_SMS / cg && p.m_blocks > 1 &&
                   (long long)(TUNED_SMS / cg) * p.NS * (a.K1 + a.K2 + a.K3) * 2 > (48LL << 20);
    p.relu = a.relu;
    p.l2norm = a.l2norm;
    // instruction descriptor, kind::f16: D fp32 (bit 4), A and B bf16 (bits 7, 10), both K-major,
    // N >> 3 at bits [17,23), M >> 4 at bits [24,29); M = 256 for a CTA pair
    p.idesc = (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(p.CN >> 3) << 17) |
              ((uint32_t)((BM * cg) >> 4) << 24);
    return true;
}

// The plan launch_gemm_tc will use: CTA pairs when the shape allows and the caller does not forbid it.
bool plan_auto(const GemmArgs &a, const GemmTune &t, TcParams &p, int &smem_bytes, const char **why)
{
    // Pairs pay when the GEMM is tensor-bound (measured on B200: +12-14 % at config 3's shapes); on
    // the HBM-bound shapes (arithmetic intensity K N / (K + N) below ~160 flop per byte moved, e.g.
    // 256 x 256) single-CTA tiles keep more independent tiles in flight and are 15-35 % faster.
    const long long Kt = a.K1 + a.K2 + a.K3;
    const bool tensor_bound = Kt * a.N >= 160 * (Kt + a.N);
    if ((t.cg == 2 || (t.cg == 0 && tensor_bound)) && plan(a, 2, t.gx, t.bres, p, smem_bytes, nullptr)) return true;
    if (t.cg == 2) {
        if (why) *why = "shape not supported by the CTA-pair kernel";
        return false;
    }
    return plan(a, 1, t.gx, t.bres, p, smem_bytes, why);
}

template <int CG, int NCH>
cudaError_t launch_cg(GemmTcState *st, const TcParams &p, int smem, cudaStream_t s, const CUtensorMap &tmA1,
                      const CUtensorMap &tmA2, const CUtensorMap &tmA3, const CUtensorMap &tmB,
                      const CUtensorMap &tmOut)
{
    if (!st->attr_set[CG - 1][NCH - 1]) {
        cudaError_t e = cudaFuncSetAttribute(gemm_tc_kernel<CG, NCH>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             SMEM_LIMIT);
        if (e != cudaSuccess) return e;
        st->attr_set[CG - 1][NCH - 1] = true;
    }
    cudaLaunchConfig_t cfg{};
    cfg.blockDim = dim3(NUM_THREADS);
    cfg.dynamicSmemBytes = (size_t)smem;
    cfg.stream = s;
    cudaLaunchAttribute attr[2];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)p.cluster;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    // grid-wide norm exchange: the CTAs wait on each other, so the whole grid must be co-resident --
    // a cooperative launch makes that a guarantee (it does not start until every CTA has an SM).
    // gx == 2 asks for a plain launch (profilers that cannot replay a cooperative one): co-residency then
    // rests on the persistent grid having the device to itself, and a wait that outlasts ~2 s traps.
    attr[1].id = cudaLaunchAttributeCooperative;
    attr[1].val.cooperative = 1;
    cfg.attrs = attr;
    cfg.numAttrs = p.gx == 1 ? 2 : 1;

    // co-resident clusters of this shape (cached: the query costs a driver call)
    int max_clusters = st->clusters[CG - 1][NCH - 1][p.cluster];
    if (max_clusters == 0) {
        cfg.gridDim = dim3((unsigned)(st->num_sms / p.cluster * p.cluster));
        cfg.dynamicSmemBytes = SMEM_LIMIT;
        if (cudaOccupancyMaxActiveClusters(&max_clusters, gemm_tc_kernel<CG, NCH>, &cfg) != cudaSuccess ||
            max_clusters < 1) {
            cudaGetLastError();
            max_clusters = st->num_sms / p.cluster;
        }
        st->clusters[CG - 1][NCH - 1][p.cluster] = max_clusters;
        cfg.dynamicSmemBytes = (size_t)smem;
    }
    const int units_per_cluster = p.cluster / CG;
    const long long tiles = p.m_blocks * p.n_slabs;
    long long units = (long long)max_clusters * units_per_cluster;
    if (units > tiles) units = tiles;
    units = units / p.n_slabs * p.n_slabs;
    if (units < p.n_slabs) units = p.n_slabs;
    if (p.gx && units * CG > st->num_sms) return cudaErrorLaunchOutOfResources;   // (never: one CTA per SM)
    if (p.tile_major) units = tiles;
    cfg.gridDim = dim3((unsigned)(units * CG));
    return cudaLaunchKernelEx(&cfg, gemm_tc_kernel<CG, NCH>, tmA1, tmA2, tmA3, tmB, tmOut, p);
}

}  // namespace

const ::CUtensorMap_st *gemm_tc_map(GemmTcState *st, const void *ptr, long long rows, int cols, int box_rows, int ld,
                                  bool f32)
{
    return st ? get_map(st, ptr, rows, cols, box_rows, ld, f32) : nullptr;
}

bool gemm_tc_supported(const GemmArgs &a, const GemmTune &t, const char **why)
{
    TcParams p;
    int smem = 0;
    if (!plan_auto(a, t, p, smem, why)) return false;
    if (!encode_fn()) {
        if (why) *why = "cuTensorMapEncodeTiled is not available from this driver";
        return false;
    }
    return true;
}

cudaError_t launch_gemm_tc(const GemmArgs &a, const GemmTune &t, GemmTcState *st, cudaStream_t s, int *launches)
{
    TcParams p;
    int smem = 0;
    if (!st) return cudaErrorInvalidValue;
    if (!plan_auto(a, t, p, smem, nullptr)) return cudaErrorNotSupported;
    // (maps are copied out of the cache: a later get_map may evict the entry a pointer refers to)
    const CUtensorMap *m = get_map(st, a.A1, a.M, a.K1, BM);
    if (!m) return cudaErrorInvalidValue;
    const CUtensorMap tmA1 = *m;
    CUtensorMap tmA2 = tmA1, tmA3 = tmA1;
    if (a.K2 > 0) {
        if (!(m = get_map(st, a.A2, a.M, a.K2, BM))) return cudaErrorInvalidValue;
        tmA2 = *m;
    }
    if (a.K3 > 0) {
        if (!(m = get_map(st, a.A3, a.M, a.K3, BM))) return cudaErrorInvalidValue;
        tmA3 = *m;
    }
    if (!(m = get_map(st, a.B, a.b_rows > 0 ? a.b_rows : a.N, a.K1 + a.K2 + a.K3, p.CN / p.cg, a.ldb)))
        return cudaErrorInvalidValue;
    const CUtensorMap tmB = *m;
    // (the selection epilogue stores nothing: its output map is never used)
    CUtensorMap tmOut = tmA1;
    if (!a.sel_state) {
        if (!(m = get_map(st, a.out, a.M, a.N, 32, 0, a.out_f32 != 0))) return cudaErrorInvalidValue;
        tmOut = *m;
    }
    if (launches) ++*launches;
    if (p.gx) {
        // exchange buffers of the grid-wide row-norm exchange: one per stream this context has used
        // (launches on different streams may overlap in time); arrival counters are zeroed before
        // every launch, in stream order
        void *mem = nullptr;
        for (const auto &g : st->gx)
            if (g.s == s) mem = g.mem;
        if (!mem) {
            cudaError_t e = cudaMalloc(&mem, st->gx_buf_bytes + st->gx_cnt_bytes);
            if (e != cudaSuccess) return e;
            st->gx.push_back({s, mem});
        }
        p.gx_buf = static_cast<float *>(mem);
        p.gx_cnt = reinterpret_cast<unsigned *>(static_cast<char *>(mem) + st->gx_buf_bytes);
        cudaError_t e = cudaMemsetAsync(p.gx_cnt, 0, st->gx_cnt_bytes, s);
        if (e != cudaSuccess) return e;
    }
    if (p.cg == 2)
        return p.nchunks == 2 ? launch_cg<2, 2>(st, p, smem, s, tmA1, tmA2, tmA3, tmB, tmOut)
                              : launch_cg<2, 1>(st, p, smem, s, tmA1, tmA2, tmA3, tmB, tmOut);
    return p.nchunks == 2 ? launch_cg<1, 2>(st, p, smem, s, tmA1, tmA2, tmA3, tmB, tmOut)
                          : launch_cg<1, 1>(st, p, smem, s, tmA1, tmA2, tmA3, tmB, tmOut);
}

}  // namespace pinsage

// internal.h -- declarations shared by the translation units of libpinsage.so.
// Product code (CUDA path). Shares nothing with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <stddef.h>
#include <stdint.h>

struct CUtensorMap_st;   // (cuda.h's tensor map; only gemm_*.cu include the driver header)

namespace pinsage {

// SM count of the part the size heuristics were tuned on (B200: 148).  Heuristics only -- grids and buffers that
// must match the device are sized from the context's num_sms.
constexpr int TUNED_SMS = 148;


enum class DType : int { BF16 = 0, F32 = 1 };

inline size_t elem_size(DType t) { return t == DType::BF16 ? 2 : 4; }

// out[M x N] = epi(A1[M x K1] * B[:, 0:K1]^T + A2[M x K2] * B[:, K1:K1+K2]^T + bias)
// B is [N x (K1+K2)] row-major ("out x in"), i.e. K-major.  K2 == 0 -> single segment.
// epi: +addend (if non-null) -> +bias (if non-null) -> ReLU (if relu) -> row L2 normalisation (if l2norm) -> round to dtype.
struct GemmArgs {
    int64_t M = 0;
    int32_t K1 = 0, K2 = 0, N = 0;
    const void *A1 = nullptr;
    const void *A2 = nullptr;
    int32_t K3 = 0;                 // tcgen05 kernel only: a third K segment A3 [M x K3] against
    const void *A3 = nullptr;       // B[:, K1+K2 : K1+K2+K3] (the hub term of the hub-split pool)
    const void *B = nullptr;
    int64_t b_rows = 0;             // rows of B that exist (0 = N); rows b_rows .. N-1 read as zero
    int32_t ldb = 0;                // row stride of B in elements; 0 = K1 + K2 (B may be a column
                                    // block of a wider matrix, e.g. W1 / W2 inside W)
    const void *addend = nullptr;   // optional [M x N] (dtype, row stride N) added to the product in
                                    // fp32 before bias / ReLU: the pooled W2-projection of the
                                    // linear-pool schedule
    const float *bias = nullptr;
    int relu = 0;
    int l2norm = 0;
    // top-K selection epilogue (tcgen05 kernel only, see topk.cu): instead of storing the product,
    // every score that beats row q's current k-th key is appended to q's candidate buffer.  Columns are
    // candidates sel_id0 + [0, b_rows).  out is not written.
    unsigned long long *sel_state = nullptr;
    int *sel_cnt = nullptr;
    int32_t sel_k = 0;
    int64_t sel_id0 = 0;
    int out_f32 = 0;                // tcgen05 kernel only: store the result as fp32 (top-K scores; split fp32 mode)
    void *out = nullptr;
};

// ---- gemm_simt.cu: SIMT fp32-FMA GEMM (the F32 mode; also the BF16 reference kernels) ----------
// ztmp: fp32 scratch of M*N floats, required iff l2norm (un-normalised z lives there).
cudaError_t launch_gemm_simt(DType dt, const GemmArgs &a, float *ztmp, cudaStream_t s, int *launches);
size_t gemm_simt_scratch_bytes(const GemmArgs &a);

// ---- gemm_tcgen05.cu: tcgen05 / TMEM / TMA GEMM, bf16 in, fp32 accumulate ----------------------
// Diagnostic knobs (context options "gemm_cg", "gemm_gx"; tests and profiling only).
struct GemmTune {
    int cg = 0;    // 0 = automatic (CTA pairs, cta_group::2, when the GEMM is tensor-bound), 1 = single-CTA
                   // tiles only, 2 = CTA pairs or fail
    int gx = 1;    // row-norm GEMMs wider than 512 columns: 1 = 256-column slabs, the norms exchanged through
                   // global memory between co-resident CTA pairs, cooperative launch; 2 = the same with a
                   // plain launch (Nsight Compute cannot replay a cooperative one; a wait that outlasts
                   // ~2 s traps instead of hanging); 0 = 512-column slabs exchanged inside a cluster
    int bres = 1;  // 1 = keep the CTA's share of B in shared memory when it fits (short K), 0 = always stream it
};
// Per-context state of the launcher: function attributes already set, co-resident cluster counts, the
// exchange buffers of the grid-wide row-norm exchange (one per stream used, sized from the SM count),
// cached tensor maps.  Owned by the pinsage_ctx, freed with it; not thread-safe (neither is a context).
struct GemmTcState;
GemmTcState *gemm_tc_state_create(int num_sms);
void gemm_tc_state_destroy(GemmTcState *st);
// Shapes outside the compiled set: gemm_tc_supported is false / launch returns cudaErrorNotSupported
// (the caller reports PINSAGE_ERR_UNSUPPORTED_SHAPE).
bool gemm_tc_supported(const GemmArgs &a, const GemmTune &t, const char **why);
cudaError_t launch_gemm_tc(const GemmArgs &a, const GemmTune &t, GemmTcState *st, cudaStream_t s, int *launches);
// A (cached) tensor map of the row-major matrix [rows x cols] at ptr (bf16, or fp32 with f32), box =
// box_rows x 128 bytes, SWIZZLE_128B; ld = row stride in elements (0 = cols).  Null when the driver entry
// point is missing or the encoding fails.  The pointer is valid until the next call on this state.
const ::CUtensorMap_st *gemm_tc_map(GemmTcState *st, const void *ptr, long long rows, int cols, int box_rows, int ld,
                                  bool f32);

// ---- gemm_head.cu: S4 -> S5 in one launch, the intermediate a kept in an L2-resident scratch -------------
bool head_tc_supported(int32_t d, int32_t g1, int32_t d_out);
size_t head_tc_scratch_bytes(int32_t g1, int num_sms);
cudaError_t launch_head_tc(GemmTcState *st, int64_t M, int32_t d, int32_t g1, int32_t d_out, const void *H,
                           const void *G1, const float *g, const void *G2, void *out, void *scratch, int num_sms,
                           cudaStream_t s, int *launches, bool pairs = true);
// The same launch with the scratch in a file-scope __device__ array (no allocation anywhere): gemm_head.cu
size_t head_static_scratch_bytes();
cudaError_t launch_head_tc_static(GemmTcState *st, int64_t M, int32_t d, int32_t g1, int32_t d_out, const void *H,
                                  const void *G1, const float *g, const void *G2, void *out, int num_sms,
                                  cudaStream_t s, int *launches, bool *too_big);

// ---- split_f32.cu: fp32 operands as K-concatenated bf16 planes (fp32 mode on the tensor cores) ----
// out [rows x 6 (K1 + K2)] bf16 from [S1 | S2] (fp32, row strides ld1 / ld2; all multiples of 4).
// is_b selects the plane order of the B operand, so that A' . B'^T sums the six leading terms.
cudaError_t launch_split3(bool is_b, const float *S1, int32_t K1, int64_t ld1, const float *S2, int32_t K2,
                          int64_t ld2, int64_t rows, void *out, cudaStream_t s, int *launches);

// ---- pool.cu ------------------------------------------------------------------------------------
// slab_bytes: 0 = whole rows (one pass); 32 / 64 / 128 = column-slab passes that keep the gathered
// sub-table L2-resident (ignored when pool_slab_ok is false for the shape).
// mode: 0 importance (weighted sum), 1 element-wise mean, 2 element-wise max (w unused for 1, 2).
cudaError_t launch_pool(DType dt, int mode, int64_t n_dst, int32_t T, int32_t m, const void *P,
                        const int32_t *idx, const float *w, void *out, int slab_bytes, cudaStream_t s,
                        int *launches, int skip_neg = 0, void *hubA = nullptr, int H = 0);
// skip_neg: entries with idx < 0 are not gathered; hubA (rows of >= 272 bytes only): such an entry
// -(r + 1) adds its weight to A[v, r] instead, A [n_dst x H] bf16 (the hub-split pool, hubs.cu)
bool pool_hub_fused_ok(DType dt, int32_t m);
bool pool_slab_ok(DType dt, int32_t T, int32_t m, int slab_bytes);
cudaError_t launch_normalize_counts(int64_t N, int32_t T, const int32_t *counts, float *w,
                                    cudaStream_t s, int *launches);
// first_bad: device int64, set to the smallest offending flat position or -1
cudaError_t launch_validate(int64_t n_dst, int64_t n_src, int32_t T, const int32_t *idx,
                            const float *w, long long *first_bad, cudaStream_t s, int *launches);

// ---- calib.cu: calibration kernels of the roofline report (not on the product path) ---------------
cudaError_t launch_calib(int kind, const void *buf, size_t bytes, int row_bytes, long long n_src, long long n_dst,
                         int T, void *out, int num_sms, cudaStream_t s, int *launches);

// ---- hubs.cu: the hub part of the pool on skewed graphs as a GEMM (see the file header) ----------
cudaError_t launch_hub_select(const int32_t *idx, int64_t N, int32_t T, int64_t n_src, int32_t H,
                              int32_t *counts, int32_t *rank, void *cand, int32_t *hub_ids, long long *info,
                              int64_t *sampled, cudaStream_t s, int *launches);
size_t hub_cand_bytes();
cudaError_t launch_hub_remap(const int32_t *idx, const int32_t *rank, int64_t total, int32_t *out,
                             cudaStream_t s, int *launches);
cudaError_t launch_hub_remap_sub(const int32_t *list, int64_t n, const int32_t *idx, int32_t T, const int32_t *rank,
                                 int32_t *idx_loc, cudaStream_t s, int *launches);
cudaError_t launch_hub_localize(const int32_t *hub_ids, int32_t H, const unsigned char *mark, const int32_t *pos,
                                int32_t *hub_loc, cudaStream_t s, int *launches);
cudaError_t launch_hub_matrix(const int32_t *idxm, const float *w, int64_t rows, int32_t T, int32_t H,
                              int mean, void *A, cudaStream_t s, int *launches);
cudaError_t launch_hub_gather(const void *P, const int32_t *hub_ids, int32_t H, int32_t pw, void *Ph,
                              cudaStream_t s, int *launches);
cudaError_t launch_hub_weights(const void *W, int32_t kw, const float *G, int32_t H, int32_t d, void *Wext,
                               cudaStream_t s, int *launches);

// ---- walks.cu: importance-based neighbourhoods by simulated random walks ------------------------
// walk_slots: shared-memory key slots per node (0 = n_walks * walk_len outside [1, 2048]).
int walk_slots(int32_t n_walks, int32_t walk_len);
cudaError_t launch_walk_neighbourhoods(int64_t N, const int64_t *row_ptr, const int32_t *col_idx,
                                       int32_t n_walks, int32_t walk_len, int32_t T, uint64_t seed,
                                       int32_t *nbr_idx, int32_t *counts, cudaStream_t s, int *launches);

// ---- subset.cu: K-hop sets of a minibatch and re-indexed sub-tables (Algorithm 2 l.1-7) ----------
long long subset_blocks(int64_t N);
cudaError_t subset_mark_targets(const int32_t *targets, int64_t M, int64_t N, unsigned char *mark,
                                long long *first_bad, cudaStream_t s, int *launches);
cudaError_t subset_expand(const int32_t *list, int64_t n, const int32_t *idx, int32_t T,
                          unsigned char *mark_prev, cudaStream_t s, int *launches);
cudaError_t subset_compact(const unsigned char *mark, int64_t N, long long *counts, int32_t *list,
                           int32_t *pos, bool scatter, cudaStream_t s, int *launches);
cudaError_t subset_gather_rows(const void *src, const int32_t *ids, const int32_t *map, int64_t n,
                               size_t row_bytes, void *dst, cudaStream_t s, int *launches);
cudaError_t subset_remap_tables(const int32_t *list, int64_t n, const int32_t *idx, const float *w,
                                int32_t T, const int32_t *pos_prev, int32_t *idx_loc, float *w_loc,
                                cudaStream_t s, int *launches);

// ---- keys of the top-K lookup (shared by topk.cu and the selection epilogue of the tcgen05 GEMM) ----
//     key = orderable(score) << 32 | (0xFFFFFFFF - id)        (larger key = better: score desc, id asc)
// Per-query state: TK_TOTAL keys -- the running list (sorted descending at its last merge) in [0, k),
// zeros up to TK_LIST, the candidate buffer in [TK_LIST, TK_LIST + cnt[q]).
constexpr int TK_LIST = 1024;              // k <= TK_LIST
constexpr int TK_TOTAL = 2 * TK_LIST;      // running list + candidate buffer
#ifdef __CUDACC__
__device__ __forceinline__ unsigned ord_f32(float x)       // order-preserving map fp32 -> uint32
{
    const unsigned u = __float_as_uint(x);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float unord_f32(unsigned o)
{
    return __uint_as_float((o & 0x80000000u) ? (o & 0x7fffffffu) : ~o);
}
__device__ __forceinline__ unsigned long long make_key(float score, long long id)
{
    return ((unsigned long long)ord_f32(score) << 32) | (unsigned long long)(0xFFFFFFFFu - (unsigned)id);
}
#endif

// ---- topk.cu: running top-k lists for the exact nearest-neighbour lookup ---------------------------
size_t topk_state_bytes(int64_t nq);   // per-query running lists + buffers; zero it before the first block
// only: optional byte mask [nq]; queries with only[q] == 0 are skipped (the redo of overflowed blocks)
cudaError_t launch_topk_merge(const float *scores, int64_t nq, int64_t ld, int32_t nb, int64_t id0,
                              int32_t k, void *state, const unsigned char *only, cudaStream_t s,
                              int *launches);
// After a block of candidates went through the selection epilogue: per query, if its buffer
// overflowed (cnt > TK_LIST) the block's entries are dropped (cnt restored from cnt_prev), ovf[q] = 1
// and *any = 1 -- the caller redoes that block for those queries from stored scores; otherwise
// ovf[q] = 0 and a buffer at least merge_at full is merged into the list (new k-th key).
// cnt_prev [nq] ints (device), equal to the counters before the block; updated for the next block.
cudaError_t launch_topk_maintain(void *state, int64_t nq, int32_t k, int32_t merge_at, int *cnt_prev,
                                 unsigned char *ovf, int *any, cudaStream_t s, int *launches);
cudaError_t launch_topk_finish(const void *state, int64_t nq, int32_t k, int32_t *idx, float *score,
                               cudaStream_t s, int *launches);

}  // namespace pinsage

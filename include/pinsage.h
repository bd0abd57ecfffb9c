/*
 * pinsage.h -- C-ABI of the B200-native (sm_100a) PinSage layer-wise inference library.
 *
 * The path (citations are /root/reference/PAPER.md = arXiv 1806.01973, line:section):
 *
 *   for k = 1..K over ALL N nodes                       (stacking, :126; Alg. 2 l.8-14 :155-164)
 *     S1  P   = ReLU(H_{k-1} Q^T + q)      once per node    (Alg. 1 l.1 dense part :114; sec. 3.4 job 1 :218)
 *     S2  n_v = sum_t nbr_w[v,t] P[nbr_idx[v,t]]            (Alg. 1 l.1 gamma :114, importance pooling :124;
 *                                                            sec. 3.4 job 2 :219)
 *     S3  z_v = ReLU(W [H_{k-1,v} ; n_v] + w)               (Alg. 1 l.2 :115, self first)
 *         H_k[v] = z_v / ||z_v||_2   (zero row stays zero)  (Alg. 1 l.3 :116)
 *   S4  a   = ReLU(H_K G1^T + g)                            (Alg. 2 l.16 :166)
 *   S5  out = a G2^T                                        (same line; no bias / activation / norm after G2)
 *
 * Conventions
 *   - Plain C99. No exceptions cross the boundary; every call returns a pinsage_status and
 *     leaves a message retrievable with pinsage_last_error().  There is NO CPU fallback:
 *     a non-sm_100 device gives PINSAGE_ERR_ARCH.
 *   - Matrices are row-major.  Parameter matrices are in the paper's orientation, "out x in":
 *     Q [m x d_in] applied as Q h (:114), W [d x (d_in+m)] (:115), G1 [g1 x d], G2 [d_out x g1] (:166).
 *   - dtype selects storage of features, weights, intermediates and outputs:
 *     PINSAGE_BF16 (bf16 storage, tcgen05 tensor-core GEMMs, fp32 accumulate, one RNE rounding at each
 *     of P, n, H_k, a, out) or PINSAGE_F32 (fp32 storage, IEEE fp32 FMA arithmetic).  Biases and
 *     neighbour weights are always fp32, neighbour ids int32.
 *   - Pointers are DEVICE pointers unless a parameter is documented "host or device".
 *     All pointers must be 16-byte aligned; every feature dimension must be a multiple of 8.
 *   - The caller owns every buffer passed in.  The library never frees or keeps caller pointers
 *     beyond the stream-ordered completion of the call.  Compute calls are asynchronous on the
 *     context's stream unless documented otherwise.
 *   - 0 <= nbr_idx < N is a precondition of the hot path (checked only by pinsage_validate_graph
 *     or when the context option "check_indices" is 1).  Self references and repeated ids are
 *     legal; a short neighbourhood is padded with any valid id and weight 0.
 *   - nbr_w is used as given (weighted SUM).  The paper's weighted mean = rows that sum to 1,
 *     e.g. produced by pinsage_normalize_counts.
 *   - Identical inputs give bit-identical outputs run to run (no floating-point atomics, fixed summation
 *     order).  pinsage_embed_all, pinsage_layer + pinsage_head, and pinsage_embed_nodes give the same bits
 *     for the same node, whatever the chunking and wherever the buffers live.
 *   - A context is not thread-safe: calls on one context must be serialised by the caller; different
 *     contexts (one per device or stream) may be used from different threads.
 */
#ifndef PINSAGE_H_
#define PINSAGE_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    PINSAGE_OK = 0,
    PINSAGE_ERR_INVALID_ARG = 1,       /* null pointer, non-positive size, inconsistent dims, bad overlap */
    PINSAGE_ERR_UNSUPPORTED_SHAPE = 2, /* a dimension outside what the kernels are built for */
    PINSAGE_ERR_MISALIGNED = 3,        /* pointer not 16-byte aligned */
    PINSAGE_ERR_BAD_INDEX = 4,         /* nbr_idx outside [0, N) found by validation */
    PINSAGE_ERR_OOM = 5,               /* workspace allocation failed / caller workspace too small */
    PINSAGE_ERR_CUDA = 6,              /* CUDA runtime / driver error, text in pinsage_last_error */
    PINSAGE_ERR_ARCH = 7               /* device is not compute capability 10.x */
} pinsage_status;

typedef enum { PINSAGE_BF16 = 0, PINSAGE_F32 = 1 } pinsage_dtype;

typedef struct pinsage_ctx pinsage_ctx; /* opaque */

/* One CONVOLVE layer's parameters.  Device pointers. */
typedef struct {
    int32_t d_in, m, d; /* Q:[m x d_in]  W:[d x (d_in+m)] */
    const void *Q;      /* dtype */
    const float *q;     /* [m] fp32 */
    const void *W;      /* dtype */
    const float *w;     /* [d] fp32 */
} pinsage_layer_params;

/* Head parameters G1, g, G2.  Device pointers. */
typedef struct {
    int32_t d, g1, d_out; /* G1:[g1 x d]  G2:[d_out x g1] */
    const void *G1;       /* dtype */
    const float *g;       /* [g1] fp32 */
    const void *G2;       /* dtype */
} pinsage_head_params;

/* ---- context ------------------------------------------------------------------------------ */

/* Creates a context on `device`.  `cuda_stream` (a cudaStream_t, may be NULL = the legacy default
 * stream) is borrowed: all work is enqueued there.  Fails with PINSAGE_ERR_ARCH unless the device is
 * compute capability 10.x.  *out is NULL on failure. */
pinsage_status pinsage_create(pinsage_ctx **out, int device, void *cuda_stream);

/* Synchronises the context's stream and releases everything the context owns. NULL is a no-op. */
void pinsage_destroy(pinsage_ctx *ctx);

/* Context-owned, NUL-terminated message of the last failing call ("" if none). With ctx == NULL
 * returns the message of the last failed pinsage_create on this thread. */
const char *pinsage_last_error(const pinsage_ctx *ctx);

/* Static version string, e.g. "pinsage-b200 0.1.0 (sm_100a)". */
const char *pinsage_version(void);

/* Integer options (key, value).  Unknown key or value out of range -> PINSAGE_ERR_INVALID_ARG.
 *
 *   "gemm_impl"      0 = tcgen05 tensor-core GEMMs (default), 1 = SIMT reference kernels
 *   "f32_split"      PINSAGE_F32 GEMMs on the tensor cores: both operands split into three bf16 planes
 *                    (x = x0 + x1 + x2 exactly), the six products with i + j <= 2 summed by one tcgen05 GEMM
 *                    over a six times longer K (fp32 accumulate, error ~1e-6 relative; 5-7 x the SIMT
 *                    kernel): -1 = when rows x N x K >= 2^28 and the shape is covered (default; "rows" are
 *                    those of the whole call -- N nodes -- not of a chunk or of a sub-graph, so every
 *                    chunking and pinsage_embed_nodes make the same choice), 0 = never (SIMT fp32 FMA
 *                    kernels), 1 = always; a GEMM the split path does not cover (K % 4 != 0, the
 *                    linear-pool addend) is then PINSAGE_ERR_UNSUPPORTED_SHAPE.  Ignored when gemm_impl = 1.
 *   "check_indices"  1 = every pinsage_pool / layer / embed_all / embed_nodes call validates nbr_idx
 *                    first (synchronous), default 0
 *   "overlap"        1 = pinsage_layer / embed_all run S2 of chunk c+1 and S3 of chunk c on two streams
 *                    (default 0: measured no faster on B200, the pool's CTAs fill the device first)
 *   "mem_limit_mb"   bytes (in MiB) of device memory pinsage_embed_all may plan with for its workspace and
 *                    staging; 0 (default) = what cudaMemGetInfo reports free at the call, less a margin.
 *                    The plan keeps P and one H resident (none when a device `out` as wide as every layer
 *                    can serve as H), stages host inputs whole when that fits and streams them through
 *                    rings of chunk slots otherwise, and halves the chunk (down to 16384 rows) before it
 *                    gives up with PINSAGE_ERR_OOM.
 *   "pool_mode"      the aggregator gamma of Alg. 1 l.1 used by pinsage_pool / layer / embed_all /
 *                    embed_nodes: 0 = importance pooling, the weighted sum (default); 1 = element-wise
 *                    mean, 2 = element-wise max of the T projected neighbour rows (the paper's ablation
 *                    variants; nbr_w is not read, but must still be a valid pointer)
 *   "linear_pool"    pinsage_layer / embed_all / embed_nodes schedule: pool the W2-projection P W2^T
 *                    (width d) and add it to H W1^T in the S3 epilogue, instead of pooling P (width m) --
 *                    the same function in real arithmetic, m / d times fewer gathered bytes: -1 = when
 *                    m > d (default), 0 never, 1 always.  Not used with pool_mode 2 (max is not linear).
 *   "pool_hubs"      skewed graphs (BF16, importance pooling, m <= d schedule): the entries of the neighbour
 *                    lists that point at the H most listed nodes ("hubs", found from a sample of the lists)
 *                    are not gathered; their term  A (P_hub W2^T),  A[u, h] = the summed weight of u's
 *                    entries naming hub h (summed in table order), enters S3 as a third K segment on the
 *                    tensor cores (A and P_hub W2^T rounded to bf16, exact products, fp32 sum).  The same
 *                    function in real arithmetic and the same error level as the plain pool (which rounds
 *                    all of n to bf16), but a different rounding.  0 = off, H = 64 .. 512 (multiple of 64)
 *                    = on, -1 = on (H = 256) when the sampled hubs hold at least a third of all entries
 *                    (one stream synchronisation per call).  Power-law config: 1.45 x faster.
 *   "topk_fused"     pinsage_topk: 1 (default) = once every running list is full, scores are tested against
 *                    the query's k-th score in the GEMM's epilogue and only the keepers leave the SM (no
 *                    fp32 score matrix in HBM); 0 = every block of scores is stored and scanned by a
 *                    second kernel.  Same result.
 *   "profile"        1 = bracket every kernel launch of the path with CUDA events on its stream, see
 *                    pinsage_profile_read (default 0)
 *
 * Diagnostic keys (tests and profiling; not part of the stable interface, results are unchanged):
 *   "debug_poison"   1 = pinsage_embed_all fills every buffer with NaN patterns the moment the plan says it
 *                    is dead (P after a layer's last pool, the pooled and head chunks after their consumer,
 *                    a replaced H, ring slots): a read that the aliasing rules forbid shows in the output
 *   "gemm_cg"        tcgen05 tile owner: 0 = automatic (CTA pairs, cta_group::2, 256-row tiles, when the
 *                    GEMM is tensor-bound), 1 = single CTAs only, 2 = CTA pairs or UNSUPPORTED_SHAPE
 *   "gemm_gx"        row norms of S3 wider than 512 columns: 1 (default) = exchanged through global memory
 *                    between the co-resident CTA pairs of a cooperative launch; 2 = the same with a plain
 *                    launch (Nsight Compute cannot replay a cooperative one; a wait longer than ~2 s traps);
 *                    0 = exchanged inside a thread-block cluster (512-column slabs)
 *   "head_fused"     1 (default) = the head runs as one launch where the shape allows (BF16, g1 and d_out
 *                    <= 256: the intermediate a = ReLU(h G1^T + g) stays in an L2-resident scratch and never
 *                    reaches HBM; CTA pairs that keep the weights in shared memory for the whole launch where
 *                    those fit, else single CTAs that stream them), 2 = the single-CTA form only, 0 = always S4
 *                    and S5 as two GEMM launches.  Same bits in every form.
 *   "gemm_bres"      1 (default) = a GEMM with short K keeps each CTA's share of its weight slab in shared
 *                    memory for the whole launch and streams only the activations; 0 = always stream both
 *   "pool_slab"      column-slab width in bytes of the S2 pool: -1 automatic (default: 128-byte slabs when
 *                    P exceeds L2 but n_src x 128 bytes fits in 0.7 of it), 0 = whole rows, 32 / 64 / 128 */
pinsage_status pinsage_set_option(pinsage_ctx *ctx, const char *key, int64_t value);

/* Number of kernels this context has launched so far (for launch accounting in benchmarks). */
int64_t pinsage_launch_count(const pinsage_ctx *ctx);

/* Context-owned description of the memory plan the last pinsage_embed_all call chose, e.g.
 * "chunk=1048576 chunks=48 H=out feats=staged tables=ring out=ring workspace=... staging=... hubs=off"
 * (hubs=H when the hub-split pool was taken; "" before the first call).  Valid until the next pinsage_embed_all on this context. */
const char *pinsage_last_plan(const pinsage_ctx *ctx);

/* Per-kernel device time gathered while option "profile" is 1.  Synchronises the context's streams,
 * then sums the event-measured duration of every launch of `kind` (in layer `layer`, 1-based; 0 = all
 * layers; the head carries the last layer's number) since the last reset into *total_ms and their number
 * into *launches (HOST pointers).  kind: 0 = S2 pool (with the hub preparation of "pool_hubs"), 1 = S1
 * (also pinsage_dense and the score GEMMs of pinsage_topk), 2 = S3, 3 = S4, 4 = S5, 5 = the P W2^T
 * projection of the linear-pool schedule, -1 = reset the records (outputs are then 0). */
pinsage_status pinsage_profile_read(pinsage_ctx *ctx, int32_t kind, int32_t layer, double *total_ms,
                                    int64_t *launches);

/* ---- the steps of the path, one call each ------------------------------------------------- */

/* S1 / S4 / S5: out[M x n_out] = act(A[M x k] * Wt[n_out x k]^T + bias).
 * bias may be NULL (S5).  relu: 0/1.  A, Wt, out: dtype.  PAPER.md:114, :166. */
pinsage_status pinsage_dense(pinsage_ctx *ctx, pinsage_dtype dtype, int64_t M, int32_t k,
                             int32_t n_out, const void *A, const void *Wt, const float *bias,
                             int32_t relu, void *out);

/* S2: n[v] = sum_{t<T} nbr_w[v,t] * P[nbr_idx[v,t], :] for v in [0, n_dst), fp32 accumulation in the
 * order t = 0..T-1.  P:[n_src x m] dtype (randomly accessed); nbr_idx/nbr_w:[n_dst x T];
 * n:[n_dst x m] dtype.  1 <= T <= 1024.  PAPER.md:114, :124, :219. */
pinsage_status pinsage_pool(pinsage_ctx *ctx, pinsage_dtype dtype, int64_t n_dst, int64_t n_src,
                            int32_t T, int32_t m, const void *P, const int32_t *nbr_idx,
                            const float *nbr_w, void *n);

/* S3: out[v] = normalise(ReLU(W [H[v] ; n[v]] + w)), W:[d x (d_in+m)] read as two K-segments
 * (no concat is materialised).  H:[M x d_in], n:[M x m], out:[M x d], all dtype.
 * out == H is allowed iff d == d_in (in-place layer k >= 2).  PAPER.md:115-116.
 * H == NULL with d_in == 0 drops the self segment (W:[d x m]): a destination type without a
 * representation of its own, as the boards of the paper's bipartite pin-board graph (:216-221);
 * with pinsage_dense and pinsage_pool (n_dst != n_src) this composes the alternating layers. */
pinsage_status pinsage_combine(pinsage_ctx *ctx, pinsage_dtype dtype, int64_t M, int32_t d_in,
                               int32_t m, int32_t d, const void *H, const void *n, const void *W,
                               const float *w, void *out);

/* ---- the entry points BASELINE.json names ------------------------------------------------- */

/* One CONVOLVE layer over all N nodes: S1 -> S2 -> S3.  feats:[N x d_in], out:[N x d].
 * Workspace (P [N x m] + one chunk of n) is ctx-owned when ws == NULL, else the caller's
 * (ws_bytes >= pinsage_layer_workspace_bytes, 256-byte aligned; too small -> PINSAGE_ERR_OOM).
 * out == feats is allowed iff d == d_in.  Alg. 1; schedule sec. 3.4 :214-221. */
pinsage_status pinsage_layer(pinsage_ctx *ctx, pinsage_dtype dtype, int64_t N, int32_t T,
                             const void *feats, const int32_t *nbr_idx, const float *nbr_w,
                             const pinsage_layer_params *params, void *out, void *ws,
                             size_t ws_bytes);

size_t pinsage_layer_workspace_bytes(pinsage_dtype dtype, int64_t N, int32_t T,
                                     const pinsage_layer_params *params);

/* Head: S4 -> S5 in node chunks.  h:[N x d] -> out:[N x d_out].  Alg. 2 l.16. */
pinsage_status pinsage_head(pinsage_ctx *ctx, pinsage_dtype dtype, int64_t N, const void *h,
                            const pinsage_head_params *params, void *out);

/* The head for callers that must not allocate (CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): the same one-launch S4 -> S5 kernel as pinsage_head's default form, same bits, with its scratch
 * (the a = ReLU(h G1^T + g) tiles in flight) in a file-scope __device__ array of 29 097 984 bytes (148 SMs x 3
 * tiles x 128 rows x 256 bf16 values) that every GPU loading the library holds until the process exits.  The
 * call itself makes no cudaMalloc / cudaFree and creates no events; the first call on a device resolves the
 * array's address (cudaGetSymbolAddress) and sets a function attribute -- make it once before capturing.
 * Limits: PINSAGE_BF16 only, g1 <= 256, d_out <= 256, N < 2^31, and g1 x SMs within the array (any g1 <= 256 on
 * a 148-SM part); anything else -> PINSAGE_ERR_UNSUPPORTED_SHAPE, nothing launched.  All device pointers.
 * The array is shared by every call in the process and keeps the last call's contents (nothing needs to start
 * at zero: a tile is always written before it is read).  Calls that overlap on the GPU -- two streams, two
 * contexts -- race on it: serialise them.  The "profile" option records nothing here.  PAPER.md:166. */
pinsage_status pinsage_head_static(pinsage_ctx *ctx, pinsage_dtype dtype, int64_t N, const void *h,
                                   const pinsage_head_params *params, void *out);

/* K layers + head over all N nodes with the chunked layer driver (Alg. 2 l.8-17 with S^(k) = V).
 * feats:[N x layers[0].d_in], nbr_idx / nbr_w:[N x T], out:[N x head->d_out] may each be DEVICE or
 * HOST pointers (detected with cudaPointerGetAttributes; host buffers should be pinned for speed):
 * host inputs are copied to device staging owned by the context and a host `out` is filled by a
 * device-to-host copy, all inside this call.  `layers` (array of K structs) and `head` are host
 * structs holding device pointers.  chunk_nodes = destination rows per S2/S3 chunk (0 = automatic).
 * If any buffer is a host pointer the call synchronises the stream before returning; with device
 * buffers only it is asynchronous. */
pinsage_status pinsage_embed_all(pinsage_ctx *ctx, pinsage_dtype dtype, int64_t N, int32_t T,
                                 int32_t K, const void *feats, const int32_t *nbr_idx,
                                 const float *nbr_w, const pinsage_layer_params *layers,
                                 const pinsage_head_params *head, void *out, int64_t chunk_nodes);

/* Targeted / incremental inference = Algorithm 2 on a minibatch: embeds only the M
 * nodes listed in `targets` (device int32 [M], ids in [0, N), repeats allowed) by building their K-hop
 * sets S^(K) = targets, S^(k-1) = S^(k) U N(S^(k)) (l.1-7), re-indexing the sub-tables (:182) and running
 * the same S1-S5 kernels on the closure only.  All pointers are DEVICE pointers; feats / nbr_idx / nbr_w
 * describe the whole graph as in pinsage_embed_all; out:[M x head->d_out], row j = embedding of
 * targets[j], bit-identical to row targets[j] of pinsage_embed_all.  The call synchronises the stream
 * K + 1 times (set sizes are read back); scratch is context-owned.  A target outside [0, N) gives
 * PINSAGE_ERR_BAD_INDEX. */
pinsage_status pinsage_embed_nodes(pinsage_ctx *ctx, pinsage_dtype dtype, int64_t N, int32_t T,
                                   int32_t K, const void *feats, const int32_t *nbr_idx,
                                   const float *nbr_w, const pinsage_layer_params *layers,
                                   const pinsage_head_params *head, int64_t M, const int32_t *targets,
                                   void *out);

/* Exact K-nearest-neighbour lookup in the embedding space (PAPER.md:225 sec. 3.5; :289: top K = 500
 * neighbours of a query among 5 million candidates) -- the exact form of what the paper serves
 * approximately with LSH.  "Nearest" = largest inner product z_q . z_i, the score the loss ranks by
 * (Eq. 1); ties go to the smaller id; the query is not excluded.  Q:[nq x d], Z:[N x d] dtype (device);
 * out_idx:[nq x k] int32, out_score:[nq x k] fp32 (device), each row ordered by (score descending, id
 * ascending).  Scores are fp32 accumulations of the exact bf16 / fp32 products (tcgen05 GEMM in BF16
 * mode; the split tcgen05 GEMM or the SIMT kernel in F32 mode, option "f32_split"), compared as IEEE
 * values.  1 <= k <= min(N, 1024).  With N beyond one candidate block (up to 65 536) and option
 * "topk_fused" on, the call synchronises the context's stream once before it returns (it reads back
 * which blocks, if any, overflowed a candidate buffer and must be redone); otherwise asynchronous. */
pinsage_status pinsage_topk(pinsage_ctx *ctx, pinsage_dtype dtype, int64_t nq, int64_t N, int32_t d,
                            const void *Q, const void *Z, int32_t k, int32_t *out_idx, float *out_score);

/* ---- helpers ------------------------------------------------------------------------------ */

/* nbr_w[v,t] = (float)counts[v,t] / (float)(sum_t counts[v,t]) in IEEE binary32 (L1-normalised visit
 * counts).  counts:[N x T] int32 >= 0 with a positive row sum. */
pinsage_status pinsage_normalize_counts(pinsage_ctx *ctx, int64_t N, int32_t T,
                                        const int32_t *counts, float *nbr_w);

/* Importance-based neighbourhoods: for every node u simulate n_walks random walks
 * that start at u and take walk_len steps to a uniformly chosen out-neighbour (a node without
 * out-neighbours ends the walk), count the arrivals at every node v != u, and keep the T most visited
 * nodes (ties to the smaller id) in that order; a node with fewer than T distinct visited nodes is
 * padded with (id u, count 0).  The graph is a CSR adjacency: row_ptr [N+1] int64 (row_ptr[0] = 0,
 * non-decreasing), col_idx [row_ptr[N]] int32 in [0, N) -- device pointers, as are the outputs
 * nbr_idx / counts [N x T] int32.  Draws are a counter-based function of (seed, u, walk, step), so the
 * result does not depend on scheduling (readings B1-B5).  counts feeds
 * pinsage_normalize_counts.  1 <= n_walks * walk_len <= 2048 (else PINSAGE_ERR_UNSUPPORTED_SHAPE). */
pinsage_status pinsage_build_neighbourhoods(pinsage_ctx *ctx, int64_t N, const int64_t *row_ptr,
                                            const int32_t *col_idx, int32_t n_walks, int32_t walk_len,
                                            int32_t T, uint64_t seed, int32_t *nbr_idx, int32_t *counts);

/* Synchronous.  Checks 0 <= nbr_idx[i] < n_src for all n_dst*T entries and that every weight is
 * finite.  *first_bad (HOST pointer) receives the flat position of the first offender or -1;
 * returns PINSAGE_ERR_BAD_INDEX if there is one. */
pinsage_status pinsage_validate_graph(pinsage_ctx *ctx, int64_t n_dst, int64_t n_src, int32_t T,
                                      const int32_t *nbr_idx, const float *nbr_w,
                                      int64_t *first_bad);

/* Measurement aid, not a step of the path ("how to report the pool honestly"): what
 * this device delivers to the access patterns of the S2 pool, so that the pool can be
 * reported against physical ceilings of the day instead of a copy rate.
 *   kind 0 (m1): read-only streaming reduction over table_bytes bytes of `table`; `out` needs
 *                num_sms x 8 x 256 x 16 bytes (303 104 x 16 on a 148-SM part).
 *   kind 1 (m2 / m3): un-weighted random-row gather: for each of n_dst destinations, T rows of row_bytes
 *                (256, 512, 1024 or 2048) bytes at hashed positions of `table` (table_bytes / row_bytes rows)
 *                are XOR-summed into out [n_dst x row_bytes].  A table far larger than L2 gives the random-row
 *                ceiling from HBM (m2), a table that fits L2 the L2 / LSU ceiling (m3).
 * Device pointers, 16-byte aligned.  Synchronous: one warm-up launch, then `reps` launches between two CUDA
 * events on the context's stream; *ms (HOST pointer) = average milliseconds per launch. */
pinsage_status pinsage_calibrate(pinsage_ctx *ctx, int32_t kind, const void *table, size_t table_bytes,
                                 int32_t row_bytes, int64_t n_dst, int32_t T, void *out, size_t out_bytes,
                                 int32_t reps, double *ms);

#ifdef __cplusplus
}
#endif
#endif /* PINSAGE_H_ */

// api.cu -- the C-ABI of include/pinsage.h: context, argument checking, the layer driver (S6).
// Every step of the path runs in this library's own kernels (pool.cu, gemm_tcgen05.cu,
// gemm_simt.cu); there is no CPU or vendor-library fallback.
#include "../../include/pinsage.h"
#include "internal.h"

#include <algorithm>
#include <functional>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include <nvtx3/nvToolsExt.h>   // header-only; ranges cost a pointer test when no tool is attached

using namespace pinsage;

struct pinsage_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    cudaStream_t aux = nullptr;      // second stream for S2 / S3 overlap
    cudaStream_t h2d = nullptr;      // copy streams of the host-buffer pipeline (pinsage_embed_all)
    cudaStream_t d2h = nullptr;
    std::vector<cudaEvent_t> pipe_events;   // per-chunk "input landed" / "output ready" events
    cudaEvent_t ev_pool[2] = {nullptr, nullptr};
    cudaEvent_t ev_gemm[2] = {nullptr, nullptr};
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
    int num_sms = 0;
    int gemm_impl = 0;               // 0 tcgen05, 1 SIMT reference
    GemmTune tune;                   // tcgen05 diagnostic knobs ("gemm_cg", "gemm_gx")
    GemmTcState *tc = nullptr;       // launcher state: function attributes, exchange buffers, tensor maps
    int cur_layer = 0;               // 1-based layer of the running call (NVTX range names only)
    int64_t m_hint = 0;              // rows the GEMMs of the running call would have on the whole graph
                                     // (pinsage_embed_nodes: same kernel choice as pinsage_embed_all)
    int check_indices = 0;
    int overlap = 0;
    int poison = 0;                  // debug: buffers are filled with NaN patterns the moment they are dead
    int64_t mem_limit = 0;           // bytes the context may own for one call (0 = what the device has free)
    int pool_mode = 0;               // aggregator gamma: 0 importance, 1 mean, 2 max
    int linear_pool = -1;            // pool the W2-projection (width d) instead of P (width m):
                                     // -1 automatic (when m > d), 0 never, 1 always
    int pool_slab = -1;              // -1 automatic, 0 off, 32 / 64 / 128 forced slab width in bytes
    size_t l2_bytes = 0;
    int launches = 0;
    int64_t total_launches = 0;
    void *ws = nullptr;              // context-owned workspace
    size_t ws_bytes = 0;
    void *stage = nullptr;           // device staging for host inputs / outputs
    size_t stage_bytes = 0;
    long long *d_first_bad = nullptr;
    int pool_hubs = -1;              // hub-split pool (hubs.cu): 0 off, -1 automatic (default), H = 64..512 forced
    struct HubState {                // valid during one pinsage_embed_all call
        int H = 0;
        const int32_t *src_idx = nullptr;   // the caller's table the remapped one stands for
        const int32_t *idxm = nullptr;      // remapped table: hub entries are -(rank + 1)
        const int32_t *hub_ids = nullptr;
        void *A = nullptr;                  // [chunk x H] bf16
        void *Ph = nullptr;                 // [H x m] bf16: the hub rows of P
        float *G = nullptr;                 // [H x d] fp32: P_hub W2^T
        void *Wext = nullptr;               // [d x (d_in + m + H)] bf16: [W1 | W2 | G^T]
    } hub;
    void *hub_buf = nullptr, *hub_tab = nullptr;   // selection scratch; remapped table + per-layer matrices
    size_t hub_bytes = 0, hub_tab_bytes = 0;
    void *hub_sample = nullptr;      // sampled rows of a host table
    size_t hub_sample_bytes = 0;
    long long *hub_info_h = nullptr; // pinned: {hubs found, sampled entries they hold}
    cudaEvent_t ev_hub = nullptr;
    int topk_fused = 1;              // pinsage_topk: select in the GEMM epilogue (1) or in a second pass over stored scores (0)
    int f32_split = -1;              // fp32 GEMMs on the tensor cores by bf16 splitting: -1 automatic, 0 never, 1 always
    void *split_buf = nullptr;       // bf16 planes of the operands of a split fp32 GEMM (grown on demand)
    size_t split_bytes = 0;
    int head_fused = 1;              // S4 -> S5 in one launch where the shape allows (gemm_head.cu); 2 = its single-CTA form only
    void *head_scratch = nullptr;    // its L2-resident scratch for the a tiles
    size_t head_scratch_bytes = 0;
    void *subA = nullptr, *subB = nullptr;   // scratch of pinsage_embed_nodes (sets / compact tensors)
    size_t subA_bytes = 0, subB_bytes = 0;
    // optional per-kernel timing ("profile" option): event pairs around every launch
    int profile = 0;
    std::vector<cudaEvent_t> prof_events;
    struct ProfRec { int kind, layer; int e0, e1; };
    std::vector<ProfRec> prof_recs;
    size_t prof_used = 0;
    std::string err;
    std::string plan;                // description of the last pinsage_embed_all memory plan
};

namespace {

thread_local std::string g_create_err;

pinsage_status fail(pinsage_ctx *ctx, pinsage_status st, const char *fmt, ...)
{
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    if (ctx)
        ctx->err = buf;
    else
        g_create_err = buf;
    return st;
}

#define PS_CUDA(ctx, expr)                                                                   \
    do {                                                                                     \
        cudaError_t e_ = (expr);                                                             \
        if (e_ != cudaSuccess)                                                               \
            return fail(ctx, e_ == cudaErrorMemoryAllocation ? PINSAGE_ERR_OOM               \
                                                             : PINSAGE_ERR_CUDA,             \
                        "%s: %s", #expr, cudaGetErrorString(e_));                            \
    } while (0)

#define PS_TRY(expr)                          \
    do {                                      \
        pinsage_status st_ = (expr);          \
        if (st_ != PINSAGE_OK) return st_;    \
    } while (0)

struct DeviceGuard {
    int prev = -1;
    explicit DeviceGuard(int dev)
    {
        cudaGetDevice(&prev);
        if (prev != dev) cudaSetDevice(dev);
        else prev = -1;
    }
    ~DeviceGuard()
    {
        if (prev >= 0) cudaSetDevice(prev);
    }
};

// NVTX range "S<step> <what>" around the launches of one step: makes an nsys / ncu
// capture self-describing.  No tool attached: nvtxRangePush is a null-pointer test.
struct StepRange {
    StepRange(const char *fmt, ...)
    {
        char buf[96];
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(buf, sizeof buf, fmt, ap);
        va_end(ap);
        nvtxRangePushA(buf);
    }
    ~StepRange() { nvtxRangePop(); }
};

// Kernel choices that depend on the problem size (the fp32 GEMM: split tensor-core path or SIMT) are
// taken from the rows of the CALL, not of the chunk or sub-graph a launch happens to cover, so that
// every chunking and pinsage_embed_nodes (hint = the whole graph's N) give the same bits.
struct HintGuard {
    pinsage_ctx *c;
    int64_t prev;
    HintGuard(pinsage_ctx *ctx, int64_t rows);
    ~HintGuard();
};

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

HintGuard::HintGuard(pinsage_ctx *ctx, int64_t rows) : c(ctx), prev(ctx->m_hint) { ctx->m_hint = std::max(prev, rows); }
HintGuard::~HintGuard() { c->m_hint = prev; }

bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

pinsage_status check_dtype(pinsage_ctx *ctx, pinsage_dtype dt)
{
    if (dt != PINSAGE_BF16 && dt != PINSAGE_F32)
        return fail(ctx, PINSAGE_ERR_INVALID_ARG, "unknown dtype %d", (int)dt);
    return PINSAGE_OK;
}

pinsage_status check_dim(pinsage_ctx *ctx, const char *name, int64_t v)
{
    if (v <= 0) return fail(ctx, PINSAGE_ERR_INVALID_ARG, "%s = %lld must be positive", name, (long long)v);
    if (v % 8 != 0)
        return fail(ctx, PINSAGE_ERR_UNSUPPORTED_SHAPE, "%s = %lld must be a multiple of 8", name,
                    (long long)v);
    if (v > 8192)
        return fail(ctx, PINSAGE_ERR_UNSUPPORTED_SHAPE, "%s = %lld exceeds 8192", name, (long long)v);
    return PINSAGE_OK;
}

pinsage_status check_ptr(pinsage_ctx *ctx, const char *name, const void *p)
{
    if (!p) return fail(ctx, PINSAGE_ERR_INVALID_ARG, "%s is NULL", name);
    if (!aligned16(p)) return fail(ctx, PINSAGE_ERR_MISALIGNED, "%s is not 16-byte aligned", name);
    return PINSAGE_OK;
}

bool overlaps(const void *a, size_t na, const void *b, size_t nb)
{
    const char *pa = static_cast<const char *>(a), *pb = static_cast<const char *>(b);
    return pa < pb + nb && pb < pa + na;
}

pinsage_status ensure_ws(pinsage_ctx *ctx, size_t bytes)
{
    if (bytes <= ctx->ws_bytes) return PINSAGE_OK;
    if (ctx->ws) {
        PS_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
        PS_CUDA(ctx, cudaStreamSynchronize(ctx->aux));
        cudaFree(ctx->ws);
        ctx->ws = nullptr;
        ctx->ws_bytes = 0;
    }
    cudaError_t e = cudaMalloc(&ctx->ws, bytes);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return fail(ctx, PINSAGE_ERR_OOM, "workspace of %zu bytes: %s", bytes, cudaGetErrorString(e));
    }
    ctx->ws_bytes = bytes;
    return PINSAGE_OK;
}

pinsage_status ensure_stage(pinsage_ctx *ctx, size_t bytes)
{
    if (bytes <= ctx->stage_bytes) return PINSAGE_OK;
    if (ctx->stage) {
        PS_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
        cudaFree(ctx->stage);
        ctx->stage = nullptr;
        ctx->stage_bytes = 0;
    }
    cudaError_t e = cudaMalloc(&ctx->stage, bytes);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return fail(ctx, PINSAGE_ERR_OOM, "staging of %zu bytes: %s", bytes, cudaGetErrorString(e));
    }
    ctx->stage_bytes = bytes;
    return PINSAGE_OK;
}

// Column-slab width for the pool (pool.cu): slabs pay off when P does not fit L2 but a 128-byte
// column slab of it does.  Measured on B200: a slab sub-table of up to ~64 MB
// is gathered at 14.8 TB/s (whole rows from HBM: 8-9.5 TB/s), the gain fades by ~90 MB, and slabs
// narrower than the 128-byte L2 line never win (L2 allocates whole lines, requests double).
int pick_slab(const pinsage_ctx *ctx, DType dt, int64_t n_src, int32_t T, int32_t m)
{
    if (ctx->pool_slab == 0) return 0;
    if (ctx->pool_slab > 0) return pool_slab_ok(dt, T, m, ctx->pool_slab) ? ctx->pool_slab : 0;
    const size_t row = (size_t)m * elem_size(dt);
    if ((size_t)n_src * row <= ctx->l2_bytes / 2) return 0;      // whole table is L2-resident anyway
    if (pool_slab_ok(dt, T, m, 128) && (size_t)n_src * 128 <= ctx->l2_bytes / 10 * 7) return 128;
    return 0;
}

pinsage_status ensure_buf(pinsage_ctx *ctx, void **buf, size_t *cap, size_t bytes, const char *what)
{
    if (bytes <= *cap) return PINSAGE_OK;
    if (*buf) {
        PS_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
        cudaFree(*buf);
        *buf = nullptr;
        *cap = 0;
    }
    cudaError_t e = cudaMalloc(buf, bytes);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return fail(ctx, PINSAGE_ERR_OOM, "%s of %zu bytes: %s", what, bytes, cudaGetErrorString(e));
    }
    *cap = bytes;
    return PINSAGE_OK;
}

// kinds of pinsage_profile_read: the steps of the path; PROF_DENSE also takes pinsage_dense and the score
// GEMMs of pinsage_topk, PROF_AUX the P W2^T projection of the linear-pool schedule
enum ProfKind { PROF_POOL = 0, PROF_DENSE = 1, PROF_COMBINE = 2, PROF_HEAD1 = 3, PROF_HEAD2 = 4, PROF_AUX = 5,
                PROF_KINDS = 6 };

// Records an event on stream s (profile mode only) and returns its slot, or -1.
int prof_mark(pinsage_ctx *ctx, cudaStream_t s)
{
    if (!ctx->profile) return -1;
    if (ctx->prof_used == ctx->prof_events.size()) {
        cudaEvent_t e;
        if (cudaEventCreate(&e) != cudaSuccess) return -1;
        ctx->prof_events.push_back(e);
    }
    const int slot = (int)ctx->prof_used++;
    cudaEventRecord(ctx->prof_events[slot], s);
    return slot;
}

void prof_close(pinsage_ctx *ctx, int kind, int e0, cudaStream_t s)
{
    if (e0 < 0) return;
    const int e1 = prof_mark(ctx, s);
    if (e1 >= 0) ctx->prof_recs.push_back({kind, ctx->cur_layer, e0, e1});
}

void count_launches(pinsage_ctx *ctx)
{
    ctx->total_launches += ctx->launches;
    ctx->launches = 0;
}

// The fp32 GEMM on the tensor cores (split_f32.cu): both operands as K-concatenated bf16 planes in a
// context-owned buffer, A in row blocks so that the buffer stays bounded, one tcgen05 GEMM with fp32
// output per block.  *done = false when the shape is outside what the split path covers (the caller
// falls back to the SIMT kernel).
constexpr size_t SPLIT_A_BYTES = 256u << 20;    // planes of one row block of A

// Whether the split path takes this GEMM; fills the bf16 GEMM of one row block (pointers unset).
bool split_covers(const pinsage_ctx *ctx, const GemmArgs &a, cudaStream_t s, GemmArgs &g, int64_t &blk)
{
    const int kt = a.K1 + a.K2;
    const int ldb = a.ldb ? a.ldb : kt;
    if (a.addend || a.K1 % 4 || a.K2 % 4 || ldb % 4 || !aligned16(a.A1) || !aligned16(a.B) ||
        (a.K2 && !aligned16(a.A2)) || (long long)kt * 6 > 0x7fffffffLL || s != ctx->stream)
        return false;
    const size_t row_bytes = (size_t)kt * 6 * 2;
    blk = (int64_t)(SPLIT_A_BYTES / row_bytes) / 256 * 256;
    blk = std::min<int64_t>(std::max<int64_t>(blk, 256), a.M);
    if (a.sel_state && blk < a.M) return false;                 // (the selection epilogue numbers rows from 0)
    g = GemmArgs{};
    g.M = blk;
    g.K1 = kt * 6;
    g.N = a.N;
    g.b_rows = a.b_rows ? a.b_rows : a.N;
    g.bias = a.bias;
    g.relu = a.relu;
    g.l2norm = a.l2norm;
    g.out_f32 = 1;
    g.sel_state = a.sel_state;
    g.sel_cnt = a.sel_cnt;
    g.sel_k = a.sel_k;
    g.sel_id0 = a.sel_id0;
    g.A1 = g.B = g.out = reinterpret_cast<void *>(16);          // (shape check only)
    GemmArgs tail = g;
    tail.M = a.M % blk ? a.M % blk : blk;
    return gemm_tc_supported(g, ctx->tune, nullptr) && gemm_tc_supported(tail, ctx->tune, nullptr);
}

bool split_wanted(const pinsage_ctx *ctx, DType dt, const GemmArgs &a)
{
    return dt == DType::F32 && ctx->gemm_impl == 0 &&
           (ctx->f32_split == 1 ||
            (ctx->f32_split == -1 &&
             (double)std::max<int64_t>(a.M, ctx->m_hint) * a.N * (a.K1 + a.K2) >= (double)(1 << 28)));
}

pinsage_status run_gemm_split(pinsage_ctx *ctx, const GemmArgs &a, cudaStream_t s, int kind, bool *done)
{
    *done = false;
    GemmArgs g;
    int64_t blk = 0;
    if (!split_covers(ctx, a, s, g, blk)) return PINSAGE_OK;
    const int kt = a.K1 + a.K2;
    const int ldb = a.ldb ? a.ldb : kt;
    const int64_t b_rows = g.b_rows;
    const size_t row_bytes = (size_t)kt * 6 * 2;
    const size_t b_bytes = align_up((size_t)b_rows * row_bytes, 256);
    const size_t need = b_bytes + (size_t)blk * row_bytes;
    if (need > ctx->split_bytes) {
        PS_CUDA(ctx, cudaStreamSynchronize(s));
        if (ctx->split_buf) cudaFree(ctx->split_buf);
        ctx->split_buf = nullptr;
        ctx->split_bytes = 0;
        PS_CUDA(ctx, cudaMalloc(&ctx->split_buf, need));
        ctx->split_bytes = need;
    }
    char *Bp = static_cast<char *>(ctx->split_buf), *Ap = Bp + b_bytes;
    const int e0 = prof_mark(ctx, s);
    cudaError_t e = launch_split3(true, static_cast<const float *>(a.B), kt, ldb, nullptr, 0, 0, b_rows, Bp, s,
                                  &ctx->launches);
    for (int64_t r0 = 0; r0 < a.M && e == cudaSuccess; r0 += blk) {
        const int64_t rows = std::min<int64_t>(blk, a.M - r0);
        e = launch_split3(false, static_cast<const float *>(a.A1) + r0 * a.K1, a.K1, a.K1,
                          a.K2 ? static_cast<const float *>(a.A2) + r0 * a.K2 : nullptr, a.K2, a.K2, rows, Ap, s,
                          &ctx->launches);
        if (e != cudaSuccess) break;
        g.M = rows;
        g.A1 = Ap;
        g.B = Bp;
        g.out = static_cast<float *>(a.out) + r0 * a.N;
        e = launch_gemm_tc(g, ctx->tune, ctx->tc, s, &ctx->launches);
    }
    prof_close(ctx, kind, e0, s);
    count_launches(ctx);
    PS_CUDA(ctx, e);
    *done = true;
    return PINSAGE_OK;
}

// One GEMM of the path on stream s. scratch: fp32 [M x N] for the SIMT norm pass / tcgen05 partials.
pinsage_status run_gemm(pinsage_ctx *ctx, DType dt, const GemmArgs &a, void *scratch,
                        size_t scratch_bytes, cudaStream_t s, int prof_kind = -1)
{
    if (a.M == 0) return PINSAGE_OK;
    const bool simt = dt == DType::F32 || ctx->gemm_impl == 1;
    const int kind = prof_kind >= 0 ? prof_kind : a.l2norm ? PROF_COMBINE : PROF_DENSE;
    if (split_wanted(ctx, dt, a)) {
        bool done = false;
        PS_TRY(run_gemm_split(ctx, a, s, kind, &done));
        if (done) return PINSAGE_OK;
        if (ctx->f32_split == 1)
            return fail(ctx, PINSAGE_ERR_UNSUPPORTED_SHAPE,
                        "f32_split = 1: shape outside the split fp32 GEMM (M=%lld K1=%d K2=%d N=%d)",
                        (long long)a.M, a.K1, a.K2, a.N);
    }
    if (simt) {
        if (a.sel_state || a.K3)
            return fail(ctx, PINSAGE_ERR_CUDA, "internal: selection epilogue / third K segment on the SIMT path");
        const size_t need = gemm_simt_scratch_bytes(a);
        if (need > scratch_bytes)
            return fail(ctx, PINSAGE_ERR_OOM, "internal: SIMT scratch %zu > %zu", need, scratch_bytes);
        const int e0 = prof_mark(ctx, s);
        cudaError_t e = launch_gemm_simt(dt, a, static_cast<float *>(scratch), s, &ctx->launches);
        prof_close(ctx, kind, e0, s);
        count_launches(ctx);
        PS_CUDA(ctx, e);
        return PINSAGE_OK;
    }
    const char *why = nullptr;
    if (!gemm_tc_supported(a, ctx->tune, &why))
        return fail(ctx, PINSAGE_ERR_UNSUPPORTED_SHAPE, "tcgen05 GEMM: %s (M=%lld K1=%d K2=%d N=%d)",
                    why ? why : "unsupported shape", (long long)a.M, a.K1, a.K2, a.N);
    const int e0 = prof_mark(ctx, s);
    cudaError_t e = launch_gemm_tc(a, ctx->tune, ctx->tc, s, &ctx->launches);
    prof_close(ctx, kind, e0, s);
    count_launches(ctx);
    PS_CUDA(ctx, e);
    return PINSAGE_OK;
}

// The head of `rows` rows: out = ReLU(h G1^T + g) G2^T.  One launch with the intermediate
// kept in an L2-resident scratch where the fused kernel covers the shape (BF16 on the tcgen05 path, g1 and
// d_out <= 256), else S4 into `abuf` [rows x g1] and S5 from it: the same bits either way.
pinsage_status run_head(pinsage_ctx *ctx, DType dt, int64_t rows, const void *h, const pinsage_head_params *head,
                        void *abuf, void *out, cudaStream_t s)
{
    if (rows == 0) return PINSAGE_OK;
    if (ctx->head_fused && dt == DType::BF16 && ctx->gemm_impl == 0 && head_tc_supported(head->d, head->g1, head->d_out)) {
        PS_TRY(ensure_buf(ctx, &ctx->head_scratch, &ctx->head_scratch_bytes, head_tc_scratch_bytes(256, ctx->num_sms),
                          "head scratch"));
        const int e0 = prof_mark(ctx, s);
        cudaError_t e = launch_head_tc(ctx->tc, rows, head->d, head->g1, head->d_out, h, head->G1, head->g, head->G2, out,
                                       ctx->head_scratch, ctx->num_sms, s, &ctx->launches, ctx->head_fused != 2);
        prof_close(ctx, PROF_HEAD1, e0, s);
        count_launches(ctx);
        PS_CUDA(ctx, e);
        return PINSAGE_OK;
    }
    GemmArgs g;
    g.M = rows; g.K1 = head->d; g.N = head->g1; g.A1 = h;
    g.B = head->G1; g.bias = head->g; g.relu = 1; g.out = abuf;
    PS_TRY(run_gemm(ctx, dt, g, nullptr, 0, s, PROF_HEAD1));
    GemmArgs g2;
    g2.M = rows; g2.K1 = head->g1; g2.N = head->d_out; g2.A1 = abuf; g2.B = head->G2; g2.out = out;
    PS_TRY(run_gemm(ctx, dt, g2, nullptr, 0, s, PROF_HEAD2));
    if (ctx->poison) PS_CUDA(ctx, cudaMemsetAsync(abuf, 0xFF, (size_t)rows * head->g1 * elem_size(dt), s));
    return PINSAGE_OK;
}

size_t gemm_scratch_bytes(const pinsage_ctx *ctx, DType dt, const GemmArgs &a)
{
    const bool simt = dt == DType::F32 || (ctx && ctx->gemm_impl == 1);
    return simt ? align_up(gemm_simt_scratch_bytes(a), 256) : 0;   // (the tcgen05 kernel needs none)
}

pinsage_status check_layer_params(pinsage_ctx *ctx, const pinsage_layer_params *p, const char *what)
{
    if (!p) return fail(ctx, PINSAGE_ERR_INVALID_ARG, "%s is NULL", what);
    PS_TRY(check_dim(ctx, "d_in", p->d_in));
    PS_TRY(check_dim(ctx, "m", p->m));
    PS_TRY(check_dim(ctx, "d", p->d));
    PS_TRY(check_ptr(ctx, "Q", p->Q));
    PS_TRY(check_ptr(ctx, "q", p->q));
    PS_TRY(check_ptr(ctx, "W", p->W));
    PS_TRY(check_ptr(ctx, "w", p->w));
    return PINSAGE_OK;
}

pinsage_status check_head_params(pinsage_ctx *ctx, const pinsage_head_params *p)
{
    if (!p) return fail(ctx, PINSAGE_ERR_INVALID_ARG, "head params are NULL");
    PS_TRY(check_dim(ctx, "head.d", p->d));
    PS_TRY(check_dim(ctx, "head.g1", p->g1));
    PS_TRY(check_dim(ctx, "head.d_out", p->d_out));
    PS_TRY(check_ptr(ctx, "G1", p->G1));
    PS_TRY(check_ptr(ctx, "g", p->g));
    PS_TRY(check_ptr(ctx, "G2", p->G2));
    return PINSAGE_OK;
}

pinsage_status check_graph_args(pinsage_ctx *ctx, int64_t N, int32_t T)
{
    if (N < 1 || N >= (1LL << 31))
        return fail(ctx, PINSAGE_ERR_INVALID_ARG, "N = %lld outside [1, 2^31)", (long long)N);
    if (T < 1 || T > 1024) return fail(ctx, PINSAGE_ERR_INVALID_ARG, "T = %d outside [1, 1024]", T);
    return PINSAGE_OK;
}

pinsage_status maybe_validate(pinsage_ctx *ctx, int64_t n_dst, int64_t n_src, int32_t T,
                              const int32_t *idx, const float *w)
{
    if (!ctx->check_indices) return PINSAGE_OK;
    int64_t bad = -1;
    return pinsage_validate_graph(ctx, n_dst, n_src, T, idx, w, &bad);
}

// Destination rows per S2/S3 chunk.  Automatic: as many rows as keep one chunk buffer (rows x
// row_bytes) within 1 GiB, at least 131072 -- measured on B200: few
// large launches beat many small ones (fewer wave tails in the pool, fewer partial waves of
// 128-row tiles in the persistent GEMM), and chunk buffers of this size cost < 1 % of HBM.
int64_t auto_chunk(int64_t N, int64_t requested, size_t row_bytes)
{
    int64_t c = requested > 0
                    ? requested
                    : std::max<int64_t>(131072, (int64_t)((size_t(1) << 30) / std::max<size_t>(row_bytes, 1)));
    c = std::min<int64_t>(c, N);
    if (c < N) c = std::max<int64_t>(128, c / 128 * 128);  // keep chunk starts on GEMM tile edges
    return c;
}

// The linear-pool schedule: W [h ; sum_t a_t p_t] = W1 h + sum_t a_t (W2 p_t), exact in real
// arithmetic because the pool is linear (not so for the element-wise max).  Pooling the projected
// rows P' = P W2^T (width d) instead of P (width m) divides the gathered bytes by m / d -- 2x at the
// paper's own geometry, m = 2048, d = 1024 -- for the same flops.
bool use_linear_pool(const pinsage_ctx *ctx, const pinsage_layer_params *lp)
{
    if (!ctx || ctx->pool_mode == 2 || ctx->linear_pool == 0) return false;
    return ctx->linear_pool == 1 || lp->m > lp->d;
}

// The pool kernels cover rows of at most 256 16-byte chunks (4096 bytes: 2048 bf16 / 1024 fp32 values).
// Checked before anything is enqueued, for the row width the chosen schedule pools.
pinsage_status check_pool_width(pinsage_ctx *ctx, DType dt, const pinsage_layer_params *lp)
{
    const int32_t pw = use_linear_pool(ctx, lp) ? lp->d : lp->m;
    if ((size_t)pw * elem_size(dt) > 4096)
        return fail(ctx, PINSAGE_ERR_UNSUPPORTED_SHAPE,
                    "pooled rows of %d %s values exceed 4096 bytes (m = %d, d = %d)", pw,
                    dt == DType::BF16 ? "bf16" : "fp32", lp->m, lp->d);
    return PINSAGE_OK;
}

// Where the chunk loops of a layer get a chunk's inputs from and what happens around its steps.  Every
// member may be empty: the arrays are then device arrays addressed by row offset.  pinsage_embed_all
// fills them in when inputs arrive from the host (staged whole, or streamed through a ring of chunk
// slots), and to run the head of a chunk right after its last S3.
struct ChunkIO {
    // before / after S1 of source chunk c (layer 1 of a host-feature call): the chunk's rows
    std::function<pinsage_status(int64_t c, const void **src)> s1_in;
    std::function<pinsage_status(int64_t c)> s1_done;
    // before / after S2 of chunk c, on the pool's stream: the chunk's (id, weight) rows -- ids already
    // remapped when hub_remapped (the hub-split pool on tables that came from the host)
    std::function<pinsage_status(int64_t c, cudaStream_t ps, const int32_t **idx, const float **w)> tables_in;
    std::function<pinsage_status(int64_t c, cudaStream_t ps)> tables_done;
    bool hub_remapped = false;
    // before S3 of chunk c: the chunk's own previous representations (the self segment)
    std::function<pinsage_status(int64_t c, const void **self)> self_in;
    // after S3 of chunk c: its self rows are consumed, its output rows exist
    std::function<pinsage_status(int64_t c, int64_t r0, int64_t rows)> after_chunk;
};

// S2 + S3 over all destination rows in chunks; pool of chunk c+1 may overlap combine of chunk c.
// Hin [N x d_in] (read), P [N x pw] (read), Hout [N x d] (written; may alias Hin iff d == d_in).
// pw = m (P = projections, n is the second K segment of S3) or, in the linear-pool schedule, d
// (P = projections times W2^T, n is an addend of S3).  nbuf: two chunk buffers [chunk x pw].
pinsage_status pool_combine_chunks(pinsage_ctx *ctx, DType dt, int64_t N, int32_t T,
                                   const pinsage_layer_params *lp, const void *Hin, const void *P,
                                   const int32_t *idx, const float *w, void *Hout, int64_t chunk,
                                   void *nbuf0, void *nbuf1, void *scratch, size_t scratch_bytes,
                                   int64_t n_src, const ChunkIO &io)
{
    if (n_src < 0) n_src = N;                // rows of P; N = destination rows
    const size_t es = elem_size(dt);
    const bool linear = use_linear_pool(ctx, lp);
    const int32_t pw = linear ? lp->d : lp->m;
    const int64_t nchunks = (N + chunk - 1) / chunk;
    const bool two = ctx->overlap && nchunks > 1;
    void *nb[2] = {nbuf0, two ? nbuf1 : nbuf0};
    if (two) {
        PS_CUDA(ctx, cudaEventRecord(ctx->ev_fork, ctx->stream));
        PS_CUDA(ctx, cudaStreamWaitEvent(ctx->aux, ctx->ev_fork, 0));
    }
    cudaStream_t ps = two ? ctx->aux : ctx->stream;
    // hub-split pool (hubs.cu): the gather skips the hub entries; their term enters S3 as a third K
    // segment A [rows x H] against G = P_hub W2^T, appended to the layer's W once per layer
    const bool hubs = ctx->hub.H > 0 && (io.hub_remapped || idx == ctx->hub.src_idx) && !two && !linear &&
                      dt == DType::BF16 && ctx->pool_mode == 0;
    const int H = ctx->hub.H;
    if (hubs) {
        const int pe0 = prof_mark(ctx, ps);
        cudaError_t e = launch_hub_gather(P, ctx->hub.hub_ids, H, pw, ctx->hub.Ph, ps, &ctx->launches);
        prof_close(ctx, PROF_POOL, pe0, ps);
        count_launches(ctx);
        PS_CUDA(ctx, e);
        GemmArgs gg;                              // G [H x d] = P_hub W2^T in fp32
        gg.M = H;
        gg.K1 = lp->m;
        gg.N = lp->d;
        gg.A1 = ctx->hub.Ph;
        gg.B = static_cast<const char *>(lp->W) + (size_t)lp->d_in * es;
        gg.ldb = lp->d_in + lp->m;
        gg.out_f32 = 1;
        gg.out = ctx->hub.G;
        PS_TRY(run_gemm(ctx, dt, gg, nullptr, 0, ps, PROF_POOL));
        e = launch_hub_weights(lp->W, lp->d_in + lp->m, ctx->hub.G, H, lp->d, ctx->hub.Wext, ps, &ctx->launches);
        count_launches(ctx);
        PS_CUDA(ctx, e);
    }
    for (int64_t c = 0; c < nchunks; ++c) {
        const int64_t r0 = c * chunk, rows = std::min(chunk, N - r0);
        const int b = (int)(c & 1);
        if (two && c >= 2) PS_CUDA(ctx, cudaStreamWaitEvent(ps, ctx->ev_gemm[b], 0));
        const int32_t *ic = hubs && !io.hub_remapped ? ctx->hub.idxm + (size_t)r0 * T : idx + (size_t)r0 * T;
        const float *wc = w + (size_t)r0 * T;
        if (io.tables_in) PS_TRY(io.tables_in(c, ps, &ic, &wc));
        {
            StepRange r2("S2 pool k=%d rows %lld+%lld", ctx->cur_layer, (long long)r0, (long long)rows);
            const int pe0 = prof_mark(ctx, ps);
            cudaError_t e;
            if (hubs) {
                const bool fusedA = pool_hub_fused_ok(dt, pw);     // the gather kernel also writes A
                e = launch_pool(dt, 0, rows, T, pw, P, ic, wc, nb[b], 0, ps, &ctx->launches, 1,
                                fusedA ? ctx->hub.A : nullptr, H);
                if (e == cudaSuccess && !fusedA)
                    e = launch_hub_matrix(ic, wc, rows, T, H, 0, ctx->hub.A, ps, &ctx->launches);
            } else {
                e = launch_pool(dt, ctx->pool_mode, rows, T, pw, P, ic, wc, nb[b], pick_slab(ctx, dt, n_src, T, pw), ps,
                                &ctx->launches);
            }
            prof_close(ctx, PROF_POOL, pe0, ps);
            count_launches(ctx);
            PS_CUDA(ctx, e);
        }
        if (io.tables_done) PS_TRY(io.tables_done(c, ps));
        if (two) {
            PS_CUDA(ctx, cudaEventRecord(ctx->ev_pool[b], ps));
            PS_CUDA(ctx, cudaStreamWaitEvent(ctx->stream, ctx->ev_pool[b], 0));
        }
        const void *self = static_cast<const char *>(Hin) + (size_t)r0 * lp->d_in * es;
        if (io.self_in) PS_TRY(io.self_in(c, &self));
        GemmArgs g;
        g.M = rows;
        g.K1 = lp->d_in;
        g.N = lp->d;
        g.A1 = self;
        g.B = lp->W;
        if (linear) {                        // z = H W1^T + pooled(P W2^T) + w
            g.ldb = lp->d_in + lp->m;
            g.addend = nb[b];
        } else {                             // z = H W1^T + n W2^T + w: two K segments
            g.K2 = lp->m;
            g.A2 = nb[b];
            if (hubs) {                          // ... + A (P_hub W2^T): the hub term as a third one
                g.K3 = H;
                g.A3 = ctx->hub.A;
                g.B = ctx->hub.Wext;
                g.ldb = lp->d_in + lp->m + H;
            }
        }
        g.bias = lp->w;
        g.relu = 1;
        g.l2norm = 1;
        g.out = static_cast<char *>(Hout) + (size_t)r0 * lp->d * es;
        {
            StepRange r3("S3 combine k=%d rows %lld+%lld", ctx->cur_layer, (long long)r0, (long long)rows);
            PS_TRY(run_gemm(ctx, dt, g, scratch, scratch_bytes, ctx->stream));
        }
        if (two) PS_CUDA(ctx, cudaEventRecord(ctx->ev_gemm[b], ctx->stream));
        if (ctx->poison)                     // the pooled chunk is dead once S3 has consumed it
            PS_CUDA(ctx, cudaMemsetAsync(nb[b], 0xFF, (size_t)rows * pw * es, ctx->stream));
        if (io.after_chunk) PS_TRY(io.after_chunk(c, r0, rows));
    }
    if (two) {
        PS_CUDA(ctx, cudaEventRecord(ctx->ev_join, ps));
        PS_CUDA(ctx, cudaStreamWaitEvent(ctx->stream, ctx->ev_join, 0));
    }
    if (ctx->poison)                         // P is dead once the layer's last pool has run
        PS_CUDA(ctx, cudaMemsetAsync(const_cast<void *>(P), 0xFF, (size_t)n_src * pw * es, ctx->stream));
    return PINSAGE_OK;
}

struct LayerWs {
    size_t P_off, Pc_off, n0_off, n1_off, scratch_off, scratch_bytes, total;
};

// Workspace of one layer.  Standard schedule: P [N x m] | n chunk(s) [chunk x m] | scratch.
// Linear-pool schedule: P' [N x d] | projection chunk Pc [chunk x m] | n chunk(s) [chunk x d] | scratch.
LayerWs plan_layer_ws(const pinsage_ctx *ctx, DType dt, int64_t N, const pinsage_layer_params *lp,
                      int64_t chunk)
{
    const size_t es = elem_size(dt);
    const bool linear = use_linear_pool(ctx, lp);
    const int32_t pw = linear ? lp->d : lp->m;
    LayerWs p{};
    size_t off = 0;
    p.P_off = off;
    off += align_up((size_t)N * pw * es, 256);
    p.Pc_off = off;
    if (linear) off += align_up((size_t)chunk * lp->m * es, 256);
    p.n0_off = off;
    off += align_up((size_t)chunk * pw * es, 256);
    p.n1_off = p.n0_off;                       // second chunk buffer only for the two-stream schedule
    if (ctx && ctx->overlap) {
        p.n1_off = off;
        off += align_up((size_t)chunk * pw * es, 256);
    }
    GemmArgs g1;
    g1.M = linear ? chunk : N; g1.K1 = lp->d_in; g1.N = lp->m; g1.relu = 1;
    GemmArgs g3;
    g3.M = chunk; g3.K1 = lp->d_in; g3.K2 = linear ? 0 : lp->m; g3.N = lp->d; g3.relu = 1; g3.l2norm = 1;
    p.scratch_bytes = std::max(gemm_scratch_bytes(ctx, dt, g1), gemm_scratch_bytes(ctx, dt, g3));
    p.scratch_off = off;
    off += p.scratch_bytes;
    p.total = off;
    return p;
}

// S1 of one layer on a planned workspace: P = ReLU(src Q^T + q) over the n_src source rows -- in one
// launch, or chunk by chunk when the features arrive from the host (io.s1_in) or the linear-pool
// schedule projects P W2^T per chunk.
pinsage_status project_chunks(pinsage_ctx *ctx, DType dt, int64_t n_src, const pinsage_layer_params *lp,
                              const void *src_feats, char *ws, const LayerWs &plan, int64_t chunk,
                              const ChunkIO &io)
{
    const size_t es = elem_size(dt);
    const bool linear = use_linear_pool(ctx, lp);
    const int64_t s1_rows = (io.s1_in || linear) ? chunk : n_src;
    for (int64_t r0 = 0, c = 0; r0 < n_src; r0 += s1_rows, ++c) {
        const void *src = static_cast<const char *>(src_feats) + (size_t)r0 * lp->d_in * es;
        if (io.s1_in) PS_TRY(io.s1_in(c, &src));
        GemmArgs g;
        g.M = std::min(s1_rows, n_src - r0);
        g.K1 = lp->d_in;
        g.N = lp->m;
        g.A1 = src;
        g.B = lp->Q;
        g.bias = lp->q;
        g.relu = 1;
        g.out = linear ? ws + plan.Pc_off : ws + plan.P_off + (size_t)r0 * lp->m * es;
        StepRange r1("S1 project k=%d rows %lld+%lld", ctx->cur_layer, (long long)r0, (long long)g.M);
        PS_TRY(run_gemm(ctx, dt, g, ws + plan.scratch_off, plan.scratch_bytes, ctx->stream));
        if (io.s1_done) PS_TRY(io.s1_done(c));
        if (linear) {                          // P'[chunk] = P[chunk] W2^T (W2 = columns d_in.. of W)
            GemmArgs g2;
            g2.M = g.M;
            g2.K1 = lp->m;
            g2.N = lp->d;
            g2.A1 = ws + plan.Pc_off;
            g2.B = static_cast<const char *>(lp->W) + (size_t)lp->d_in * es;
            g2.ldb = lp->d_in + lp->m;
            g2.out = ws + plan.P_off + (size_t)r0 * lp->d * es;
            PS_TRY(run_gemm(ctx, dt, g2, ws + plan.scratch_off, plan.scratch_bytes, ctx->stream, PROF_AUX));
        }
    }
    return PINSAGE_OK;
}

// One layer: S1 over the source rows, then the S2 / S3 chunk loop over the N destination rows.
// n_src / src_feats (targeted inference): the source rows S1 projects differ from the destination rows,
// whose own previous representations are `feats`.
pinsage_status layer_on_ws(pinsage_ctx *ctx, DType dt, int64_t N, int32_t T, const void *feats,
                           const int32_t *idx, const float *w, const pinsage_layer_params *lp,
                           void *out, char *ws, const LayerWs &plan, int64_t chunk, int64_t n_src = -1,
                           const void *src_feats = nullptr, const ChunkIO &io = ChunkIO())
{
    if (n_src < 0) {
        n_src = N;
        src_feats = feats;
    }
    PS_TRY(project_chunks(ctx, dt, n_src, lp, src_feats, ws, plan, chunk, io));
    return pool_combine_chunks(ctx, dt, N, T, lp, feats, ws + plan.P_off, idx, w, out, chunk,
                               ws + plan.n0_off, ws + plan.n1_off, ws + plan.scratch_off,
                               plan.scratch_bytes, n_src, io);
}

// Grows the per-chunk event pool of the host-buffer pipeline to n events.
pinsage_status ensure_pipe_events(pinsage_ctx *ctx, size_t n)
{
    while (ctx->pipe_events.size() < n) {
        cudaEvent_t e;
        PS_CUDA(ctx, cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        ctx->pipe_events.push_back(e);
    }
    return PINSAGE_OK;
}

// ---- host buffers of pinsage_embed_all ---------------------------------------------------------------
// An input [N x row_bytes] that lives in host memory reaches the kernels chunk by chunk through device
// slots: `depth` = number of chunks (the array is staged whole: copied once, valid for the rest of the
// call) or a small ring that every pass over the chunks re-fills.  Copies run on the context's h2d stream;
// `landed[slot]` orders a chunk's consumer behind its copy, `freed[slot]` the next copy into a slot
// behind the slot's last consumer.  (cudaStreamWaitEvent looks at the LAST record of an event, so a
// slot's `freed` is always recorded before the copy that waits for it is enqueued.)
struct HostSrc {
    const char *host = nullptr;
    char *dev = nullptr;
    size_t row_bytes = 0;
    int64_t N = 0, chunk = 0, nchunks = 0;
    int depth = 0;
    bool whole = false, loaded = false;
    cudaEvent_t *landed = nullptr, *freed = nullptr;
    std::vector<char> used;                     // slot has had a consumer whose `freed` was recorded

    bool active() const { return host != nullptr; }
    int slot(int64_t c) const { return (int)(c % depth); }
    char *ptr(int64_t c) const { return dev + (size_t)slot(c) * chunk * row_bytes; }

    pinsage_status copy(pinsage_ctx *ctx, int64_t c)
    {
        const int sl = slot(c);
        const int64_t r0 = c * chunk, rows = std::min(chunk, N - r0);
        if (used[sl]) PS_CUDA(ctx, cudaStreamWaitEvent(ctx->h2d, freed[sl], 0));
        PS_CUDA(ctx, cudaMemcpyAsync(ptr(c), host + (size_t)r0 * row_bytes, (size_t)rows * row_bytes,
                                     cudaMemcpyHostToDevice, ctx->h2d));
        PS_CUDA(ctx, cudaEventRecord(landed[sl], ctx->h2d));
        return PINSAGE_OK;
    }
    // start of a pass over the chunks 0 .. nchunks-1: the first `depth` copies
    pinsage_status begin_pass(pinsage_ctx *ctx)
    {
        if (!active() || loaded) return PINSAGE_OK;
        for (int64_t c = 0; c < std::min<int64_t>(depth, nchunks); ++c) PS_TRY(copy(ctx, c));
        return PINSAGE_OK;
    }
    // consumer side, on stream s: chunk c's rows
    pinsage_status acquire(pinsage_ctx *ctx, int64_t c, cudaStream_t s, const void **p)
    {
        if (!loaded) PS_CUDA(ctx, cudaStreamWaitEvent(s, landed[slot(c)], 0));
        *p = ptr(c);
        return PINSAGE_OK;
    }
    // the consumer of chunk c has been enqueued on s: a ring slot may take chunk c + depth
    pinsage_status release(pinsage_ctx *ctx, int64_t c, cudaStream_t s)
    {
        if (whole) {
            if (c == nchunks - 1) loaded = true;
            return PINSAGE_OK;
        }
        const int sl = slot(c);
        if (ctx->poison) PS_CUDA(ctx, cudaMemsetAsync(ptr(c), 0xFF, (size_t)chunk * row_bytes, s));
        PS_CUDA(ctx, cudaEventRecord(freed[sl], s));
        used[sl] = 1;
        if (c + depth < nchunks) PS_TRY(copy(ctx, c + depth));
        return PINSAGE_OK;
    }
};

// The output [N x row_bytes] of a call whose `out` is host memory: two chunk slots on the device, each
// copied home on the d2h stream while the next chunk is computed into the other.
struct HostSink {
    char *host = nullptr, *dev = nullptr;
    size_t row_bytes = 0;
    int64_t chunk = 0;
    cudaEvent_t ready[2] = {nullptr, nullptr}, copied[2] = {nullptr, nullptr};
    bool used[2] = {false, false};

    bool active() const { return host != nullptr; }
    char *ptr(int64_t c) const { return dev + (size_t)(c & 1) * chunk * row_bytes; }
    pinsage_status acquire(pinsage_ctx *ctx, int64_t c, cudaStream_t s)
    {
        if (used[c & 1]) PS_CUDA(ctx, cudaStreamWaitEvent(s, copied[c & 1], 0));
        return PINSAGE_OK;
    }
    pinsage_status release(pinsage_ctx *ctx, int64_t c, int64_t r0, int64_t rows, cudaStream_t s)
    {
        const int sl = (int)(c & 1);
        PS_CUDA(ctx, cudaEventRecord(ready[sl], s));
        PS_CUDA(ctx, cudaStreamWaitEvent(ctx->d2h, ready[sl], 0));
        PS_CUDA(ctx, cudaMemcpyAsync(host + (size_t)r0 * row_bytes, ptr(c), (size_t)rows * row_bytes,
                                     cudaMemcpyDeviceToHost, ctx->d2h));
        PS_CUDA(ctx, cudaEventRecord(copied[sl], ctx->d2h));
        used[sl] = true;
        return PINSAGE_OK;
    }
};

// ---- memory plan of pinsage_embed_all -------------------------------------------
// Resident by necessity: P (the one randomly accessed array) and one H buffer -- none when the caller's
// device `out` can serve as H (every layer as wide as the output: same row stride, and a chunk's out rows
// are written after its H rows were consumed) -- plus a second H only when layer widths change.
// Everything else is per chunk.  Host inputs are staged whole when that fits (tables first: every layer
// reads them; then the features: layer 1 reads them twice), else streamed through rings of RING chunk
// slots per pass; a host output always leaves through two chunk slots.  When the plan does not fit the
// budget (free device memory, or the "mem_limit_mb" option) the chunk is halved, down to 16384 rows.
constexpr int RING = 3;

struct EmbedPlan {
    int64_t chunk = 0, nchunks = 0;
    bool H_is_out = false, need_Hb = false, feats_whole = false, tabs_whole = false;
    size_t max_layer_ws = 0, H_bytes = 0, a_bytes = 0, ws_total = 0;
    size_t feats_off = 0, idx_off = 0, w_off = 0, out_off = 0, stage_total = 0;
};

pinsage_status plan_embed(pinsage_ctx *ctx, DType dt, int64_t N, int32_t T, int32_t K,
                          const pinsage_layer_params *layers, const pinsage_head_params *head, int64_t chunk_nodes,
                          bool h_feats, bool h_idx, bool h_w, bool h_out, EmbedPlan &pl)
{
    const size_t es = elem_size(dt);
    const bool any_host = h_feats || h_idx || h_w || h_out;
    // what this call may own: the device's free memory plus what the context already holds for it
    size_t free_b = 0, total_b = 0;
    PS_CUDA(ctx, cudaMemGetInfo(&free_b, &total_b));
    size_t budget = free_b + ctx->ws_bytes + ctx->stage_bytes;
    budget -= std::min(budget, std::max<size_t>(budget / 64, (size_t)128 << 20));     // allocator slack
    if (ctx->mem_limit > 0) budget = std::min(budget, (size_t)ctx->mem_limit);
    int32_t w_max = head->g1, d_max = 0;
    pl.H_is_out = !h_out;
    for (int k = 0; k < K; ++k) {
        w_max = std::max(w_max, layers[k].m);
        d_max = std::max(d_max, layers[k].d);
        pl.H_is_out = pl.H_is_out && layers[k].d == head->d_out;
        if (k > 0) pl.need_Hb = pl.need_Hb || layers[k].d != layers[k].d_in;
    }
    pl.H_bytes = align_up((size_t)N * d_max * es, 256);
    int64_t chunk = auto_chunk(N, chunk_nodes, (size_t)w_max * es);
    // host buffers: at least ~8 chunks so that copies and kernels overlap chunk by chunk
    if (any_host && chunk_nodes == 0)
        chunk = std::min<int64_t>(chunk, std::max<int64_t>(32768, ((N + 7) / 8 + 127) / 128 * 128));
    size_t least = 0;
    for (;;) {
        pl.chunk = chunk;
        pl.nchunks = (N + chunk - 1) / chunk;
        pl.max_layer_ws = 0;
        for (int k = 0; k < K; ++k)
            pl.max_layer_ws = std::max(pl.max_layer_ws, plan_layer_ws(ctx, dt, N, &layers[k], chunk).total);
        pl.a_bytes = align_up((size_t)chunk * head->g1 * es, 256);
        pl.ws_total = pl.max_layer_ws + pl.H_bytes * ((pl.H_is_out ? 0 : 1) + (pl.need_Hb ? 1 : 0)) + pl.a_bytes;
        const size_t feats_row = (size_t)layers[0].d_in * es, tab_row = (size_t)T * 4, out_row = (size_t)head->d_out * es;
        auto bytes = [&](bool on, bool whole, size_t row) -> size_t {
            if (!on) return 0;
            return align_up(whole ? (size_t)N * row : (size_t)std::min<int64_t>(RING, pl.nchunks) * chunk * row, 256);
        };
        // whole staging where it fits: the tables first (read by every layer), then the features
        for (int mode = 0; mode < 3; ++mode) {
            pl.tabs_whole = mode < 2;
            pl.feats_whole = mode < 1;
            size_t off = 0;
            pl.feats_off = off; off += bytes(h_feats, pl.feats_whole, feats_row);
            pl.idx_off = off;   off += bytes(h_idx, pl.tabs_whole, tab_row);
            pl.w_off = off;     off += bytes(h_w, pl.tabs_whole, tab_row);
            pl.out_off = off;   off += h_out ? align_up((size_t)2 * chunk * out_row, 256) : 0;
            pl.stage_total = off;
            if (pl.ws_total + pl.stage_total <= budget) return PINSAGE_OK;
            least = pl.ws_total + pl.stage_total;
        }
        if (chunk_nodes > 0) break;                        // the caller fixed the chunk
        const int64_t smaller = std::max<int64_t>(16384, chunk / 2 / 128 * 128);
        if (smaller >= chunk) break;
        chunk = smaller;
    }
    return fail(ctx, PINSAGE_ERR_OOM,
                "embed_all needs at least %zu bytes of device memory (P [N x m] and H [N x d] must be resident; "
                "chunk of %lld rows) but only %zu are available%s",
                least, (long long)chunk, budget, ctx->mem_limit > 0 ? " (option mem_limit_mb)" : "");
}

// The context's workspace and staging allocations at the planned sizes.  When one of them has to grow,
// an oversized other one is released first, so that the pair never holds more than the plan.
pinsage_status fit_buffers(pinsage_ctx *ctx, size_t ws_need, size_t stage_need)
{
    const bool grow = ws_need > ctx->ws_bytes || stage_need > ctx->stage_bytes;
    if (grow) {
        PS_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
        PS_CUDA(ctx, cudaStreamSynchronize(ctx->aux));
        if (ctx->ws && ctx->ws_bytes != ws_need) {
            cudaFree(ctx->ws);
            ctx->ws = nullptr;
            ctx->ws_bytes = 0;
        }
        if (ctx->stage && ctx->stage_bytes != stage_need) {
            cudaFree(ctx->stage);
            ctx->stage = nullptr;
            ctx->stage_bytes = 0;
        }
    }
    PS_TRY(ensure_ws(ctx, ws_need));
    if (stage_need) PS_TRY(ensure_stage(ctx, stage_need));
    return PINSAGE_OK;
}

// ---- hub-split pool: shared by pinsage_layer, pinsage_embed_all and pinsage_embed_nodes, which must
// take the same decision and pick the same hubs for their results to agree bit for bit ------------------
struct HubPlan {                 // layout of ctx->hub_buf for one call
    int H = 0;
    int32_t *counts = nullptr, *rank = nullptr, *hub_ids = nullptr, *hub_loc = nullptr, *idxm = nullptr;
    void *cand = nullptr;
    long long *info = nullptr;
    void *A = nullptr, *Ph = nullptr, *Wext = nullptr;
    float *G = nullptr;
    int64_t sampled = 0;         // entries of the sample
};

struct HubReset {                // the hub state is valid during one call only
    pinsage_ctx *c;
    ~HubReset() { c->hub = pinsage_ctx::HubState{}; }
};

// Whether the hub-split pool can apply to a call at all: the option, BF16 importance pooling on the
// tcgen05 path, one stream, at least one layer on the m <= d schedule, a table of at least 2^22 entries.
// Depends on the whole graph and the options only, never on chunks or on which nodes are embedded.
bool hub_eligible(const pinsage_ctx *ctx, DType dt, int64_t N, int32_t T, int32_t K, const pinsage_layer_params *layers)
{
    if (ctx->pool_hubs == 0 || dt != DType::BF16 || ctx->pool_mode != 0 || ctx->gemm_impl != 0 || ctx->overlap ||
        N * (int64_t)T < (1 << 22))
        return false;
    for (int k = 0; k < K; ++k)
        if (!use_linear_pool(ctx, &layers[k])) return true;
    return false;
}

// Picks the hubs of the whole graph's table for a call that runs `layers`, in two steps so that the one
// read-back of the automatic mode hides behind work enqueued in between (S1 of the first layer):
//   hub_select_begin   histogram of a sample of the lists (every (N / 16384)-th row: `sample` is the
//                      device table itself with sample_n = N, or the gathered sample rows with sample_n =
//                      their number), candidates, the H most listed ids and their ranks; asynchronous
//   hub_select_finish  *use = the split is taken: forced, or -- automatic mode -- the sampled hubs hold a
//                      third of the sampled entries (waits for the selection only, not for the stream);
//                      then the storage of the split: [the remapped whole table,] A, P_hub, G, [W | G^T]
// a_rows: rows of the per-chunk matrix A.  want_table: room for the remapped whole table (device tables).
pinsage_status hub_select_begin(pinsage_ctx *ctx, DType dt, int64_t N, int32_t T, int32_t K,
                                const pinsage_layer_params *layers, const int32_t *sample, int64_t sample_n, HubPlan &hp)
{
    hp = HubPlan{};
    if (!hub_eligible(ctx, dt, N, T, K, layers)) return PINSAGE_OK;
    // automatic: 256 hubs (config 4, step ms with H = 64 / 128 / 192 / 256: 131.7 / 119.6 / 118.4 / 117.4)
    const int H = ctx->pool_hubs > 0 ? ctx->pool_hubs : 256;
    const size_t nB = align_up((size_t)N * 4, 256), candB = align_up(hub_cand_bytes(), 256);
    const size_t idsB = align_up((size_t)H * 4, 256);
    PS_TRY(ensure_buf(ctx, &ctx->hub_buf, &ctx->hub_bytes, 2 * nB + candB + 2 * idsB + 256, "hub selection scratch"));
    if (!ctx->hub_info_h) {
        PS_CUDA(ctx, cudaMallocHost(reinterpret_cast<void **>(&ctx->hub_info_h), 16));
        PS_CUDA(ctx, cudaEventCreateWithFlags(&ctx->ev_hub, cudaEventDisableTiming));
    }
    char *hb = static_cast<char *>(ctx->hub_buf);
    hp.H = H;
    hp.counts = reinterpret_cast<int32_t *>(hb);
    hp.rank = reinterpret_cast<int32_t *>(hb + nB);
    hp.cand = hb + 2 * nB;
    hp.hub_ids = reinterpret_cast<int32_t *>(hb + 2 * nB + candB);
    hp.hub_loc = reinterpret_cast<int32_t *>(hb + 2 * nB + candB + idsB);
    hp.info = reinterpret_cast<long long *>(hb + 2 * nB + candB + 2 * idsB);
    StepRange r("hub selection");
    cudaError_t e = launch_hub_select(sample, sample_n, T, N, H, hp.counts, hp.rank, hp.cand, hp.hub_ids, hp.info,
                                      &hp.sampled, ctx->stream, &ctx->launches);
    count_launches(ctx);
    PS_CUDA(ctx, e);
    if (ctx->pool_hubs < 0) {
        PS_CUDA(ctx, cudaMemcpyAsync(ctx->hub_info_h, hp.info, 16, cudaMemcpyDeviceToHost, ctx->stream));
        PS_CUDA(ctx, cudaEventRecord(ctx->ev_hub, ctx->stream));
    }
    return PINSAGE_OK;
}

pinsage_status hub_select_finish(pinsage_ctx *ctx, int64_t N, int32_t T, int32_t K, const pinsage_layer_params *layers,
                                 int64_t a_rows, bool want_table, HubPlan &hp, bool *use)
{
    *use = false;
    if (hp.H == 0) return PINSAGE_OK;
    *use = true;
    if (ctx->pool_hubs < 0) {              // automatic: worth it when the hubs hold a third of the entries
        PS_CUDA(ctx, cudaEventSynchronize(ctx->ev_hub));
        *use = ctx->hub_info_h[0] > 0 && 3 * ctx->hub_info_h[1] >= hp.sampled;
    }
    if (!*use) return PINSAGE_OK;
    int32_t m_max = 0, dd_max = 0, kw_max = 0;
    for (int k = 0; k < K; ++k) {
        if (use_linear_pool(ctx, &layers[k])) continue;
        m_max = std::max(m_max, layers[k].m);
        dd_max = std::max(dd_max, layers[k].d);
        kw_max = std::max(kw_max, layers[k].d_in + layers[k].m);
    }
    const int H = hp.H;
    const size_t tabB = want_table ? align_up((size_t)N * T * 4, 256) : 0;
    const size_t AB = align_up((size_t)a_rows * H * 2, 256), PhB = align_up((size_t)H * m_max * 2, 256);
    const size_t GB = align_up((size_t)H * dd_max * 4, 256);
    const size_t WB = align_up((size_t)dd_max * (kw_max + H) * 2, 256);
    const size_t need = tabB + AB + PhB + GB + WB;
    if (need > ctx->hub_tab_bytes) {       // no room left for the split's storage: the plain pool (a different
        size_t free_b = 0, total_b = 0;    // rounding of the same function) instead of PINSAGE_ERR_OOM
        if (cudaMemGetInfo(&free_b, &total_b) != cudaSuccess || need > free_b + ctx->hub_tab_bytes ||
            (ctx->mem_limit > 0 && need > (size_t)ctx->mem_limit)) {
            cudaGetLastError();
            *use = false;
            return PINSAGE_OK;
        }
    }
    PS_TRY(ensure_buf(ctx, &ctx->hub_tab, &ctx->hub_tab_bytes, need, "hub-split pool storage"));
    char *after = static_cast<char *>(ctx->hub_tab);
    hp.idxm = reinterpret_cast<int32_t *>(after);
    after += tabB;
    hp.A = after;
    hp.Ph = after + AB;
    hp.G = reinterpret_cast<float *>(after + AB + PhB);
    hp.Wext = after + AB + PhB + GB;
    return PINSAGE_OK;
}

void hub_activate(pinsage_ctx *ctx, const HubPlan &hp, const int32_t *src_idx, const int32_t *idxm,
                  const int32_t *hub_ids)
{
    ctx->hub.H = hp.H;
    ctx->hub.src_idx = src_idx;
    ctx->hub.idxm = idxm;
    ctx->hub.hub_ids = hub_ids;
    ctx->hub.A = hp.A;
    ctx->hub.Ph = hp.Ph;
    ctx->hub.G = hp.G;
    ctx->hub.Wext = hp.Wext;
}

// whole-graph calls: hub entries of the table become -(rank + 1) in a remapped copy
pinsage_status hub_remap_whole(pinsage_ctx *ctx, const HubPlan &hp, const int32_t *idx, int64_t N, int32_t T)
{
    cudaError_t e = launch_hub_remap(idx, hp.rank, N * (int64_t)T, hp.idxm, ctx->stream, &ctx->launches);
    count_launches(ctx);
    PS_CUDA(ctx, e);
    hub_activate(ctx, hp, idx, hp.idxm, hp.hub_ids);
    return PINSAGE_OK;
}

bool is_host_ptr(const void *p)
{
    cudaPointerAttributes at;
    cudaError_t e = cudaPointerGetAttributes(&at, p);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return true;  // unregistered pageable host memory
    }
    return at.type == cudaMemoryTypeHost || at.type == cudaMemoryTypeUnregistered;
}

}  // namespace

extern "C" {

const char *pinsage_version(void) { return "pinsage-b200 0.1.0 (sm_100a)"; }

const char *pinsage_last_error(const pinsage_ctx *ctx)
{
    return ctx ? ctx->err.c_str() : g_create_err.c_str();
}

pinsage_status pinsage_create(pinsage_ctx **out, int device, void *cuda_stream)
{
    if (!out) return fail(nullptr, PINSAGE_ERR_INVALID_ARG, "out is NULL");
    *out = nullptr;
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return fail(nullptr, PINSAGE_ERR_CUDA, "cudaGetDeviceCount: %s", cudaGetErrorString(e));
    }
    if (device < 0 || device >= ndev)
        return fail(nullptr, PINSAGE_ERR_INVALID_ARG, "device %d of %d", device, ndev);
    cudaDeviceProp prop;
    e = cudaGetDeviceProperties(&prop, device);
    if (e != cudaSuccess)
        return fail(nullptr, PINSAGE_ERR_CUDA, "cudaGetDeviceProperties: %s", cudaGetErrorString(e));
    if (prop.major != 10)
        return fail(nullptr, PINSAGE_ERR_ARCH,
                    "device %d is sm_%d%d; this library is built for sm_100a only", device,
                    prop.major, prop.minor);
    pinsage_ctx *ctx = new (std::nothrow) pinsage_ctx;
    if (!ctx) return fail(nullptr, PINSAGE_ERR_OOM, "host allocation failed");
    ctx->device = device;
    ctx->stream = static_cast<cudaStream_t>(cuda_stream);
    ctx->num_sms = prop.multiProcessorCount;
    ctx->l2_bytes = (size_t)prop.l2CacheSize;
    DeviceGuard guard(device);
    bool ok = cudaStreamCreateWithFlags(&ctx->aux, cudaStreamNonBlocking) == cudaSuccess;
    ok = ok && cudaStreamCreateWithFlags(&ctx->h2d, cudaStreamNonBlocking) == cudaSuccess;
    ok = ok && cudaStreamCreateWithFlags(&ctx->d2h, cudaStreamNonBlocking) == cudaSuccess;
    for (int i = 0; i < 2 && ok; ++i) {
        ok = ok && cudaEventCreateWithFlags(&ctx->ev_pool[i], cudaEventDisableTiming) == cudaSuccess;
        ok = ok && cudaEventCreateWithFlags(&ctx->ev_gemm[i], cudaEventDisableTiming) == cudaSuccess;
    }
    ok = ok && cudaEventCreateWithFlags(&ctx->ev_fork, cudaEventDisableTiming) == cudaSuccess;
    ok = ok && cudaEventCreateWithFlags(&ctx->ev_join, cudaEventDisableTiming) == cudaSuccess;
    ok = ok && cudaMalloc(&ctx->d_first_bad, sizeof(long long)) == cudaSuccess;
    ok = ok && (ctx->tc = gemm_tc_state_create(ctx->num_sms)) != nullptr;
    if (!ok) {
        e = cudaGetLastError();
        pinsage_destroy(ctx);
        return fail(nullptr, PINSAGE_ERR_CUDA, "context setup: %s", cudaGetErrorString(e));
    }
    *out = ctx;
    return PINSAGE_OK;
}

void pinsage_destroy(pinsage_ctx *ctx)
{
    if (!ctx) return;
    DeviceGuard guard(ctx->device);
    cudaStreamSynchronize(ctx->stream);
    if (ctx->aux) {
        cudaStreamSynchronize(ctx->aux);
        cudaStreamDestroy(ctx->aux);
    }
    for (cudaStream_t st : {ctx->h2d, ctx->d2h})
        if (st) {
            cudaStreamSynchronize(st);
            cudaStreamDestroy(st);
        }
    for (cudaEvent_t e : ctx->pipe_events) cudaEventDestroy(e);
    for (int i = 0; i < 2; ++i) {
        if (ctx->ev_pool[i]) cudaEventDestroy(ctx->ev_pool[i]);
        if (ctx->ev_gemm[i]) cudaEventDestroy(ctx->ev_gemm[i]);
    }
    if (ctx->ev_fork) cudaEventDestroy(ctx->ev_fork);
    if (ctx->ev_join) cudaEventDestroy(ctx->ev_join);
    if (ctx->ws) cudaFree(ctx->ws);
    if (ctx->stage) cudaFree(ctx->stage);
    if (ctx->d_first_bad) cudaFree(ctx->d_first_bad);
    if (ctx->split_buf) cudaFree(ctx->split_buf);
    if (ctx->hub_buf) cudaFree(ctx->hub_buf);
    if (ctx->hub_tab) cudaFree(ctx->hub_tab);
    if (ctx->head_scratch) cudaFree(ctx->head_scratch);
    if (ctx->hub_sample) cudaFree(ctx->hub_sample);
    if (ctx->hub_info_h) cudaFreeHost(ctx->hub_info_h);
    if (ctx->ev_hub) cudaEventDestroy(ctx->ev_hub);
    gemm_tc_state_destroy(ctx->tc);
    if (ctx->subA) cudaFree(ctx->subA);
    if (ctx->subB) cudaFree(ctx->subB);
    for (cudaEvent_t e : ctx->prof_events) cudaEventDestroy(e);
    cudaGetLastError();
    delete ctx;
}

pinsage_status pinsage_set_option(pinsage_ctx *ctx, const char *key, int64_t value)
{
    if (!ctx) return PINSAGE_ERR_INVALID_ARG;
    if (!key) return fail(ctx, PINSAGE_ERR_INVALID_ARG, "key is NULL");
    if (!strcmp(key, "gemm_impl")) {
        if (value != 0 && value != 1)
            return fail(ctx, PINSAGE_ERR_INVALID_ARG, "gemm_impl must be 0 or 1");
        ctx->gemm_impl = (int)value;
    } else if (!strcmp(key, "gemm_cg")) {
        if (value < 0 || value > 2) return fail(ctx, PINSAGE_ERR_INVALID_ARG, "gemm_cg must be 0, 1 or 2");
        ctx->tune.cg = (int)value;
    } else if (!strcmp(key, "head_fused")) {
        if (value < 0 || value > 2) return fail(ctx, PINSAGE_ERR_INVALID_ARG, "head_fused = %lld outside {0, 1, 2}", (long long)value);
        ctx->head_fused = (int)value;
    } else if (!strcmp(key, "gemm_bres")) {
        if (value != 0 && value != 1) return fail(ctx, PINSAGE_ERR_INVALID_ARG, "gemm_bres must be 0 or 1");
        ctx->tune.bres = (int)value;
    } else if (!strcmp(key, "gemm_gx")) {
        if (value < 0 || value > 2) return fail(ctx, PINSAGE_ERR_INVALID_ARG, "gemm_gx must be 0, 1 or 2");
        ctx->tune.gx = (int)value;
    } else if (!strcmp(key, "check_indices")) {
        ctx->check_indices = value != 0;
    } else if (!strcmp(key, "overlap")) {
        ctx->overlap = value != 0;
    } else if (!strcmp(key, "debug_poison")) {
        ctx->poison = value != 0;
    } else if (!strcmp(key, "mem_limit_mb")) {
        if (value < 0) return fail(ctx, PINSAGE_ERR_INVALID_ARG, "mem_limit_mb must be >= 0");
        ctx->mem_limit = value << 20;
    } else if (!strcmp(key, "pool_mode")) {
        if (value < 0 || value > 2) return fail(ctx, PINSAGE_ERR_INVALID_ARG, "pool_mode must be 0, 1 or 2");
        ctx->pool_mode = (int)value;
    } else if (!strcmp(key, "linear_pool")) {
        if (value < -1 || value > 1) return fail(ctx, PINSAGE_ERR_INVALID_ARG, "linear_pool must be -1, 0 or 1");
        ctx->linear_pool = (int)value;
    } else if (!strcmp(key, "pool_slab")) {
        if (value != -1 && value != 0 && value != 32 && value != 64 && value != 128)
            return fail(ctx, PINSAGE_ERR_INVALID_ARG, "pool_slab must be -1, 0, 32, 64 or 128");
        ctx->pool_slab = (int)value;
    } else if (!strcmp(key, "pool_hubs")) {
        if (value != -1 && value != 0 && (value < 64 || value > 512 || value % 64))
            return fail(ctx, PINSAGE_ERR_INVALID_ARG, "pool_hubs must be -1, 0 or a multiple of 64 in [64, 512]");
        ctx->pool_hubs = (int)value;
    } else if (!strcmp(key, "topk_fused")) {
        ctx->topk_fused = value != 0;
    } else if (!strcmp(key, "f32_split")) {
        if (value < -1 || value > 1) return fail(ctx, PINSAGE_ERR_INVALID_ARG, "f32_split must be -1, 0 or 1");
        ctx->f32_split = (int)value;
    } else if (!strcmp(key, "profile")) {
        ctx->profile = value != 0;
    } else {
        return fail(ctx, PINSAGE_ERR_INVALID_ARG, "unknown option '%s'", key);
    }
    return PINSAGE_OK;
}

int64_t pinsage_launch_count(const pinsage_ctx *ctx) { return ctx ? ctx->total_launches : 0; }

const char *pinsage_last_plan(const pinsage_ctx *ctx) { return ctx ? ctx->plan.c_str() : ""; }

pinsage_status pinsage_profile_read(pinsage_ctx *ctx, int32_t kind, int32_t layer, double *total_ms,
                                    int64_t *launches)
{
    if (!ctx) return PINSAGE_ERR_INVALID_ARG;
    DeviceGuard guard(ctx->device);
    if (kind < -1 || kind >= PROF_KINDS || !total_ms || !launches)
        return fail(ctx, PINSAGE_ERR_INVALID_ARG, "profile_read: bad kind or NULL output");
    PS_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    PS_CUDA(ctx, cudaStreamSynchronize(ctx->aux));
    double ms = 0.0;
    int64_t n = 0;
    for (const auto &r : ctx->prof_recs) {
        if (r.kind != kind || (layer > 0 && r.layer != layer)) continue;
        float t = 0.f;
        PS_CUDA(ctx, cudaEventElapsedTime(&t, ctx->prof_events[r.e0], ctx->prof_events[r.e1]));
        ms += t;
        ++n;
    }
    *total_ms = ms;
    *launches = n;
    if (kind == -1) {  // reset
        ctx->prof_recs.clear();
        ctx->prof_used = 0;
    }
    return PINSAGE_OK;
}

pinsage_status pinsage_dense(pinsage_ctx *ctx, pinsage_dtype dtype, int64_t M, int32_t k,
                             int32_t n_out, const void *A, const void *Wt, const float *bias,
                             int32_t relu, void *out)
{
    if (!ctx) return PINSAGE_ERR_INVALID_ARG;
    DeviceGuard guard(ctx->device);
    PS_TRY(check_dtype(ctx, dtype));
    if (M < 0) return fail(ctx, PINSAGE_ERR_INVALID_ARG, "M = %lld is negative", (long long)M);
    PS_TRY(check_dim(ctx, "k", k));
    PS_TRY(check_dim(ctx, "n_out", n_out));
    PS_TRY(check_ptr(ctx, "A", A));
    PS_TRY(check_ptr(ctx, "Wt", Wt));
    PS_TRY(check_ptr(ctx, "out", out));
    if (bias && !aligned16(bias)) return fail(ctx, PINSAGE_ERR_MISALIGNED, "bias is not 16-byte aligned");
    const DType dt = static_cast<DType>(dtype);
    const size_t es = elem_size(dt);
    if (overlaps(A, (size_t)M * k * es, out, (size_t)M * n_out * es))
        return fail(ctx, PINSAGE_ERR_INVALID_ARG, "out overlaps A");
    GemmArgs g;
    g.M = M; g.K1 = k; g.N = n_out; g.A1 = A; g.B = Wt; g.bias = bias; g.relu = relu != 0; g.out = out;
    const size_t sb = gemm_scratch_bytes(ctx, dt, g);
    PS_TRY(ensure_ws(ctx, sb));
    return run_gemm(ctx, dt, g, ctx->ws, ctx->ws_bytes, ctx->stream);
}

pinsage_status pinsage_pool(pinsage_ctx *ctx, pinsage_dtype dtype, int64_t n_dst, int64_t n_src,
                            int32_t T, int32_t m, const void *P, const int32_t *nbr_idx,
                            const float *nbr_w, void *n)
{
    if (!ctx) return PINSAGE_ERR_INVALID_ARG;
    DeviceGuard guard(ctx->device);
    PS_TRY(check_dtype(ctx, dtype));
    if (n_dst < 0) return fail(ctx, PINSAGE_ERR_INVALID_ARG, "n_dst is negative");
    PS_TRY(check_graph_args(ctx, n_src, T));
    PS_TRY(check_dim(ctx, "m", m));
    if ((size_t)m * elem_size(static_cast<DType>(dtype)) > 4096)
        return fail(ctx, PINSAGE_ERR_UNSUPPORTED_SHAPE, "pool: rows of %d values exceed 4096 bytes", m);
    if (n_dst == 0) return PINSAGE_OK;
    PS_TRY(check_ptr(ctx, "P", P));
    PS_TRY(check_ptr(ctx, "nbr_idx", nbr_idx));
    PS_TRY(check_ptr(ctx, "nbr_w", nbr_w));
    PS_TRY(check_ptr(ctx, "n", n));
    const DType dt = static_cast<DType>(dtype);
    const size_t es = elem_size(dt);
    if (overlaps(P, (size_t)n_src * m * es, n, (size_t)n_dst * m * es))
        return fail(ctx, PINSAGE_ERR_INVALID_ARG, "n overlaps P");
    PS_TRY(maybe_validate(ctx, n_dst, n_src, T, nbr_idx, nbr_w));
    const int pe0 = prof_mark(ctx, ctx->stream);
    cudaError_t e = launch_pool(dt, ctx->pool_mode, n_dst, T, m, P, nbr_idx, nbr_w, n, pick_slab(ctx, dt, n_src, T, m),
                                ctx->stream, &ctx->launches);
    prof_close(ctx, PROF_POOL, pe0, ctx->stream);
    count_launches(ctx);
    if (e == cudaErrorNotSupported)
        return fail(ctx, PINSAGE_ERR_UNSUPPORTED_SHAPE, "pool: row of %d elements is too wide", m);
    PS_CUDA(ctx, e);
    return PINSAGE_OK;
}

pinsage_status pinsage_combine(pinsage_ctx *ctx, pinsage_dtype dtype, int64_t M, int32_t d_in,
                               int32_t m, int32_t d, const void *H, const void *n, const void *W,
                               const float *w, void *out)
{
    if (!ctx) return PINSAGE_ERR_INVALID_ARG;
    DeviceGuard guard(ctx->device);
    PS_TRY(check_dtype(ctx, dtype));
    if (M < 0) return fail(ctx, PINSAGE_ERR_INVALID_ARG, "M is negative");
    // d_in == 0 with H == NULL: a destination without a representation of its own (a feature-less
    // node type of a bipartite graph): z = ReLU(W n + w), W:[d x m]
    const bool no_self = d_in == 0 && H == nullptr;
    if (!no_self) {
        PS_TRY(check_dim(ctx, "d_in", d_in));
        PS_TRY(check_ptr(ctx, "H", H));
    }
    PS_TRY(check_dim(ctx, "m", m));
    PS_TRY(check_dim(ctx, "d", d));
    PS_TRY(check_ptr(ctx, "n", n));
    PS_TRY(check_ptr(ctx, "W", W));
    PS_TRY(check_ptr(ctx, "w", w));
    PS_TRY(check_ptr(ctx, "out", out));
    const DType dt = static_cast<DType>(dtype);
    const size_t es = elem_size(dt);
    if (no_self) {
    } else if (out == H) {
        if (d != d_in) return fail(ctx, PINSAGE_ERR_INVALID_ARG, "out == H requires d == d_in");
    } else if (overlaps(H, (size_t)M * d_in * es, out, (size_t)M * d * es)) {
        return fail(ctx, PINSAGE_ERR_INVALID_ARG, "out partially overlaps H");
    }
    if (overlaps(n, (size_t)M * m * es, out, (size_t)M * d * es))
        return fail(ctx, PINSAGE_ERR_INVALID_ARG, "out overlaps n");
    GemmArgs g;
    g.M = M; g.N = d; g.B = W; g.bias = w;
    g.relu = 1; g.l2norm = 1; g.out = out;
    if (no_self) {
        g.K1 = m; g.A1 = n;
    } else {
        g.K1 = d_in; g.K2 = m; g.A1 = H; g.A2 = n;
    }
    PS_TRY(ensure_ws(ctx, gemm_scratch_bytes(ctx, dt, g)));
    return run_gemm(ctx, dt, g, ctx->ws, ctx->ws_bytes, ctx->stream);
}

size_t pinsage_layer_workspace_bytes(pinsage_dtype dtype, int64_t N, int32_t T,
                                     const pinsage_layer_params *params)
{
    (void)T;
    if (!params || N <= 0 || (dtype != PINSAGE_BF16 && dtype != PINSAGE_F32)) return 0;
    // sized for the larger (SIMT reference) scratch so that either gemm_impl fits
    pinsage_ctx probe;
    probe.gemm_impl = 1;
    probe.overlap = 1;
    const DType dt = static_cast<DType>(dtype);
    const int64_t chunk = auto_chunk(N, 0, (size_t)params->m * elem_size(dt));
    size_t need = 0;
    for (int lin = 0; lin <= 1; ++lin) {       // whichever schedule the context options select
        probe.linear_pool = lin;
        need = std::max(need, plan_layer_ws(&probe, dt, N, params, chunk).total);
    }
    return need;
}

pinsage_status pinsage_layer(pinsage_ctx *ctx, pinsage_dtype dtype, int64_t N, int32_t T,
                             const void *feats, const int32_t *nbr_idx, const float *nbr_w,
                             const pinsage_layer_params *params, void *out, void *ws,
                             size_t ws_bytes)
{
    if (!ctx) return PINSAGE_ERR_INVALID_ARG;
    DeviceGuard guard(ctx->device);
    PS_TRY(check_dtype(ctx, dtype));
    PS_TRY(check_graph_args(ctx, N, T));
    PS_TRY(check_layer_params(ctx, params, "params"));
    PS_TRY(check_ptr(ctx, "feats", feats));
    PS_TRY(check_ptr(ctx, "nbr_idx", nbr_idx));
    PS_TRY(check_ptr(ctx, "nbr_w", nbr_w));
    PS_TRY(check_ptr(ctx, "out", out));
    const DType dt = static_cast<DType>(dtype);
    const size_t es = elem_size(dt);
    PS_TRY(check_pool_width(ctx, dt, params));
    if (out == feats) {
        if (params->d != params->d_in)
            return fail(ctx, PINSAGE_ERR_INVALID_ARG, "out == feats requires d == d_in");
    } else if (overlaps(feats, (size_t)N * params->d_in * es, out, (size_t)N * params->d * es)) {
        return fail(ctx, PINSAGE_ERR_INVALID_ARG, "out partially overlaps feats");
    }
    const int64_t chunk = auto_chunk(N, 0, (size_t)params->m * es);
    const LayerWs plan = plan_layer_ws(ctx, dt, N, params, chunk);
    char *base;
    if (ws) {
        if ((reinterpret_cast<uintptr_t>(ws) & 255u) != 0)
            return fail(ctx, PINSAGE_ERR_MISALIGNED, "ws is not 256-byte aligned");
        if (ws_bytes < plan.total)
            return fail(ctx, PINSAGE_ERR_OOM, "ws_bytes = %zu < required %zu", ws_bytes, plan.total);
        base = static_cast<char *>(ws);
    } else {
        PS_TRY(ensure_ws(ctx, plan.total));
        base = static_cast<char *>(ctx->ws);
    }
    PS_TRY(maybe_validate(ctx, N, N, T, nbr_idx, nbr_w));
    HintGuard hint(ctx, N);
    ctx->cur_layer = 1;
    HubReset hub_reset{ctx};
    HubPlan hp;
    bool use = false;
    PS_TRY(hub_select_begin(ctx, dt, N, T, 1, params, nbr_idx, N, hp));
    PS_TRY(project_chunks(ctx, dt, N, params, feats, base, plan, chunk, ChunkIO()));   // (hides the read-back)
    PS_TRY(hub_select_finish(ctx, N, T, 1, params, chunk, true, hp, &use));
    if (use) PS_TRY(hub_remap_whole(ctx, hp, nbr_idx, N, T));
    return pool_combine_chunks(ctx, dt, N, T, params, feats, base + plan.P_off, nbr_idx, nbr_w, out, chunk,
                               base + plan.n0_off, base + plan.n1_off, base + plan.scratch_off, plan.scratch_bytes, N,
                               ChunkIO());
}

pinsage_status pinsage_head(pinsage_ctx *ctx, pinsage_dtype dtype, int64_t N, const void *h,
                            const pinsage_head_params *params, void *out)
{
    if (!ctx) return PINSAGE_ERR_INVALID_ARG;
    DeviceGuard guard(ctx->device);
    PS_TRY(check_dtype(ctx, dtype));
    if (N < 1) return fail(ctx, PINSAGE_ERR_INVALID_ARG, "N must be positive");
    PS_TRY(check_head_params(ctx, params));
    PS_TRY(check_ptr(ctx, "h", h));
    PS_TRY(check_ptr(ctx, "out", out));
    const DType dt = static_cast<DType>(dtype);
    const size_t es = elem_size(dt);
    if (overlaps(h, (size_t)N * params->d * es, out, (size_t)N * params->d_out * es))
        return fail(ctx, PINSAGE_ERR_INVALID_ARG, "out overlaps h");
    const int64_t chunk = auto_chunk(N, 0, (size_t)params->g1 * es);
    const size_t a_bytes = align_up((size_t)chunk * params->g1 * es, 256);
    PS_TRY(ensure_ws(ctx, a_bytes));
    HintGuard hint(ctx, N);
    for (int64_t r0 = 0; r0 < N; r0 += chunk) {
        const int64_t rows = std::min(chunk, N - r0);
        StepRange r45("S4+S5 head rows %lld+%lld", (long long)r0, (long long)rows);
        PS_TRY(run_head(ctx, dt, rows, static_cast<const char *>(h) + (size_t)r0 * params->d * es, params, ctx->ws,
                        static_cast<char *>(out) + (size_t)r0 * params->d_out * es, ctx->stream));
    }
    return PINSAGE_OK;
}

// The head without any allocation: one launch of the fused S4 -> S5 kernel with its scratch in a file-scope
// __device__ array (gemm_head.cu).  No cudaMalloc / cudaFree / event creation on this path, whatever the
// context's options say (no profile records, no workspace growth).
pinsage_status pinsage_head_static(pinsage_ctx *ctx, pinsage_dtype dtype, int64_t N, const void *h,
                                   const pinsage_head_params *params, void *out)
{
    if (!ctx) return PINSAGE_ERR_INVALID_ARG;
    DeviceGuard guard(ctx->device);
    PS_TRY(check_dtype(ctx, dtype));
    if (N < 1) return fail(ctx, PINSAGE_ERR_INVALID_ARG, "N must be positive");
    PS_TRY(check_head_params(ctx, params));
    PS_TRY(check_ptr(ctx, "h", h));
    PS_TRY(check_ptr(ctx, "out", out));
    const DType dt = static_cast<DType>(dtype);
    if (dt != DType::BF16 || !head_tc_supported(params->d, params->g1, params->d_out))
        return fail(ctx, PINSAGE_ERR_UNSUPPORTED_SHAPE,
                    "pinsage_head_static covers BF16 heads with g1 <= 256 and d_out <= 256 (the one-launch kernel); "
                    "got dtype %d, d = %d, g1 = %d, d_out = %d", (int)dtype, params->d, params->g1, params->d_out);
    if (N >= (1LL << 31)) return fail(ctx, PINSAGE_ERR_INVALID_ARG, "N = %lld outside [1, 2^31)", (long long)N);
    const size_t es = elem_size(dt);
    if (overlaps(h, (size_t)N * params->d * es, out, (size_t)N * params->d_out * es))
        return fail(ctx, PINSAGE_ERR_INVALID_ARG, "out overlaps h");
    StepRange r45("S4+S5 head (static scratch) rows 0+%lld", (long long)N);
    bool too_big = false;
    cudaError_t e = launch_head_tc_static(ctx->tc, N, params->d, params->g1, params->d_out, h, params->G1, params->g,
                                          params->G2, out, ctx->num_sms, ctx->stream, &ctx->launches, &too_big);
    count_launches(ctx);
    if (too_big)
        return fail(ctx, PINSAGE_ERR_UNSUPPORTED_SHAPE,
                    "pinsage_head_static: g1 = %d on %d SMs needs %zu bytes of scratch, the static array holds %zu",
                    params->g1, ctx->num_sms, head_tc_scratch_bytes(params->g1, ctx->num_sms), head_static_scratch_bytes());
    PS_CUDA(ctx, e);
    return PINSAGE_OK;
}

pinsage_status pinsage_embed_all(pinsage_ctx *ctx, pinsage_dtype dtype, int64_t N, int32_t T,
                                 int32_t K, const void *feats, const int32_t *nbr_idx,
                                 const float *nbr_w, const pinsage_layer_params *layers,
                                 const pinsage_head_params *head, void *out, int64_t chunk_nodes)
{
    if (!ctx) return PINSAGE_ERR_INVALID_ARG;
    DeviceGuard guard(ctx->device);
    PS_TRY(check_dtype(ctx, dtype));
    PS_TRY(check_graph_args(ctx, N, T));
    if (K < 1 || K > 64) return fail(ctx, PINSAGE_ERR_INVALID_ARG, "K = %d outside [1, 64]", K);
    if (chunk_nodes < 0) return fail(ctx, PINSAGE_ERR_INVALID_ARG, "chunk_nodes is negative");
    if (!layers) return fail(ctx, PINSAGE_ERR_INVALID_ARG, "layers is NULL");
    for (int k = 0; k < K; ++k) {
        PS_TRY(check_layer_params(ctx, &layers[k], "layers[k]"));
        if (k > 0 && layers[k].d_in != layers[k - 1].d)
            return fail(ctx, PINSAGE_ERR_INVALID_ARG, "layers[%d].d_in = %d != layers[%d].d = %d", k,
                        layers[k].d_in, k - 1, layers[k - 1].d);
    }
    PS_TRY(check_head_params(ctx, head));
    if (head->d != layers[K - 1].d)
        return fail(ctx, PINSAGE_ERR_INVALID_ARG, "head.d = %d != layers[K-1].d = %d", head->d,
                    layers[K - 1].d);
    PS_TRY(check_ptr(ctx, "feats", feats));
    PS_TRY(check_ptr(ctx, "nbr_idx", nbr_idx));
    PS_TRY(check_ptr(ctx, "nbr_w", nbr_w));
    PS_TRY(check_ptr(ctx, "out", out));
    const DType dt = static_cast<DType>(dtype);
    const size_t es = elem_size(dt);
    for (int k = 0; k < K; ++k) PS_TRY(check_pool_width(ctx, dt, &layers[k]));
    HintGuard hint(ctx, N);
    const size_t feats_bytes = (size_t)N * layers[0].d_in * es;
    const size_t tab_bytes = (size_t)N * T * 4;
    const size_t out_bytes = (size_t)N * head->d_out * es;
    if (overlaps(feats, feats_bytes, out, out_bytes))
        return fail(ctx, PINSAGE_ERR_INVALID_ARG, "out overlaps feats");

    // ---- where the arrays live, and the memory plan -------------------------------------------------
    const bool h_feats = is_host_ptr(feats), h_idx = is_host_ptr(nbr_idx), h_w = is_host_ptr(nbr_w);
    const bool h_out = is_host_ptr(out);
    const bool any_host = h_feats || h_idx || h_w || h_out;
    EmbedPlan pl;
    PS_TRY(plan_embed(ctx, dt, N, T, K, layers, head, chunk_nodes, h_feats, h_idx, h_w, h_out, pl));
    const int64_t chunk = pl.chunk, nchunks = pl.nchunks;
    {
        char buf[256];
        snprintf(buf, sizeof buf, "chunk=%lld chunks=%lld H=%s%s feats=%s tables=%s out=%s workspace=%zu staging=%zu",
                 (long long)chunk, (long long)nchunks, pl.H_is_out ? "out" : "workspace", pl.need_Hb ? "+second" : "",
                 !h_feats ? "device" : pl.feats_whole ? "staged" : "ring", !(h_idx || h_w) ? "device" : pl.tabs_whole ? "staged" : "ring",
                 h_out ? "ring" : "device", pl.ws_total, pl.stage_total);
        ctx->plan = buf;
    }
    PS_TRY(fit_buffers(ctx, pl.ws_total, pl.stage_total));
    char *ws = static_cast<char *>(ctx->ws);
    char *stage = static_cast<char *>(ctx->stage);
    char *Ha = pl.H_is_out ? static_cast<char *>(out) : ws + pl.max_layer_ws;
    char *Hb = pl.need_Hb ? ws + pl.max_layer_ws + (pl.H_is_out ? 0 : pl.H_bytes) : nullptr;
    char *abuf = ws + pl.max_layer_ws + pl.H_bytes * ((pl.H_is_out ? 0 : 1) + (pl.need_Hb ? 1 : 0));

    // ---- host inputs / output: slots, events, the first copies (features first, then the tables: layer
    // 1's S1 launches chase the feature chunks, its S2 / S3 the table chunks) --------------------------
    HostSrc sF, sI, sW;
    HostSink sO;
    if (any_host) {
        auto setup = [&](HostSrc &h, const void *p, size_t row_bytes, bool whole, size_t off) {
            h.host = static_cast<const char *>(p);
            h.dev = stage + off;
            h.row_bytes = row_bytes;
            h.N = N;
            h.chunk = chunk;
            h.nchunks = nchunks;
            h.whole = whole;
            h.depth = whole ? (int)nchunks : (int)std::min<int64_t>(RING, nchunks);
            h.used.assign((size_t)h.depth, 0);
        };
        if (h_feats) setup(sF, feats, (size_t)layers[0].d_in * es, pl.feats_whole, pl.feats_off);
        if (h_idx) setup(sI, nbr_idx, (size_t)T * 4, pl.tabs_whole, pl.idx_off);
        if (h_w) setup(sW, nbr_w, (size_t)T * 4, pl.tabs_whole, pl.w_off);
        size_t n_ev = 4;
        for (HostSrc *h : {&sF, &sI, &sW}) n_ev += h->active() ? 2 * (size_t)h->depth : 0;
        PS_TRY(ensure_pipe_events(ctx, n_ev));
        cudaEvent_t *ev = ctx->pipe_events.data();
        for (HostSrc *h : {&sF, &sI, &sW})
            if (h->active()) {
                h->landed = ev;
                h->freed = ev + h->depth;
                ev += 2 * h->depth;
            }
        if (h_out) {
            sO.host = static_cast<char *>(out);
            sO.dev = stage + pl.out_off;
            sO.row_bytes = (size_t)head->d_out * es;
            sO.chunk = chunk;
            sO.ready[0] = ev[0]; sO.ready[1] = ev[1]; sO.copied[0] = ev[2]; sO.copied[1] = ev[3];
        }
        // the staging slots may still be read by kernels of an earlier call on the compute stream
        PS_CUDA(ctx, cudaEventRecord(ctx->ev_fork, ctx->stream));
        PS_CUDA(ctx, cudaStreamWaitEvent(ctx->h2d, ctx->ev_fork, 0));
        PS_CUDA(ctx, cudaStreamWaitEvent(ctx->d2h, ctx->ev_fork, 0));
    }

    // ---- validation on request (whole tables: host tables are checked chunk by chunk as they land) ----
    if (ctx->check_indices && !h_idx && !h_w) PS_TRY(maybe_validate(ctx, N, N, T, nbr_idx, nbr_w));

    // ---- hub-split pool (skewed graphs; hubs.cu): pick the hubs from a sample of the lists.  Device
    // tables are remapped into a copy; tables from the host are remapped in their staging slots. -------
    HubReset hub_reset{ctx};
    bool hubs_on = false;
    HubPlan hp;
    {
        const int64_t rows_s = std::min<int64_t>(N, 16384), stride = N / rows_s;
        const int32_t *sample = nbr_idx;
        int64_t sample_n = N;
        if (h_idx && hub_eligible(ctx, dt, N, T, K, layers)) {
            // every stride-th row of the host table, as the device path samples it: one strided copy
            PS_TRY(ensure_buf(ctx, &ctx->hub_sample, &ctx->hub_sample_bytes, (size_t)rows_s * T * 4, "hub sample"));
            PS_CUDA(ctx, cudaMemcpy2DAsync(ctx->hub_sample, (size_t)T * 4, nbr_idx, (size_t)stride * T * 4,
                                           (size_t)T * 4, (size_t)rows_s, cudaMemcpyHostToDevice, ctx->stream));
            sample = static_cast<const int32_t *>(ctx->hub_sample);
            sample_n = rows_s;
        }
        PS_TRY(hub_select_begin(ctx, dt, N, T, K, layers, sample, sample_n, hp));
    }
    // (hub_select_finish follows S1 of the first layer, which hides the selection's read-back)
    auto hub_finish = [&]() -> pinsage_status {
        PS_TRY(hub_select_finish(ctx, N, T, K, layers, chunk, !h_idx, hp, &hubs_on));
        if (hubs_on && !h_idx) PS_TRY(hub_remap_whole(ctx, hp, nbr_idx, N, T));
        else if (hubs_on) hub_activate(ctx, hp, nullptr, nullptr, hp.hub_ids);
        return PINSAGE_OK;
    };

    // ---- per-chunk plumbing of the layers -------------------------------------------------------------
    const char *Hlast = nullptr;               // the last layer's output buffer (set when the loop reaches it)
    void *d_out = h_out ? nullptr : out;
    int layer = 0;                             // 0-based layer the lambdas below act for
    std::vector<char> remapped((size_t)nchunks, 0), validated((size_t)nchunks, 0);
    ChunkIO io;
    if (h_feats) {
        io.s1_in = [&](int64_t c, const void **src) { return sF.acquire(ctx, c, ctx->stream, src); };
        io.s1_done = [&](int64_t c) { return sF.release(ctx, c, ctx->stream); };
    }
    io.tables_in = [&](int64_t c, cudaStream_t ps, const int32_t **ic, const float **wc) -> pinsage_status {
        const int64_t r0 = c * chunk, rows = std::min(chunk, N - r0);
        const void *p = nullptr;
        if (h_idx) {
            PS_TRY(sI.acquire(ctx, c, ps, &p));
            *ic = static_cast<const int32_t *>(p);
        }
        if (h_w) {
            PS_TRY(sW.acquire(ctx, c, ps, &p));
            *wc = static_cast<const float *>(p);
        }
        if (ctx->check_indices && (h_idx || h_w) && !validated[(size_t)c]) {
            if (ps != ctx->stream) {           // (the validation kernel runs on the context's main stream)
                if (h_idx) PS_TRY(sI.acquire(ctx, c, ctx->stream, &p));
                if (h_w) PS_TRY(sW.acquire(ctx, c, ctx->stream, &p));
            }
            int64_t bad = -1;                  // (synchronous; ids are still the caller's here)
            pinsage_status st = pinsage_validate_graph(ctx, rows, N, T, *ic, *wc, &bad);
            if (st != PINSAGE_OK) return st;
            validated[(size_t)c] = 1;
        }
        if (io.hub_remapped && !(sI.whole && remapped[(size_t)c])) {
            // in place in the staging slot (once when the table is staged whole, every pass through a ring)
            int32_t *slot = const_cast<int32_t *>(*ic);
            cudaError_t e = launch_hub_remap(slot, hp.rank, rows * (int64_t)T, slot, ps, &ctx->launches);
            count_launches(ctx);
            PS_CUDA(ctx, e);
            remapped[(size_t)c] = 1;
        }
        return PINSAGE_OK;
    };
    io.tables_done = [&](int64_t c, cudaStream_t ps) -> pinsage_status {
        if (h_idx) PS_TRY(sI.release(ctx, c, ps));
        if (h_w) PS_TRY(sW.release(ctx, c, ps));
        return PINSAGE_OK;
    };
    if (!h_idx && !h_w) {
        io.tables_in = nullptr;
        io.tables_done = nullptr;
    }
    io.self_in = [&](int64_t c, const void **self) -> pinsage_status {
        if (layer == 0 && h_feats) return sF.acquire(ctx, c, ctx->stream, self);
        return PINSAGE_OK;
    };
    // after S3 of chunk c: (layer 1, streamed features) the slot is free; (last layer) the head of the
    // chunk -- the intermediate a never exists in full, and a host `out` streams home during the layer
    io.after_chunk = [&](int64_t c, int64_t r0, int64_t rows) -> pinsage_status {
        if (layer == 0 && h_feats) PS_TRY(sF.release(ctx, c, ctx->stream));
        if (layer != K - 1) return PINSAGE_OK;
        StepRange r45("S4+S5 head rows %lld+%lld", (long long)r0, (long long)rows);
        if (h_out) PS_TRY(sO.acquire(ctx, c, ctx->stream));
        PS_TRY(run_head(ctx, dt, rows, Hlast + (size_t)r0 * head->d * es, head, abuf,
                        h_out ? sO.ptr(c) : static_cast<char *>(d_out) + (size_t)r0 * head->d_out * es, ctx->stream));
        if (h_out) PS_TRY(sO.release(ctx, c, r0, rows, ctx->stream));
        return PINSAGE_OK;
    };

    const void *Hin = h_feats ? nullptr : feats;
    char *Hcur = nullptr;
    for (int k = 0; k < K; ++k) {
        const pinsage_layer_params *lp = &layers[k];
        const LayerWs plan = plan_layer_ws(ctx, dt, N, lp, chunk);
        ctx->cur_layer = k + 1;
        layer = k;
        char *Hout;
        if (k == 0) Hout = Ha;
        else if (lp->d == lp->d_in) Hout = Hcur;           // in place (S1 has consumed all of H first)
        else Hout = (Hcur == Ha) ? Hb : Ha;
        if (k == K - 1) Hlast = Hout;
        // aliasing rules, as assertions: a layer runs in place only at equal widths;
        // `out` doubles as H only when every row of H has out's stride; two H buffers otherwise
        if ((Hout == Hcur && lp->d != lp->d_in) || (pl.H_is_out && lp->d != head->d_out) ||
            (Hout != Hcur && k > 0 && !Hb))
            return fail(ctx, PINSAGE_ERR_CUDA, "internal: buffer aliasing rule violated in layer %d", k + 1);
        ChunkIO lio = io;
        if (k > 0 || !h_feats) {
            lio.s1_in = nullptr;
            lio.s1_done = nullptr;
        }
        if (k == 0) PS_TRY(sF.begin_pass(ctx));                     // pass 1: S1 behind the feature chunks
        PS_TRY(project_chunks(ctx, dt, N, lp, Hin, ws, plan, chunk, lio));
        if (k == 0) {
            PS_TRY(hub_finish());
            io.hub_remapped = lio.hub_remapped = hubs_on && h_idx;
            ctx->plan += hubs_on ? " hubs=" + std::to_string(hp.H) : std::string(" hubs=off");
        }
        if (k == 0 && !sF.whole) PS_TRY(sF.begin_pass(ctx));        // streamed features, pass 2: the self rows of S3
        PS_TRY(sI.begin_pass(ctx));                                 // (no-ops for device arrays and for
        PS_TRY(sW.begin_pass(ctx));                                 //  tables already staged whole)
        PS_TRY(pool_combine_chunks(ctx, dt, N, T, lp, Hin, ws + plan.P_off, nbr_idx, nbr_w, Hout, chunk,
                                   ws + plan.n0_off, ws + plan.n1_off, ws + plan.scratch_off, plan.scratch_bytes,
                                   N, lio));
        if (ctx->poison && Hcur && Hout != Hcur)   // the previous H is dead once S1 and every S3 of this layer ran
            PS_CUDA(ctx, cudaMemsetAsync(Hcur, 0xFF, (size_t)N * lp->d_in * es, ctx->stream));
        Hcur = Hout;
        Hin = Hout;
    }
    if (any_host) {
        PS_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
        PS_CUDA(ctx, cudaStreamSynchronize(ctx->h2d));
        PS_CUDA(ctx, cudaStreamSynchronize(ctx->d2h));
    }
    return PINSAGE_OK;
}

pinsage_status pinsage_embed_nodes(pinsage_ctx *ctx, pinsage_dtype dtype, int64_t N, int32_t T,
                                   int32_t K, const void *feats, const int32_t *nbr_idx,
                                   const float *nbr_w, const pinsage_layer_params *layers,
                                   const pinsage_head_params *head, int64_t M, const int32_t *targets,
                                   void *out)
{
    if (!ctx) return PINSAGE_ERR_INVALID_ARG;
    DeviceGuard guard(ctx->device);
    PS_TRY(check_dtype(ctx, dtype));
    PS_TRY(check_graph_args(ctx, N, T));
    if (K < 1 || K > 64) return fail(ctx, PINSAGE_ERR_INVALID_ARG, "K = %d outside [1, 64]", K);
    if (M < 1 || M >= (1LL << 31)) return fail(ctx, PINSAGE_ERR_INVALID_ARG, "M = %lld outside [1, 2^31)", (long long)M);
    if (!layers) return fail(ctx, PINSAGE_ERR_INVALID_ARG, "layers is NULL");
    for (int k = 0; k < K; ++k) {
        PS_TRY(check_layer_params(ctx, &layers[k], "layers[k]"));
        if (k > 0 && layers[k].d_in != layers[k - 1].d)
            return fail(ctx, PINSAGE_ERR_INVALID_ARG, "layers[%d].d_in != layers[%d].d", k, k - 1);
    }
    PS_TRY(check_head_params(ctx, head));
    if (head->d != layers[K - 1].d) return fail(ctx, PINSAGE_ERR_INVALID_ARG, "head.d != layers[K-1].d");
    PS_TRY(check_ptr(ctx, "feats", feats));
    PS_TRY(check_ptr(ctx, "nbr_idx", nbr_idx));
    PS_TRY(check_ptr(ctx, "nbr_w", nbr_w));
    PS_TRY(check_ptr(ctx, "targets", targets));
    PS_TRY(check_ptr(ctx, "out", out));
    const DType dt = static_cast<DType>(dtype);
    const size_t es = elem_size(dt);
    for (int k = 0; k < K; ++k) PS_TRY(check_pool_width(ctx, dt, &layers[k]));
    HintGuard hint(ctx, N);
    cudaStream_t st = ctx->stream;
    PS_TRY(maybe_validate(ctx, N, N, T, nbr_idx, nbr_w));

    // ---- phase A: the sets S^(K) = targets, S^(k-1) = S^(k) U N(S^(k))  (Alg. 2 l.1-7) ---------------
    const long long nb = subset_blocks(N);
    const size_t markB = align_up((size_t)N, 256), i32B = align_up((size_t)N * 4, 256);
    const size_t cntB = align_up((size_t)(nb + 1) * 8, 256);
    PS_TRY(ensure_buf(ctx, &ctx->subA, &ctx->subA_bytes, (size_t)(K + 1) * (markB + 2 * i32B) + cntB,
                      "embed_nodes set storage"));
    char *A = static_cast<char *>(ctx->subA);
    auto mark = [&](int k) { return reinterpret_cast<unsigned char *>(A + (size_t)k * markB); };
    auto list = [&](int k) { return reinterpret_cast<int32_t *>(A + (size_t)(K + 1) * markB + (size_t)k * i32B); };
    auto pos = [&](int k) { return reinterpret_cast<int32_t *>(A + (size_t)(K + 1) * (markB + i32B) + (size_t)k * i32B); };
    long long *counts = reinterpret_cast<long long *>(A + (size_t)(K + 1) * (markB + 2 * i32B));
    PS_CUDA(ctx, cudaMemsetAsync(A, 0, (size_t)(K + 1) * markB, st));
    PS_CUDA(ctx, subset_mark_targets(targets, M, N, mark(K), ctx->d_first_bad, st, &ctx->launches));
    std::vector<int64_t> n(K + 1, 0);
    for (int k = K; k >= 0; --k) {
        PS_CUDA(ctx, subset_compact(mark(k), N, counts, nullptr, nullptr, false, st, &ctx->launches));
        long long host[2] = {0, 0};
        PS_CUDA(ctx, cudaMemcpyAsync(&host[0], counts + nb, 8, cudaMemcpyDeviceToHost, st));
        PS_CUDA(ctx, cudaMemcpyAsync(&host[1], ctx->d_first_bad, 8, cudaMemcpyDeviceToHost, st));
        PS_CUDA(ctx, cudaStreamSynchronize(st));
        if (k == K && host[1] != 0x7fffffffffffffffLL) {
            count_launches(ctx);
            return fail(ctx, PINSAGE_ERR_BAD_INDEX, "targets[%lld] is outside [0, %lld)", host[1], (long long)N);
        }
        n[k] = host[0];
        PS_CUDA(ctx, subset_compact(mark(k), N, counts, list(k), pos(k), true, st, &ctx->launches));
        if (k > 0) PS_CUDA(ctx, subset_expand(list(k), n[k], nbr_idx, T, mark(k - 1), st, &ctx->launches));
    }
    count_launches(ctx);

    // ---- phase B: compact tensors, sized from the set sizes ----------------------------------------------
    size_t Hmax = (size_t)n[0] * layers[0].d_in * es, selfmax = 0, tabmax = 0, wsmax = 0;
    std::vector<int64_t> chunk(K + 1, 0);
    for (int k = 1; k <= K; ++k) {
        const pinsage_layer_params *lp = &layers[k - 1];
        Hmax = std::max(Hmax, (size_t)n[k] * lp->d * es);
        selfmax = std::max(selfmax, (size_t)n[k] * lp->d_in * es);
        tabmax = std::max(tabmax, (size_t)n[k] * T * 4);
        chunk[k] = auto_chunk(n[k], 0, (size_t)std::max(lp->m, lp->d) * es);
        wsmax = std::max(wsmax, plan_layer_ws(ctx, dt, n[k - 1], lp, chunk[k]).total);
    }
    // the hub-split pool, if the whole graph would take it: same hubs, same split, same bits as the rows
    // of pinsage_embed_all
    HubReset hub_reset{ctx};
    HubPlan hp;
    bool use_hubs = false;
    PS_TRY(hub_select_begin(ctx, dt, N, T, K, layers, nbr_idx, N, hp));
    PS_TRY(hub_select_finish(ctx, N, T, K, layers, *std::max_element(chunk.begin() + 1, chunk.end()), false, hp,
                             &use_hubs));
    const size_t aB = align_up((size_t)n[K] * head->g1 * es, 256), oB = align_up((size_t)n[K] * head->d_out * es, 256);
    Hmax = align_up(Hmax, 256); selfmax = align_up(selfmax, 256); tabmax = align_up(tabmax, 256);
    wsmax = align_up(wsmax, 256);
    PS_TRY(ensure_buf(ctx, &ctx->subB, &ctx->subB_bytes, 2 * Hmax + selfmax + 2 * tabmax + wsmax + aB + oB,
                      "embed_nodes compact tensors"));
    char *B = static_cast<char *>(ctx->subB);
    char *Hbuf[2] = {B, B + Hmax};
    char *Hself = B + 2 * Hmax;
    int32_t *idx_loc = reinterpret_cast<int32_t *>(Hself + selfmax);
    float *w_loc = reinterpret_cast<float *>(Hself + selfmax + tabmax);
    char *lws = Hself + selfmax + 2 * tabmax;
    char *abuf = lws + wsmax, *obuf = abuf + aB;

    // h^(0) = x on S^(0)  (Alg. 2 l.8), then CONVOLVE level by level on the re-indexed sub-graph (l.9-14)
    PS_CUDA(ctx, subset_gather_rows(feats, list(0), nullptr, n[0], (size_t)layers[0].d_in * es, Hbuf[0], st,
                                    &ctx->launches));
    int cur = 0;
    for (int k = 1; k <= K; ++k) {
        const pinsage_layer_params *lp = &layers[k - 1];
        PS_CUDA(ctx, subset_remap_tables(list(k), n[k], nbr_idx, nbr_w, T, pos(k - 1), idx_loc, w_loc, st,
                                         &ctx->launches));
        PS_CUDA(ctx, subset_gather_rows(Hbuf[cur], list(k), pos(k - 1), n[k], (size_t)lp->d_in * es, Hself, st,
                                        &ctx->launches));
        ctx->hub.H = 0;
        if (use_hubs && !use_linear_pool(ctx, lp)) {
            // entries that name a hub of the whole graph become -(rank + 1); the hubs' rows of the compact
            // P are found through the previous set's positions
            PS_CUDA(ctx, launch_hub_remap_sub(list(k), n[k], nbr_idx, T, hp.rank, idx_loc, st, &ctx->launches));
            PS_CUDA(ctx, launch_hub_localize(hp.hub_ids, hp.H, mark(k - 1), pos(k - 1), hp.hub_loc, st, &ctx->launches));
            hub_activate(ctx, hp, idx_loc, idx_loc, hp.hub_loc);
        }
        count_launches(ctx);
        const LayerWs plan = plan_layer_ws(ctx, dt, n[k - 1], lp, chunk[k]);
        ctx->cur_layer = k;
        PS_TRY(layer_on_ws(ctx, dt, n[k], T, Hself, idx_loc, w_loc, lp, Hbuf[cur ^ 1], lws, plan, chunk[k],
                           n[k - 1], Hbuf[cur]));
        cur ^= 1;
    }
    // head on S^(K) (l.15-17), then one row per requested target, in the caller's order
    PS_TRY(run_head(ctx, dt, n[K], Hbuf[cur], head, abuf, obuf, st));
    PS_CUDA(ctx, subset_gather_rows(obuf, targets, pos(K), M, (size_t)head->d_out * es, out, st, &ctx->launches));
    count_launches(ctx);
    return PINSAGE_OK;
}

pinsage_status pinsage_topk(pinsage_ctx *ctx, pinsage_dtype dtype, int64_t nq, int64_t N, int32_t d,
                            const void *Q, const void *Z, int32_t k, int32_t *out_idx, float *out_score)
{
    if (!ctx) return PINSAGE_ERR_INVALID_ARG;
    DeviceGuard guard(ctx->device);
    PS_TRY(check_dtype(ctx, dtype));
    if (nq < 1 || nq >= (1LL << 31)) return fail(ctx, PINSAGE_ERR_INVALID_ARG, "nq = %lld outside [1, 2^31)", (long long)nq);
    if (N < 1 || N >= (1LL << 31)) return fail(ctx, PINSAGE_ERR_INVALID_ARG, "N = %lld outside [1, 2^31)", (long long)N);
    if (k < 1 || k > N) return fail(ctx, PINSAGE_ERR_INVALID_ARG, "k = %d outside [1, N]", k);
    if (k > 1024) return fail(ctx, PINSAGE_ERR_UNSUPPORTED_SHAPE, "k = %d exceeds 1024", k);
    PS_TRY(check_dim(ctx, "d", d));
    PS_TRY(check_ptr(ctx, "Q", Q));
    PS_TRY(check_ptr(ctx, "Z", Z));
    PS_TRY(check_ptr(ctx, "out_idx", out_idx));
    PS_TRY(check_ptr(ctx, "out_score", out_score));
    // many queries: groups of 16 384, so that the candidate blocks stay wide (>= 16 384 candidates
    // per GEMM) and the per-block bookkeeping small; the groups are independent lookups
    constexpr int64_t Q_GROUP = 16384;
    if (nq > Q_GROUP) {
        const size_t esz = elem_size(static_cast<DType>(dtype));
        for (int64_t q0 = 0; q0 < nq; q0 += Q_GROUP) {
            const int64_t n = std::min(Q_GROUP, nq - q0);
            PS_TRY(pinsage_topk(ctx, dtype, n, N, d, static_cast<const char *>(Q) + (size_t)q0 * d * esz, Z, k,
                                out_idx + (size_t)q0 * k, out_score + (size_t)q0 * k));
        }
        return PINSAGE_OK;
    }
    const DType dt = static_cast<DType>(dtype);
    const size_t es = elem_size(dt);
    // candidate block: as wide as keeps the fp32 score block within 1 GiB, a multiple of 256, <= 65536
    int64_t NB = std::min<int64_t>(65536, std::max<int64_t>(256, ((int64_t)1 << 28) / nq / 256 * 256));
    // (whole waves: a CTA pair owns one 256-candidate slab for all queries, num_sms / 2 pairs run at a time)
    const int64_t wave = (int64_t)(ctx->num_sms / 2) * 256;
    if (NB >= wave) NB = NB / wave * wave;
    NB = std::min<int64_t>(NB, (N + 7) / 8 * 8);
    const int64_t n_blocks = (N + NB - 1) / NB;
    const size_t score_bytes = align_up((size_t)nq * NB * 4, 256), key_bytes = align_up(topk_state_bytes(nq), 256);
    const size_t prev_bytes = align_up((size_t)nq * 4, 256), any_bytes = align_up((size_t)n_blocks * 4, 256);
    const size_t ovf_bytes = align_up((size_t)n_blocks * nq, 256);
    GemmArgs probe;
    probe.M = nq; probe.K1 = d; probe.N = (int32_t)NB; probe.out_f32 = 1;
    probe.A1 = Q; probe.B = Z;
    const size_t scratch = gemm_scratch_bytes(ctx, dt, probe);
    PS_TRY(ensure_ws(ctx, score_bytes + key_bytes + prev_bytes + any_bytes + ovf_bytes + scratch));
    char *ws = static_cast<char *>(ctx->ws);
    float *scores = reinterpret_cast<float *>(ws);
    void *keys = ws + score_bytes;
    int *cnts = reinterpret_cast<int *>(static_cast<unsigned long long *>(keys) + (size_t)nq * TK_TOTAL);
    int *cnt_prev = reinterpret_cast<int *>(ws + score_bytes + key_bytes);
    int *any = reinterpret_cast<int *>(ws + score_bytes + key_bytes + prev_bytes);
    unsigned char *ovf = reinterpret_cast<unsigned char *>(ws + score_bytes + key_bytes + prev_bytes + any_bytes);
    char *gscratch = ws + score_bytes + key_bytes + prev_bytes + any_bytes + ovf_bytes;
    // Selection in the GEMM epilogue (no score round trip through HBM) once every list is full and its
    // k-th score is a useful threshold: after the first block (two for k > 512; a block then adds about
    // k / blocks-seen keys per query to a 1024-key buffer).  A buffer that overflows anyway is detected
    // on the device and that (block, query) is redone from stored scores after the pass.
    probe.sel_state = static_cast<unsigned long long *>(keys);
    probe.sel_cnt = cnts;
    probe.sel_k = k;
    bool fused = ctx->topk_fused && ctx->gemm_impl == 0;
    if (fused && dt == DType::BF16) fused = gemm_tc_supported(probe, ctx->tune, nullptr);
    if (fused && dt == DType::F32) {
        GemmArgs g6;
        int64_t blk = 0;
        fused = split_wanted(ctx, dt, probe) && split_covers(ctx, probe, ctx->stream, g6, blk);
    }
    const int64_t warm = k <= TK_LIST / 2 ? 1 : 2;
    PS_CUDA(ctx, cudaMemsetAsync(keys, 0, topk_state_bytes(nq), ctx->stream));
    PS_CUDA(ctx, cudaMemsetAsync(any, 0, (size_t)n_blocks * 4, ctx->stream));
    auto block_args = [&](int64_t b, int64_t &nb, int64_t &nb_pad) {
        const int64_t c0 = b * NB;
        nb = std::min(NB, N - c0);
        nb_pad = (nb + 7) / 8 * 8;
        GemmArgs g;                                   // scores[nq x nb_pad] = Q Z[c0 .. c0+nb)^T, fp32
        g.M = nq; g.K1 = d; g.N = (int32_t)nb_pad; g.A1 = Q;
        g.B = static_cast<const char *>(Z) + (size_t)c0 * d * es;
        g.b_rows = nb;
        g.out = scores;
        g.out_f32 = 1;
        return g;
    };
    for (int64_t b = 0; b < n_blocks; ++b) {
        int64_t nb = 0, nb_pad = 0;
        GemmArgs g = block_args(b, nb, nb_pad);
        cudaError_t e;
        bool fb = fused && b >= warm;
        if (fb) {
            g.sel_state = static_cast<unsigned long long *>(keys);
            g.sel_cnt = cnts;
            g.sel_k = k;
            g.sel_id0 = b * NB;
            GemmArgs g6;
            int64_t blk = 0;
            fb = dt == DType::BF16 ? gemm_tc_supported(g, ctx->tune, nullptr)      // (a ragged last block)
                                   : split_wanted(ctx, dt, g) && split_covers(ctx, g, ctx->stream, g6, blk);
            if (!fb) g.sel_state = nullptr;
        }
        if (fb) {
            PS_TRY(run_gemm(ctx, dt, g, gscratch, scratch, ctx->stream));
            e = launch_topk_maintain(keys, nq, k, 3 * TK_LIST / 8, cnt_prev, ovf + (size_t)b * nq, any + b,
                                     ctx->stream, &ctx->launches);
        } else {
            PS_TRY(run_gemm(ctx, dt, g, gscratch, scratch, ctx->stream));
            e = launch_topk_merge(scores, nq, nb_pad, (int32_t)nb, b * NB, k, keys, nullptr, ctx->stream,
                                  &ctx->launches);
            // before a block that selects in the epilogue: merge every buffer, so that the k-th key is
            // that of everything seen so far (the scan leaves it as of its last in-kernel merge)
            if (e == cudaSuccess && fused && b + 1 >= warm && b + 1 < n_blocks)
                e = launch_topk_maintain(keys, nq, k, 0, cnt_prev, ovf + (size_t)b * nq, any + b, ctx->stream,
                                         &ctx->launches);
        }
        count_launches(ctx);
        PS_CUDA(ctx, e);
    }
    if (fused && n_blocks > warm) {                   // redo what overflowed (normally nothing)
        std::vector<int> any_h((size_t)n_blocks);
        PS_CUDA(ctx, cudaMemcpyAsync(any_h.data(), any, (size_t)n_blocks * 4, cudaMemcpyDeviceToHost, ctx->stream));
        PS_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
        for (int64_t b = warm; b < n_blocks; ++b) {
            if (!any_h[(size_t)b]) continue;
            int64_t nb = 0, nb_pad = 0;
            GemmArgs g = block_args(b, nb, nb_pad);
            PS_TRY(run_gemm(ctx, dt, g, gscratch, scratch, ctx->stream));
            cudaError_t e = launch_topk_merge(scores, nq, nb_pad, (int32_t)nb, b * NB, k, keys,
                                              ovf + (size_t)b * nq, ctx->stream, &ctx->launches);
            count_launches(ctx);
            PS_CUDA(ctx, e);
        }
    }
    cudaError_t e = launch_topk_finish(keys, nq, k, out_idx, out_score, ctx->stream, &ctx->launches);
    count_launches(ctx);
    PS_CUDA(ctx, e);
    return PINSAGE_OK;
}

pinsage_status pinsage_normalize_counts(pinsage_ctx *ctx, int64_t N, int32_t T,
                                        const int32_t *counts, float *nbr_w)
{
    if (!ctx) return PINSAGE_ERR_INVALID_ARG;
    DeviceGuard guard(ctx->device);
    PS_TRY(check_graph_args(ctx, N, T));
    PS_TRY(check_ptr(ctx, "counts", counts));
    PS_TRY(check_ptr(ctx, "nbr_w", nbr_w));
    cudaError_t e = launch_normalize_counts(N, T, counts, nbr_w, ctx->stream, &ctx->launches);
    count_launches(ctx);
    PS_CUDA(ctx, e);
    return PINSAGE_OK;
}

pinsage_status pinsage_build_neighbourhoods(pinsage_ctx *ctx, int64_t N, const int64_t *row_ptr,
                                            const int32_t *col_idx, int32_t n_walks, int32_t walk_len,
                                            int32_t T, uint64_t seed, int32_t *nbr_idx, int32_t *counts)
{
    if (!ctx) return PINSAGE_ERR_INVALID_ARG;
    DeviceGuard guard(ctx->device);
    PS_TRY(check_graph_args(ctx, N, T));
    if (n_walks < 1 || walk_len < 1)
        return fail(ctx, PINSAGE_ERR_INVALID_ARG, "n_walks = %d and walk_len = %d must be positive", n_walks, walk_len);
    if (walk_slots(n_walks, walk_len) == 0)
        return fail(ctx, PINSAGE_ERR_UNSUPPORTED_SHAPE, "n_walks * walk_len = %lld exceeds 2048",
                    (long long)n_walks * walk_len);
    PS_TRY(check_ptr(ctx, "row_ptr", row_ptr));
    PS_TRY(check_ptr(ctx, "nbr_idx", nbr_idx));
    PS_TRY(check_ptr(ctx, "counts", counts));
    // col_idx may be NULL for a graph without edges (it is then never dereferenced)
    cudaError_t e = launch_walk_neighbourhoods(N, row_ptr, col_idx, n_walks, walk_len, T, seed, nbr_idx,
                                               counts, ctx->stream, &ctx->launches);
    count_launches(ctx);
    PS_CUDA(ctx, e);
    return PINSAGE_OK;
}

pinsage_status pinsage_calibrate(pinsage_ctx *ctx, int32_t kind, const void *table, size_t table_bytes,
                                 int32_t row_bytes, int64_t n_dst, int32_t T, void *out, size_t out_bytes,
                                 int32_t reps, double *ms)
{
    if (!ctx) return PINSAGE_ERR_INVALID_ARG;
    DeviceGuard guard(ctx->device);
    if (!ms) return fail(ctx, PINSAGE_ERR_INVALID_ARG, "ms is NULL");
    *ms = 0.0;
    PS_TRY(check_ptr(ctx, "table", table));
    PS_TRY(check_ptr(ctx, "out", out));
    if (reps < 1 || reps > 1000) return fail(ctx, PINSAGE_ERR_INVALID_ARG, "reps = %d outside [1, 1000]", reps);
    int64_t n_src = 0;
    if (kind == 0) {
        if (table_bytes < 16 || out_bytes < (size_t)ctx->num_sms * 8 * 256 * 16)
            return fail(ctx, PINSAGE_ERR_INVALID_ARG, "calibrate m1: out needs %zu bytes",
                        (size_t)ctx->num_sms * 8 * 256 * 16);
    } else if (kind == 1) {
        if (row_bytes != 256 && row_bytes != 512 && row_bytes != 1024 && row_bytes != 2048)
            return fail(ctx, PINSAGE_ERR_UNSUPPORTED_SHAPE, "calibrate: row_bytes must be 256, 512, 1024 or 2048");
        n_src = (int64_t)(table_bytes / (size_t)row_bytes);
        if (n_src < 1 || n_src >= (1LL << 31) || n_dst < 1 || T < 1 || T > 1024)
            return fail(ctx, PINSAGE_ERR_INVALID_ARG, "calibrate: bad table size, n_dst or T");
        if (out_bytes < (size_t)n_dst * row_bytes)
            return fail(ctx, PINSAGE_ERR_INVALID_ARG, "calibrate: out needs n_dst x row_bytes bytes");
    } else {
        return fail(ctx, PINSAGE_ERR_INVALID_ARG, "calibrate: kind must be 0 (stream) or 1 (gather)");
    }
    cudaEvent_t e0, e1;
    PS_CUDA(ctx, cudaEventCreate(&e0));
    PS_CUDA(ctx, cudaEventCreate(&e1));
    cudaError_t e = cudaSuccess;
    for (int r = -1; r < reps && e == cudaSuccess; ++r) {          // one untimed warm-up launch
        if (r == 0) e = cudaEventRecord(e0, ctx->stream);
        if (e == cudaSuccess)
            e = launch_calib(kind, table, table_bytes, row_bytes, n_src, n_dst, T, out, ctx->num_sms, ctx->stream,
                             &ctx->launches);
    }
    if (e == cudaSuccess) e = cudaEventRecord(e1, ctx->stream);
    if (e == cudaSuccess) e = cudaEventSynchronize(e1);
    float t = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&t, e0, e1);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    count_launches(ctx);
    PS_CUDA(ctx, e);
    *ms = (double)t / reps;
    return PINSAGE_OK;
}

pinsage_status pinsage_validate_graph(pinsage_ctx *ctx, int64_t n_dst, int64_t n_src, int32_t T,
                                      const int32_t *nbr_idx, const float *nbr_w,
                                      int64_t *first_bad)
{
    if (!ctx) return PINSAGE_ERR_INVALID_ARG;
    DeviceGuard guard(ctx->device);
    if (!first_bad) return fail(ctx, PINSAGE_ERR_INVALID_ARG, "first_bad is NULL");
    *first_bad = -1;
    if (n_dst < 0) return fail(ctx, PINSAGE_ERR_INVALID_ARG, "n_dst is negative");
    PS_TRY(check_graph_args(ctx, n_src, T));
    if (n_dst == 0) return PINSAGE_OK;
    PS_TRY(check_ptr(ctx, "nbr_idx", nbr_idx));
    PS_TRY(check_ptr(ctx, "nbr_w", nbr_w));
    cudaError_t e = launch_validate(n_dst, n_src, T, nbr_idx, nbr_w, ctx->d_first_bad, ctx->stream,
                                    &ctx->launches);
    count_launches(ctx);
    PS_CUDA(ctx, e);
    long long bad = -1;
    PS_CUDA(ctx, cudaMemcpyAsync(&bad, ctx->d_first_bad, sizeof bad, cudaMemcpyDeviceToHost, ctx->stream));
    PS_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    *first_bad = bad;
    if (bad >= 0)
        return fail(ctx, PINSAGE_ERR_BAD_INDEX,
                    "entry %lld (node %lld, slot %lld) has an id outside [0, %lld) or a non-finite weight",
                    bad, bad / T, bad % T, (long long)n_src);
    return PINSAGE_OK;
}

}  // extern "C"

/*
 * pinsage_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * A plain, slow, obviously-correct fp64 CPU statement of what the PinSage
 * inference hot path computes, written from the paper text
 * (/root/reference/PAPER.md = arXiv 1806.01973).  Only tests/, bench.py's
 * cpu_baseline / --impl reference leg and __graft_entry__.smoke() may call it.
 * It shares no code, header, table or helper with the CUDA path under
 * paper_1806_01973_b200/csrc/ and neither includes the other.
 *
 * What is implemented (every function cites the passage it follows):
 *   Algorithm 1 CONVOLVE
 *     line 1: n_u = gamma({ReLU(Q h_v + q) | v in N(u)}, alpha)        :114
 *             gamma = importance pooling = weighted mean with the
 *             L1-normalised visit counts as weights                     :120-124
 *     line 2: z_u = ReLU(W concat(h_u, n_u) + w)   (self first)         :115
 *     line 3: z_u = z_u / ||z_u||_2                                     :116
 *   Stacking K layers, layer 0 = input features    PAPER.md:126, Alg.2 l.8-14 :155-164
 *   Head z_u = G2 ReLU(G1 h_u^(K) + g)             PAPER.md:166 (Alg.2 l.16), :130
 *   Layer-wise ("MapReduce") schedule: project every node once, then join
 *   + pool per destination                         PAPER.md:214-221 (sec. 3.4)
 *
 * Readings where the paper is silent / garbled:
 *   A2  alpha[v][t] = (float)c[v][t] / (float)(sum_t c[v][t]) in IEEE binary32,
 *       then used as given: the pool is a weighted SUM with weights summing to 1.
 *   A3  ||z|| == 0  ->  the zero row (no NaN).
 *   A5  concat order [h_u ; n_u]: the first d_in columns of W act on self.
 *   A6  head has one bias (g, on G1), no activation / normalisation after G2.
 *   A18 every matrix is stored "out x in" row-major, applied as M * vector.
 *
 * Parity pins (tests/test_oracle_pins.py, none of them re-types these loops):
 *   numpy fp64 relu(H @ Q.T + q) for the dense steps; scipy.sparse SpMM for the
 *   pool; hand-computed worked example (tests/golden/worked_example.txt);
 *   closed forms (identity layer, graph-free self-loop MLP, sparse power step,
 *   positive-scale invariance); invariants (unit rows, alpha rows sum to 1,
 *   neighbour-order and node-relabelling invariance, entry splitting);
 *   brute-force recursion over the K-hop tree == literal == layer-wise.
 *   Nothing here is "parity unpinned".
 *
 * All arrays are row-major double unless stated; indices are int32 in [0, N).
 * Build: gcc -O2 -std=c99 -ffp-contract=off -fopenmp -shared -fPIC (see oracle.py).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifdef _OPENMP
#include <omp.h>
#endif

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

static double relu(double x) { return x > 0.0 ? x : 0.0; }

/* y[j] = ReLU(sum_i M[j][i] x[i] + b[j]),  M is [rows x cols] "out x in".
 * b may be NULL (no bias); act = 0 disables the ReLU.                      */
static void affine(const double *M, const double *b, int rows, int cols,
                   const double *x, int act, double *y)
{
    for (int j = 0; j < rows; ++j) {
        double s = 0.0;
        for (int i = 0; i < cols; ++i)
            s += M[(size_t)j * cols + i] * x[i];
        if (b)
            s += b[j];
        y[j] = act ? relu(s) : s;
    }
}

/* PAPER.md:120-124 + reading A2.  counts [N x T] int32 -> alpha [N x T] float. */
void oracle_normalize_counts(int64_t N, int32_t T, const int32_t *counts, float *alpha)
{
    for (int64_t v = 0; v < N; ++v) {
        int64_t tot = 0;
        for (int t = 0; t < T; ++t)
            tot += counts[v * T + t];
        float ftot = (float)tot;
        for (int t = 0; t < T; ++t)   /* a node that visited nobody (reading B4) has all-zero weights */
            alpha[v * T + t] = tot > 0 ? (float)counts[v * T + t] / ftot : 0.0f;
    }
}

/*
 * Algorithm 1 CONVOLVE for ONE node, literally.
 *   h_u      [d_in]       current representation of u
 *   h_nbr    [T x d_in]   current representations of v_0..v_{T-1} in N(u)
 *   alpha    [T]          neighbour weights
 *   Q [m x d_in], q [m], W [d x (d_in+m)], w [d]
 *   out      [d]
 * scratch must hold 2*m + d_in + m doubles (p_t, n, concat).
 */
void oracle_convolve_node(int32_t T, int32_t d_in, int32_t m, int32_t d,
                          const double *h_u, const double *h_nbr, const double *alpha,
                          const double *Q, const double *q, const double *W, const double *w,
                          double *out, double *scratch)
{
    double *p = scratch;          /* [m]        */
    double *n = scratch + m;      /* [m]        */
    double *cat = scratch + 2 * m; /* [d_in + m] */
    for (int j = 0; j < m; ++j)
        n[j] = 0.0;
    /* line 1: project each neighbour through Q (ReLU inside, A19), weight, sum */
    for (int t = 0; t < T; ++t) {
        affine(Q, q, m, d_in, h_nbr + (size_t)t * d_in, 1, p);
        for (int j = 0; j < m; ++j)
            n[j] += alpha[t] * p[j];
    }
    /* line 2: concat(self, neighbourhood), W, ReLU */
    for (int i = 0; i < d_in; ++i)
        cat[i] = h_u[i];
    for (int j = 0; j < m; ++j)
        cat[d_in + j] = n[j];
    affine(W, w, d, d_in + m, cat, 1, out);
    /* line 3: L2 normalise (A3: zero row stays zero) */
    double ss = 0.0;
    for (int j = 0; j < d; ++j)
        ss += out[j] * out[j];
    double nrm = sqrt(ss);
    if (nrm > 0.0)
        for (int j = 0; j < d; ++j)
            out[j] /= nrm;
}

/* Mode A: one layer, literal Algorithm 1 applied node by node over all N nodes
 * (every neighbour projection is recomputed for every (u,t) occurrence).     */
void oracle_layer_literal(int64_t N, int32_t T, int32_t d_in, int32_t m, int32_t d,
                          const double *H, const int32_t *idx, const float *alpha,
                          const double *Q, const double *q, const double *W, const double *w,
                          double *out)
{
#pragma omp parallel
    {
        double *scratch = (double *)malloc(sizeof(double) * (size_t)(3 * m + d_in));
        double *nbr = (double *)malloc(sizeof(double) * (size_t)T * d_in);
        double *a = (double *)malloc(sizeof(double) * (size_t)T);
#pragma omp for schedule(static)
        for (int64_t u = 0; u < N; ++u) {
            for (int t = 0; t < T; ++t) {
                memcpy(nbr + (size_t)t * d_in, H + (size_t)idx[u * T + t] * d_in,
                       sizeof(double) * (size_t)d_in);
                a[t] = (double)alpha[u * T + t];
            }
            oracle_convolve_node(T, d_in, m, d, H + (size_t)u * d_in, nbr, a, Q, q, W, w,
                                 out + (size_t)u * d, scratch);
        }
        free(scratch);
        free(nbr);
        free(a);
    }
}

/* S1 (PAPER.md:114 dense part; sec. 3.4 job 1 :218): P[v] = ReLU(Q H[v] + q), once per node.
 * Also serves the head's dense layers (act / bias switchable).                */
void oracle_dense(int64_t N, int32_t d_in, int32_t d_out, const double *H,
                  const double *M, const double *b, int32_t act, double *P)
{
#pragma omp parallel for schedule(static)
    for (int64_t v = 0; v < N; ++v)
        affine(M, b, d_out, d_in, H + (size_t)v * d_in, act, P + (size_t)v * d_out);
}

/* S2 (PAPER.md:114 gamma, :124; sec. 3.4 job 2 :219): n[v] = sum_t alpha[v][t] * P[idx[v][t]]. */
void oracle_pool(int64_t N, int32_t T, int32_t m, const double *P,
                 const int32_t *idx, const float *alpha, double *n)
{
#pragma omp parallel for schedule(static)
    for (int64_t v = 0; v < N; ++v) {
        double *nv = n + (size_t)v * m;
        for (int j = 0; j < m; ++j)
            nv[j] = 0.0;
        for (int t = 0; t < T; ++t) {
            const double *pr = P + (size_t)idx[v * T + t] * m;
            double a = (double)alpha[v * T + t];
            for (int j = 0; j < m; ++j)
                nv[j] += a * pr[j];
        }
    }
}

/* The ablation aggregators of PAPER.md:262-263 (gamma "e.g., a element-wise mean or weighted sum",
 * :118): gamma = 1 element-wise MEAN of the T projected neighbour rows (weights unused),
 * gamma = 2 element-wise MAX.  gamma = 0 is importance pooling (oracle_pool).  alpha may be NULL
 * for gamma != 0.  T >= 1. */
void oracle_pool_gamma(int64_t N, int32_t T, int32_t m, const double *P, const int32_t *idx,
                       const float *alpha, int32_t gamma, double *n)
{
    if (gamma == 0) {
        oracle_pool(N, T, m, P, idx, alpha, n);
        return;
    }
#pragma omp parallel for schedule(static)
    for (int64_t v = 0; v < N; ++v) {
        double *nv = n + (size_t)v * m;
        const double *p0 = P + (size_t)idx[v * T] * m;
        for (int j = 0; j < m; ++j)
            nv[j] = p0[j];
        for (int t = 1; t < T; ++t) {
            const double *pr = P + (size_t)idx[v * T + t] * m;
            for (int j = 0; j < m; ++j) {
                if (gamma == 1)
                    nv[j] += pr[j];
                else if (pr[j] > nv[j])
                    nv[j] = pr[j];
            }
        }
        if (gamma == 1)
            for (int j = 0; j < m; ++j)
                nv[j] /= (double)T;
    }
}

/* S3: out[v] = normalise(ReLU(W concat(H[v], n[v]) + w)). */
void oracle_combine(int64_t N, int32_t d_in, int32_t m, int32_t d,
                    const double *H, const double *n, const double *W, const double *w,
                    double *out)
{
#pragma omp parallel
    {
        double *cat = (double *)malloc(sizeof(double) * (size_t)(d_in + m));
#pragma omp for schedule(static)
        for (int64_t v = 0; v < N; ++v) {
            double *o = out + (size_t)v * d;
            memcpy(cat, H + (size_t)v * d_in, sizeof(double) * (size_t)d_in);
            memcpy(cat + d_in, n + (size_t)v * m, sizeof(double) * (size_t)m);
            affine(W, w, d, d_in + m, cat, 1, o);
            double ss = 0.0;
            for (int j = 0; j < d; ++j)
                ss += o[j] * o[j];
            double nrm = sqrt(ss);
            if (nrm > 0.0)
                for (int j = 0; j < d; ++j)
                    o[j] /= nrm;
        }
        free(cat);
    }
}

/* Mode B: one layer in the layer-wise schedule of sec. 3.4:
 * project every node once, then pool + combine per destination.  Same per-output
 * arithmetic and loop order as the literal form, so the two agree bit for bit.
 * P_ws [N x m] and n_ws [N x m] are caller-provided workspaces.               */
void oracle_layer_layerwise(int64_t N, int32_t T, int32_t d_in, int32_t m, int32_t d,
                            const double *H, const int32_t *idx, const float *alpha,
                            const double *Q, const double *q, const double *W, const double *w,
                            double *out, double *P_ws, double *n_ws)
{
    oracle_dense(N, d_in, m, H, Q, q, 1, P_ws);
    oracle_pool(N, T, m, P_ws, idx, alpha, n_ws);
    oracle_combine(N, d_in, m, d, H, n_ws, W, w, out);
}

/* Head (Alg. 2 l.16; A6): out[v] = G2 ReLU(G1 h[v] + g). */
void oracle_head(int64_t N, int32_t d, int32_t g1, int32_t d_out, const double *H,
                 const double *G1, const double *g, const double *G2, double *out)
{
#pragma omp parallel
    {
        double *a = (double *)malloc(sizeof(double) * (size_t)g1);
#pragma omp for schedule(static)
        for (int64_t v = 0; v < N; ++v) {
            affine(G1, g, g1, d, H + (size_t)v * d, 1, a);
            affine(G2, NULL, d_out, g1, a, 0, out + (size_t)v * d_out);
        }
        free(a);
    }
}

/*
 * Mode R: brute-force recursion over the K-hop computation tree (Fig. 1,
 * PAPER.md:39; Alg. 2 l.8-14 with no sharing of any intermediate):
 *   rec(u,0) = x_u ;  rec(u,k) = CONVOLVE_k(rec(u,k-1), {rec(v_t,k-1)}).
 * Cost O(T^K) per node: tiny inputs only.
 * dims[0..K] = d_0, d_1, ..., d_K ; ms[k-1] = m of layer k;
 * Qs/qs/Ws/ws are arrays of K pointers.  out [dims[k]].
 */
void oracle_rec(int64_t u, int32_t k, int32_t T, const int32_t *dims, const int32_t *ms,
                const double *X, const int32_t *idx, const float *alpha,
                const double *const *Qs, const double *const *qs,
                const double *const *Ws, const double *const *ws, double *out)
{
    if (k == 0) {
        memcpy(out, X + (size_t)u * dims[0], sizeof(double) * (size_t)dims[0]);
        return;
    }
    int32_t d_in = dims[k - 1], d = dims[k], m = ms[k - 1];
    double *h_u = (double *)malloc(sizeof(double) * (size_t)d_in);
    double *nbr = (double *)malloc(sizeof(double) * (size_t)T * d_in);
    double *a = (double *)malloc(sizeof(double) * (size_t)T);
    double *scratch = (double *)malloc(sizeof(double) * (size_t)(3 * m + d_in));
    oracle_rec(u, k - 1, T, dims, ms, X, idx, alpha, Qs, qs, Ws, ws, h_u);
    for (int t = 0; t < T; ++t) {
        oracle_rec(idx[u * T + t], k - 1, T, dims, ms, X, idx, alpha, Qs, qs, Ws, ws,
                   nbr + (size_t)t * d_in);
        a[t] = (double)alpha[u * T + t];
    }
    oracle_convolve_node(T, d_in, m, d, h_u, nbr, a, Qs[k - 1], qs[k - 1], Ws[k - 1], ws[k - 1],
                         out, scratch);
    free(h_u);
    free(nbr);
    free(a);
    free(scratch);
}

/* ---------------------------------------------------------------------------------------------
 * Importance-based neighbourhoods: "we simulate random walks starting from
 * node u and compute the L1-normalized visit count of nodes visited by the random walk.  The
 * neighborhood of u is then defined as the top T nodes with the highest normalized visit counts".
 * The paper gives no walk parameters (it cites Pixie [14]); readings B1-B5 of DESIGN.md:
 *   B1 the graph is a CSR adjacency (row_ptr [N+1] int64, col_idx [E] int32), any ids in [0, N);
 *   B2 n_walks walks per node, each restarting at u and taking walk_len steps to a uniformly
 *      chosen out-neighbour of the current node; a node without out-neighbours ends the walk;
 *   B3 every arrival at a node v != u is one visit (u is never its own neighbour);
 *   B4 keep the T most visited, ties to the smaller id, in that order; fewer than T distinct
 *      visited nodes: pad with id u and count 0 (weight 0, reading A7);
 *   B5 randomness is counter-based, a function of (seed, u, walk, step) only:
 *      key = mix(seed + 0x100000001B3 * u), x = mix(key ^ (walk << 32 | step)), mix = the
 *      splitmix64 finaliser; choice = ((x >> 32) * degree) >> 32.
 * counts are the raw integer visit counts; the L1 normalisation is oracle_normalize_counts.
 * -------------------------------------------------------------------------------------------- */
static uint64_t walk_mix(uint64_t z)
{
    z += 0x9E3779B97F4A7C15ULL;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}

static int cmp_i32(const void *a, const void *b)
{
    int32_t x = *(const int32_t *)a, y = *(const int32_t *)b;
    return (x > y) - (x < y);
}

typedef struct { int32_t id, count; } visit_t;

static int cmp_visit(const void *a, const void *b)   /* count descending, then id ascending */
{
    const visit_t *x = (const visit_t *)a, *y = (const visit_t *)b;
    if (x->count != y->count) return (x->count < y->count) - (x->count > y->count);
    return (x->id > y->id) - (x->id < y->id);
}

void oracle_walk_neighbourhoods(int64_t N, const int64_t *row_ptr, const int32_t *col_idx,
                                int32_t n_walks, int32_t walk_len, int32_t T, uint64_t seed,
                                int32_t *nbr_idx, int32_t *counts)
{
#pragma omp parallel
    {
        int32_t *seen = (int32_t *)malloc(sizeof(int32_t) * (size_t)n_walks * walk_len + 4);
        visit_t *vis = (visit_t *)malloc(sizeof(visit_t) * ((size_t)n_walks * walk_len + 1));
#pragma omp for schedule(dynamic, 64)
        for (int64_t u = 0; u < N; ++u) {
            const uint64_t key = walk_mix(seed + 0x100000001B3ULL * (uint64_t)u);
            size_t ns = 0;
            for (int32_t r = 0; r < n_walks; ++r) {
                int64_t cur = u;
                for (int32_t s = 0; s < walk_len; ++s) {
                    const int64_t beg = row_ptr[cur], deg = row_ptr[cur + 1] - beg;
                    if (deg <= 0) break;                                         /* B2 */
                    const uint64_t x = walk_mix(key ^ (((uint64_t)r << 32) | (uint64_t)s));
                    const uint64_t pick = ((x >> 32) * (uint64_t)deg) >> 32;     /* B5 */
                    cur = col_idx[beg + (int64_t)pick];
                    if (cur != u) seen[ns++] = (int32_t)cur;                     /* B3 */
                }
            }
            qsort(seen, ns, sizeof(int32_t), cmp_i32);
            size_t nv = 0;
            for (size_t i = 0; i < ns;) {
                size_t j = i;
                while (j < ns && seen[j] == seen[i]) ++j;
                vis[nv].id = seen[i];
                vis[nv].count = (int32_t)(j - i);
                ++nv;
                i = j;
            }
            qsort(vis, nv, sizeof(visit_t), cmp_visit);                          /* B4 */
            for (int32_t t = 0; t < T; ++t) {
                nbr_idx[u * T + t] = (size_t)t < nv ? vis[t].id : (int32_t)u;
                counts[u * T + t] = (size_t)t < nv ? vis[t].count : 0;
            }
        }
        free(seen);
        free(vis);
    }
}

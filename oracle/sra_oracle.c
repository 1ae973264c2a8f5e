/* CPU fp64 oracle for Sparse Reference Attention (SRA), plain C.   *** TEST INFRASTRUCTURE ***
 *
 * Same definition as oracle/sra_oracle.py (mask reading in
 * SURVEY.md section 8c / DESIGN.md), written as scalar loops so that it is affordable at the
 * paper-sized workloads: every output row depends only on its own Q row and the K/V rows it
 * may see, so computing a *subset* of rows (or of key columns, for dK/dV) is exact, not an
 * approximation.  The mask is the predicate is_visible(i, j) below - it knows nothing about
 * tiles or schedules.  Everything is fp64; bf16 inputs are upcast exactly; no intermediate is
 * rounded; no blocking, fusion or reordering beyond "for each row, for each visible key".
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may load this.  It shares no code with the CUDA path.
 *
 * Two optional restrictions of the mask, the same readings as oracle/sra_oracle.py (A8, A12, A17):
 *   valid[]  ("skip invalid reference tokens"): an invalid reference token is nobody's key and its
 *            own row is empty (O = 0, LSE = -inf, zero gradients); one flag array per context or one per batch item;
 *   frames + window ("restricts each frame's receptive field to a local neighborhood"): a generation
 *            row of frame f sees only the generation keys of frames [f - w, f + w] (and every reference key).
 *
 * Row/column index convention: global index t in [0, Ng+Nr): t < Ng is generation token t,
 * otherwise reference token t-Ng.  Tensors are [B, N, H, d] bf16 bit patterns, d contiguous.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

static double bf16_to_f64(uint16_t b) {
    uint32_t u = ((uint32_t)b) << 16;
    float f;
    memcpy(&f, &u, 4);
    return (double)f;
}

/* block(t) = k with off[k] <= t < off[k+1]  (t is a reference-token index) */
static int block_of(int t, const int32_t* off, int n_blk) {
    for (int k = 0; k < n_blk; ++k)
        if (off[k] <= t && t < off[k + 1]) return k;
    return -1;
}

/* Optional restrictions of the mask (NULL / window < 0 = absent). */
typedef struct {
    const uint8_t* valid;   /* Nr flags of the current batch item, or NULL */
    const int32_t* fr;      /* n_fr + 1 generation frame offsets, or NULL */
    int n_fr, window;
} mask_opt_t;

/* The SRA mask M[i][j]:  G rows see G u R;  R rows see only their own R block.
 * With valid[]: an invalid reference token loses its column and its row.  With a window: G -> G only
 * between frames at distance <= window. */
static int is_visible(int i, int j, int Ng, const int32_t* off, int n_blk, const mask_opt_t* m) {
    if (m && m->valid) {
        if (i >= Ng && !m->valid[i - Ng]) return 0;
        if (j >= Ng && !m->valid[j - Ng]) return 0;
    }
    if (i < Ng) {
        if (j < Ng && m && m->fr && m->window >= 0) {
            int d = block_of(i, m->fr, m->n_fr) - block_of(j, m->fr, m->n_fr);
            if (d < 0) d = -d;
            return d <= m->window;
        }
        return 1;
    }
    if (j < Ng) return 0;
    return block_of(i - Ng, off, n_blk) == block_of(j - Ng, off, n_blk);
}

typedef struct {
    int B, H, d, Ng, Nr, n_blk;
    const int32_t* off;
    double scale;
    mask_opt_t m;
} shape_t;

/* fp64 copy of one (b,h) slice of a [G ; R] pair of tensors -> [Ng+Nr][d] */
static double* load_head(const uint16_t* gen, const uint16_t* ref, const shape_t* s, int b, int h) {
    int n = s->Ng + s->Nr, d = s->d;
    double* x = (double*)malloc((size_t)n * d * sizeof(double));
    if (!x) return NULL;
    for (int t = 0; t < n; ++t) {
        const uint16_t* src;
        if (t < s->Ng) src = gen ? gen + (((size_t)b * s->Ng + t) * s->H + h) * d : NULL;
        else           src = ref ? ref + (((size_t)b * s->Nr + (t - s->Ng)) * s->H + h) * d : NULL;
        for (int c = 0; c < d; ++c) x[(size_t)t * d + c] = src ? bf16_to_f64(src[c]) : 0.0;
    }
    return x;
}

static double dot(const double* a, const double* b, int d) {
    double acc = 0.0;
    for (int c = 0; c < d; ++c) acc += a[c] * b[c];
    return acc;
}

/* One output row: O_i = sum_j P_ij V_j,  LSE_i = max + log(sum), over visible j.  s_buf: n doubles.
 * A row with no visible key (an invalid reference token, reading A8) gives O = 0, LSE = -inf. */
static void forward_row(int i, const double* Q, const double* K, const double* V, const shape_t* s,
                        double* s_buf, double* o_row, double* lse) {
    int n = s->Ng + s->Nr, d = s->d;
    double mx = -INFINITY;
    int seen = 0;
    for (int j = 0; j < n; ++j) {
        if (!is_visible(i, j, s->Ng, s->off, s->n_blk, &s->m)) continue;
        s_buf[j] = s->scale * dot(Q + (size_t)i * d, K + (size_t)j * d, d);
        if (s_buf[j] > mx) mx = s_buf[j];
        seen = 1;
    }
    for (int c = 0; c < d; ++c) o_row[c] = 0.0;
    if (!seen) { *lse = -INFINITY; return; }
    double z = 0.0;
    for (int j = 0; j < n; ++j) {
        if (!is_visible(i, j, s->Ng, s->off, s->n_blk, &s->m)) continue;
        double e = exp(s_buf[j] - mx);
        z += e;
        for (int c = 0; c < d; ++c) o_row[c] += e * V[(size_t)j * d + c];
    }
    for (int c = 0; c < d; ++c) o_row[c] /= z;
    *lse = mx + log(z);
}

int sra_oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* mask options of batch item b: valid is [Nr] (valid_batch_stride == 0, shared by the batch) or [B][Nr]
 * (valid_batch_stride == Nr, one mask per batch item - reading A12) */
static mask_opt_t mask_of(const uint8_t* valid, int valid_batch_stride, const int32_t* fr, int n_fr, int window, int b) {
    mask_opt_t m;
    m.valid = valid ? valid + (size_t)b * valid_batch_stride : NULL;
    m.fr = (fr && window >= 0) ? fr : NULL;
    m.n_fr = n_fr;
    m.window = window;
    return m;
}

/* Forward for a list of rows, all batches and heads.
 * o_out [B][n_rows][H][d] fp64, lse_out [B][H][n_rows] fp64.  q_ref may be NULL iff no row >= Ng.
 * valid / fr / window: optional mask restrictions (see is_visible); NULL, NULL, -1 = plain SRA. */
int sra_oracle_forward_rows_ex(const uint16_t* q_gen, const uint16_t* k_gen, const uint16_t* v_gen,
                               const uint16_t* q_ref, const uint16_t* k_ref, const uint16_t* v_ref,
                               int B, int H, int d, int Ng, int Nr, const int32_t* off, int n_blk,
                               double scale, const int32_t* rows, int n_rows,
                               const uint8_t* valid, int valid_batch_stride, const int32_t* fr, int n_fr, int window,
                               double* o_out, double* lse_out) {
    shape_t s = {B, H, d, Ng, Nr, n_blk, off, scale, {NULL, NULL, 0, -1}};
    int n = Ng + Nr;
    for (int r = 0; r < n_rows; ++r) {
        if (rows[r] < 0 || rows[r] >= n) return -1;
        if (rows[r] >= Ng && !q_ref) return -1;
    }
    int err = 0;
    for (int b = 0; b < B; ++b) {
        s.m = mask_of(valid, valid_batch_stride, fr, n_fr, window, b);
        for (int h = 0; h < H; ++h) {
            double* Q = load_head(q_gen, q_ref, &s, b, h);
            double* K = load_head(k_gen, k_ref, &s, b, h);
            double* V = load_head(v_gen, v_ref, &s, b, h);
            if (!Q || !K || !V) { free(Q); free(K); free(V); return -2; }
#pragma omp parallel
            {
                double* s_buf = (double*)malloc((size_t)n * sizeof(double));
                if (!s_buf) {
#pragma omp atomic write
                    err = -2;
                } else {
#pragma omp for schedule(dynamic, 1)
                    for (int r = 0; r < n_rows; ++r) {
                        double* o_row = o_out + (((size_t)b * n_rows + r) * H + h) * d;
                        forward_row(rows[r], Q, K, V, &s, s_buf, o_row,
                                    lse_out + ((size_t)b * H + h) * n_rows + r);
                    }
                    free(s_buf);
                }
            }
            free(Q); free(K); free(V);
        }
    }
    return err;
}

int sra_oracle_forward_rows(const uint16_t* q_gen, const uint16_t* k_gen, const uint16_t* v_gen,
                            const uint16_t* q_ref, const uint16_t* k_ref, const uint16_t* v_ref,
                            int B, int H, int d, int Ng, int Nr, const int32_t* off, int n_blk,
                            double scale, const int32_t* rows, int n_rows,
                            double* o_out, double* lse_out) {
    return sra_oracle_forward_rows_ex(q_gen, k_gen, v_gen, q_ref, k_ref, v_ref, B, H, d, Ng, Nr, off, n_blk, scale,
                                      rows, n_rows, NULL, 0, NULL, 0, -1, o_out, lse_out);
}

/* Full forward of ONE (b,h): o [n][d], lse [n]  (n = Ng+Nr, rows [G ; R]). */
int sra_oracle_forward_head_ex(const uint16_t* q_gen, const uint16_t* k_gen, const uint16_t* v_gen,
                               const uint16_t* q_ref, const uint16_t* k_ref, const uint16_t* v_ref,
                               int B, int H, int d, int Ng, int Nr, const int32_t* off, int n_blk,
                               double scale, int b, int h,
                               const uint8_t* valid, int valid_batch_stride, const int32_t* fr, int n_fr, int window,
                               double* o, double* lse) {
    shape_t s = {B, H, d, Ng, Nr, n_blk, off, scale, {NULL, NULL, 0, -1}};
    s.m = mask_of(valid, valid_batch_stride, fr, n_fr, window, b);
    int n = Ng + Nr, err = 0;
    double* Q = load_head(q_gen, q_ref, &s, b, h);
    double* K = load_head(k_gen, k_ref, &s, b, h);
    double* V = load_head(v_gen, v_ref, &s, b, h);
    if (!Q || !K || !V) { free(Q); free(K); free(V); return -2; }
#pragma omp parallel
    {
        double* s_buf = (double*)malloc((size_t)n * sizeof(double));
        if (!s_buf) {
#pragma omp atomic write
            err = -2;
        } else {
#pragma omp for schedule(dynamic, 16)
            for (int i = 0; i < n; ++i) forward_row(i, Q, K, V, &s, s_buf, o + (size_t)i * d, lse + i);
            free(s_buf);
        }
    }
    free(Q); free(K); free(V);
    return err;
}

int sra_oracle_forward_head(const uint16_t* q_gen, const uint16_t* k_gen, const uint16_t* v_gen,
                            const uint16_t* q_ref, const uint16_t* k_ref, const uint16_t* v_ref,
                            int B, int H, int d, int Ng, int Nr, const int32_t* off, int n_blk,
                            double scale, int b, int h, double* o, double* lse) {
    return sra_oracle_forward_head_ex(q_gen, k_gen, v_gen, q_ref, k_ref, v_ref, B, H, d, Ng, Nr, off, n_blk, scale, b, h,
                                      NULL, 0, NULL, 0, -1, o, lse);
}

/* Backward of ONE (b,h), for a subset of query rows (dQ) and a subset of key columns (dK, dV).
 *   D_i = sum_c dO_ic O_ic;  P_ij = exp(S_ij - LSE_i);  dP_ij = dO_i . V_j;  dS_ij = P_ij (dP_ij - D_i)
 *   dQ_i = s sum_j dS_ij K_j;   dK_j = s sum_i dS_ij Q_i;   dV_j = sum_i P_ij dO_i     (visible pairs only)
 * o/lse are the full-head forward results from sra_oracle_forward_head[_ex] under the SAME mask options (every row
 * that sees a requested key needs its own LSE and D).  rows/cols are global indices; dq [n_rows][d], dk/dv [n_cols][d].
 * Pass rows == NULL && n_rows == n (resp. cols) for "all".  Empty rows and invisible keys get zero gradients. */
int sra_oracle_backward_head_ex(const uint16_t* q_gen, const uint16_t* k_gen, const uint16_t* v_gen,
                                const uint16_t* q_ref, const uint16_t* k_ref, const uint16_t* v_ref,
                                const uint16_t* do_gen, const uint16_t* do_ref,
                                int B, int H, int d, int Ng, int Nr, const int32_t* off, int n_blk,
                                double scale, int b, int h, const double* o, const double* lse,
                                const int32_t* rows, int n_rows, const int32_t* cols, int n_cols,
                                const uint8_t* valid, int valid_batch_stride, const int32_t* fr, int n_fr, int window,
                                double* dq, double* dk, double* dv) {
    shape_t s = {B, H, d, Ng, Nr, n_blk, off, scale, {NULL, NULL, 0, -1}};
    s.m = mask_of(valid, valid_batch_stride, fr, n_fr, window, b);
    const mask_opt_t* m = &s.m;
    int n = Ng + Nr;
    double* Q = load_head(q_gen, q_ref, &s, b, h);
    double* K = load_head(k_gen, k_ref, &s, b, h);
    double* V = load_head(v_gen, v_ref, &s, b, h);
    double* dO = load_head(do_gen, do_ref, &s, b, h);
    double* D = (double*)malloc((size_t)n * sizeof(double));
    if (!Q || !K || !V || !dO || !D) { free(Q); free(K); free(V); free(dO); free(D); return -2; }
#pragma omp parallel for schedule(static)
    for (int i = 0; i < n; ++i) D[i] = dot(dO + (size_t)i * d, o + (size_t)i * d, d);

#pragma omp parallel for schedule(dynamic, 1)
    for (int r = 0; r < n_rows; ++r) {
        int i = rows ? rows[r] : r;
        double* dq_row = dq + (size_t)r * d;
        for (int c = 0; c < d; ++c) dq_row[c] = 0.0;
        for (int j = 0; j < n; ++j) {
            if (!is_visible(i, j, Ng, off, n_blk, m)) continue;
            double p = exp(scale * dot(Q + (size_t)i * d, K + (size_t)j * d, d) - lse[i]);
            double dp = dot(dO + (size_t)i * d, V + (size_t)j * d, d);
            double ds = p * (dp - D[i]);
            for (int c = 0; c < d; ++c) dq_row[c] += scale * ds * K[(size_t)j * d + c];
        }
    }
#pragma omp parallel for schedule(dynamic, 1)
    for (int r = 0; r < n_cols; ++r) {
        int j = cols ? cols[r] : r;
        double* dk_row = dk + (size_t)r * d;
        double* dv_row = dv + (size_t)r * d;
        for (int c = 0; c < d; ++c) { dk_row[c] = 0.0; dv_row[c] = 0.0; }
        for (int i = 0; i < n; ++i) {
            if (!is_visible(i, j, Ng, off, n_blk, m)) continue;
            double p = exp(scale * dot(Q + (size_t)i * d, K + (size_t)j * d, d) - lse[i]);
            double dp = dot(dO + (size_t)i * d, V + (size_t)j * d, d);
            double ds = p * (dp - D[i]);
            for (int c = 0; c < d; ++c) {
                dv_row[c] += p * dO[(size_t)i * d + c];
                dk_row[c] += scale * ds * Q[(size_t)i * d + c];
            }
        }
    }
    free(Q); free(K); free(V); free(dO); free(D);
    return 0;
}

int sra_oracle_backward_head(const uint16_t* q_gen, const uint16_t* k_gen, const uint16_t* v_gen,
                             const uint16_t* q_ref, const uint16_t* k_ref, const uint16_t* v_ref,
                             const uint16_t* do_gen, const uint16_t* do_ref,
                             int B, int H, int d, int Ng, int Nr, const int32_t* off, int n_blk,
                             double scale, int b, int h, const double* o, const double* lse,
                             const int32_t* rows, int n_rows, const int32_t* cols, int n_cols,
                             double* dq, double* dk, double* dv) {
    return sra_oracle_backward_head_ex(q_gen, k_gen, v_gen, q_ref, k_ref, v_ref, do_gen, do_ref, B, H, d, Ng, Nr, off,
                                       n_blk, scale, b, h, o, lse, rows, n_rows, cols, n_cols, NULL, 0, NULL, 0, -1,
                                       dq, dk, dv);
}

/* pairs = number of (i,j) with M[i][j]=1, counted by enumeration of the predicate (for small n) */
long long sra_oracle_count_pairs_ex(int Ng, int Nr, const int32_t* off, int n_blk, const uint8_t* valid,
                                    const int32_t* fr, int n_fr, int window) {
    mask_opt_t m = mask_of(valid, 0, fr, n_fr, window, 0);
    long long cnt = 0;
    int n = Ng + Nr;
    for (int i = 0; i < n; ++i)
        for (int j = 0; j < n; ++j) cnt += is_visible(i, j, Ng, off, n_blk, &m);
    return cnt;
}

long long sra_oracle_count_pairs(int Ng, int Nr, const int32_t* off, int n_blk) {
    return sra_oracle_count_pairs_ex(Ng, Nr, off, n_blk, NULL, NULL, 0, -1);
}

/*
 * qp_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU fp64 implementation of stage I of QuickProbs 2 ("Posterior
 * probability matrices are calculated for all sequence pairs on the basis of hidden Markov model and partition
 * function. The matrices are further employed to establish maximum expected accuracy alignments. Alignment
 * scores are used to estimate pairwise distances"), PAPER.md:59 (sparse form) and PAPER.md:69 (the partition
 * function uses a substitution matrix, gap penalties and a temperature).
 *
 * The paper prints no recurrence, so each function follows the reading fixed in SURVEY.md section 8(c)
 * (repeated in DESIGN.md "Readings"): c-1 the generic weighted pair automaton in natural-log space, c-2 the
 * root-mean-square combination, the threshold, the max-plus expected-accuracy recurrence and the distance.
 * The method reaches an exact result (posterior marginals of two fully specified models), so this file is that
 * definition written out: textbook O(n*m) log-space forward/backward, no blocking, no scaling tricks, no
 * reordering. It shares no code with the CUDA path (paper_1512_07437_b200/csrc) and must only be used by
 * tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs.
 *
 * Pins (tests/test_oracle_pins.py): brute-force path enumeration (n,m <= 5), logZ_f == logZ_b, per-row
 * marginal identity over all state planes, transposition symmetry, 1x1 and 1x2 closed forms, background
 * normalisation invariance, PF reversal symmetry, T->0 limit against textbook Gotoh, MEA brute force.
 * Parity unpinned against the paper itself: the constants, the RMS rule, tau and the distance formula are
 * readings (SURVEY.md 8(c) c-4 #1,#6,#7,#9) -- no QuickProbs binary or dataset is available.
 *
 * OpenMP is used only across independent pairs in qpo_run (schedule(dynamic)); every per-pair routine is serial.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define QPO_MAX_INS 2

typedef struct {
    int32_t n_ins;            /* G: 1 or 2                                   */
    int32_t alphabet;         /* A                                           */
    const double *log_match;  /* A*A natural-log match weights lm[a][b]      */
    const double *log_ins;    /* A   natural-log insert weights lx[a]=ly[a]  */
    double t_MM, t_MI[QPO_MAX_INS], t_II[QPO_MAX_INS], t_IM[QPO_MAX_INS];
    double init_M, init_I[QPO_MAX_INS], end_M, end_I[QPO_MAX_INS];
} qpo_model;

static const double NEG_INF = -INFINITY;

/* a (+) b = log(exp a + exp b), with log 0 = -inf handled explicitly */
static double lse(double a, double b)
{
    if (a == NEG_INF) return b;
    if (b == NEG_INF) return a;
    double hi = a > b ? a : b, lo = a > b ? b : a;
    return hi + log1p(exp(lo - hi));
}

/* plane index helpers: planes are (n+1) x (m+1), state order M, X_1..X_G, Y_1..Y_G */
#define IDX(i, j) ((size_t)(i) * (size_t)(m + 1) + (size_t)(j))

int qpo_num_states(const qpo_model *mdl) { return 1 + 2 * mdl->n_ins; }

/*
 * Forward recurrence, SURVEY.md 8(c) c-1:
 *   F_M (i,j) = lm[x_i][y_j] + ( [i=1,j=1] init_M (+) t_MM + F_M(i-1,j-1)
 *                                (+)_g t_IM[g] + F_Xg(i-1,j-1)  (+)_g t_IM[g] + F_Yg(i-1,j-1) ),  -inf if i=0 or j=0
 *   F_Xg(i,j) = lx[x_i] + ( [i=1,j=0] init_I[g] (+) t_MI[g] + F_M(i-1,j) (+) t_II[g] + F_Xg(i-1,j) ),  -inf if i=0
 *   F_Yg(i,j) = ly[y_j] + ( [i=0,j=1] init_I[g] (+) t_MI[g] + F_M(i,j-1) (+) t_II[g] + F_Yg(i,j-1) ),  -inf if j=0
 *   logZ_f    = (+)_s F_s(n,m) + end_s
 * F holds S planes; returns logZ_f.
 */
double qpo_forward(const qpo_model *mdl, const uint8_t *x, int n, const uint8_t *y, int m, double *F)
{
    const int G = mdl->n_ins, A = mdl->alphabet;
    const size_t pl = (size_t)(n + 1) * (size_t)(m + 1);
    double *FM = F;
    for (int i = 0; i <= n; ++i) {
        for (int j = 0; j <= m; ++j) {
            /* M */
            double v = NEG_INF;
            if (i >= 1 && j >= 1) {
                double acc = (i == 1 && j == 1) ? mdl->init_M : NEG_INF;
                acc = lse(acc, mdl->t_MM + FM[IDX(i - 1, j - 1)]);
                for (int g = 0; g < G; ++g) {
                    acc = lse(acc, mdl->t_IM[g] + F[(1 + g) * pl + IDX(i - 1, j - 1)]);
                    acc = lse(acc, mdl->t_IM[g] + F[(1 + G + g) * pl + IDX(i - 1, j - 1)]);
                }
                v = mdl->log_match[(size_t)x[i - 1] * A + y[j - 1]] + acc;
            }
            FM[IDX(i, j)] = v;
            /* X_g : consumes x_i */
            for (int g = 0; g < G; ++g) {
                double u = NEG_INF;
                if (i >= 1) {
                    double acc = (i == 1 && j == 0) ? mdl->init_I[g] : NEG_INF;
                    acc = lse(acc, mdl->t_MI[g] + FM[IDX(i - 1, j)]);
                    acc = lse(acc, mdl->t_II[g] + F[(1 + g) * pl + IDX(i - 1, j)]);
                    u = mdl->log_ins[x[i - 1]] + acc;
                }
                F[(1 + g) * pl + IDX(i, j)] = u;
            }
            /* Y_g : consumes y_j */
            for (int g = 0; g < G; ++g) {
                double u = NEG_INF;
                if (j >= 1) {
                    double acc = (i == 0 && j == 1) ? mdl->init_I[g] : NEG_INF;
                    acc = lse(acc, mdl->t_MI[g] + FM[IDX(i, j - 1)]);
                    acc = lse(acc, mdl->t_II[g] + F[(1 + G + g) * pl + IDX(i, j - 1)]);
                    u = mdl->log_ins[y[j - 1]] + acc;
                }
                F[(1 + G + g) * pl + IDX(i, j)] = u;
            }
        }
    }
    double z = FM[IDX(n, m)] + mdl->end_M;
    for (int g = 0; g < G; ++g) {
        z = lse(z, F[(1 + g) * pl + IDX(n, m)] + mdl->end_I[g]);
        z = lse(z, F[(1 + G + g) * pl + IDX(n, m)] + mdl->end_I[g]);
    }
    return z;
}

/*
 * Backward recurrence, SURVEY.md 8(c) c-1:
 *   B_s(n,m)  = end_s
 *   B_M (i,j) = [i<n,j<m]( t_MM + lm[x_{i+1}][y_{j+1}] + B_M(i+1,j+1) )
 *               (+)_g [i<n]( t_MI[g] + lx[x_{i+1}] + B_Xg(i+1,j) ) (+)_g [j<m]( t_MI[g] + ly[y_{j+1}] + B_Yg(i,j+1) )
 *   B_Xg(i,j) = [i<n,j<m]( t_IM[g] + lm[..] + B_M(i+1,j+1) ) (+) [i<n]( t_II[g] + lx[x_{i+1}] + B_Xg(i+1,j) )
 *   B_Yg(i,j) = [i<n,j<m]( t_IM[g] + lm[..] + B_M(i+1,j+1) ) (+) [j<m]( t_II[g] + ly[y_{j+1}] + B_Yg(i,j+1) )
 *   logZ_b    = ( init_M + lm[x_1][y_1] + B_M(1,1) ) (+)_g ( init_I[g] + lx[x_1] + B_Xg(1,0) )
 *               (+)_g ( init_I[g] + ly[y_1] + B_Yg(0,1) )
 * B holds S planes; returns logZ_b.
 */
double qpo_backward(const qpo_model *mdl, const uint8_t *x, int n, const uint8_t *y, int m, double *B)
{
    const int G = mdl->n_ins, A = mdl->alphabet;
    const size_t pl = (size_t)(n + 1) * (size_t)(m + 1);
    double *BM = B;
    for (int i = n; i >= 0; --i) {
        for (int j = m; j >= 0; --j) {
            if (i == n && j == m) {
                BM[IDX(i, j)] = mdl->end_M;
                for (int g = 0; g < G; ++g) {
                    B[(1 + g) * pl + IDX(i, j)] = mdl->end_I[g];
                    B[(1 + G + g) * pl + IDX(i, j)] = mdl->end_I[g];
                }
                continue;
            }
            double diag = NEG_INF; /* lm[x_{i+1}][y_{j+1}] + B_M(i+1,j+1) */
            if (i < n && j < m) diag = mdl->log_match[(size_t)x[i] * A + y[j]] + BM[IDX(i + 1, j + 1)];
            double bm = (diag == NEG_INF) ? NEG_INF : mdl->t_MM + diag;
            for (int g = 0; g < G; ++g) {
                double down = NEG_INF, right = NEG_INF; /* into X_g at (i+1,j); into Y_g at (i,j+1) */
                if (i < n) down = mdl->log_ins[x[i]] + B[(1 + g) * pl + IDX(i + 1, j)];
                if (j < m) right = mdl->log_ins[y[j]] + B[(1 + G + g) * pl + IDX(i, j + 1)];
                bm = lse(bm, mdl->t_MI[g] + down);
                bm = lse(bm, mdl->t_MI[g] + right);
                B[(1 + g) * pl + IDX(i, j)] = lse(mdl->t_IM[g] + diag, mdl->t_II[g] + down);
                B[(1 + G + g) * pl + IDX(i, j)] = lse(mdl->t_IM[g] + diag, mdl->t_II[g] + right);
            }
            BM[IDX(i, j)] = bm;
        }
    }
    double z = mdl->init_M + mdl->log_match[(size_t)x[0] * A + y[0]] + BM[IDX(1, 1)];
    for (int g = 0; g < G; ++g) {
        z = lse(z, mdl->init_I[g] + mdl->log_ins[x[0]] + B[(1 + g) * pl + IDX(1, 0)]);
        z = lse(z, mdl->init_I[g] + mdl->log_ins[y[0]] + B[(1 + G + g) * pl + IDX(0, 1)]);
    }
    return z;
}

/*
 * P_model(i,j) = exp( F_M(i,j) + B_M(i,j) - logZ_f ), 1<=i<=n, 1<=j<=m  (c-1, last line).
 * P is n*m row-major (0-based). F/B are caller scratch of S*(n+1)*(m+1) doubles (kept for the plane pins).
 */
void qpo_posterior(const qpo_model *mdl, const uint8_t *x, int n, const uint8_t *y, int m, double *F, double *B,
                   double *P, double *logZ_f, double *logZ_b)
{
    double zf = qpo_forward(mdl, x, n, y, m, F);
    double zb = qpo_backward(mdl, x, n, y, m, B);
    for (int i = 1; i <= n; ++i)
        for (int j = 1; j <= m; ++j)
            P[(size_t)(i - 1) * m + (j - 1)] = exp(F[IDX(i, j)] + B[IDX(i, j)] - zf);
    if (logZ_f) *logZ_f = zf;
    if (logZ_b) *logZ_b = zb;
}

/* c-2: P = sqrt( (P_hmm^2 + P_pf^2) / 2 ) */
void qpo_combine(const double *Ph, const double *Pp, size_t cells, double *P)
{
    for (size_t c = 0; c < cells; ++c) P[c] = sqrt((Ph[c] * Ph[c] + Pp[c] * Pp[c]) / 2.0);
}

/* c-2: A(0,.)=A(.,0)=0; A(i,j)=max(A(i-1,j-1)+P(i,j), A(i-1,j), A(i,j-1)) over the dense un-thresholded P. */
double qpo_mea(const double *P, int n, int m)
{
    double *A = (double *)calloc((size_t)(n + 1) * (size_t)(m + 1), sizeof(double));
    for (int i = 1; i <= n; ++i)
        for (int j = 1; j <= m; ++j) {
            double a = A[IDX(i - 1, j - 1)] + P[(size_t)(i - 1) * m + (j - 1)];
            if (A[IDX(i - 1, j)] > a) a = A[IDX(i - 1, j)];
            if (A[IDX(i, j - 1)] > a) a = A[IDX(i, j - 1)];
            A[IDX(i, j)] = a;
        }
    double r = A[IDX(n, m)];
    free(A);
    return r;
}

/* c-2: d_xy = 1 - A(n,m) / min(n,m) */
double qpo_distance(double mea, int n, int m) { return 1.0 - mea / (double)(n < m ? n : m); }

/*
 * One pair, both models: dense combined P (n*m, optional Ph/Pp), logZ4 = {hmm fwd, hmm bwd, pf fwd, pf bwd},
 * returns the distance. Returns NaN on allocation failure.
 */
double qpo_pair(const qpo_model *hmm, const qpo_model *pf, const uint8_t *x, int n, const uint8_t *y, int m,
                double *P, double *Ph_out, double *Pp_out, double *logZ4)
{
    const size_t cells = (size_t)n * (size_t)m, pl = (size_t)(n + 1) * (size_t)(m + 1);
    const int Smax = 1 + 2 * QPO_MAX_INS;
    double *F = (double *)malloc(sizeof(double) * pl * Smax), *B = (double *)malloc(sizeof(double) * pl * Smax);
    double *Ph = Ph_out ? Ph_out : (double *)malloc(sizeof(double) * cells);
    double *Pp = Pp_out ? Pp_out : (double *)malloc(sizeof(double) * cells);
    double d = NAN, z[4] = {0, 0, 0, 0};
    if (F && B && Ph && Pp) {
        qpo_posterior(hmm, x, n, y, m, F, B, Ph, &z[0], &z[1]);
        qpo_posterior(pf, x, n, y, m, F, B, Pp, &z[2], &z[3]);
        qpo_combine(Ph, Pp, cells, P);
        d = qpo_distance(qpo_mea(P, n, m), n, m);
    }
    if (logZ4) memcpy(logZ4, z, sizeof z);
    free(F);
    free(B);
    if (!Ph_out) free(Ph);
    if (!Pp_out) free(Pp);
    return d;
}

/* ------------------------------------------------------------------------------------------------------------
 * All listed pairs: distances + per-pair CSR of entries P >= tau (c-2 "CSR keeps P(i,j) >= tau,
 * columns ascending, values unmodified"). Results live in a handle because nnz is not known in advance.
 * ---------------------------------------------------------------------------------------------------------- */
typedef struct {
    int64_t n_pairs;
    int32_t **row_ptr; /* per pair: n_p+1 local offsets */
    int32_t **col;     /* per pair: nnz_p 0-based columns */
    double **val;      /* per pair: nnz_p values (fp64, unmodified) */
    int32_t *n_rows;
    double *dist;      /* per pair */
    double *logZ;      /* per pair x 4 */
    double **dense;    /* per pair dense P or NULL */
    int threads;
    double seconds;
} qpo_result;

static double now_s(void)
{
#ifdef _OPENMP
    return omp_get_wtime();
#else
    return 0.0;
#endif
}

qpo_result *qpo_run(const qpo_model *hmm, const qpo_model *pf, double tau, const uint8_t *seqs,
                    const int64_t *offsets, const int32_t *pairs, int64_t n_pairs, int keep_dense, int threads)
{
    qpo_result *r = (qpo_result *)calloc(1, sizeof *r);
    r->n_pairs = n_pairs;
    r->row_ptr = (int32_t **)calloc((size_t)n_pairs, sizeof(void *));
    r->col = (int32_t **)calloc((size_t)n_pairs, sizeof(void *));
    r->val = (double **)calloc((size_t)n_pairs, sizeof(void *));
    r->dense = (double **)calloc((size_t)n_pairs, sizeof(void *));
    r->n_rows = (int32_t *)calloc((size_t)n_pairs, sizeof(int32_t));
    r->dist = (double *)calloc((size_t)n_pairs, sizeof(double));
    r->logZ = (double *)calloc((size_t)n_pairs * 4, sizeof(double));
#ifdef _OPENMP
    if (threads > 0) omp_set_num_threads(threads);
    r->threads = threads > 0 ? threads : omp_get_max_threads();
#else
    r->threads = 1;
#endif
    double t0 = now_s();
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t p = 0; p < n_pairs; ++p) {
        int32_t xi = pairs[2 * p], yi = pairs[2 * p + 1];
        const uint8_t *x = seqs + offsets[xi], *y = seqs + offsets[yi];
        int n = (int)(offsets[xi + 1] - offsets[xi]), m = (int)(offsets[yi + 1] - offsets[yi]);
        double *P = (double *)malloc(sizeof(double) * (size_t)n * (size_t)m);
        r->dist[p] = qpo_pair(hmm, pf, x, n, y, m, P, NULL, NULL, r->logZ + 4 * p);
        int32_t *rp = (int32_t *)malloc(sizeof(int32_t) * (size_t)(n + 1));
        int64_t nnz = 0;
        for (int i = 0; i < n; ++i)
            for (int j = 0; j < m; ++j) nnz += (P[(size_t)i * m + j] >= tau);
        int32_t *cc = (int32_t *)malloc(sizeof(int32_t) * (size_t)(nnz ? nnz : 1));
        double *vv = (double *)malloc(sizeof(double) * (size_t)(nnz ? nnz : 1));
        int32_t q = 0;
        for (int i = 0; i < n; ++i) {
            rp[i] = q;
            for (int j = 0; j < m; ++j)
                if (P[(size_t)i * m + j] >= tau) {
                    cc[q] = j;
                    vv[q] = P[(size_t)i * m + j];
                    ++q;
                }
        }
        rp[n] = q;
        r->n_rows[p] = n;
        r->row_ptr[p] = rp;
        r->col[p] = cc;
        r->val[p] = vv;
        if (keep_dense) r->dense[p] = P; else free(P);
    }
    r->seconds = now_s() - t0;
    return r;
}

int64_t qpo_result_nnz(const qpo_result *r, int64_t p) { return r->row_ptr[p][r->n_rows[p]]; }
int32_t qpo_result_rows(const qpo_result *r, int64_t p) { return r->n_rows[p]; }
int qpo_result_threads(const qpo_result *r) { return r->threads; }
double qpo_result_seconds(const qpo_result *r) { return r->seconds; }
double qpo_result_dist(const qpo_result *r, int64_t p) { return r->dist[p]; }
void qpo_result_logZ(const qpo_result *r, int64_t p, double *out4) { memcpy(out4, r->logZ + 4 * p, 4 * sizeof(double)); }

void qpo_result_csr(const qpo_result *r, int64_t p, int32_t *row_ptr, int32_t *col, double *val)
{
    int n = r->n_rows[p];
    int64_t nnz = r->row_ptr[p][n];
    memcpy(row_ptr, r->row_ptr[p], sizeof(int32_t) * (size_t)(n + 1));
    memcpy(col, r->col[p], sizeof(int32_t) * (size_t)nnz);
    memcpy(val, r->val[p], sizeof(double) * (size_t)nnz);
}

int qpo_result_dense(const qpo_result *r, int64_t p, double *out, int64_t cells)
{
    if (!r->dense[p]) return -1;
    memcpy(out, r->dense[p], sizeof(double) * (size_t)cells);
    return 0;
}

void qpo_result_free(qpo_result *r)
{
    if (!r) return;
    for (int64_t p = 0; p < r->n_pairs; ++p) {
        free(r->row_ptr[p]);
        free(r->col[p]);
        free(r->val[p]);
        free(r->dense[p]);
    }
    free(r->row_ptr);
    free(r->col);
    free(r->val);
    free(r->dense);
    free(r->n_rows);
    free(r->dist);
    free(r->logZ);
    free(r);
}

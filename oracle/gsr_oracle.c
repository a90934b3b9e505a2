/*
 * gsr_oracle.c -- CPU ORACLE for the Gaia AVU-GSR hot path.  TEST INFRASTRUCTURE ONLY.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may load this library.  It shares no code, header, table or helper with the CUDA path
 * (paper_2212_11675_b200/csrc) and neither includes the other.
 *
 * Plain, slow, serial C following the paper in its own order and notation:
 *   - matrix in the paper's compressed form A_d / M_i / I_c      (section 3)
 *   - aprod mode 1  b[i] += sum_k A_d[i*Npar+k] * x[col(i,k)]    (Algorithm 1)
 *   - aprod mode 2  x[col(i,k)] += A_d[i*Npar+k] * b[i]          (Algorithm 2)
 *   - preconditioner: p_j = 1/||A_j||_2, columns scaled in place
 *   - LSQR: the paper cites Paige & Saunders 1982 and prints only the
 *     loop skeleton (Algorithm 3); the recurrences below are the published
 *     algorithm, damp = 0, written in DESIGN.md's notation (reading C3).
 *
 * Rounding (readings A6, A14): a row sum (24 terms) is a plain fp64 accumulator in
 * storage order, compiled with -ffp-contract=off (no FMA).  Every long sum (each x[col] of
 * aprod2, every norm, column sums of squares) is accumulated in long double (x87 80-bit) so
 * that the oracle is the more exact side at 1e8 rows.
 *
 * Pins (tests/test_oracle_*.py): scipy CSR rebuilt from the raw arrays, unit-vector probes,
 * adjoint identity, dense lstsq / normal equations on tiny systems, Krylov-subspace
 * minimiser at fixed k, consistent-system recovery, block-diagonal per-star 5x5 solves,
 * unit column norms, scipy.sparse.linalg.lsqr as a black box.
 * Constraint equations (row f3): extra CSR rows below the observations, pinned by the dense
 * augmented matrix (tests/test_constraints.py).
 * Standard errors (row f1): Paige & Saunders' var_j = sum_k (w_j/rho_k)^2, pinned by
 * diag((A^T A)^-1) on tiny systems run to finite termination.
 * Timing-only OpenMP build (-DORC_OPENMP -fopenmp -> libgsr_oracle_omp.so): the same file with
 * the paper's own CPU scheme: aprod1 as a `parallel for` over rows; aprod2 with
 * one contiguous, star-aligned row range per thread, the astrometric columns owned by the range
 * and thread-private accumulators for the replicated attitude + instrumental + global slice,
 * combined in thread order.  Used by bench.py's all-core cpu_baseline and by the full-size
 * parity legs; tests/test_oracle_omp.py checks it against the serial build (1e-13).  The
 * serial build is the definition.
 * parity unpinned: the authors' own "modified" LSQR and their variance formula, covariances,
 * constraints (PAPER.md:27, 65, 67 give no formula) -- covariances / constraints not implemented.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef ORC_OPENMP
#include <omp.h>
#endif

/* threads the build uses (1: the serial definition) */
int orc_threads(void) {
#ifdef ORC_OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

#define N_ASTRO 5
#define N_AXES 3
#define N_PAR_AXIS 4
#define N_ATT (N_AXES * N_PAR_AXIS)
#define N_INSTR 6
#define N_GLOB 1
#define N_PAR 24

typedef struct {
    int64_t n_rows;  /* m */
    int64_t n_stars; /* S */
    int64_t n_dfa;   /* D = N_DFA, degrees of freedom per attitude axis */
    int64_t n_instr; /* I */
} orc_dims;

typedef struct {
    int32_t istop;
    int32_t istop_natural; /* first rule 1-6 that fired (0 if none); = istop unless forced */
    int64_t itn;
    int64_t itn_natural;   /* iteration at which istop_natural fired (0 if none) */
    double rnorm, arnorm, anorm, acond, xnorm, bnorm;
} orc_result;

static int64_t n_cols(const orc_dims* d) { return 5 * d->n_stars + 3 * d->n_dfa + d->n_instr + 1; }

/* Constraint equations: "to find a unique solution, an additional number of constraint equations
 * have to be set"; both aprod modes end with a "constraints computation"
 * (Algorithms 1 and 2).  The paper does not give their structure, so
 * they are n_con extra rows in general CSR form appended below the m observation rows: row m+r
 * has coefficients val[e] at columns col[e], e in [row_ptr[r], row_ptr[r+1]).  Set once per call
 * by the Python wrapper (the oracle is single-threaded test infrastructure); n_con = 0: none. */
typedef struct {
    int64_t n_con;
    const int64_t* row_ptr;
    const int32_t* col;
    double* val;
} orc_con;
static orc_con g_con = {0, NULL, NULL, NULL};
void orc_set_constraints(int64_t n_con, const int64_t* row_ptr, const int32_t* col, double* val) {
    g_con.n_con = n_con;
    g_con.row_ptr = row_ptr;
    g_con.col = col;
    g_con.val = val;
}

/* Column of stored coefficient k of row i.  Section 3 and the index
 * expressions of Algorithm 1: astrometric x[j+offset[i]], offset = 5*star;
 * attitude k2 = j1*N_DFA + offset[i], x[j2+k2]; instrumental
 * x[F(i,j)+offset] with F = I_c; global x[j+offset]. */
static int64_t col_of(const orc_dims* d, const int32_t* star_idx, const int32_t* att_start,
                      const int32_t* instr_col, int64_t i, int k) {
    const int64_t off_att = N_ASTRO * d->n_stars;
    const int64_t off_instr = off_att + N_AXES * d->n_dfa;
    const int64_t off_glob = off_instr + d->n_instr;
    if (k < N_ASTRO) return N_ASTRO * (int64_t)star_idx[i] + k;
    if (k < N_ASTRO + N_ATT) {
        int j1 = (k - N_ASTRO) / N_PAR_AXIS, j2 = (k - N_ASTRO) % N_PAR_AXIS;
        return off_att + j1 * d->n_dfa + att_start[i] + j2;
    }
    if (k < N_ASTRO + N_ATT + N_INSTR) return off_instr + instr_col[N_INSTR * i + (k - N_ASTRO - N_ATT)];
    return off_glob;
}

/* 0 if the index arrays describe a legal system, else a negative code naming the fault. */
int orc_validate(const orc_dims* d, const int32_t* star_idx, const int32_t* att_start,
                 const int32_t* instr_col) {
    if (d->n_rows < 0 || d->n_stars < 1 || d->n_dfa < 4 || d->n_instr < 1) return -1;
    for (int64_t i = 0; i < d->n_rows; ++i) {
        if (star_idx[i] < 0 || star_idx[i] >= d->n_stars) return -2;
        if (i > 0 && star_idx[i] < star_idx[i - 1]) return -3;
        if (att_start[i] < 0 || att_start[i] > d->n_dfa - 4) return -4;
        for (int j = 0; j < N_INSTR; ++j)
            if (instr_col[N_INSTR * i + j] < 0 || instr_col[N_INSTR * i + j] >= d->n_instr) return -5;
    }
    return 0;
}

/* The 24 (column, value) pairs of rows [row0, row0+nrows). */
void orc_expand_rows(const orc_dims* d, const int32_t* star_idx, const int32_t* att_start,
                     const int32_t* instr_col, const double* A_d, int64_t row0, int64_t nrows,
                     int64_t* cols, double* vals) {
    for (int64_t r = 0; r < nrows; ++r)
        for (int k = 0; k < N_PAR; ++k) {
            cols[N_PAR * r + k] = col_of(d, star_idx, att_start, instr_col, row0 + r, k);
            vals[N_PAR * r + k] = A_d[N_PAR * (row0 + r) + k];
        }
}

/* aprod mode 1: b[i] = b[i] + sum.  One accumulator per row,
 * k = 0..23 in storage order (reading A6).  If scale != NULL it receives
 * |b0[i]| + sum_k |A_d*x| (the component-wise error scale of reading A13). */
void orc_aprod1(const orc_dims* d, const int32_t* star_idx, const int32_t* att_start,
                const int32_t* instr_col, const double* A_d, const double* x, double* b,
                double* scale) {
#ifdef ORC_OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (int64_t i = 0; i < d->n_rows; ++i) {
        double sum = 0.0, asum = 0.0;
        const int64_t k0 = i * N_PAR;
        for (int k = 0; k < N_PAR; ++k) {
            double t = A_d[k0 + k] * x[col_of(d, star_idx, att_start, instr_col, i, k)];
            sum = sum + t;
            asum = asum + fabs(t);
        }
        if (scale) scale[i] = fabs(b[i]) + asum;
        b[i] = b[i] + sum;
    }
    for (int64_t r = 0; r < g_con.n_con; ++r) { /* constraints computation */
        const int64_t i = d->n_rows + r;
        double sum = 0.0, asum = 0.0;
        for (int64_t e = g_con.row_ptr[r]; e < g_con.row_ptr[r + 1]; ++e) {
            double t = g_con.val[e] * x[g_con.col[e]];
            sum = sum + t;
            asum = asum + fabs(t);
        }
        if (scale) scale[i] = fabs(b[i]) + asum;
        b[i] = b[i] + sum;
    }
}

/* aprod mode 2: x[col] = x[col] + A_d[k]*b[i], rows in order,
 * each x[col] accumulated in long double (reading A14) and rounded once at the end. */
void orc_aprod2(const orc_dims* d, const int32_t* star_idx, const int32_t* att_start,
                const int32_t* instr_col, const double* A_d, const double* b, double* x,
                double* scale) {
    const int64_t n = n_cols(d);
    long double* acc = (long double*)malloc(sizeof(long double) * (size_t)n);
    long double* aacc = scale ? (long double*)malloc(sizeof(long double) * (size_t)n) : NULL;
    for (int64_t j = 0; j < n; ++j) {
        acc[j] = x[j];
        if (aacc) aacc[j] = fabs(x[j]);
    }
#ifdef ORC_OPENMP
    {   /* timing build: star-aligned row range per thread */
        const int nt = omp_get_max_threads();
        const int64_t n_astro = N_ASTRO * d->n_stars, n_rep = n - n_astro;
        int64_t* lo = (int64_t*)malloc(sizeof(int64_t) * (size_t)(nt + 1));
        for (int t = 0; t <= nt; ++t) {
            int64_t r = d->n_rows * t / nt;
            while (r > 0 && r < d->n_rows && star_idx[r] == star_idx[r - 1]) ++r;
            lo[t] = r;
        }
        long double* priv = (long double*)calloc((size_t)(nt * n_rep), sizeof(long double));
        long double* apriv = aacc ? (long double*)calloc((size_t)(nt * n_rep), sizeof(long double)) : NULL;
#pragma omp parallel num_threads(nt)
        {
            const int t = omp_get_thread_num();
            long double* pr = priv + (size_t)t * n_rep;
            long double* apr = apriv ? apriv + (size_t)t * n_rep : NULL;
            for (int64_t i = lo[t]; i < lo[t + 1]; ++i) {
                const int64_t k0 = i * N_PAR;
                for (int k = 0; k < N_PAR; ++k) {
                    int64_t c = col_of(d, star_idx, att_start, instr_col, i, k);
                    double tt = A_d[k0 + k] * b[i];
                    if (c < n_astro) {          /* owned by this range: rows are star-aligned */
                        acc[c] += tt;
                        if (aacc) aacc[c] += fabs(tt);
                    } else {
                        pr[c - n_astro] += tt;
                        if (apr) apr[c - n_astro] += fabs(tt);
                    }
                }
            }
        }
        for (int t = 0; t < nt; ++t)            /* replicated slice, combined in thread order */
            for (int64_t j = 0; j < n_rep; ++j) {
                acc[n_astro + j] += priv[(size_t)t * n_rep + j];
                if (aacc) aacc[n_astro + j] += apriv[(size_t)t * n_rep + j];
            }
        free(lo);
        free(priv);
        free(apriv);
    }
#else
    for (int64_t i = 0; i < d->n_rows; ++i) {
        const int64_t k0 = i * N_PAR;
        for (int k = 0; k < N_PAR; ++k) {
            int64_t c = col_of(d, star_idx, att_start, instr_col, i, k);
            double t = A_d[k0 + k] * b[i];
            acc[c] += t;
            if (aacc) aacc[c] += fabs(t);
        }
    }
#endif
    for (int64_t r = 0; r < g_con.n_con; ++r) /* constraints computation */
        for (int64_t e = g_con.row_ptr[r]; e < g_con.row_ptr[r + 1]; ++e) {
            double t = g_con.val[e] * b[d->n_rows + r];
            acc[g_con.col[e]] += t;
            if (aacc) aacc[g_con.col[e]] += fabs(t);
        }
    for (int64_t j = 0; j < n; ++j) {
        x[j] = (double)acc[j];
        if (aacc) scale[j] = (double)aacc[j];
    }
    free(acc);
    free(aacc);
}

/* q_j = sum_i A_ij^2 (long double), the squared column norms of PAPER.md:43. */
void orc_colsumsq(const orc_dims* d, const int32_t* star_idx, const int32_t* att_start,
                  const int32_t* instr_col, const double* A_d, double* q) {
    const int64_t n = n_cols(d);
    long double* acc = (long double*)calloc((size_t)n, sizeof(long double));
#ifdef ORC_OPENMP
    {   /* timing build: same partition as orc_aprod2 */
        const int nt = omp_get_max_threads();
        const int64_t n_astro = N_ASTRO * d->n_stars, n_rep = n - n_astro;
        int64_t* lo = (int64_t*)malloc(sizeof(int64_t) * (size_t)(nt + 1));
        for (int t = 0; t <= nt; ++t) {
            int64_t r = d->n_rows * t / nt;
            while (r > 0 && r < d->n_rows && star_idx[r] == star_idx[r - 1]) ++r;
            lo[t] = r;
        }
        long double* priv = (long double*)calloc((size_t)(nt * n_rep), sizeof(long double));
#pragma omp parallel num_threads(nt)
        {
            const int t = omp_get_thread_num();
            long double* pr = priv + (size_t)t * n_rep;
            for (int64_t i = lo[t]; i < lo[t + 1]; ++i)
                for (int k = 0; k < N_PAR; ++k) {
                    double a = A_d[i * N_PAR + k];
                    int64_t c = col_of(d, star_idx, att_start, instr_col, i, k);
                    if (c < n_astro) acc[c] += (long double)a * a;
                    else pr[c - n_astro] += (long double)a * a;
                }
        }
        for (int t = 0; t < nt; ++t)
            for (int64_t j = 0; j < n_rep; ++j) acc[n_astro + j] += priv[(size_t)t * n_rep + j];
        free(lo);
        free(priv);
    }
#else
    for (int64_t i = 0; i < d->n_rows; ++i)
        for (int k = 0; k < N_PAR; ++k) {
            double a = A_d[i * N_PAR + k];
            acc[col_of(d, star_idx, att_start, instr_col, i, k)] += (long double)a * a;
        }
#endif
    for (int64_t e = 0; g_con.n_con > 0 && e < g_con.row_ptr[g_con.n_con]; ++e)
        acc[g_con.col[e]] += (long double)g_con.val[e] * g_con.val[e];
    for (int64_t j = 0; j < n; ++j) q[j] = (double)acc[j];
    free(acc);
}

/* Preconditioner (reading A7): p_j = 1/sqrt(q_j), 1 for an empty column;
 * every stored coefficient is multiplied by p[col] in place.  p has n entries. */
void orc_precondition(const orc_dims* d, const int32_t* star_idx, const int32_t* att_start,
                      const int32_t* instr_col, double* A_d, double* p) {
    const int64_t n = n_cols(d);
    orc_colsumsq(d, star_idx, att_start, instr_col, A_d, p);
    for (int64_t j = 0; j < n; ++j) p[j] = p[j] > 0.0 ? 1.0 / sqrt(p[j]) : 1.0;
#ifdef ORC_OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (int64_t i = 0; i < d->n_rows; ++i)
        for (int k = 0; k < N_PAR; ++k)
            A_d[i * N_PAR + k] = A_d[i * N_PAR + k] * p[col_of(d, star_idx, att_start, instr_col, i, k)];
    for (int64_t e = 0; g_con.n_con > 0 && e < g_con.row_ptr[g_con.n_con]; ++e)
        g_con.val[e] = g_con.val[e] * p[g_con.col[e]];
}

static double sumsq(const double* v, int64_t len) {
    long double s = 0.0L;
#ifdef ORC_OPENMP
#pragma omp parallel for schedule(static) reduction(+ : s)
#endif
    for (int64_t j = 0; j < len; ++j) s += (long double)v[j] * v[j];
    return (double)s;
}
static double nrm2(const double* v, int64_t len) {
    long double s = 0.0L;
#ifdef ORC_OPENMP
#pragma omp parallel for schedule(static) reduction(+ : s)
#endif
    for (int64_t j = 0; j < len; ++j) s += (long double)v[j] * v[j];
    return (double)sqrtl(s);
}
static double hyp(double a, double b) { return sqrt(a * a + b * b); } /* reading A15 */
/* v[i] = c * v[i] or v[i] / c, element-wise (same rounding in both builds) */
static void scal(double* v, int64_t len, double c, int divide) {
#ifdef ORC_OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (int64_t i = 0; i < len; ++i) v[i] = divide ? v[i] / c : c * v[i];
}

/* Damping (row f4; Paige & Saunders 1982, section 2 of the algorithm paper): with damp > 0 LSQR
 * minimises || [A; damp I] x - [b; 0] ||.  The paper does not use it (damp = 0, the default);
 * set by the Python wrapper around a call, like the constraints. */
static double g_damp = 0.0;
void orc_set_damp(double damp) { g_damp = damp; }

/* LSQR, Paige & Saunders 1982 (cited PAPER.md:27, 699-700), damp = 0; reading C3.
 * force_itnlim != 0 (reading A9): rules 1-6 are evaluated and recorded in *_natural but only
 * the iteration limit ends the loop.  hist (may be NULL) receives per iteration
 * [rnorm, arnorm, anorm, acond, xnorm, alpha, beta] (7 doubles each, itnlim rows). */
/* var (may be NULL): on return var[j] = sum over the iterations of (w_j / rho)^2, the LSQR
 * estimate of diag((A^T A)^-1) from which standard errors follow ("Variances ... computation",
 * Algorithm 3 line 17; the paper gives no formula: Paige & Saunders' one). */
int orc_lsqr_var(const orc_dims* d, const int32_t* star_idx, const int32_t* att_start,
                 const int32_t* instr_col, const double* A_d, const double* b, double* x,
                 int64_t itnlim, double atol, double btol, double conlim, int force_itnlim,
                 orc_result* res, double* hist, double* var) {
    const int64_t m = d->n_rows + g_con.n_con, n = n_cols(d);   /* b, u: observations then constraints */
    if (var)
        for (int64_t j = 0; j < n_cols(d); ++j) var[j] = 0.0;
    double* u = (double*)malloc(sizeof(double) * (size_t)(m > 0 ? m : 1));
    double* v = (double*)calloc((size_t)n, sizeof(double));
    double* w = (double*)malloc(sizeof(double) * (size_t)n);
    const double ctol = conlim > 0.0 ? 1.0 / conlim : 0.0;
    double anorm = 0, acond = 0, ddnorm = 0, xxnorm = 0, z = 0, cs2 = -1, sn2 = 0;
    double alpha = 0, beta, rhobar, phibar, bnorm, rnorm, arnorm = 0, xnorm = 0;
    const double damp = g_damp;
    double res2 = 0.0; /* sum of psi^2: the part of the residual that the damping rows hold */
    int istop = 0;
    int64_t itn = 0;
    memset(res, 0, sizeof(*res));
    for (int64_t j = 0; j < n; ++j) x[j] = 0.0;
    memcpy(u, b, sizeof(double) * (size_t)m);
    beta = nrm2(u, m);
    bnorm = beta;
    res->bnorm = bnorm;
    if (beta == 0.0) goto done_trivial; /* x = 0 is the exact solution: istop 0 */
    scal(u, m, beta, 1);
    /* "aprod 2 call (calculation of the initial solution)", Algorithm 3 line 6 */
    orc_aprod2(d, star_idx, att_start, instr_col, A_d, u, v, NULL);
    alpha = nrm2(v, n);
    if (alpha == 0.0) {
        res->rnorm = beta;
        goto done_trivial;
    }
    for (int64_t j = 0; j < n; ++j) v[j] = v[j] / alpha;
    memcpy(w, v, sizeof(double) * (size_t)n);
    rhobar = alpha;
    phibar = beta;
    rnorm = beta;
    arnorm = alpha * beta;

    while (1) {
        itn += 1;
        /* bidiagonalisation: u = A v - alpha u ; v = A^T u - beta v   (Alg. 3 lines 11, 15) */
        scal(u, m, -alpha, 0);
        orc_aprod1(d, star_idx, att_start, instr_col, A_d, v, u, NULL);
        beta = nrm2(u, m);
        if (beta > 0.0) {
            scal(u, m, beta, 1);
            anorm = hyp(hyp(anorm, alpha), beta);
            if (damp > 0.0) anorm = hyp(anorm, damp);
            for (int64_t j = 0; j < n; ++j) v[j] = -beta * v[j];
            orc_aprod2(d, star_idx, att_start, instr_col, A_d, u, v, NULL);
            alpha = nrm2(v, n);
            if (alpha > 0.0)
                for (int64_t j = 0; j < n; ++j) v[j] = v[j] / alpha;
        }
        /* plane rotation eliminating the damping parameter (only when damp > 0) */
        double rhobar1 = rhobar, psi = 0.0;
        if (damp > 0.0) {
            rhobar1 = hyp(rhobar, damp);
            double cs1 = rhobar / rhobar1, sn1 = damp / rhobar1;
            psi = sn1 * phibar;
            phibar = cs1 * phibar;
        }
        /* plane rotation eliminating beta */
        double rho = hyp(rhobar1, beta);
        double cs = rhobar1 / rho, sn = beta / rho;
        double theta = sn * alpha;
        rhobar = -cs * alpha;
        double phi = cs * phibar;
        phibar = sn * phibar;
        double tau = sn * phi;
        /* update x and w */
        double t1 = phi / rho, t2 = -theta / rho;
        ddnorm = ddnorm + sumsq(w, n) / (rho * rho); /* reading A10 */
        if (var)
            for (int64_t j = 0; j < n; ++j) {
                double dk = w[j] / rho;
                var[j] = var[j] + dk * dk;
            }
        for (int64_t j = 0; j < n; ++j) {
            x[j] = x[j] + t1 * w[j];
            w[j] = v[j] + t2 * w[j];
        }
        /* second rotation: estimate of ||x|| */
        double delta = sn2 * rho;
        double gambar = -cs2 * rho;
        double rhs = phi - delta * z;
        double zbar = rhs / gambar;
        xnorm = sqrt(xxnorm + zbar * zbar);
        double gamma = hyp(gambar, theta);
        cs2 = gambar / gamma;
        sn2 = theta / gamma;
        z = rhs / gamma;
        xxnorm = xxnorm + z * z;
        /* norms and stopping tests */
        acond = anorm * sqrt(ddnorm);
        res2 = res2 + psi * psi;
        rnorm = damp > 0.0 ? sqrt(phibar * phibar + res2) : phibar;
        arnorm = alpha * fabs(tau);
        double test1 = rnorm / bnorm;
        double test2 = (anorm * rnorm > 0.0) ? arnorm / (anorm * rnorm) : INFINITY; /* A8 */
        double test3 = 1.0 / acond;
        double t1c = test1 / (1.0 + anorm * xnorm / bnorm);
        double rtol = btol + atol * anorm * xnorm / bnorm;
        int nat = 0;
        if (1.0 + test3 <= 1.0) nat = 6;
        if (1.0 + test2 <= 1.0) nat = 5;
        if (1.0 + t1c <= 1.0) nat = 4;
        if (test3 <= ctol) nat = 3;
        if (test2 <= atol) nat = 2;
        if (test1 <= rtol) nat = 1;
        if (nat != 0 && res->istop_natural == 0) {
            res->istop_natural = nat;
            res->itn_natural = itn;
        }
        if (hist) {
            double* h = hist + 7 * (itn - 1);
            h[0] = rnorm; h[1] = arnorm; h[2] = anorm; h[3] = acond; h[4] = xnorm;
            h[5] = alpha; h[6] = beta;
        }
        if (itn >= itnlim) istop = 7;
        if (!force_itnlim && nat != 0) istop = nat;
        if (istop != 0) break;
    }
    res->istop = istop;
    res->itn = itn;
    res->rnorm = rnorm;
    res->arnorm = arnorm;
    res->anorm = anorm;
    res->acond = acond;
    res->xnorm = xnorm;
    if (res->istop_natural == 0 && istop != 7) res->istop_natural = istop;
    free(u); free(v); free(w);
    return 0;
done_trivial:
    res->istop = 0;
    res->itn = 0;
    free(u); free(v); free(w);
    return 0;
}

int orc_lsqr(const orc_dims* d, const int32_t* star_idx, const int32_t* att_start,
             const int32_t* instr_col, const double* A_d, const double* b, double* x,
             int64_t itnlim, double atol, double btol, double conlim, int force_itnlim,
             orc_result* res, double* hist) {
    return orc_lsqr_var(d, star_idx, att_start, instr_col, A_d, b, x, itnlim, atol, btol, conlim,
                        force_itnlim, res, hist, NULL);
}

/* Standard errors of the unknowns (Paige & Saunders): se_j = rnorm * sqrt(var_j / dof),
 * dof = m - n if m > n, else 1; for a column-scaled system multiplied by p_j like the solution
 * ("also ... the standard errors").  p may be NULL. */
void orc_standard_errors(int64_t m, int64_t n, double rnorm, const double* var, const double* p,
                         double* se) {
    const double dof = m > n ? (double)(m - n) : 1.0;
    for (int64_t j = 0; j < n; ++j) {
        double e = rnorm * sqrt(var[j] / dof);
        se[j] = p ? p[j] * e : e;
    }
}

/* x = p (.) z : "we re-multiply the solution ... by the preconditioning vector p" */
void orc_unscale(int64_t n, const double* p, double* x) {
    for (int64_t j = 0; j < n; ++j) x[j] = p[j] * x[j];
}

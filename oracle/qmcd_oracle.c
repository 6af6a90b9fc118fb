/*
 * qmcd_oracle.c -- TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, obviously-correct CPU fp64 oracle for the hot path of
 * arXiv 1708.00744 ("Delayed Slater determinant update algorithms for high
 * efficiency quantum Monte Carlo").  It shares no code, header, table or
 * helper with the CUDA path under paper_1708_00744_b200/csrc/ and neither
 * imports the other.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call this file.
 *
 * Citations are lines of /root/reference/PAPER.md.
 *
 * Notation (the paper's own symbols clash, PAPER.md:57
 * uses k for the electron and PAPER.md:80-87 use k for the rank):
 *   N      electrons = matrix order
 *   A      Slater matrix, A[i][k] = phi_i(r_k): row = orbital,
 *          column = electron
 *   B      explicit inverse of A, row-major
 *   j      moved electron: column of A, row of B
 *   v      the NEW column j of A (orbitals at the new position)
 *   u      = v - A[:,j], the column change
 *   K      delay; m = moves currently queued, 0 <= m <= K
 *   J, C, W  queued electron indices, their new columns (one per row of C),
 *          and the rows J of the STALE inverse B0 (one per row of W)
 *   S      = I_m + V'A^-1 U of Eq. 3 = W C^T  (derived below)
 *
 * Three independent paths (plus path 3, the lock-step variant of PAPER.md:97-99,
 * which is path 2 with every proposal occupying a queue slot, and path 4, path 2
 * with the slot-replacement accept for a repeated electron -- pin P12):
 *   path 0  the plain definition: explicit LU determinants / inverse
 *           (PAPER.md:55,57 -- "p ~ det(A_new)/det(A)").
 *   path 1  classic rank-1 Sherman-Morrison, Eqs. 1-2.
 *   path 2  delayed rank-K: Eq. 3 look-ahead + Eq. 4 Woodbury flush
 *           (PAPER.md:78-93).
 * The method is exact, so path 0 is the definition of truth and
 * paths 1-2 must agree with it to rounding.  Pins: tests/test_oracle_pins.py.
 * Parity unpinned: nothing (every function below has a pin there; path 3: P11;
 * orc_residual: test_residual_known_nonzero_values_order_and_sign -- known non-zero
 * residuals, A.B versus B.A, negative entries, NaN).
 *
 * No blocking, fusion or reordering beyond what the formulas state; the only
 * parallelism is an OpenMP "parallel for" over independent walkers in the
 * batch driver (PAPER.md:99 -- walkers are independent), which changes no
 * arithmetic.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_OK 0
#define ORC_ESINGULAR (-1)
#define ORC_EINVAL (-2)
#define ORC_ENOMEM (-3)

/* ------------------------------------------------------------------ */
/* LU with partial pivoting (textbook Doolittle, Golub & Van Loan --    */
/* the paper's ref [21]).  a is n x n row-major, factored */
/* in place: unit-lower L below the diagonal, U on and above it.       */
/* piv[k] = row swapped with k at step k.  Returns the permutation     */
/* sign (+1/-1), or 0 if an exact zero pivot is met.                   */
/* ------------------------------------------------------------------ */
int orc_lu_factor(int n, double *a, int *piv)
{
    int sign = 1;
    for (int k = 0; k < n; ++k) {
        int p = k;
        double best = fabs(a[(size_t)k * n + k]);
        for (int i = k + 1; i < n; ++i) {
            double x = fabs(a[(size_t)i * n + k]);
            if (x > best) { best = x; p = i; }
        }
        piv[k] = p;
        if (best == 0.0) return 0;
        if (p != k) {
            for (int c = 0; c < n; ++c) {
                double t = a[(size_t)k * n + c];
                a[(size_t)k * n + c] = a[(size_t)p * n + c];
                a[(size_t)p * n + c] = t;
            }
            sign = -sign;
        }
        double d = a[(size_t)k * n + k];
        for (int i = k + 1; i < n; ++i) {
            double l = a[(size_t)i * n + k] / d;
            a[(size_t)i * n + k] = l;
            for (int c = k + 1; c < n; ++c)
                a[(size_t)i * n + c] -= l * a[(size_t)k * n + c];
        }
    }
    return sign;
}

/* Solve (LU) X = RHS for nrhs right-hand sides stored as the COLUMNS of the
 * row-major n x nrhs array x (overwritten with the solution). */
void orc_lu_solve(int n, const double *lu, const int *piv, double *x, int nrhs)
{
    for (int k = 0; k < n; ++k) {           /* apply the row swaps */
        int p = piv[k];
        if (p != k)
            for (int c = 0; c < nrhs; ++c) {
                double t = x[(size_t)k * nrhs + c];
                x[(size_t)k * nrhs + c] = x[(size_t)p * nrhs + c];
                x[(size_t)p * nrhs + c] = t;
            }
    }
    for (int i = 0; i < n; ++i)             /* L y = Pb (unit lower) */
        for (int k = 0; k < i; ++k) {
            double l = lu[(size_t)i * n + k];
            for (int c = 0; c < nrhs; ++c)
                x[(size_t)i * nrhs + c] -= l * x[(size_t)k * nrhs + c];
        }
    for (int i = n - 1; i >= 0; --i) {      /* U x = y */
        for (int k = i + 1; k < n; ++k) {
            double u = lu[(size_t)i * n + k];
            for (int c = 0; c < nrhs; ++c)
                x[(size_t)i * nrhs + c] -= u * x[(size_t)k * nrhs + c];
        }
        double d = lu[(size_t)i * n + i];
        for (int c = 0; c < nrhs; ++c) x[(size_t)i * nrhs + c] /= d;
    }
}

/* sign and log|det| of the n x n row-major matrix a (not modified).
 * "explicit recalculation of the determinant is O(N^3)". */
int orc_slogdet(int n, const double *a, int *sign_out, double *logabs_out)
{
    double *w = (double *)malloc(sizeof(double) * (size_t)n * n);
    int *piv = (int *)malloc(sizeof(int) * (size_t)(n > 0 ? n : 1));
    if (!w || !piv) { free(w); free(piv); return ORC_ENOMEM; }
    memcpy(w, a, sizeof(double) * (size_t)n * n);
    int sign = orc_lu_factor(n, w, piv);
    double la = 0.0;
    if (sign == 0) {
        la = -INFINITY;
    } else {
        for (int k = 0; k < n; ++k) {
            double d = w[(size_t)k * n + k];
            if (d < 0) { sign = -sign; d = -d; }
            la += log(d);
        }
    }
    *sign_out = sign;
    *logabs_out = la;
    free(w); free(piv);
    return ORC_OK;
}

/* Explicit inverse by LU: solve A X = I.  PAPER.md:63 ("explicit copy of
 * the matrix inverse"). */
int orc_inverse(int n, const double *a, double *ainv)
{
    double *w = (double *)malloc(sizeof(double) * (size_t)n * n);
    int *piv = (int *)malloc(sizeof(int) * (size_t)(n > 0 ? n : 1));
    if (!w || !piv) { free(w); free(piv); return ORC_ENOMEM; }
    memcpy(w, a, sizeof(double) * (size_t)n * n);
    int sign = orc_lu_factor(n, w, piv);
    if (sign == 0) { free(w); free(piv); return ORC_ESINGULAR; }
    memset(ainv, 0, sizeof(double) * (size_t)n * n);
    for (int i = 0; i < n; ++i) ainv[(size_t)i * n + i] = 1.0;
    orc_lu_solve(n, w, piv, ainv, n);
    free(w); free(piv);
    return ORC_OK;
}

/* ------------------------------------------------------------------ */
/* Path 0: the plain definition.  R = det(A with column j := v)/det(A) */
/* (A_new = A + u v_k', p ~ det(A_new)/det(A)), each      */
/* determinant by explicit LU, compared through sign and log|det|.     */
/* ------------------------------------------------------------------ */
int orc_ratio_bruteforce(int n, const double *A, int j, const double *v, double *R_out)
{
    if (j < 0 || j >= n) return ORC_EINVAL;
    double *An = (double *)malloc(sizeof(double) * (size_t)n * n);
    if (!An) return ORC_ENOMEM;
    memcpy(An, A, sizeof(double) * (size_t)n * n);
    for (int i = 0; i < n; ++i) An[(size_t)i * n + j] = v[i];
    int s0, s1; double l0, l1;
    int rc = orc_slogdet(n, A, &s0, &l0);
    if (rc == ORC_OK) rc = orc_slogdet(n, An, &s1, &l1);
    free(An);
    if (rc != ORC_OK) return rc;
    if (s0 == 0) return ORC_ESINGULAR;
    *R_out = (s1 == 0) ? 0.0 : (double)(s0 * s1) * exp(l1 - l0);
    return ORC_OK;
}

/* ------------------------------------------------------------------ */
/* Path 1: classic rank-1 Sherman-Morrison.           */
/*                                                                    */
/* Eq. 1 with u = v - A[:,j] and the paper's v_k = e_j:                */
/*   R = 1 + e_j' B u = 1 + B[j,:].v - B[j,:].A[:,j] = B[j,:].v        */
/* because B A = I gives B[j,:].A[:,j] = 1.                            */
/* ------------------------------------------------------------------ */
double orc_sm_ratio(int n, const double *B, int j, const double *v)
{
    double r = 0.0;
    for (int k = 0; k < n; ++k) r += B[(size_t)j * n + k] * v[k];
    return r;
}

/* Eq. 2 with the same substitution: B u = B v - e_j and 1 + e_j'Bu = R, so
 *   B_new = B - (B v - e_j) (B[j,:]) / R      using the OLD row j. */
int orc_sm_accept(int n, double *B, int j, const double *v)
{
    double *x = (double *)malloc(sizeof(double) * (size_t)n);
    double *rowj = (double *)malloc(sizeof(double) * (size_t)n);
    if (!x || !rowj) { free(x); free(rowj); return ORC_ENOMEM; }
    for (int i = 0; i < n; ++i) {
        double s = 0.0;
        for (int k = 0; k < n; ++k) s += B[(size_t)i * n + k] * v[k];
        x[i] = s;
    }
    double R = x[j];
    x[j] -= 1.0;
    memcpy(rowj, B + (size_t)j * n, sizeof(double) * (size_t)n);
    for (int i = 0; i < n; ++i)
        for (int k = 0; k < n; ++k)
            B[(size_t)i * n + k] -= x[i] * rowj[k] / R;
    free(x); free(rowj);
    return (R == 0.0 || !isfinite(R)) ? ORC_ESINGULAR : ORC_OK;
}

/* ------------------------------------------------------------------ */
/* Path 2: delayed rank-K.                            */
/*                                                                    */
/* Let A0/B0 be the matrix/inverse at the last flush and (J, C) the    */
/* queue of accepted moves (distinct electrons j_i with new columns    */
/* v_i = C[i,:]).  In the paper's Eq. 3/4 notation U = [v_i - A0[:,j_i]]*/
/* (N x m) and V = [e_{j_i}] (N x m).  Because B0 A0[:,j] = e_j,        */
/*     B0 U = B0 C^T - E_J        (E_J[:,i] = e_{j_i})                 */
/* so  S := I_m + V' B0 U = I_m + (W C^T - I_m) = W C^T,               */
/* with W[a,:] = B0[j_a,:] the queued rows of the stale inverse.       */
/* Eq. 3: det S = det(A_m)/det(A0).                                    */
/*                                                                    */
/* Ratio of a further proposal (j, v) against the CURRENT matrix A_m:  */
/*   R = e_j' A_m^-1 v, and Eq. 4 gives                                */
/*   A_m^-1 = B0 - (B0 C^T - E_J) S^-1 W, hence                        */
/*   R = d - p' S^-1 q,  d = B0[j,:].v,                                */
/*       p_i = B0[j,:].C[i,:] - delta(j, j_i),  q_a = W[a,:].v.        */
/* (Equivalently det S_{m+1}/det S_m, the paper's look-ahead           */
/* determinant ratio.)                                 */
/* The oracle keeps S itself and LU-solves S c = q for every proposal  */
/* -- it never maintains S^-1 incrementally.                           */
/* ------------------------------------------------------------------ */
typedef struct orc_delayed {
    int n, K, m;
    double *B;      /* n x n, BORROWED, updated in place at flush       */
    double *C;      /* K x n  queued new columns, one per row           */
    double *W;      /* K x n  rows J of the stale inverse               */
    double *S;      /* K x K  (leading dimension K), S = W C^T          */
    int *J;         /* K      queued electron indices                   */
    /* staged by ratio for a possible accept */
    int sj;         /* staged electron, -1 if none                      */
    double *sv;     /* n   staged v                                     */
    double *sp;     /* K   B0[j,:].C[i,:]  (WITHOUT the delta term)     */
    double *sq;     /* K   W[a,:].v                                     */
    double sd;      /*     B0[j,:].v                                    */
    double sR;
    long n_flush;
    int replace;    /* slot-replacement accept for a repeated electron (path 4) */
} orc_delayed;

void orc_delayed_destroy(orc_delayed *h)
{
    if (!h) return;
    free(h->C); free(h->W); free(h->S); free(h->J);
    free(h->sv); free(h->sp); free(h->sq);
    free(h);
}

orc_delayed *orc_delayed_create(int n, int K, double *B)
{
    if (n < 1 || K < 1 || K > n || !B) return NULL;
    orc_delayed *h = (orc_delayed *)calloc(1, sizeof(*h));
    if (!h) return NULL;
    h->n = n; h->K = K; h->m = 0; h->B = B; h->sj = -1;
    h->C = (double *)malloc(sizeof(double) * (size_t)K * n);
    h->W = (double *)malloc(sizeof(double) * (size_t)K * n);
    h->S = (double *)malloc(sizeof(double) * (size_t)K * K);
    h->J = (int *)malloc(sizeof(int) * (size_t)K);
    h->sv = (double *)malloc(sizeof(double) * (size_t)n);
    h->sp = (double *)malloc(sizeof(double) * (size_t)K);
    h->sq = (double *)malloc(sizeof(double) * (size_t)K);
    if (!h->C || !h->W || !h->S || !h->J || !h->sv || !h->sp || !h->sq) {
        orc_delayed_destroy(h);
        return NULL;
    }
    return h;
}

int orc_delayed_pending(const orc_delayed *h) { return h->m; }
long orc_delayed_flush_count(const orc_delayed *h) { return h->n_flush; }

/* Look-ahead ratio -- see the derivation above. */
int orc_delayed_ratio(orc_delayed *h, int j, const double *v, double *R_out)
{
    const int n = h->n, m = h->m, K = h->K;
    if (j < 0 || j >= n) return ORC_EINVAL;
    const double *rowj = h->B + (size_t)j * n;        /* B0[j,:] (stale) */
    double d = 0.0;
    for (int k = 0; k < n; ++k) d += rowj[k] * v[k];
    double R = d;
    for (int i = 0; i < m; ++i) {
        double s = 0.0, t = 0.0;
        for (int k = 0; k < n; ++k) s += rowj[k] * h->C[(size_t)i * n + k];
        for (int k = 0; k < n; ++k) t += h->W[(size_t)i * n + k] * v[k];
        h->sp[i] = s;
        h->sq[i] = t;
    }
    if (m > 0) {
        /* solve S c = q by LU on a copy of the leading m x m block */
        double *lu = (double *)malloc(sizeof(double) * (size_t)m * m);
        double *c = (double *)malloc(sizeof(double) * (size_t)m);
        int *piv = (int *)malloc(sizeof(int) * (size_t)m);
        if (!lu || !c || !piv) { free(lu); free(c); free(piv); return ORC_ENOMEM; }
        for (int a = 0; a < m; ++a)
            for (int i = 0; i < m; ++i) lu[(size_t)a * m + i] = h->S[(size_t)a * K + i];
        for (int a = 0; a < m; ++a) c[a] = h->sq[a];
        int sign = orc_lu_factor(m, lu, piv);
        if (sign == 0) { free(lu); free(c); free(piv); return ORC_ESINGULAR; }
        orc_lu_solve(m, lu, piv, c, 1);
        double corr = 0.0;
        for (int i = 0; i < m; ++i) {
            double p = h->sp[i] - ((h->J[i] == j) ? 1.0 : 0.0);
            corr += p * c[i];
        }
        R = d - corr;
        free(lu); free(c); free(piv);
    }
    memcpy(h->sv, v, sizeof(double) * (size_t)n);
    h->sj = j; h->sd = d; h->sR = R;
    *R_out = R;
    return ORC_OK;
}

/* Eq. 4: B <- B0 - (B0 C^T - E_J) S^-1 W, any 1 <= m <= K. */
int orc_delayed_flush(orc_delayed *h)
{
    const int n = h->n, m = h->m, K = h->K;
    if (m == 0) return ORC_OK;
    double *lu = (double *)malloc(sizeof(double) * (size_t)m * m);
    double *Y = (double *)malloc(sizeof(double) * (size_t)m * n);
    double *T = (double *)malloc(sizeof(double) * (size_t)n * m);
    int *piv = (int *)malloc(sizeof(int) * (size_t)m);
    if (!lu || !Y || !T || !piv) { free(lu); free(Y); free(T); free(piv); return ORC_ENOMEM; }
    for (int a = 0; a < m; ++a)
        for (int i = 0; i < m; ++i) lu[(size_t)a * m + i] = h->S[(size_t)a * K + i];
    int sign = orc_lu_factor(m, lu, piv);
    if (sign == 0) { free(lu); free(Y); free(T); free(piv); return ORC_ESINGULAR; }
    memcpy(Y, h->W, sizeof(double) * (size_t)m * n);       /* S Y = W */
    orc_lu_solve(m, lu, piv, Y, n);
    for (int i = 0; i < n; ++i)                             /* T = B0 C^T - E_J */
        for (int a = 0; a < m; ++a) {
            double s = 0.0;
            for (int k = 0; k < n; ++k) s += h->B[(size_t)i * n + k] * h->C[(size_t)a * n + k];
            if (h->J[a] == i) s -= 1.0;
            T[(size_t)i * m + a] = s;
        }
    for (int i = 0; i < n; ++i)                             /* B = B0 - T Y */
        for (int a = 0; a < m; ++a) {
            double t = T[(size_t)i * m + a];
            for (int k = 0; k < n; ++k) h->B[(size_t)i * n + k] -= t * Y[(size_t)a * n + k];
        }
    h->m = 0;
    h->sj = -1;
    h->n_flush += 1;
    free(lu); free(Y); free(T); free(piv);
    return ORC_OK;
}

/* Queue the staged move ("A group of accepted changes is queued
 * ... until a preset limit of unapplied moves K is reached").  Appends
 * (j, v, B0[j,:]) and the new row/column/corner of S = W C^T.  When m reaches
 * K the queue is applied (Eq. 4).  Returns 1 if a flush was performed here.
 *
 * Same electron accepted twice inside one window (the paper is silent;
 * DESIGN.md reading G7): two queue entries with equal j would make S
 * singular, so the queue is flushed first and the move is then queued with
 * m = 0 against the fresh inverse (mathematically neutral). */
int orc_delayed_accept(orc_delayed *h)
{
    const int n = h->n, K = h->K;
    if (h->sj < 0) return ORC_EINVAL;
    int j = h->sj, flushed = 0;
    if (h->sR == 0.0 || !isfinite(h->sR)) return ORC_ESINGULAR;
    if (h->replace)
        for (int a = 0; a < h->m; ++a)
            if (h->J[a] == j) {
                /* Path 4 (reading G7, second alternative; the paper is silent,
                 * PAPER.md:84): electron j_a moved again before the queue was applied.  The
                 * current matrix is A0 with column j_a = the NEWEST accepted column, so the
                 * queue entry keeps its slot and its row W[a,:] = B0[j_a,:] and only its column
                 * changes: C[a,:] <- v.  S = W C^T is then rebuilt from its definition (plain
                 * loops, no incremental trick); nothing is flushed and m is unchanged. */
                const int m = h->m;
                memcpy(h->C + (size_t)a * n, h->sv, sizeof(double) * (size_t)n);
                for (int x = 0; x < m; ++x)
                    for (int i = 0; i < m; ++i) {
                        double t = 0.0;
                        for (int k = 0; k < n; ++k) t += h->W[(size_t)x * n + k] * h->C[(size_t)i * n + k];
                        h->S[(size_t)x * K + i] = t;
                    }
                h->sj = -1;
                return 0;
            }
    for (int i = 0; i < h->m; ++i)
        if (h->J[i] == j) {                 /* repeated electron: flush first */
            double *v = (double *)malloc(sizeof(double) * (size_t)n);
            if (!v) return ORC_ENOMEM;
            memcpy(v, h->sv, sizeof(double) * (size_t)n);
            int rc = orc_delayed_flush(h);
            double R;
            if (rc == ORC_OK) rc = orc_delayed_ratio(h, j, v, &R);
            free(v);
            if (rc != ORC_OK) return rc;
            flushed = 1;
            break;
        }
    int m = h->m;
    const double *rowj = h->B + (size_t)j * n;
    /* S[a][m] = W[a,:].v = q_a ; S[m][i] = B0[j,:].C[i,:] ; S[m][m] = d */
    for (int a = 0; a < m; ++a) h->S[(size_t)a * K + m] = h->sq[a];
    for (int i = 0; i < m; ++i) h->S[(size_t)m * K + i] = h->sp[i];
    h->S[(size_t)m * K + m] = h->sd;
    h->J[m] = j;
    memcpy(h->C + (size_t)m * n, h->sv, sizeof(double) * (size_t)n);
    memcpy(h->W + (size_t)m * n, rowj, sizeof(double) * (size_t)n);
    h->m = m + 1;
    h->sj = -1;
    if (h->m == K) {
        int rc = orc_delayed_flush(h);
        if (rc != ORC_OK) return rc;
        flushed = 1;
    }
    return flushed;
}

void orc_delayed_reject(orc_delayed *h) { h->sj = -1; }

/* Read-only views for the pins (P5: det S_m = product of the window's
 * accepted ratios, Eq. 3). */
const double *orc_delayed_S(const orc_delayed *h) { return h->S; }
const int *orc_delayed_J(const orc_delayed *h) { return h->J; }

/* ------------------------------------------------------------------ */
/* Batch driver: `batch` independent walkers, n_moves    */
/* proposals each; move t proposes electron j = (j_begin + t) mod n    */
/* with new column proposals[t][b][:].                                 */
/*   path    1 = rank-1 Sherman-Morrison, 2 = delayed rank-K           */
/*   mode    0 = accept iff mask[t][b] != 0                            */
/*           1 = Metropolis: accept iff uniforms[t][b] < min(1, R^2)   */
/*               (BASELINE.json configs[2]; reading G11)     */
/*   final_flush  apply whatever is still queued at the end            */
/* Outputs R_out[t][b], acc_out[t][b]; B is updated in place.          */
/* Returns 0 or the first error code met.                              */
/* ------------------------------------------------------------------ */
int orc_run(int path, int batch, int n, int K, int n_moves, int j_begin,
            double *B, const double *proposals, const unsigned char *mask,
            const double *uniforms, int mode, int final_flush,
            double *R_out, unsigned char *acc_out, int *threads_used)
{
    if ((path != 1 && path != 2) || batch < 1 || n < 1 || n_moves < 0) return ORC_EINVAL;
    if (mode == 0 && !mask) return ORC_EINVAL;
    if (mode == 1 && !uniforms) return ORC_EINVAL;
    int err = ORC_OK;
    int nthreads = 1;
#ifdef _OPENMP
    nthreads = omp_get_max_threads();
    if (nthreads > batch) nthreads = batch;
#endif
    if (threads_used) *threads_used = nthreads;
#pragma omp parallel for schedule(dynamic, 1) num_threads(nthreads)
    for (int b = 0; b < batch; ++b) {
        double *Bb = B + (size_t)b * n * n;
        orc_delayed *h = NULL;
        int rc = ORC_OK;
        if (path == 2) {
            h = orc_delayed_create(n, K, Bb);
            if (!h) rc = ORC_EINVAL;
        }
        for (int t = 0; t < n_moves && rc == ORC_OK; ++t) {
            int j = (j_begin + t) % n;
            const double *v = proposals + ((size_t)t * batch + b) * n;
            double R;
            if (path == 1) R = orc_sm_ratio(n, Bb, j, v);
            else rc = orc_delayed_ratio(h, j, v, &R);
            if (rc != ORC_OK) break;
            int acc;
            if (mode == 0) {
                acc = mask[(size_t)t * batch + b] != 0;
            } else {
                double pacc = R * R;
                if (pacc > 1.0) pacc = 1.0;
                acc = uniforms[(size_t)t * batch + b] < pacc;
            }
            R_out[(size_t)t * batch + b] = R;
            acc_out[(size_t)t * batch + b] = (unsigned char)acc;
            if (acc) {
                if (path == 1) rc = orc_sm_accept(n, Bb, j, v);
                else { rc = orc_delayed_accept(h); if (rc > 0) rc = ORC_OK; }
            } else if (path == 2) {
                orc_delayed_reject(h);
            }
        }
        if (path == 2 && h) {
            if (rc == ORC_OK && final_flush) rc = orc_delayed_flush(h);
            orc_delayed_destroy(h);
        }
        if (rc != ORC_OK) {
#pragma omp critical
            { if (err == ORC_OK) err = rc; }
        }
    }
    return err;
}

/* ------------------------------------------------------------------ */
/* Path 3: the lock-step variant of PAPER.md:97-99.  */
/* "Rejected moves can be treated similarly to an accepted move, only  */
/* substituting the unchanged matrix columns": EVERY     */
/* proposal occupies a slot of the queue.  An accepted proposal queues */
/* its new column v; a rejected one queues the column the electron     */
/* already has, A_cur[:,j] (a zero column of the paper's U, so it      */
/* changes neither the determinant nor the inverse).  The queue is     */
/* therefore full after exactly K proposals for every walker, and all  */
/* walkers apply Eq. 4 at the same time ("the number of   */
/* operations is fixed").  Written literally: it needs the current     */
/* Slater matrix A (row-major, [batch][n][n], updated in place with    */
/* the accepted columns) to know the unchanged column.                 */
/* mode / mask / uniforms / outputs / final_flush as in orc_run.       */
/* ------------------------------------------------------------------ */
int orc_run_lockstep(int batch, int n, int K, int n_moves, int j_begin,
                     double *A, double *B, const double *proposals,
                     const unsigned char *mask, const double *uniforms, int mode,
                     int final_flush, double *R_out, unsigned char *acc_out,
                     long *flushes_out, int *threads_used)
{
    if (batch < 1 || n < 1 || n_moves < 0 || !A || !B) return ORC_EINVAL;
    if (mode == 0 && !mask) return ORC_EINVAL;
    if (mode == 1 && !uniforms) return ORC_EINVAL;
    int err = ORC_OK;
    int nthreads = 1;
#ifdef _OPENMP
    nthreads = omp_get_max_threads();
    if (nthreads > batch) nthreads = batch;
#endif
    if (threads_used) *threads_used = nthreads;
#pragma omp parallel for schedule(dynamic, 1) num_threads(nthreads)
    for (int b = 0; b < batch; ++b) {
        double *Ab = A + (size_t)b * n * n;
        double *Bb = B + (size_t)b * n * n;
        double *col = (double *)malloc((size_t)n * sizeof(double));
        orc_delayed *h = orc_delayed_create(n, K, Bb);
        int rc = (h && col) ? ORC_OK : ORC_EINVAL;
        for (int t = 0; t < n_moves && rc == ORC_OK; ++t) {
            int j = (j_begin + t) % n;
            const double *v = proposals + ((size_t)t * batch + b) * n;
            double R;
            rc = orc_delayed_ratio(h, j, v, &R);
            if (rc != ORC_OK) break;
            int acc;
            if (mode == 0) {
                acc = mask[(size_t)t * batch + b] != 0;
            } else {
                double pacc = R * R;
                if (pacc > 1.0) pacc = 1.0;
                acc = uniforms[(size_t)t * batch + b] < pacc;
            }
            R_out[(size_t)t * batch + b] = R;
            acc_out[(size_t)t * batch + b] = (unsigned char)acc;
            if (acc) {
                for (int i = 0; i < n; ++i) Ab[(size_t)i * n + j] = v[i];
            } else {
                /* the slot takes the unchanged column */
                double R1;
                for (int i = 0; i < n; ++i) col[i] = Ab[(size_t)i * n + j];
                rc = orc_delayed_ratio(h, j, col, &R1);
                if (rc != ORC_OK) break;
            }
            rc = orc_delayed_accept(h);      /* flushes when all K slots are taken */
            if (rc > 0) rc = ORC_OK;
        }
        if (h) {
            if (rc == ORC_OK && final_flush) rc = orc_delayed_flush(h);
            if (flushes_out) flushes_out[b] = orc_delayed_flush_count(h);
            orc_delayed_destroy(h);
        }
        free(col);
        if (rc != ORC_OK) {
#pragma omp critical
            { if (err == ORC_OK) err = rc; }
        }
    }
    return err;
}

/* Path 4 switch: with `on` != 0, accepting an electron that is already queued replaces the
 * column of its queue slot instead of flushing first (see orc_delayed_accept). */
void orc_delayed_set_replace(orc_delayed *h, int on) { h->replace = on ? 1 : 0; }

/* ------------------------------------------------------------------ */
/* Batch driver with an ARBITRARY electron sequence jseq[t] (the same  */
/* for every walker) -- needed to exercise a repeated electron inside  */
/* one window.  replace = 0: path 2 as it stands (flush first, G7);    */
/* replace = 1: path 4 (slot replacement).  Other arguments as in      */
/* orc_run; flushes_out[b] = number of Eq.-4 applications of walker b. */
/* ------------------------------------------------------------------ */
int orc_run_jseq(int batch, int n, int K, int n_moves, const int *jseq, int replace,
                 double *B, const double *proposals, const unsigned char *mask,
                 const double *uniforms, int mode, int final_flush,
                 double *R_out, unsigned char *acc_out, long *flushes_out, int *threads_used)
{
    if (batch < 1 || n < 1 || n_moves < 0 || !B || (n_moves > 0 && !jseq)) return ORC_EINVAL;
    if (mode == 0 && !mask) return ORC_EINVAL;
    if (mode == 1 && !uniforms) return ORC_EINVAL;
    int err = ORC_OK;
    int nthreads = 1;
#ifdef _OPENMP
    nthreads = omp_get_max_threads();
    if (nthreads > batch) nthreads = batch;
#endif
    if (threads_used) *threads_used = nthreads;
#pragma omp parallel for schedule(dynamic, 1) num_threads(nthreads)
    for (int b = 0; b < batch; ++b) {
        int rc = ORC_OK;
        orc_delayed *h = orc_delayed_create(n, K, B + (size_t)b * n * n);
        if (!h) rc = ORC_EINVAL;
        else orc_delayed_set_replace(h, replace);
        for (int t = 0; t < n_moves && rc == ORC_OK; ++t) {
            const double *v = proposals + ((size_t)t * batch + b) * n;
            double R;
            rc = orc_delayed_ratio(h, jseq[t], v, &R);
            if (rc != ORC_OK) break;
            int acc;
            if (mode == 0) acc = mask[(size_t)t * batch + b] != 0;
            else { double pa = R * R; if (pa > 1.0) pa = 1.0; acc = uniforms[(size_t)t * batch + b] < pa; }
            if (R_out) R_out[(size_t)t * batch + b] = R;
            if (acc_out) acc_out[(size_t)t * batch + b] = (unsigned char)acc;
            if (acc) { int r2 = orc_delayed_accept(h); if (r2 < 0) rc = r2; }
            else orc_delayed_reject(h);
        }
        if (rc == ORC_OK && final_flush) rc = orc_delayed_flush(h);
        if (h && flushes_out) flushes_out[b] = orc_delayed_flush_count(h);
        if (h) orc_delayed_destroy(h);
        if (rc != ORC_OK) {
#pragma omp critical
            { if (err == ORC_OK) err = rc; }
        }
    }
    return err;
}

/* max |A B - I| over all entries (the residual named by BASELINE.json's
 * north_star: "Ainv to max|A.Ainv - I| <= 1e-8 after every flush"). */
double orc_residual(int n, const double *A, const double *B)
{
    double worst = 0.0;
    for (int i = 0; i < n; ++i)
        for (int c = 0; c < n; ++c) {
            double s = 0.0;
            for (int k = 0; k < n; ++k) s += A[(size_t)i * n + k] * B[(size_t)k * n + c];
            if (i == c) s -= 1.0;
            s = fabs(s);
            if (s > worst || s != s) worst = s;
        }
    return worst;
}

int orc_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

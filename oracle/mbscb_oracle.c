/*
 * mbscb_oracle.c — CPU ORACLE.  TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, obviously-correct fp64 implementation of what the hot path
 * computes: transient slab-geometry S_N transport, simple corner balance (SCB)
 * in space and multiple balance (MB) in time, iterated either by one-cell
 * inversion (OCI, parallel block Jacobi) or by source iteration (SI, sweeps).
 * Written from /root/reference/PAPER.md (cited below as P:<line>) in the
 * paper's order and notation.  It shares no code, header, table or helper with
 * the CUDA path under paper_2305_13555_b200/, and neither imports the other.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load this library.
 *
 * What pins it (tests/test_oracle_pins.py, `-m "not gpu"`):
 *   - quadrature: identities + numpy's leggauss
 *   - the 4x4 A+- / b+- / c+- : a whole-problem dense system assembled in the
 *     test directly from the balance equations (4)-(7),(10),(11) and solved
 *     with numpy (brute force), on tiny S2/S4 problems
 *   - MB time stepping: 0-D closed form; SCB space: steady attenuation closed
 *     form; pure absorber -> exp(-Sigma x/mu) at 2nd order
 *   - infinite-medium steady phi = Q/(Sigma-Sigma_s); OCI == SI; particle
 *     balance; LU vs numpy.linalg; spectral radii
 *   - stopping rule: the (d, r) an iteration returns vs numpy max-norms of phi
 *     re-formed from the angular fluxes (maxima placed in a k slot of an
 *     interior cell), and the three branches of converged() with the d = tol r
 *     boundary located by nextafter
 * Parity unpinned (no value printed in the paper): iteration counts and the
 * absolute flux values of the five BASELINE configs (oracle-vs-GPU only).
 *
 * Conventions where the paper is silent or garbled:
 *   angles ascending in mu; reflecting partner of m is N-1-m; reflecting
 *   boundaries are lagged one iteration in both OCI and SI; convergence is
 *   max|phi_new-phi_old| <= tol * max|phi_new| over all cells and four slots,
 *   tested after every iteration; tol < 0 never converges; the iterate is
 *   carried from step to step.
 *
 * Unknown layout in a cell (eqs. 23-24): index 4m+s, m the angle,
 * s in {0:(k,L), 1:(k,R), 2:(k+1/2,L), 3:(k+1/2,R)}.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

enum { ORC_BC_VACUUM = 0, ORC_BC_INCIDENT_ISOTROPIC = 1, ORC_BC_REFLECTING = 2 };

typedef struct {
    int64_t J;          /* cells */
    int32_t N;          /* angles */
    int32_t n;          /* 4N unknowns per cell */
    double v, dt;
    double *dx, *sig, *sigs;          /* [J] */
    int32_t bcL, bcR;
    double bcLv, bcRv;
    double *mu, *w;                   /* [N] Gauss-Legendre, ascending */
    double *psi_prev;                 /* [J][N][2]  psi_{m,k-1/2,j,(L,R)} */
    double *Q;                        /* [J][4] */
    double *Psi, *Psi_old;            /* [J][n] current / previous iterate */
    double *phi, *phi_old;            /* [J][4] */
    int64_t nblk;                     /* distinct (dx,Sigma,Sigma_s) triples */
    int64_t *blk;                     /* [J] -> block id */
    double *LU;                       /* [nblk][n][n] packed L\U, row major */
    int32_t *piv;                     /* [nblk][n] */
    int32_t ready;
    int32_t threads;
} orc_ctx;

/* ------------------------------------------------------------------ */
/* Gauss-Legendre quadrature on [-1,1] ("Gauss Legendre quadrature was
 * used in all"; weights sum to 2, matching the 1/2 in eq. (1)).
 * Newton iteration on the Legendre polynomial P_N via its three-term
 * recurrence; nodes returned ascending.                                  */
void orc_gauss_legendre(int32_t N, double *mu, double *w)
{
    const double pi = 3.14159265358979323846264338327950288;
    for (int32_t i = 0; i < N; ++i) {
        /* i-th root counted from the largest */
        double x = cos(pi * (i + 0.75) / (N + 0.5));
        double dp = 1.0;
        for (int it = 0; it < 100; ++it) {
            double p0 = 1.0, p1 = x;              /* P_0, P_1 */
            for (int32_t k = 2; k <= N; ++k) {
                double pk = ((2.0 * k - 1.0) * x * p1 - (k - 1.0) * p0) / k;
                p0 = p1;
                p1 = pk;
            }
            /* P_N'(x) = N (x P_N - P_{N-1}) / (x^2 - 1) */
            dp = N * (x * p1 - p0) / (x * x - 1.0);
            double dxn = p1 / dp;
            x -= dxn;
            if (fabs(dxn) < 1e-16) break;
        }
        {   /* re-evaluate the derivative at the converged root */
            double p0 = 1.0, p1 = x;
            for (int32_t k = 2; k <= N; ++k) {
                double pk = ((2.0 * k - 1.0) * x * p1 - (k - 1.0) * p0) / k;
                p0 = p1;
                p1 = pk;
            }
            dp = N * (x * p1 - p0) / (x * x - 1.0);
        }
        mu[N - 1 - i] = x;
        w[N - 1 - i] = 2.0 / ((1.0 - x * x) * dp * dp);
    }
}

/* ------------------------------------------------------------------ */
/* The local 4x4 matrix of eqs. (13) (mu>0) and (16) (mu<0),
 * rows 3 (and the duplicated row of (16)) repaired from eqs. (6),(7),(9),(11)
 * (readings G1-G3).  Row major, unknowns
 * [psi_{k,L}, psi_{k,R}, psi_{k+1/2,L}, psi_{k+1/2,R}].
 *
 *   mu>0: diagonal (mu + dx Sigma)/2 ; mu<0: diagonal (-mu + dx Sigma)/2
 *   off-diagonals keep the signed mu.                                     */
void orc_A4(double mu, double dx, double sig, double v, double dt, double *A)
{
    double diag = (mu > 0.0) ? (mu + dx * sig) / 2.0 : (-mu + dx * sig) / 2.0;
    double a_half = dx / (2.0 * v * dt);     /* dx/(2 v dt) */
    double a_full = dx / (v * dt);           /* dx/(v dt)   */
    /* row 0: eq. (4) */
    A[0] = diag;      A[1] = mu / 2.0;  A[2] = a_half;          A[3] = 0.0;
    /* row 1: eq. (5) */
    A[4] = -mu / 2.0; A[5] = diag;      A[6] = 0.0;             A[7] = a_half;
    /* row 2: eq. (6) */
    A[8] = -a_full;   A[9] = 0.0;       A[10] = a_full + diag;  A[11] = mu / 2.0;
    /* row 3: eq. (7) */
    A[12] = 0.0;      A[13] = -a_full;  A[14] = -mu / 2.0;      A[15] = a_full + diag;
}

/* ------------------------------------------------------------------ */
/* Dense LU with partial pivoting and row interchanges, as LAPACK _gesv does
 * (P:208).  A is n x n row major, overwritten by L (unit, below) and U.    */
int32_t orc_lu_factor(int32_t n, double *A, int32_t *piv)
{
    for (int32_t k = 0; k < n; ++k) {
        int32_t p = k;
        double big = fabs(A[(int64_t)k * n + k]);
        for (int32_t i = k + 1; i < n; ++i) {
            double a = fabs(A[(int64_t)i * n + k]);
            if (a > big) { big = a; p = i; }
        }
        piv[k] = p;
        if (big == 0.0) return k + 1;       /* singular */
        if (p != k) {
            for (int32_t c = 0; c < n; ++c) {
                double t = A[(int64_t)k * n + c];
                A[(int64_t)k * n + c] = A[(int64_t)p * n + c];
                A[(int64_t)p * n + c] = t;
            }
        }
        double pivot = A[(int64_t)k * n + k];
        for (int32_t i = k + 1; i < n; ++i) {
            double l = A[(int64_t)i * n + k] / pivot;
            A[(int64_t)i * n + k] = l;
            if (l != 0.0)
                for (int32_t c = k + 1; c < n; ++c)
                    A[(int64_t)i * n + c] -= l * A[(int64_t)k * n + c];
        }
    }
    return 0;
}

/* Solve (P L U) x = b in place in b. */
void orc_lu_solve(int32_t n, const double *LU, const int32_t *piv, double *b)
{
    for (int32_t k = 0; k < n; ++k) {
        int32_t p = piv[k];
        if (p != k) { double t = b[k]; b[k] = b[p]; b[p] = t; }
    }
    for (int32_t i = 1; i < n; ++i) {           /* L y = b */
        double s = b[i];
        for (int32_t k = 0; k < i; ++k) s -= LU[(int64_t)i * n + k] * b[k];
        b[i] = s;
    }
    for (int32_t i = n - 1; i >= 0; --i) {      /* U x = y */
        double s = b[i];
        for (int32_t k = i + 1; k < n; ++k) s -= LU[(int64_t)i * n + k] * b[k];
        b[i] = s / LU[(int64_t)i * n + i];
    }
}

/* ------------------------------------------------------------------ */
/* The OCI cell matrix B = A - S of eq. (19), P:147:
 *   A = blockdiag(A_1..A_N), A_m = A+ or A- by the sign of mu_m (eqs. 20,21);
 *   S couples equal slots of all angles: S[(m,s),(n,s)] = dx Sigma_s/4 * w_n
 *   (eq. 22; slot structure from the per-corner scattering term of
 *   eqs. (4)-(7), reading G5).                                            */
void orc_cell_matrix(int32_t N, const double *mu, const double *w, double dx, double sig,
                     double sigs, double v, double dt, double *B)
{
    int32_t n = 4 * N;
    memset(B, 0, sizeof(double) * (size_t)n * n);
    for (int32_t m = 0; m < N; ++m) {
        double A[16];
        orc_A4(mu[m], dx, sig, v, dt, A);
        for (int r = 0; r < 4; ++r)
            for (int c = 0; c < 4; ++c)
                B[(int64_t)(4 * m + r) * n + (4 * m + c)] = A[4 * r + c];
    }
    for (int32_t m = 0; m < N; ++m)
        for (int s = 0; s < 4; ++s)
            for (int32_t nn = 0; nn < N; ++nn)
                B[(int64_t)(4 * m + s) * n + (4 * nn + s)] -= dx * sigs / 4.0 * w[nn];
}

/* ------------------------------------------------------------------ */
orc_ctx *orc_create(int64_t J, const double *dx, const double *sig, const double *sigs, double v,
                    double dt, int32_t N, int32_t bcL, double bcLv, int32_t bcR, double bcRv)
{
    if (J < 1 || N < 2 || (N & 1) || !(v > 0.0) || !(dt > 0.0) || !dx || !sig || !sigs) return NULL;
    for (int64_t j = 0; j < J; ++j)
        if (!(dx[j] > 0.0) || !(sig[j] >= 0.0) || !(sigs[j] >= 0.0)) return NULL;
    orc_ctx *c = (orc_ctx *)calloc(1, sizeof(orc_ctx));
    c->J = J; c->N = N; c->n = 4 * N; c->v = v; c->dt = dt;
    c->bcL = bcL; c->bcR = bcR; c->bcLv = bcLv; c->bcRv = bcRv;
    size_t sJ = sizeof(double) * (size_t)J;
    c->dx = (double *)malloc(sJ);   memcpy(c->dx, dx, sJ);
    c->sig = (double *)malloc(sJ);  memcpy(c->sig, sig, sJ);
    c->sigs = (double *)malloc(sJ); memcpy(c->sigs, sigs, sJ);
    c->mu = (double *)malloc(sizeof(double) * N);
    c->w = (double *)malloc(sizeof(double) * N);
    orc_gauss_legendre(N, c->mu, c->w);
    c->psi_prev = (double *)calloc((size_t)J * N * 2, sizeof(double));
    c->Q = (double *)calloc((size_t)J * 4, sizeof(double));
    c->Psi = (double *)calloc((size_t)J * c->n, sizeof(double));
    c->Psi_old = (double *)calloc((size_t)J * c->n, sizeof(double));
    c->phi = (double *)calloc((size_t)J * 4, sizeof(double));
    c->phi_old = (double *)calloc((size_t)J * 4, sizeof(double));
    c->blk = (int64_t *)calloc((size_t)J, sizeof(int64_t));
    c->threads = 1;
    return c;
}

void orc_destroy(orc_ctx *c)
{
    if (!c) return;
    free(c->dx); free(c->sig); free(c->sigs); free(c->mu); free(c->w);
    free(c->psi_prev); free(c->Q); free(c->Psi); free(c->Psi_old);
    free(c->phi); free(c->phi_old); free(c->blk); free(c->LU); free(c->piv);
    free(c);
}

void orc_set_threads(orc_ctx *c, int32_t t) { c->threads = t < 1 ? 1 : t; }

int32_t orc_threads_available(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* Form and LU-factor each distinct cell matrix once (dt is fixed, so this is
 * the paper's per-cell `gesv` factorisation hoisted out of the loops).
 * Returns 0, or 1+the first singular block.                               */
int64_t orc_setup(orc_ctx *c)
{
    int64_t J = c->J;
    int32_t n = c->n;
    /* classify cells by bitwise-equal (dx, Sigma, Sigma_s) */
    int64_t *rep = (int64_t *)malloc(sizeof(int64_t) * (size_t)J);
    int64_t nblk = 0;
    for (int64_t j = 0; j < J; ++j) {
        int64_t b = -1;
        for (int64_t q = 0; q < nblk; ++q) {
            int64_t r = rep[q];
            if (c->dx[r] == c->dx[j] && c->sig[r] == c->sig[j] && c->sigs[r] == c->sigs[j]) {
                b = q;
                break;
            }
        }
        if (b < 0) { b = nblk; rep[nblk++] = j; }
        c->blk[j] = b;
    }
    c->nblk = nblk;
    free(c->LU); free(c->piv);
    c->LU = (double *)malloc(sizeof(double) * (size_t)nblk * n * n);
    c->piv = (int32_t *)malloc(sizeof(int32_t) * (size_t)nblk * n);
    int64_t bad = 0;
#ifdef _OPENMP
#pragma omp parallel for num_threads(c->threads) schedule(dynamic, 1)
#endif
    for (int64_t q = 0; q < nblk; ++q) {
        int64_t r = rep[q];
        double *B = c->LU + (size_t)q * n * n;
        orc_cell_matrix(c->N, c->mu, c->w, c->dx[r], c->sig[r], c->sigs[r], c->v, c->dt, B);
        if (orc_lu_factor(n, B, c->piv + (size_t)q * n)) {
#ifdef _OPENMP
#pragma omp critical
#endif
            if (!bad || q + 1 < bad) bad = q + 1;
        }
    }
    free(rep);
    c->ready = (bad == 0);
    return bad;
}

/* phi = sum_n w_n psi_n per slot, eq. (18) */
static void scalar_flux(const orc_ctx *c, const double *Psi, double *phi)
{
    for (int64_t j = 0; j < c->J; ++j)
        for (int s = 0; s < 4; ++s) {
            double acc = 0.0;
            for (int32_t m = 0; m < c->N; ++m) acc += c->w[m] * Psi[j * c->n + 4 * m + s];
            phi[j * 4 + s] = acc;
        }
}

/* Initial condition psi_{m,0}(x) as corner values [J][N][2] = (L,R).
 * Also seeds the iterate: time-average and time-edge slots both start from
 * the initial corner values (reading S3).                                 */
void orc_set_flux(orc_ctx *c, const double *psi_edge)
{
    memcpy(c->psi_prev, psi_edge, sizeof(double) * (size_t)c->J * c->N * 2);
    for (int64_t j = 0; j < c->J; ++j)
        for (int32_t m = 0; m < c->N; ++m) {
            double L = psi_edge[(j * c->N + m) * 2 + 0], R = psi_edge[(j * c->N + m) * 2 + 1];
            double *x = c->Psi + j * c->n + 4 * m;
            x[0] = L; x[1] = R; x[2] = L; x[3] = R;
        }
    scalar_flux(c, c->Psi, c->phi);
}

void orc_set_source(orc_ctx *c, const double *q)
{
    if (q) memcpy(c->Q, q, sizeof(double) * (size_t)c->J * 4);
    else memset(c->Q, 0, sizeof(double) * (size_t)c->J * 4);
}

/* Angular flux incident on cell j in direction m, for the k and k+1/2 balance
 * equations.  `nbr` holds the neighbour cells' values (previous iterate for
 * OCI, P:177-181 superscript (l); the running sweep for SI);
 * `lag` holds the previous iterate, used by reflecting boundaries (S4).
 * Boundary data P:59-61; vacuum / reflecting P:31.                 */
static void incident(const orc_ctx *c, const double *nbr, const double *lag, int64_t j, int32_t m,
                     double *in_k, double *in_kh)
{
    int32_t n = c->n, N = c->N;
    if (c->mu[m] > 0.0) {
        if (j > 0) {                                   /* psi_{m,.,j-1,R}, eq. (10)/(11) */
            *in_k = nbr[(j - 1) * n + 4 * m + 1];
            *in_kh = nbr[(j - 1) * n + 4 * m + 3];
        } else if (c->bcL == ORC_BC_INCIDENT_ISOTROPIC) {
            *in_k = c->bcLv; *in_kh = c->bcLv;
        } else if (c->bcL == ORC_BC_REFLECTING) {      /* outgoing at x=0 of the mirror angle */
            *in_k = lag[0 * n + 4 * (N - 1 - m) + 0];
            *in_kh = lag[0 * n + 4 * (N - 1 - m) + 2];
        } else { *in_k = 0.0; *in_kh = 0.0; }
    } else {
        if (j < c->J - 1) {                            /* psi_{m,.,j+1,L} */
            *in_k = nbr[(j + 1) * n + 4 * m + 0];
            *in_kh = nbr[(j + 1) * n + 4 * m + 2];
        } else if (c->bcR == ORC_BC_INCIDENT_ISOTROPIC) {
            *in_k = c->bcRv; *in_kh = c->bcRv;
        } else if (c->bcR == ORC_BC_REFLECTING) {
            *in_k = lag[(c->J - 1) * n + 4 * (N - 1 - m) + 1];
            *in_kh = lag[(c->J - 1) * n + 4 * (N - 1 - m) + 3];
        } else { *in_k = 0.0; *in_kh = 0.0; }
    }
}

/* max-norms used by the stopping rule (S2) */
static void norms(const orc_ctx *c, double *d, double *r)
{
    double dm = 0.0, rm = 0.0;
    for (int64_t i = 0; i < c->J * 4; ++i) {
        double a = fabs(c->phi[i] - c->phi_old[i]);
        double b = fabs(c->phi[i]);
        if (a > dm) dm = a;
        if (b > rm) rm = b;
    }
    *d = dm; *r = rm;
}

/* One OCI iteration, eqs. (19)-(28): every cell solves
 * (A - S) Psi = c with the incident fluxes taken from the previous iterate. */
void orc_oci_iteration(orc_ctx *c, double *d, double *r)
{
    int64_t J = c->J;
    int32_t n = c->n, N = c->N;
    memcpy(c->Psi_old, c->Psi, sizeof(double) * (size_t)J * n);
    memcpy(c->phi_old, c->phi, sizeof(double) * (size_t)J * 4);
#ifdef _OPENMP
#pragma omp parallel for num_threads(c->threads) schedule(static)
#endif
    for (int64_t j = 0; j < J; ++j) {
        double *rhs = c->Psi + j * n;                  /* solved in place */
        double dxj = c->dx[j];
        double a_half = dxj / (2.0 * c->v * c->dt);
        const double *Qj = c->Q + j * 4;
        for (int32_t m = 0; m < N; ++m) {
            double in_k, in_kh;
            incident(c, c->Psi_old, c->Psi_old, j, m, &in_k, &in_kh);
            double pL = c->psi_prev[(j * N + m) * 2 + 0], pR = c->psi_prev[(j * N + m) * 2 + 1];
            double mu = c->mu[m];
            double *cm = rhs + 4 * m;
            if (mu > 0.0) {                            /* c+, eq. (27) */
                cm[0] = dxj / 4.0 * Qj[0] + a_half * pL + mu * in_k;
                cm[1] = dxj / 4.0 * Qj[1] + a_half * pR;
                cm[2] = dxj / 4.0 * Qj[2] + mu * in_kh;
                cm[3] = dxj / 4.0 * Qj[3];
            } else {                                   /* c-, eq. (28), row 3 per reading G4 */
                cm[0] = dxj / 4.0 * Qj[0] + a_half * pL;
                cm[1] = dxj / 4.0 * Qj[1] + a_half * pR - mu * in_k;
                cm[2] = dxj / 4.0 * Qj[2];
                cm[3] = dxj / 4.0 * Qj[3] - mu * in_kh;
            }
        }
        int64_t b = c->blk[j];
        orc_lu_solve(n, c->LU + (size_t)b * n * n, c->piv + (size_t)b * n, rhs);
    }
    scalar_flux(c, c->Psi, c->phi);
    norms(c, d, r);
}

/* 4x4 solve by Gaussian elimination with partial pivoting */
static void solve4(double *A, double *b)
{
    int32_t piv[4];
    orc_lu_factor(4, A, piv);
    orc_lu_solve(4, A, piv, b);
}

/* One source iteration, eqs. (12)-(18): scattering source from
 * phi^(l); each angle sweeps the cells in its direction of travel.        */
void orc_si_iteration(orc_ctx *c, double *d, double *r)
{
    int64_t J = c->J;
    int32_t n = c->n, N = c->N;
    memcpy(c->Psi_old, c->Psi, sizeof(double) * (size_t)J * n);
    memcpy(c->phi_old, c->phi, sizeof(double) * (size_t)J * 4);
#ifdef _OPENMP
#pragma omp parallel for num_threads(c->threads) schedule(static)
#endif
    for (int32_t m = 0; m < N; ++m) {
        double mu = c->mu[m];
        for (int64_t t = 0; t < J; ++t) {
            int64_t j = (mu > 0.0) ? t : J - 1 - t;    /* direction of travel */
            double dxj = c->dx[j];
            double a_half = dxj / (2.0 * c->v * c->dt);
            const double *Qj = c->Q + j * 4;
            const double *ph = c->phi_old + j * 4;     /* phi^(l) */
            double sgs = c->sigs[j];
            double in_k, in_kh;
            incident(c, c->Psi, c->Psi_old, j, m, &in_k, &in_kh);
            double pL = c->psi_prev[(j * N + m) * 2 + 0], pR = c->psi_prev[(j * N + m) * 2 + 1];
            double A[16], b[4];
            orc_A4(mu, dxj, c->sig[j], c->v, c->dt, A);
            if (mu > 0.0) {                            /* b+, eq. (14) */
                b[0] = dxj / 4.0 * (sgs * ph[0] + Qj[0]) + a_half * pL + mu * in_k;
                b[1] = dxj / 4.0 * (sgs * ph[1] + Qj[1]) + a_half * pR;
                b[2] = dxj / 4.0 * (sgs * ph[2] + Qj[2]) + mu * in_kh;
                b[3] = dxj / 4.0 * (sgs * ph[3] + Qj[3]);
            } else {                                   /* b-, eq. (17) */
                b[0] = dxj / 4.0 * (sgs * ph[0] + Qj[0]) + a_half * pL;
                b[1] = dxj / 4.0 * (sgs * ph[1] + Qj[1]) + a_half * pR - mu * in_k;
                b[2] = dxj / 4.0 * (sgs * ph[2] + Qj[2]);
                b[3] = dxj / 4.0 * (sgs * ph[3] + Qj[3]) - mu * in_kh;
            }
            solve4(A, b);
            double *x = c->Psi + j * n + 4 * m;
            x[0] = b[0]; x[1] = b[1]; x[2] = b[2]; x[3] = b[3];
        }
    }
    scalar_flux(c, c->Psi, c->phi);
    norms(c, d, r);
}

/* After convergence the time-step counter is incremented:
 * the time-edge unknowns become the previous-time-edge data.              */
static void commit(orc_ctx *c)
{
    for (int64_t j = 0; j < c->J; ++j)
        for (int32_t m = 0; m < c->N; ++m) {
            c->psi_prev[(j * c->N + m) * 2 + 0] = c->Psi[j * c->n + 4 * m + 2];
            c->psi_prev[(j * c->N + m) * 2 + 1] = c->Psi[j * c->n + 4 * m + 3];
        }
}

static int converged(double tol, double d, double r) { return tol >= 0.0 && d <= tol * r; }

/* Advance one time step.  Returns 0 converged, 1 max_iters reached (state
 * committed either way), -2 not set up.  resid = d/r (d if r == 0).       */
static int32_t step(orc_ctx *c, int which, double tol, int32_t max_iters, int32_t *iters,
                    double *resid)
{
    if (!c->ready) return -2;
    double d = 0.0, r = 0.0;
    int32_t l = 0, ok = 0;
    while (l < max_iters) {
        if (which == 0) orc_oci_iteration(c, &d, &r);
        else orc_si_iteration(c, &d, &r);
        ++l;
        if (converged(tol, d, r)) { ok = 1; break; }
    }
    commit(c);
    if (iters) *iters = l;
    if (resid) *resid = (r > 0.0) ? d / r : d;
    return ok ? 0 : 1;
}

int32_t orc_oci_step(orc_ctx *c, double tol, int32_t max_iters, int32_t *iters, double *resid)
{
    return step(c, 0, tol, max_iters, iters, resid);
}

int32_t orc_si_step(orc_ctx *c, double tol, int32_t max_iters, int32_t *iters, double *resid)
{
    return step(c, 1, tol, max_iters, iters, resid);
}

void orc_get_scalar_flux(const orc_ctx *c, double *phi)
{
    memcpy(phi, c->phi, sizeof(double) * (size_t)c->J * 4);
}
void orc_get_angular_flux(const orc_ctx *c, double *psi)
{
    memcpy(psi, c->Psi, sizeof(double) * (size_t)c->J * c->n);
}
void orc_get_quadrature(const orc_ctx *c, double *mu, double *w)
{
    memcpy(mu, c->mu, sizeof(double) * c->N);
    memcpy(w, c->w, sizeof(double) * c->N);
}
void orc_get_prev_edge_flux(const orc_ctx *c, double *psi_edge)
{
    memcpy(psi_edge, c->psi_prev, sizeof(double) * (size_t)c->J * c->N * 2);
}
/* Overwrite the iterate only (spectral-radius probes start from an error vector) */
void orc_set_iterate(orc_ctx *c, const double *psi)
{
    memcpy(c->Psi, psi, sizeof(double) * (size_t)c->J * c->n);
    scalar_flux(c, c->Psi, c->phi);
}
int64_t orc_num_blocks(const orc_ctx *c) { return c->nblk; }

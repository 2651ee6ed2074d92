/*
 * gsr_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, single-threaded FP64 CPU restatement of the hot path of the Gaia
 * AVU-GSR solver (arXiv 2308.00778, /root/reference/PAPER.md): the two sparse
 * products aprod1 / aprod2, the column preconditioning, the Eq. 4 norm and the
 * LSQR iteration of Paige & Saunders that the paper runs.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / reference
 * legs may build, load or call this file.  It shares no code, header, table or
 * helper with paper_2308_00778_b200/ (the CUDA path) and neither includes the
 * other.  Build: gcc -O2 -ffp-contract=off -shared -fPIC (no FMA contraction,
 * no reordering: every sum below is evaluated in the order it is written).
 *
 * What pins each function (tests/test_oracle_pins.py, tests/golden/):
 *   col mapping, aprod1, aprod2 : dense expansion + numpy matmul, structure
 *                                 invariants of PAPER.md:78-80, adjoint identity,
 *                                 a hand-worked fixture (tests/golden/hand_system.txt)
 *   norm (Eq. 4)                : equals the Euclidean norm; overflow-safe case
 *   precondition                : unit column norms, ||A'||_F^2 = #non-zero columns
 *   lsqr                        : dense least squares (numpy lstsq), planted
 *                                 solution, scipy.sparse.linalg.lsqr (same algorithm),
 *                                 true residual / A^T r norms per iteration, istop cases
 *   x_k, se (standard errors)   : closed form V_k (B_k^T B_k)^-1 V_k^T from a dense,
 *                                 re-orthogonalised Golub-Kahan bidiagonalisation
 *                                 (k <= 20), upper bound diag((A'^T A')^-1), scipy var
 *   cov (covariances of couples): off-diagonal entries of the same closed form (k <= 20), scaled by the
 *                                 true residual; cov(i,i) = se_i^2; symmetry in (i, j); |cov_ij| <= se_i se_j
 *
 * Matrix definition (PAPER.md:78-80 and the index expressions
 * of Algorithm 2).  Row i of A holds
 * N_par = nAstro + nAtt + nInstrPar + nGlob stored coefficients V[i*N_par + k] in the section order
 *   [ nAstro astrometric | nAtt attitude = 3 axes x 4 | nInstrPar instrumental | nGlob global ]
 * with 0 <= nAstro <= 5, nAtt = 12 or 0, 0 <= nInstrPar <= 6, nGlob >= 0 ("0 <= N_Astro <= 5",
 * "N_Att = 12", "0 <= N_Instr <= 6", N_Glob = 1 "or ... without computing a global part"; the paper also ran
 * 5 global parameters, and its 40 / 100 / 300 GB datasets solve only some of the sections,
 * PAPER.md:263).  The production layout is 5 / 12 / 6 / 1, N_par = 24.  A section of width 0 has no
 * columns.  With kA = nAstro, kT = kA + nAtt, kI = kT + nInstrPar, coefficient k sits in column
 *   k < kA : ia[i] + k                                   (ia[i] = nAstro*star(i))
 *   k < kT : offAtt + a*nDofAtt + iatt[i] + j            a=(k-kA)/4, j=(k-kA)%4;  offAtt = nAstro*nStars
 *   k < kI : offInstr + ic[i*nInstrPar + (k-kT)]         offInstr = offAtt + (nAtt ? 3*nDofAtt : 0)
 *   else   : offGlob + (k-kI)                            offGlob = offInstr + (nInstrPar ? nInstr : 0)
 *                                                        (Alg. 2 "glob": x[j + offset])
 * Constraint rows are generic sparse rows appended below
 * the observation rows, given as CSR (rowptr, col, val) with absolute columns.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define N_AXES 3
#define N_PAR_AXIS 4

typedef struct {
    int64_t n_obs;      /* observation rows m                                  */
    int64_t n_stars;    /* N_Stars                                             */
    int64_t n_dof_att;  /* N_DFA, per axis                                     */
    int64_t n_instr;    /* number of instrumental columns                      */
    int64_t n_con;      /* constraint rows                                     */
    int64_t n_glob;     /* N_Glob global columns (1 in production)*/
    double *V;          /* [n_obs*N_par] row-major A_d           */
    const int64_t *ia;  /* [n_obs]   M_i astro part: N_Astro*star, non-decreasing */
    const int64_t *iatt;/* [n_obs]   M_i attitude part: start s_i, axis 0      */
    const int32_t *ic;  /* [n_obs*N_Instr] I_c instrumental columns            */
    const int64_t *con_rowptr; /* [n_con+1]                                    */
    const int64_t *con_col;    /* [nnz] absolute columns                       */
    double *con_val;           /* [nnz]                                        */
    int64_t n_astro_par; /* N_Astro, 0..5 coefficients (and unknowns) per star */
    int64_t n_att_par;   /* N_Att, 12 (3 axes x 4) or 0                        */
    int64_t n_instr_par; /* N_Instr, 0..6 coefficients per row                 */
} gsr_oracle_system;

/* first column of the attitude, instrumental and global sections (a section of width 0 has no columns) */
static int64_t off_att(const gsr_oracle_system *S) { return S->n_astro_par * S->n_stars; }
static int64_t off_instr(const gsr_oracle_system *S) { return off_att(S) + (S->n_att_par ? N_AXES * S->n_dof_att : 0); }
static int64_t off_glob(const gsr_oracle_system *S) { return off_instr(S) + (S->n_instr_par ? S->n_instr : 0); }

int64_t gsr_oracle_ncols(const gsr_oracle_system *S) { return off_glob(S) + S->n_glob; }

static int npar(const gsr_oracle_system *S)
{
    return (int)(S->n_astro_par + S->n_att_par + S->n_instr_par + S->n_glob);
}

/* Column of stored coefficient k of observation row i (see header). */
int64_t gsr_oracle_col(const gsr_oracle_system *S, int64_t i, int k)
{
    const int kA = (int)S->n_astro_par, kT = kA + (int)S->n_att_par, kI = kT + (int)S->n_instr_par;
    if (k < kA)
        return S->ia[i] + k;
    if (k < kT) {
        int a = (k - kA) / N_PAR_AXIS, j = (k - kA) % N_PAR_AXIS;
        return off_att(S) + (int64_t)a * S->n_dof_att + S->iatt[i] + j;
    }
    if (k < kI)
        return off_instr(S) + S->ic[i * S->n_instr_par + (k - kT)];
    return off_glob(S) + (k - kI);
}

/*
 * aprod mode 1, Eq. 2 "b += A x"; Algorithm 2 left column
 * (PAPER.md:270-312): per row, sum the 24 products in k order, then
 * b[i] = b[i] + sum.  Constraint rows follow ("Constraints
 * computation", Alg. 2 o.29).  y has n_obs + n_con entries.  If abs_y != NULL it
 * receives |y_in[i]| + sum_k |V x| (the bound used by the 1e-12 tolerance).
 */
void gsr_oracle_aprod1(const gsr_oracle_system *S, const double *x, double *y, double *abs_y)
{
    const int N_PAR = npar(S);
    for (int64_t i = 0; i < S->n_obs; ++i) {
        double sum = 0.0, asum = 0.0;
        for (int k = 0; k < N_PAR; ++k) {
            double t = S->V[i * N_PAR + k] * x[gsr_oracle_col(S, i, k)];
            sum = sum + t;
            asum = asum + fabs(t);
        }
        if (abs_y)
            abs_y[i] = fabs(y[i]) + asum;
        y[i] = y[i] + sum;
    }
    for (int64_t r = 0; r < S->n_con; ++r) {
        double sum = 0.0, asum = 0.0;
        for (int64_t q = S->con_rowptr[r]; q < S->con_rowptr[r + 1]; ++q) {
            double t = S->con_val[q] * x[S->con_col[q]];
            sum = sum + t;
            asum = asum + fabs(t);
        }
        if (abs_y)
            abs_y[S->n_obs + r] = fabs(y[S->n_obs + r]) + asum;
        y[S->n_obs + r] = y[S->n_obs + r] + sum;
    }
}

/*
 * aprod mode 2, Eq. 3 "x += A^T b"; Algorithm 3 left column
 * (PAPER.md:485-576): rows in order, the 24 coefficients of a row in k order,
 * x[col] += V * y[i].  abs_x (optional) accumulates |x_in| + sum |V y|.
 */
void gsr_oracle_aprod2(const gsr_oracle_system *S, const double *y, double *x, double *abs_x)
{
    const int64_t n = gsr_oracle_ncols(S);
    const int N_PAR = npar(S);
    if (abs_x)
        for (int64_t j = 0; j < n; ++j)
            abs_x[j] = fabs(x[j]);
    for (int64_t i = 0; i < S->n_obs; ++i) {
        for (int k = 0; k < N_PAR; ++k) {
            int64_t c = gsr_oracle_col(S, i, k);
            double t = S->V[i * N_PAR + k] * y[i];
            x[c] = x[c] + t;
            if (abs_x)
                abs_x[c] = abs_x[c] + fabs(t);
        }
    }
    for (int64_t r = 0; r < S->n_con; ++r) {
        for (int64_t q = S->con_rowptr[r]; q < S->con_rowptr[r + 1]; ++q) {
            int64_t c = S->con_col[q];
            double t = S->con_val[q] * y[S->n_obs + r];
            x[c] = x[c] + t;
            if (abs_x)
                abs_x[c] = abs_x[c] + fabs(t);
        }
    }
}

/*
 * Eq. 4: |a| = max(a) * sqrt( sum_i a_i^2 / max(a)^2 ), with
 * max(a) = max_i |a_i|.  Returns 0 for the zero vector.
 */
double gsr_oracle_norm(const double *a, int64_t n)
{
    double mx = 0.0;
    for (int64_t i = 0; i < n; ++i)
        if (fabs(a[i]) > mx)
            mx = fabs(a[i]);
    if (mx == 0.0)
        return 0.0;
    double s = 0.0;
    for (int64_t i = 0; i < n; ++i) {
        double q = a[i] / mx;
        s = s + q * q;
    }
    return mx * sqrt(s);
}

/*
 * Column preconditioning (Alg. 1 l.2-3): "we
 * normalized the parameters of each column by the norm of the column itself",
 * the factors stored in p and the solution "re-multiplied by p" afterwards.
 * Reading (R1-R4): nrm_j = sqrt(sum_i A_ij^2) over all rows including
 * constraints, p_j = 1/nrm_j (1 if the column is empty), A_ij <- fl(A_ij * p_j)
 * in place.
 */
void gsr_oracle_precondition(gsr_oracle_system *S, double *p)
{
    const int64_t n = gsr_oracle_ncols(S);
    const int N_PAR = npar(S);
    for (int64_t j = 0; j < n; ++j)
        p[j] = 0.0;
    for (int64_t i = 0; i < S->n_obs; ++i)
        for (int k = 0; k < N_PAR; ++k) {
            double v = S->V[i * N_PAR + k];
            p[gsr_oracle_col(S, i, k)] += v * v;
        }
    for (int64_t r = 0; r < S->n_con; ++r)
        for (int64_t q = S->con_rowptr[r]; q < S->con_rowptr[r + 1]; ++q)
            p[S->con_col[q]] += S->con_val[q] * S->con_val[q];
    for (int64_t j = 0; j < n; ++j)
        p[j] = (p[j] > 0.0) ? 1.0 / sqrt(p[j]) : 1.0;
    for (int64_t i = 0; i < S->n_obs; ++i)
        for (int k = 0; k < N_PAR; ++k)
            S->V[i * N_PAR + k] = S->V[i * N_PAR + k] * p[gsr_oracle_col(S, i, k)];
    for (int64_t r = 0; r < S->n_con; ++r)
        for (int64_t q = S->con_rowptr[r]; q < S->con_rowptr[r + 1]; ++q)
            S->con_val[q] = S->con_val[q] * p[S->con_col[q]];
}

typedef struct {
    int32_t istop;
    int64_t itn;
    double anorm, acond, rnorm, arnorm, xnorm;
} gsr_oracle_result;

/*
 * LSQR (Paige & Saunders 1982, cited PAPER.md:34, 742-743; the loop is
 * Alg. 1 l.17-26), damp = 0, on the system as it stands in S
 * (already preconditioned or not).  Steps and notation follow SURVEY.md 8(c).3.
 * b has n_obs+n_con entries and is not modified.  z (n) receives the solution of
 * the system in S, var (n) the accumulated sum_k (w_k/rho_k)^2.  If p != NULL,
 * x = p (.) z and se = p (.) se_z (Alg. 1 l.27) are written to
 * x / se instead of z / se_z.  trace, if not NULL, receives 5 doubles per
 * iteration: rnorm, arnorm, anorm, acond, xnorm.
 */
static int lsqr_body(const gsr_oracle_system *S, const double *b, int64_t itnlim, double atol,
                     double btol, double conlim, const double *p, double *x, double *se,
                     gsr_oracle_result *R, double *trace, int64_t npairs, const int64_t *pi,
                     const int64_t *pj, double *cov);

int gsr_oracle_lsqr(const gsr_oracle_system *S, const double *b, int64_t itnlim, double atol,
                    double btol, double conlim, const double *p, double *x, double *se,
                    gsr_oracle_result *R, double *trace)
{
    return lsqr_body(S, b, itnlim, atol, btol, conlim, p, x, se, R, trace, 0, NULL, NULL, NULL);
}

/*
 * The same solve, with the covariances between chosen couples of unknowns ("the errors
 * (variances) on the unknowns and the covariances between the different couples of unknowns are
 * calculated"; Alg. 1 l.26-27).  The paper names neither the couples nor a formula
 * (reading R26): the couples (pi[q], pj[q]), q < npairs, are the caller's, and the estimate is
 * the one LSQR's variances are the diagonal of -- Paige & Saunders' sum_k d_k d_k^T with d_k = w_k/rho_k,
 * which tends to (A'^T A')^-1 -- scaled like the standard errors: with s = rnorm/sqrt(m - n) (s = rnorm
 * when m <= n),
 *     cov[q] = p_i p_j s^2 sum_k d_k[i] d_k[j],     i = pi[q], j = pj[q],
 * so that cov(i, i) = se_i^2.  Everything else is gsr_oracle_lsqr, step for step.
 */
int gsr_oracle_lsqr_cov(const gsr_oracle_system *S, const double *b, int64_t itnlim, double atol,
                        double btol, double conlim, const double *p, double *x, double *se,
                        gsr_oracle_result *R, double *trace, int64_t npairs, const int64_t *pi,
                        const int64_t *pj, double *cov)
{
    return lsqr_body(S, b, itnlim, atol, btol, conlim, p, x, se, R, trace, npairs, pi, pj, cov);
}

static int lsqr_body(const gsr_oracle_system *S, const double *b, int64_t itnlim, double atol,
                     double btol, double conlim, const double *p, double *x, double *se,
                     gsr_oracle_result *R, double *trace, int64_t npairs, const int64_t *pi,
                     const int64_t *pj, double *cov)
{
    const int64_t n = gsr_oracle_ncols(S);
    const int64_t m = S->n_obs + S->n_con;
    double *u = (double *)malloc(sizeof(double) * (size_t)(m > 0 ? m : 1));
    double *v = (double *)calloc((size_t)n, sizeof(double));
    double *w = (double *)calloc((size_t)n, sizeof(double));
    if (!u || !v || !w) {
        free(u); free(v); free(w);
        return -1;
    }
    int32_t istop = 0;
    int64_t itn = 0;
    double anorm = 0.0, acond = 0.0, ddnorm = 0.0, xxnorm = 0.0, xnorm = 0.0, z = 0.0;
    double cs2 = -1.0, sn2 = 0.0, arnorm = 0.0;
    const double ctol = (conlim > 0.0) ? 1.0 / conlim : 0.0;

    /* step 1: x = 0, var = 0, u = b, beta = |u|, u /= beta, v = A^T u, alpha = |v|, v /= alpha, w = v */
    for (int64_t j = 0; j < n; ++j) {
        x[j] = 0.0;
        se[j] = 0.0; /* holds var until the finish step */
    }
    for (int64_t q = 0; q < npairs; ++q)
        cov[q] = 0.0; /* holds sum_k d_k[i] d_k[j] until the finish step */
    memcpy(u, b, sizeof(double) * (size_t)m);
    double alpha = 0.0;
    double beta = gsr_oracle_norm(u, m);
    if (beta > 0.0) {
        for (int64_t i = 0; i < m; ++i)
            u[i] = u[i] / beta;
        gsr_oracle_aprod2(S, u, v, NULL); /* "initial solution" via aprod 2 */
        alpha = gsr_oracle_norm(v, n);
    }
    if (alpha > 0.0) {
        for (int64_t j = 0; j < n; ++j)
            v[j] = v[j] / alpha;
        memcpy(w, v, sizeof(double) * (size_t)n);
    }
    double rhobar = alpha, phibar = beta;
    const double bnorm = beta;
    double rnorm = beta;
    arnorm = alpha * beta;

    if (arnorm != 0.0) {
        while (itn < itnlim) {
            /* step 2: bidiagonalisation */
            itn = itn + 1;
            for (int64_t i = 0; i < m; ++i)
                u[i] = -alpha * u[i];
            gsr_oracle_aprod1(S, v, u, NULL);
            beta = gsr_oracle_norm(u, m);
            if (beta > 0.0) {
                for (int64_t i = 0; i < m; ++i)
                    u[i] = u[i] / beta;
                anorm = sqrt(anorm * anorm + alpha * alpha + beta * beta);
                for (int64_t j = 0; j < n; ++j)
                    v[j] = -beta * v[j];
                gsr_oracle_aprod2(S, u, v, NULL);
                alpha = gsr_oracle_norm(v, n);
                if (alpha > 0.0)
                    for (int64_t j = 0; j < n; ++j)
                        v[j] = v[j] / alpha;
            }
            /* step 3: plane rotation */
            const double rho = sqrt(rhobar * rhobar + beta * beta);
            const double cs = rhobar / rho;
            const double sn = beta / rho;
            const double theta = sn * alpha;
            rhobar = -cs * alpha;
            const double phi = cs * phibar;
            phibar = sn * phibar;
            const double tau = sn * phi;
            /* step 4: update x, w, var */
            const double t1 = phi / rho;
            const double t2 = -theta / rho;
            for (int64_t q = 0; q < npairs; ++q) { /* before w is overwritten: d_k = w_k / rho_k */
                const double di = w[pi[q]] / rho;
                const double dj = w[pj[q]] / rho;
                cov[q] = cov[q] + di * dj;
            }
            for (int64_t j = 0; j < n; ++j) {
                const double dk = w[j] / rho;
                x[j] = x[j] + t1 * w[j];
                w[j] = v[j] + t2 * w[j];
                se[j] = se[j] + dk * dk;
                ddnorm = ddnorm + dk * dk;
            }
            /* step 5: norm of x */
            const double delta = sn2 * rho;
            const double gambar = -cs2 * rho;
            const double rhs = phi - delta * z;
            const double zbar = rhs / gambar;
            xnorm = sqrt(xxnorm + zbar * zbar);
            const double gamma = sqrt(gambar * gambar + theta * theta);
            cs2 = gambar / gamma;
            sn2 = theta / gamma;
            z = rhs / gamma;
            xxnorm = xxnorm + z * z;
            /* step 6: estimates */
            acond = anorm * sqrt(ddnorm);
            rnorm = phibar;
            arnorm = alpha * fabs(tau);
            if (trace) {
                double *t = trace + 5 * (itn - 1);
                t[0] = rnorm; t[1] = arnorm; t[2] = anorm; t[3] = acond; t[4] = xnorm;
            }
            /* step 7: stopping tests, later assignments override earlier ones */
            const double test1 = rnorm / bnorm;
            const double test2 = (anorm * rnorm != 0.0) ? arnorm / (anorm * rnorm) : 0.0;
            const double test3 = 1.0 / acond;
            const double t1p = test1 / (1.0 + anorm * xnorm / bnorm);
            const double rtol = btol + atol * anorm * xnorm / bnorm;
            if (itn >= itnlim) istop = 7;
            if (1.0 + test3 <= 1.0) istop = 6;
            if (1.0 + test2 <= 1.0) istop = 5;
            if (1.0 + t1p <= 1.0) istop = 4;
            if (test3 <= ctol) istop = 3;
            if (test2 <= atol) istop = 2;
            if (test1 <= rtol) istop = 1;
            if (istop != 0)
                break;
        }
    }
    /* step 8: standard errors, then un-scaling by p */
    {
        double s = rnorm;
        if (m > n)
            s = rnorm / sqrt((double)(m - n));
        for (int64_t j = 0; j < n; ++j)
            se[j] = sqrt(se[j]) * s;
        for (int64_t q = 0; q < npairs; ++q)
            cov[q] = cov[q] * (s * s);
    }
    if (p) {
        for (int64_t j = 0; j < n; ++j) {
            x[j] = p[j] * x[j];
            se[j] = p[j] * se[j];
        }
        for (int64_t q = 0; q < npairs; ++q)
            cov[q] = p[pi[q]] * p[pj[q]] * cov[q];
    }
    R->istop = istop;
    R->itn = itn;
    R->anorm = anorm;
    R->acond = acond;
    R->rnorm = rnorm;
    R->arnorm = arnorm;
    R->xnorm = xnorm;
    free(u); free(v); free(w);
    return 0;
}

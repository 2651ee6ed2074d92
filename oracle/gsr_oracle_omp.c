/*
 * gsr_oracle_omp.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE, AND NOT THE PARITY ORACLE.
 *
 * The loops of gsr_oracle.c threaded with OpenMP the way the paper's production CPU solver is
 * (section 3.1): aprod1 is a `#pragma omp for` over the observation rows; aprod2
 * gives every thread a contiguous row range [N_t[tid][0], N_t[tid][1]) cut on star boundaries, so
 * the astrometric columns of a thread are its own, while the attitude / instrumental / global
 * columns (shared between threads) go to per-thread private accumulators that are summed in thread
 * order afterwards.  LSQR is the same Paige-Saunders recurrence on top of them.
 *
 * Used ONLY by bench.py's `cpu_baseline` / `--impl reference` legs to report the oracle on all host
 * cores; tests/test_oracle_pins.py checks it against the single-thread oracle
 * within 1e-12 * sum|terms| (aprod) and 1e-10 (LSQR x).  gsr_oracle.c stays the parity oracle.
 * Shares no code with gsr_oracle.c or with paper_2308_00778_b200/.
 * Build: gcc -O2 -fopenmp -ffp-contract=off -shared -fPIC.
 */
#include <math.h>
#include <omp.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

enum { NA = 5, NAX = 3, NPA = 4, NATT = 12, NI = 6, NF = 23 };   /* row width 23 + n_glob */

/* same leading fields as gsr_oracle_system (oracle/__init__.py passes one ctypes struct to both; the section
 * widths that follow there are 5 / 12 / 6 here, checked by the Python side) */
typedef struct {
    int64_t n_obs, n_stars, n_dof_att, n_instr, n_con, n_glob;
    double *V;
    const int64_t *ia, *iatt;
    const int32_t *ic;
    const int64_t *con_rowptr, *con_col;
    double *con_val;
} omp_system;

static int64_t ncols(const omp_system *S) { return NA * S->n_stars + NAX * S->n_dof_att + S->n_instr + S->n_glob; }

int gsr_omp_threads(void) { return omp_get_max_threads(); }
void gsr_omp_set_threads(int t) { omp_set_num_threads(t > 0 ? t : 1); }

/* Eq. 2, rows shared out with `omp for` */
void gsr_omp_aprod1(const omp_system *S, const double *x, double *y)
{
    const int64_t offAtt = NA * S->n_stars, offIns = offAtt + NAX * S->n_dof_att, offGlob = offIns + S->n_instr;
    const int NP = NF + (int)S->n_glob;
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < S->n_obs; ++i) {
        const double *v = S->V + i * NP;
        double sum = 0.0;
        for (int k = 0; k < NA; ++k) sum += v[k] * x[S->ia[i] + k];
        for (int a = 0; a < NAX; ++a)
            for (int j = 0; j < NPA; ++j) sum += v[NA + a * NPA + j] * x[offAtt + a * S->n_dof_att + S->iatt[i] + j];
        for (int j = 0; j < NI; ++j) sum += v[NA + NATT + j] * x[offIns + S->ic[i * NI + j]];
        for (int g = 0; g < S->n_glob; ++g) sum += v[NF + g] * x[offGlob + g];
        y[i] += sum;
    }
#pragma omp parallel for schedule(static)
    for (int64_t r = 0; r < S->n_con; ++r) {
        double sum = 0.0;
        for (int64_t q = S->con_rowptr[r]; q < S->con_rowptr[r + 1]; ++q) sum += S->con_val[q] * x[S->con_col[q]];
        y[S->n_obs + r] += sum;
    }
}

/* Eq. 3 with the thread ranges N_t of PAPER.md:150 */
void gsr_omp_aprod2(const omp_system *S, const double *y, double *x)
{
    const int64_t n = ncols(S), offAtt = NA * S->n_stars, offIns = offAtt + NAX * S->n_dof_att;
    const int64_t nShared = n - offAtt;
    const int NP = NF + (int)S->n_glob;
    const int T = omp_get_max_threads();
    double *priv = (double *)calloc((size_t)T * (size_t)nShared, sizeof(double));
    int64_t *Nt = (int64_t *)malloc(sizeof(int64_t) * (size_t)(T + 1));
    for (int t = 0; t <= T; ++t) {
        int64_t r = S->n_obs * t / T;
        while (r > 0 && r < S->n_obs && S->ia[r] == S->ia[r - 1]) ++r;   /* move the cut to the next star boundary */
        Nt[t] = r;
    }
#pragma omp parallel num_threads(T)
    {
        const int tid = omp_get_thread_num();
        double *p = priv + (size_t)tid * (size_t)nShared;
        for (int64_t i = Nt[tid]; i < Nt[tid + 1]; ++i) {
            const double *v = S->V + i * NP;
            const double yi = y[i];
            for (int k = 0; k < NA; ++k) x[S->ia[i] + k] += v[k] * yi;
            for (int a = 0; a < NAX; ++a)
                for (int j = 0; j < NPA; ++j) p[a * S->n_dof_att + S->iatt[i] + j] += v[NA + a * NPA + j] * yi;
            for (int j = 0; j < NI; ++j) p[(offIns - offAtt) + S->ic[i * NI + j]] += v[NA + NATT + j] * yi;
            for (int g = 0; g < S->n_glob; ++g) p[nShared - S->n_glob + g] += v[NF + g] * yi;
        }
#pragma omp barrier
#pragma omp for schedule(static)
        for (int64_t c = 0; c < nShared; ++c) {
            double s = 0.0;
            for (int t = 0; t < T; ++t) s += priv[(size_t)t * (size_t)nShared + c];
            x[offAtt + c] += s;
        }
    }
    /* constraint rows: few and wide; one thread (their columns are shared by all rows) */
    for (int64_t r = 0; r < S->n_con; ++r)
        for (int64_t q = S->con_rowptr[r]; q < S->con_rowptr[r + 1]; ++q)
            x[S->con_col[q]] += S->con_val[q] * y[S->n_obs + r];
    free(priv);
    free(Nt);
}

static double nrm2(const double *a, int64_t n)
{
    double mx = 0.0, s = 0.0;
#pragma omp parallel for reduction(max : mx) schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        const double t = fabs(a[i]);
        if (t > mx) mx = t;
    }
    if (mx == 0.0) return 0.0;
#pragma omp parallel for reduction(+ : s) schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        const double q = a[i] / mx;
        s += q * q;
    }
    return mx * sqrt(s);   /* Eq. 4 */
}

static void scal(double *a, int64_t n, double c)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) a[i] *= c;
}

typedef struct {
    int32_t istop;
    int64_t itn;
    double anorm, acond, rnorm, arnorm, xnorm;
} omp_result;

int gsr_omp_lsqr(const omp_system *S, const double *b, int64_t itnlim, double atol, double btol, double conlim,
                 const double *p, double *x, double *se, omp_result *R)
{
    const int64_t n = ncols(S), m = S->n_obs + S->n_con;
    double *u = (double *)malloc(sizeof(double) * (size_t)(m > 0 ? m : 1));
    double *v = (double *)calloc((size_t)n, sizeof(double));
    double *w = (double *)calloc((size_t)n, sizeof(double));
    if (!u || !v || !w) { free(u); free(v); free(w); return -1; }
    int32_t istop = 0;
    int64_t itn = 0;
    double anorm = 0, acond = 0, ddnorm = 0, xxnorm = 0, xnorm = 0, z = 0, cs2 = -1.0, sn2 = 0.0;
    const double ctol = conlim > 0.0 ? 1.0 / conlim : 0.0;
    memset(x, 0, sizeof(double) * (size_t)n);
    memset(se, 0, sizeof(double) * (size_t)n);
    memcpy(u, b, sizeof(double) * (size_t)m);
    double alpha = 0.0, beta = nrm2(u, m);
    if (beta > 0.0) {
        scal(u, m, 1.0 / beta);
        gsr_omp_aprod2(S, u, v);
        alpha = nrm2(v, n);
    }
    if (alpha > 0.0) {
        scal(v, n, 1.0 / alpha);
        memcpy(w, v, sizeof(double) * (size_t)n);
    }
    double rhobar = alpha, phibar = beta, rnorm = beta, arnorm = alpha * beta;
    const double bnorm = beta;
    if (arnorm != 0.0) {
        while (itn < itnlim) {
            ++itn;
            scal(u, m, -alpha);
            gsr_omp_aprod1(S, v, u);
            beta = nrm2(u, m);
            if (beta > 0.0) {
                scal(u, m, 1.0 / beta);
                anorm = sqrt(anorm * anorm + alpha * alpha + beta * beta);
                scal(v, n, -beta);
                gsr_omp_aprod2(S, u, v);
                alpha = nrm2(v, n);
                if (alpha > 0.0) scal(v, n, 1.0 / alpha);
            }
            const double rho = sqrt(rhobar * rhobar + beta * beta), cs = rhobar / rho, sn = beta / rho;
            const double theta = sn * alpha;
            rhobar = -cs * alpha;
            const double phi = cs * phibar;
            phibar = sn * phibar;
            const double tau = sn * phi, t1 = phi / rho, t2 = -theta / rho;
            double dd = 0.0;
#pragma omp parallel for reduction(+ : dd) schedule(static)
            for (int64_t j = 0; j < n; ++j) {
                const double dk = w[j] / rho;
                x[j] += t1 * w[j];
                w[j] = v[j] + t2 * w[j];
                se[j] += dk * dk;
                dd += dk * dk;
            }
            ddnorm += dd;
            const double delta = sn2 * rho, gambar = -cs2 * rho, rhs = phi - delta * z, zbar = rhs / gambar;
            xnorm = sqrt(xxnorm + zbar * zbar);
            const double gamma = sqrt(gambar * gambar + theta * theta);
            cs2 = gambar / gamma;
            sn2 = theta / gamma;
            z = rhs / gamma;
            xxnorm += z * z;
            acond = anorm * sqrt(ddnorm);
            rnorm = phibar;
            arnorm = alpha * fabs(tau);
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
            if (istop) break;
        }
    }
    double s = rnorm;
    if (m > n) s = rnorm / sqrt((double)(m - n));
    for (int64_t j = 0; j < n; ++j) {
        se[j] = sqrt(se[j]) * s;
        if (p) { x[j] *= p[j]; se[j] *= p[j]; }
    }
    R->istop = istop; R->itn = itn; R->anorm = anorm; R->acond = acond;
    R->rnorm = rnorm; R->arnorm = arnorm; R->xnorm = xnorm;
    free(u); free(v); free(w);
    return 0;
}

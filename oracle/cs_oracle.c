/*
 * cs_oracle.c -- plain, slow, obviously-correct CPU fp64 oracle for the batched spectral likelihood.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call this file.  It shares no code, header, table or constant
 * generator with the CUDA library (paper_2604_08463_b200/csrc) and neither imports the other.
 *
 * What it computes, written from the paper (arxiv 2604.08463, /root/reference/PAPER.md) with the readings
 * R1-R11 of SURVEY.md 8(c) (listed again in DESIGN.md):
 *
 *   for every pixel p whose three cluster ids are >= 0:
 *     A[f,:]  = (1, a_d(nu_f; beta_d[k0], T_d[k1]), a_s(nu_f; beta_s[k2]))        Eq. 2
 *     M       = A^T diag(Ninv) A ;  b_S = A^T diag(Ninv) d_S,  S = Q, U            PAPER.md:L233, Eq. 5
 *     s_S     = M^-1 b_S                                                            Eq. 5 / Eq. 8
 *     nll    += -1/2 sum_S b_S . s_S                                                Eq. 6 negated, const = 0, L80
 *     w_S     = Ninv * (d_S - A s_S)
 *     grad[k] += - sum_S w_S^T (dA/dtheta_k) s_S                                    Eq. 17, L241 (factor: R4)
 *     maps[:,S,p] = s_S
 *
 * No tables, no blocking, no fusion: the SED is evaluated directly per pixel, M is solved by Gaussian
 * elimination with partial pivoting, sums over pixels are accumulated in long double in pixel order.
 * Parity pins (tests/test_oracle_pins.py): a(nu0)=1, RJ limit, W A = I (Eq. 11), normal equations,
 * noiseless recovery, nfreq = ncomp reduction, central finite differences, chi^2 statistics, brute-force
 * grid argmin, Ninv scaling, K=(1,1,1) vs per-pixel gradients.  The tolerance scales absg / gscale (every T2
 * bound of the GPU tests is built from them) are pinned too: one pixel's gs against a numpy restatement of its
 * definition, absg == |grad| when every pixel is its own cluster, both as sums of the per-pixel terms over a
 * cluster's pixels, the closed form of gscale on noiseless data at the truth, and their scalings.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_NCOMP 3
#define ORC_UNITS_KCMB 0      /* default: dust and synchrotron columns carry the K_RJ -> K_CMB factor (R2) */
#define ORC_UNITS_LITERAL 1   /* Eq. 2 as corrected in R1, no unit factor */

/* exact SI constants (R3) */
static const double ORC_H = 6.62607015e-34;
static const double ORC_KB = 1.380649e-23;

typedef struct {
    int32_t nfreq;
    const double *freqs_ghz;
    double nu0_dust_ghz, nu0_sync_ghz, t_cmb_k;
    int32_t units;
} orc_model;

static double x_of(double nu_ghz, double T) { return ORC_H * nu_ghz * 1e9 / (ORC_KB * T); }

/* K_RJ -> K_CMB conversion u(nu) = (e^x - 1)^2 / (x^2 e^x), x = h nu / (k T_cmb)   (R2) */
double orc_krj2kcmb(double nu_ghz, double t_cmb) {
    double x = x_of(nu_ghz, t_cmb);
    double em1 = expm1(x);
    return em1 * em1 / (x * x * exp(x));
}

static double unit_ratio(const orc_model *m, double nu, double nu0) {
    if (m->units == ORC_UNITS_LITERAL) return 1.0;
    return orc_krj2kcmb(nu, m->t_cmb_k) / orc_krj2kcmb(nu0, m->t_cmb_k);
}

/* Dust column, Eq. 2 with the first denominator read as exp(h nu / k T_d) - 1 (R1):
 * a_d = u(nu)/u(nu0) * (nu/nu0)^(beta_d+1) * (e^{x0}-1)/(e^{x}-1). */
double orc_sed_dust(const orc_model *m, double nu, double beta_d, double T_d) {
    double nu0 = m->nu0_dust_ghz;
    double planck = expm1(x_of(nu0, T_d)) / expm1(x_of(nu, T_d));
    return unit_ratio(m, nu, nu0) * pow(nu / nu0, beta_d + 1.0) * planck;
}

/* Synchrotron column, Eq. 2: a_s = u(nu)/u(nu0) * (nu/nu0)^beta_s. */
double orc_sed_sync(const orc_model *m, double nu, double beta_s) {
    double nu0 = m->nu0_sync_ghz;
    return unit_ratio(m, nu, nu0) * pow(nu / nu0, beta_s);
}

/* d a_d / d beta_d = ln(nu/nu0) a_d */
double orc_dsed_dust_dbeta(const orc_model *m, double nu, double beta_d, double T_d) {
    return log(nu / m->nu0_dust_ghz) * orc_sed_dust(m, nu, beta_d, T_d);
}

/* d a_d / d T_d = a_d * (1/T) [ x e^x/(e^x-1) - x0 e^{x0}/(e^{x0}-1) ],  since dx/dT = -x/T */
double orc_dsed_dust_dT(const orc_model *m, double nu, double beta_d, double T_d) {
    double x = x_of(nu, T_d), x0 = x_of(m->nu0_dust_ghz, T_d);
    double t = x * exp(x) / expm1(x) - x0 * exp(x0) / expm1(x0);
    return orc_sed_dust(m, nu, beta_d, T_d) * t / T_d;
}

/* d a_s / d beta_s = ln(nu/nu0) a_s */
double orc_dsed_sync_dbeta(const orc_model *m, double nu, double beta_s) {
    return log(nu / m->nu0_sync_ghz) * orc_sed_sync(m, nu, beta_s);
}

/* Mixing matrix A [nfreq x 3] (row-major) and the three non-zero derivative columns dA [3 x nfreq]:
 * dA[0] = dA_dust/dbeta_d, dA[1] = dA_dust/dT_d, dA[2] = dA_sync/dbeta_s. */
void orc_mixing_matrix(const orc_model *m, double beta_d, double T_d, double beta_s, double *A, double *dA) {
    for (int f = 0; f < m->nfreq; ++f) {
        double nu = m->freqs_ghz[f];
        A[f * 3 + 0] = 1.0;                                   /* A_cmb = 1 in thermodynamic units, L56 */
        A[f * 3 + 1] = orc_sed_dust(m, nu, beta_d, T_d);
        A[f * 3 + 2] = orc_sed_sync(m, nu, beta_s);
        if (dA) {
            dA[0 * m->nfreq + f] = orc_dsed_dust_dbeta(m, nu, beta_d, T_d);
            dA[1 * m->nfreq + f] = orc_dsed_dust_dT(m, nu, beta_d, T_d);
            dA[2 * m->nfreq + f] = orc_dsed_sync_dbeta(m, nu, beta_s);
        }
    }
}

/* Solve the n x n system M x = rhs (nrhs right-hand sides, column j in rhs[j*n .. ]) by Gaussian
 * elimination with partial pivoting.  Returns 0, or -1 when a pivot is not positive-finite (R11). */
static int solve_small(int n, double *M, double *rhs, int nrhs) {
    for (int c = 0; c < n; ++c) {
        int piv = c;
        for (int r = c + 1; r < n; ++r)
            if (fabs(M[r * n + c]) > fabs(M[piv * n + c])) piv = r;
        if (!(fabs(M[piv * n + c]) > 0.0) || !isfinite(M[piv * n + c])) return -1;
        if (piv != c) {
            for (int k = 0; k < n; ++k) { double t = M[c * n + k]; M[c * n + k] = M[piv * n + k]; M[piv * n + k] = t; }
            for (int j = 0; j < nrhs; ++j) { double t = rhs[j * n + c]; rhs[j * n + c] = rhs[j * n + piv]; rhs[j * n + piv] = t; }
        }
        for (int r = c + 1; r < n; ++r) {
            double l = M[r * n + c] / M[c * n + c];
            for (int k = c; k < n; ++k) M[r * n + k] -= l * M[c * n + k];
            for (int j = 0; j < nrhs; ++j) rhs[j * n + r] -= l * rhs[j * n + c];
        }
    }
    for (int j = 0; j < nrhs; ++j)
        for (int r = n - 1; r >= 0; --r) {
            double t = rhs[j * n + r];
            for (int k = r + 1; k < n; ++k) t -= M[r * n + k] * rhs[j * n + k];
            rhs[j * n + r] = t / M[r * n + r];
        }
    return 0;
}

/* One pixel.  dq/du: the pixel's data per frequency (already promoted to double).  Outputs:
 * s[3][2] component amplitudes (comp-major, then Stokes), ll = -1/2 sum_S b_S.s_S,
 * g[3] = per-pixel gradient terms (beta_d, T_d, beta_s), gs[3] = cancellation-free magnitudes
 * sum_S |s_S,c| sum_f w_f |d_S,f| |da_f/dtheta|.  Returns -1 if M is singular. */
int orc_pixel(const orc_model *m, const double *ninv, const double *dq, const double *du,
              double beta_d, double T_d, double beta_s, double *s, double *ll, double *g, double *gs) {
    int F = m->nfreq;
    double A[3 * 64], dA[3 * 64];
    if (F > 64) return -2;
    orc_mixing_matrix(m, beta_d, T_d, beta_s, A, dA);
    double M[9] = {0}, Mc[9], b[6] = {0}, x[6];
    for (int f = 0; f < F; ++f)
        for (int i = 0; i < 3; ++i) {
            for (int j = 0; j < 3; ++j) M[i * 3 + j] += A[f * 3 + i] * ninv[f] * A[f * 3 + j];
            b[0 * 3 + i] += A[f * 3 + i] * ninv[f] * dq[f];
            b[1 * 3 + i] += A[f * 3 + i] * ninv[f] * du[f];
        }
    memcpy(Mc, M, sizeof M);
    memcpy(x, b, sizeof b);
    if (solve_small(3, Mc, x, 2) != 0) return -1;
    double l = 0.0;
    for (int S = 0; S < 2; ++S)
        for (int i = 0; i < 3; ++i) l += b[S * 3 + i] * x[S * 3 + i];
    *ll = -0.5 * l;
    for (int c = 0; c < 3; ++c) { s[c * 2 + 0] = x[0 * 3 + c]; s[c * 2 + 1] = x[1 * 3 + c]; }
    if (g) {
        const int comp_of[3] = {1, 1, 2};       /* beta_d, T_d act on the dust column; beta_s on synchrotron */
        for (int t = 0; t < 3; ++t) { g[t] = 0.0; if (gs) gs[t] = 0.0; }
        for (int S = 0; S < 2; ++S) {
            const double *d = S ? du : dq;
            for (int f = 0; f < F; ++f) {
                double model = 0.0;
                for (int c = 0; c < 3; ++c) model += A[f * 3 + c] * x[S * 3 + c];
                double w = ninv[f] * (d[f] - model);                       /* w_r = N^-1 (d - A s), L239 */
                for (int t = 0; t < 3; ++t) {
                    g[t] -= w * dA[t * F + f] * x[S * 3 + comp_of[t]];     /* Eq. 17 with factor 1 (R4) */
                    if (gs) gs[t] += fabs(x[S * 3 + comp_of[t]]) * ninv[f] * fabs(d[f]) * fabs(dA[t * F + f]);
                }
            }
        }
    }
    return 0;
}

/* One batch entry over a sky.
 *   d       float [nfreq, 2, npix]   (fp32 as the GPU receives it; promoted to double here)
 *   ninv    float [nfreq]
 *   idx0/1/2 int32 [npix]            cluster ids for beta_d, T_d, beta_s; -1 in any map = masked (R7)
 *   K       int32 [3]
 *   params  double [K0+K1+K2]        ordered [beta_d x K0 ; T_d x K1 ; beta_s x K2]
 *   region  uint8 [npix] or NULL, nregion >= 1
 * outputs (any may be NULL except nll):
 *   nll     double [nregion]
 *   grad    double [K0+K1+K2]
 *   maps    double [3, 2, npix]      0 at masked pixels
 *   absg    double [K0+K1+K2]        sum_p |g_p| per cluster       (tolerance rule T2)
 *   gscale  double [K0+K1+K2]        sum_p Gscale_p per cluster    (tolerance rule T2)
 * returns 0; -1 singular M somewhere (nll = +inf); -2 index out of range; -3 T_d <= 0 / non-finite parameter. */
int orc_nll_grad(const orc_model *m, int64_t npix, const float *d, const float *ninv_f,
                 const int32_t *idx0, const int32_t *idx1, const int32_t *idx2, const int32_t *K,
                 const double *params, const uint8_t *region, int32_t nregion,
                 double *nll, double *grad, double *maps, double *absg, double *gscale) {
    int F = m->nfreq;
    int64_t Ktot = (int64_t)K[0] + K[1] + K[2];
    const double *pbd = params, *pTd = params + K[0], *pbs = params + K[0] + K[1];
    for (int64_t k = 0; k < Ktot; ++k) if (!isfinite(params[k])) return -3;
    for (int32_t k = 0; k < K[1]; ++k) if (!(pTd[k] > 0.0)) return -3;
    for (int64_t p = 0; p < npix; ++p) {
        if (idx0[p] < -1 || idx0[p] >= K[0] || idx1[p] < -1 || idx1[p] >= K[1] || idx2[p] < -1 || idx2[p] >= K[2]) return -2;
        if (region && region[p] >= nregion) return -2;
    }
    double ninv[64];
    if (F > 64) return -2;
    for (int f = 0; f < F; ++f) ninv[f] = (double)ninv_f[f];

    double *ll_p = (double *)malloc(sizeof(double) * npix);
    double *g_p = (double *)malloc(sizeof(double) * npix * 3);
    double *gs_p = (double *)malloc(sizeof(double) * npix * 3);
    double *s_p = (double *)malloc(sizeof(double) * npix * 6);
    int *st_p = (int *)malloc(sizeof(int) * npix);
    int need_g = (grad || absg || gscale);

#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (int64_t p = 0; p < npix; ++p) {
        double dq[64], du[64];
        int k0 = idx0[p], k1 = idx1[p], k2 = idx2[p];
        st_p[p] = 1;                                    /* 1 = masked */
        if (k0 < 0 || k1 < 0 || k2 < 0) continue;
        for (int f = 0; f < F; ++f) {
            dq[f] = (double)d[((int64_t)f * 2 + 0) * npix + p];
            du[f] = (double)d[((int64_t)f * 2 + 1) * npix + p];
        }
        int rc = orc_pixel(m, ninv, dq, du, pbd[k0], pTd[k1], pbs[k2], s_p + 6 * p, ll_p + p,
                           need_g ? g_p + 3 * p : NULL, need_g ? gs_p + 3 * p : NULL);
        st_p[p] = rc == 0 ? 0 : 2;                      /* 2 = singular */
    }

    /* ordered accumulation onto regions and clusters, long double, pixel order */
    int rc = 0;
    long double *acc_n = (long double *)calloc(nregion, sizeof(long double));
    long double *acc_g = (long double *)calloc(Ktot ? Ktot : 1, sizeof(long double));
    long double *acc_a = (long double *)calloc(Ktot ? Ktot : 1, sizeof(long double));
    long double *acc_s = (long double *)calloc(Ktot ? Ktot : 1, sizeof(long double));
    if (maps) memset(maps, 0, sizeof(double) * 6 * npix);
    for (int64_t p = 0; p < npix; ++p) {
        if (st_p[p] == 1) continue;
        if (st_p[p] == 2) { rc = -1; continue; }
        acc_n[region ? region[p] : 0] += ll_p[p];
        if (need_g) {
            int64_t kk[3] = {idx0[p], (int64_t)K[0] + idx1[p], (int64_t)K[0] + K[1] + idx2[p]};
            for (int t = 0; t < 3; ++t) {
                acc_g[kk[t]] += g_p[3 * p + t];
                acc_a[kk[t]] += fabs(g_p[3 * p + t]);
                acc_s[kk[t]] += gs_p[3 * p + t];
            }
        }
        if (maps)
            for (int c = 0; c < 3; ++c)
                for (int S = 0; S < 2; ++S) maps[((int64_t)c * 2 + S) * npix + p] = s_p[6 * p + c * 2 + S];
    }
    for (int r = 0; r < nregion; ++r) nll[r] = rc == 0 ? (double)acc_n[r] : INFINITY;
    for (int64_t k = 0; k < Ktot; ++k) {
        if (grad) grad[k] = (double)acc_g[k];
        if (absg) absg[k] = (double)acc_a[k];
        if (gscale) gscale[k] = (double)acc_s[k];
    }
    free(acc_n); free(acc_g); free(acc_a); free(acc_s);
    free(ll_p); free(g_p); free(gs_p); free(s_p); free(st_p);
    return rc;
}

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void orc_set_num_threads(int n) {
#ifdef _OPENMP
    omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* salt_oracle.c -- fp64 CPU oracle for the SALT3 batched bandflux hot path.
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call this.
 * It shares no code, header, table or constant generator with the CUDA path
 * (paper_2504_08081_b200/csrc) and neither includes the other.
 *
 * What it is: the plain definition of the result, evaluated naively in double
 * precision in the paper's order -- every wavelength sample of every observation
 * does the full two-surface bicubic stencil, every factor is multiplied out
 * explicitly, the trapezoid rule is the literal formula.  No weight folding, no
 * phase-collapse, no hoisting, no reordering.  Passages followed:
 *
 *   PAPER.md:19-23 (Implementation)  F(p,lam) = x0 [M0 + x1 M1] exp(c CL(lam)),
 *                                    free parameters x0, x1, t0, c; p depends on z and t - t0
 *   PAPER.md:38-43                   bandflux = int F(lam) T(lam) lam/(hc) dlam
 *   PAPER.md:45                      "trapezoidal integration along the wavelength dimension"
 *   PAPER.md:47                      "dedicated interpolation routines" (SALT3, SALT3-NIR)
 *   BASELINE.json north_star         p = (t - t0)/(1+z), lam_rest = lam_obs/(1+z); bicubic on the
 *                                    (phase, wavelength) grid; zero-point normalisation; chi^2 per
 *                                    supernova; analytic gradient wrt (x0, x1, c, t0)
 *   DESIGN.md "Readings" G0-G15      everything the paper leaves open (kernel of the interpolant,
 *                                    border cells, out-of-grid = 0, colour-law continuation, AB
 *                                    zero point, constants)
 *
 * Step labels O1..O10 below are those of SURVEY.md section 8(c) / DESIGN.md "Oracle".
 *
 * Pins (tests/test_oracle_pins.py, run with -m "not gpu"): P1-P17 of DESIGN.md -- closed
 * forms (constant surface x top-hat, linear-in-phase, linear-in-wavelength surfaces, AB zero
 * point of a top-hat, colour integral), invariants (linearity in x0, affine in x1, c = 0,
 * scale invariance), interpolation identities (exact nodes, linear/quadratic reproduction,
 * the Keys a=-1/2 impulse response printed in tests/golden/keys_impulse.txt), trapezoid
 * error term, out-of-grid handling, chi^2 identities, gradient vs central differences, and
 * an exact-rational brute force on tiny grids.
 * Parity unpinned BY THE PAPER (conventions, self-consistent and tested, but not derivable
 * from PAPER.md): the AB reference spectrum of the zero point (G7) and the linear border
 * cells of the interpolant (G2).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* Physical constants (CGS, Angstrom).  O6/O8. */
#define SBO_H_PLANCK 6.62607015e-27          /* erg s */
#define SBO_C_AA 2.99792458e18               /* Angstrom / s */
#define SBO_HC (SBO_H_PLANCK * SBO_C_AA)     /* 1.9864458571489287e-8 erg Angstrom */
#define SBO_AB_FNU 3.631e-20                 /* erg / s / cm^2 / Hz : AB zero-magnitude flux density */

typedef struct {
    int32_t n_phase, n_wave;
    const double *phase;   /* [n_phase] uniform, increasing */
    const double *wave;    /* [n_wave] uniform, increasing */
    const double *m0;      /* [n_phase][n_wave] row-major, wavelength fastest */
    const double *m1;
    int32_t n_cl;          /* number of colour-law coefficients (degree n_cl-1) */
    const double *cl_coef; /* a_0 .. a_{n_cl-1} */
    double cl_wave_b, cl_wave_v, cl_lo, cl_hi;
} sbo_model;

typedef struct {
    int32_t n_bands;
    const int64_t *offset; /* [n_bands+1] */
    const double *wave;    /* observer-frame wavelength grid of each band, strictly increasing */
    const double *trans;   /* transmission at those wavelengths */
} sbo_bands;

typedef struct {
    int32_t n_sn, n_samples;
    const int32_t *obs_offset; /* [n_sn+1] */
    const double *time;        /* [n_obs_total] observer-frame time */
    const int32_t *band;       /* [n_obs_total] */
    const double *zp;          /* [n_obs_total] or NULL: no zero-point scaling */
    const double *z;           /* [n_sn] */
    const double *x0, *x1, *c, *t0; /* [n_sn*n_samples], sample fastest */
} sbo_batch;

/* ---------------------------------------------------------------------------------------
 * O2  One-dimensional interpolation operator on a uniform grid x_n = x0 + n*dx with node
 * values g_0..g_{n-1} (stride `stride` doubles apart).  Cubic convolution with the Keys
 * a = -1/2 kernel (= Catmull-Rom) in interior cells [DESIGN.md G1]; linear in the first
 * and last cell [G2]; zero outside the closed interval [x_0, x_{n-1}] [G3].  If dval is
 * non-NULL it receives d/dx of the selected cell's polynomial [G11] (0 outside).
 * ------------------------------------------------------------------------------------- */
double sbo_interp1(const double *g, int64_t stride, int32_t n, double x0, double dx, double x,
                   double *dval)
{
    double u = (x - x0) / dx;
    if (dval) *dval = 0.0;
    if (!(u >= 0.0) || !(u <= (double)(n - 1))) return 0.0; /* also rejects NaN */
    int32_t i = (int32_t)floor(u);
    if (i > n - 2) i = n - 2;
    double tau = u - (double)i;
    if (i == 0 || i == n - 2) { /* border cell: linear */
        double ga = g[(int64_t)i * stride], gb = g[(int64_t)(i + 1) * stride];
        if (dval) *dval = (gb - ga) / dx;
        return (1.0 - tau) * ga + tau * gb;
    }
    double t2 = tau * tau, t3 = t2 * tau;
    double wm1 = (-t3 + 2.0 * t2 - tau) / 2.0;
    double w0 = (3.0 * t3 - 5.0 * t2 + 2.0) / 2.0;
    double w1 = (-3.0 * t3 + 4.0 * t2 + tau) / 2.0;
    double w2 = (t3 - t2) / 2.0;
    double gm1 = g[(int64_t)(i - 1) * stride], g0 = g[(int64_t)i * stride];
    double g1 = g[(int64_t)(i + 1) * stride], g2 = g[(int64_t)(i + 2) * stride];
    if (dval) {
        double dm1 = (-3.0 * t2 + 4.0 * tau - 1.0) / 2.0;
        double d0 = (9.0 * t2 - 10.0 * tau) / 2.0;
        double d1 = (-9.0 * t2 + 8.0 * tau + 1.0) / 2.0;
        double d2 = (3.0 * t2 - 2.0 * tau) / 2.0;
        *dval = (dm1 * gm1 + d0 * g0 + d1 * g1 + d2 * g2) / dx;
    }
    return wm1 * gm1 + w0 * g0 + w1 * g1 + w2 * g2;
}

static double grid_step(const double *x, int32_t n) { return (x[n - 1] - x[0]) / (double)(n - 1); }

/* ---------------------------------------------------------------------------------------
 * O3  Surface value at (p, lam_rest): O2 along phase applied to (O2 along wavelength applied
 * to each phase row).  Only the <= 4 rows the phase stencil reads are filled; every other
 * entry of the column stays NaN so that a wrong index cannot go unnoticed.  dval_dp (may be
 * NULL) receives the derivative with respect to phase.  `which` = 0 for M0, 1 for M1.
 * ------------------------------------------------------------------------------------- */
double sbo_surface(const sbo_model *m, int32_t which, double p, double lam_rest, double *dval_dp)
{
    const double *surf = which ? m->m1 : m->m0;
    int32_t np = m->n_phase, nw = m->n_wave;
    double dp = grid_step(m->phase, np), dw = grid_step(m->wave, nw);
    if (dval_dp) *dval_dp = 0.0;
    double up = (p - m->phase[0]) / dp;
    if (!(up >= 0.0) || !(up <= (double)(np - 1))) return 0.0;
    int32_t ip = (int32_t)floor(up);
    if (ip > np - 2) ip = np - 2;
    int32_t border = (ip == 0 || ip == np - 2);
    int32_t k_lo = border ? ip : ip - 1, k_hi = border ? ip + 1 : ip + 2;
    double col[np]; /* C99 variable-length array; n_phase is small (71) */
    for (int32_t k = 0; k < np; ++k) col[k] = NAN;
    for (int32_t k = k_lo; k <= k_hi; ++k)
        col[k] = sbo_interp1(surf + (int64_t)k * nw, 1, nw, m->wave[0], dw, lam_rest, NULL);
    return sbo_interp1(col, 1, np, m->phase[0], dp, p, dval_dp);
}

/* ---------------------------------------------------------------------------------------
 * O4  Colour law CL(lam_rest): polynomial in the reduced wavelength
 * l = (lam - lam_B)/(lam_V - lam_B) inside [cl_lo, cl_hi], continued linearly (value and
 * slope matched) outside [BASELINE.json configs[0]; G5].
 * ------------------------------------------------------------------------------------- */
static double poly(const double *a, int32_t n, double x)
{
    double s = 0.0, xp = 1.0;
    for (int32_t q = 0; q < n; ++q) { s += a[q] * xp; xp *= x; }
    return s;
}
static double dpoly(const double *a, int32_t n, double x)
{
    double s = 0.0, xp = 1.0;
    for (int32_t q = 1; q < n; ++q) { s += (double)q * a[q] * xp; xp *= x; }
    return s;
}
double sbo_colour_law(const sbo_model *m, double lam_rest)
{
    double span = m->cl_wave_v - m->cl_wave_b;
    double l = (lam_rest - m->cl_wave_b) / span;
    double l_lo = (m->cl_lo - m->cl_wave_b) / span;
    double l_hi = (m->cl_hi - m->cl_wave_b) / span;
    if (l < l_lo) return poly(m->cl_coef, m->n_cl, l_lo) + dpoly(m->cl_coef, m->n_cl, l_lo) * (l - l_lo);
    if (l > l_hi) return poly(m->cl_coef, m->n_cl, l_hi) + dpoly(m->cl_coef, m->n_cl, l_hi) * (l - l_hi);
    return poly(m->cl_coef, m->n_cl, l);
}

/* O7  Literal trapezoid rule: sum_j 1/2 (g_j + g_{j+1}) (x_{j+1} - x_j).  PAPER.md:45. */
double sbo_trapz(const double *g, const double *x, int64_t n)
{
    double s = 0.0;
    for (int64_t j = 0; j + 1 < n; ++j) s += 0.5 * (g[j] + g[j + 1]) * (x[j + 1] - x[j]);
    return s;
}

/* O8  AB zero-point integral of band b: the same trapezoid applied to the AB reference
 * spectrum f_lam = 3.631e-20 c / lam^2 times T lam/(hc).  DESIGN.md G7. */
double sbo_zpab(const sbo_bands *bd, int32_t b)
{
    int64_t lo = bd->offset[b], n = bd->offset[b + 1] - lo;
    double *g = (double *)malloc(sizeof(double) * (size_t)n);
    for (int64_t j = 0; j < n; ++j) {
        double lam = bd->wave[lo + j];
        double f_ab = SBO_AB_FNU * SBO_C_AA / (lam * lam);
        g[j] = f_ab * bd->trans[lo + j] * lam / SBO_HC;
    }
    double s = sbo_trapz(g, bd->wave + lo, n);
    free(g);
    return s;
}

/* ---------------------------------------------------------------------------------------
 * One evaluation (one supernova, one parameter sample, one observation): O1, O3-O8, and the
 * four integrals of O10.  dm (may be NULL) receives d m / d(x0, x1, c, t0).
 * ------------------------------------------------------------------------------------- */
static double eval_one(const sbo_model *m, const sbo_bands *bd, double z, double t, int32_t b,
                       const double *zp, double x0, double x1, double c, double t0, double *dm)
{
    if (b < 0 || b >= bd->n_bands) {
        if (dm) dm[0] = dm[1] = dm[2] = dm[3] = NAN;
        return NAN;
    }
    int64_t lo = bd->offset[b], n = bd->offset[b + 1] - lo;
    const double *lam_obs = bd->wave + lo, *T = bd->trans + lo;
    double p = (t - t0) / (1.0 + z); /* O1 */
    double *g = (double *)malloc(sizeof(double) * (size_t)n * 5);
    double *gA = g + n, *gB = g + 2 * n, *gC = g + 3 * n, *gD = g + 4 * n;
    for (int64_t j = 0; j < n; ++j) {
        double lam_r = lam_obs[j] / (1.0 + z);          /* O1 */
        double d0 = 0.0, d1 = 0.0;
        double M0 = sbo_surface(m, 0, p, lam_r, &d0);   /* O3 */
        double M1 = sbo_surface(m, 1, p, lam_r, &d1);
        double CL = sbo_colour_law(m, lam_r);           /* O4 */
        double E = exp(c * CL);
        double F = x0 * (M0 + x1 * M1) * E;             /* O5 */
        double k = T[j] * lam_obs[j] / SBO_HC;          /* O6 */
        g[j] = F * k;
        gA[j] = M0 * E * k;
        gB[j] = M1 * E * k;
        gC[j] = CL * (M0 + x1 * M1) * E * k;
        gD[j] = (d0 + x1 * d1) * E * k;
    }
    double raw = sbo_trapz(g, lam_obs, n);              /* O7 */
    double s = 1.0;
    if (zp) s = pow(10.0, 0.4 * (*zp)) / sbo_zpab(bd, b); /* O8 */
    if (dm) {                                           /* O10 */
        double A = sbo_trapz(gA, lam_obs, n), B = sbo_trapz(gB, lam_obs, n);
        double C = sbo_trapz(gC, lam_obs, n), D = sbo_trapz(gD, lam_obs, n);
        dm[0] = s * (A + x1 * B);
        dm[1] = s * x0 * B;
        dm[2] = s * x0 * C;
        dm[3] = -(1.0 / (1.0 + z)) * s * x0 * D;
    }
    free(g);
    return raw * s;
}

/* Single evaluation exposed for the pins. */
double sbo_eval(const sbo_model *m, const sbo_bands *bd, double z, double t, int32_t b,
                int32_t use_zp, double zp, double x0, double x1, double c, double t0, double *dm)
{
    return eval_one(m, bd, z, t, b, use_zp ? &zp : NULL, x0, x1, c, t0, dm);
}

/* ---------------------------------------------------------------------------------------
 * Batched forms.  Output layout equals the CUDA library's (include/saltband.h):
 *   out_flux  : for each supernova s, [n_samples][n_obs(s)], observation fastest, starting at
 *               obs_offset[s]*n_samples
 *   out_dflux : same order, 4 doubles (x0, x1, c, t0) per evaluation         (may be NULL)
 *   out_chi2  : [n_sn*n_samples]                                             (O9)
 *   out_dchi2 : [n_sn*n_samples][4]  = -2 sum_i (f_i - m_i)/sigma_i^2 dm_i   (may be NULL)
 * flux/fluxerr may be NULL when neither chi^2 output is requested.
 * OpenMP only over the outermost (supernova, sample) loop.
 * ------------------------------------------------------------------------------------- */
int sbo_run(const sbo_model *m, const sbo_bands *bd, const sbo_batch *bt, const double *flux,
            const double *fluxerr, double *out_flux, double *out_dflux, double *out_chi2,
            double *out_dchi2)
{
    if (!m || !bd || !bt) return -1;
    if ((out_chi2 || out_dchi2) && (!flux || !fluxerr)) return -1;
    int64_t n_units = (int64_t)bt->n_sn * bt->n_samples;
    int want_grad = (out_dflux != NULL) || (out_dchi2 != NULL);
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t unit = 0; unit < n_units; ++unit) {
        int64_t s = unit / bt->n_samples, k = unit % bt->n_samples;
        int64_t o_lo = bt->obs_offset[s], n_obs = bt->obs_offset[s + 1] - o_lo;
        int64_t base = o_lo * bt->n_samples + k * n_obs;
        double chi2 = 0.0, dchi2[4] = {0.0, 0.0, 0.0, 0.0};
        for (int64_t i = 0; i < n_obs; ++i) {
            double dm[4];
            double mi = eval_one(m, bd, bt->z[s], bt->time[o_lo + i], bt->band[o_lo + i],
                                 bt->zp ? bt->zp + o_lo + i : NULL, bt->x0[unit], bt->x1[unit],
                                 bt->c[unit], bt->t0[unit], want_grad ? dm : NULL);
            if (out_flux) out_flux[base + i] = mi;
            if (out_dflux) memcpy(out_dflux + 4 * (base + i), dm, sizeof dm);
            if (out_chi2 || out_dchi2) {
                double sig = fluxerr[o_lo + i];
                double r = (flux[o_lo + i] - mi) / sig;                 /* O9 */
                chi2 += r * r;
                if (out_dchi2)
                    for (int q = 0; q < 4; ++q)
                        dchi2[q] += -2.0 * (flux[o_lo + i] - mi) / (sig * sig) * dm[q];
            }
        }
        if (out_chi2) out_chi2[unit] = chi2;
        if (out_dchi2) memcpy(out_dchi2 + 4 * unit, dchi2, sizeof dchi2);
    }
    return 0;
}

int sbo_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void sbo_set_num_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

double sbo_const_hc(void) { return SBO_HC; }

/*
 * rubix_oracle.c -- fp64 CPU ORACLE for the RUBIX hot path.  TEST INFRASTRUCTURE ONLY.
 *
 * This file is the slow, plain, by-the-definition implementation that the CUDA path is
 * compared against.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call it.  It shares no code, header, table or
 * constant generator with paper_2412_08265_b200/csrc/ and never calls into it.
 *
 * What it computes (section 3 "RUBIX Codebase"): "orientate the galaxy in the
 * field of view" -> "particles are assigned to the IFU spaxels" -> "Each star spectrum is
 * calculated as a lookup from a simple stellar population (SSP) library" -> "Doppler
 * shifted based on ... line-of-sight velocity" -> "resampling ... to match the wavelength
 * grid of the observed telescope" -> "the stellar spectra in each spaxel are summed up" ->
 * "point-spread function (PSF) and line-spread function (LSF) convolution"; and the
 * gradients "through the entire pipeline" (PAPER.md L22 abstract).  The paper gives no
 * formulas; the numerical readings are BASELINE.json:north_star and SURVEY.md section 8(c),
 * listed in DESIGN.md ("Readings of the paper").  Each function cites its row.
 *
 * Arithmetic: fp64 from the same fp32 input arrays the GPU sees (promoted on load), EXCEPT
 * the binning of step 1-2 which SURVEY.md 8(c)-2 defines in fp32 with a fixed operation
 * order so that spaxel keys can be compared bit for bit.  Build with -ffp-contract=off and
 * without -ffast-math (oracle/__init__.py does).
 *
 * Pins (tests/test_oracle_*.py, all run without a GPU): numpy.histogram2d and hand-checked
 * edges (binning); numpy.argsort(kind='stable') (sort); node reproduction, the bilinear
 * closed form and partition of unity (lookup); numpy.interp, the a+b*lambda closed form and
 * the line-centroid shift lambda(1+v/c) (Doppler/resample); superposition, permutation
 * invariance, flux conservation, brute-force Python loops (accumulate); delta response,
 * scipy.ndimage.convolve1d, numpy.convolve, flux conservation (PSF/LSF); central finite
 * differences, the dot-product test and the linear-template closed form (adjoint);
 * the prefix-integral formulation, constant / linear templates, the (1,6,1)/8 identity and
 * exact total-flux telescoping (flux-conserving resampling, tests/test_oracle_fluxcons.py);
 * numpy.interp at the doubly shifted wavelength, in log lambda, and at listed channel wavelengths
 * (redshift, log-sampled grids, explicit observed grids: tests/test_oracle_redshift.py,
 * test_oracle_loggrid.py, test_oracle_obsgrid.py), each with finite-difference and closed-form adjoint pins;
 * the bin average on log-sampled grids / listed channel wavelengths and listed SSP wavelengths (readings R20, R21:
 * particle_spectrum_general) against a prefix-integral restatement, numpy.interp on the knots, the telescoping sum,
 * constant / linear-in-x closed forms, reduction to the uniform-grid functions and central finite differences
 * (tests/test_oracle_gengrid.py).
 * No function here is "parity unpinned".
 *
 * No blocking, fusion or reordering beyond the definitions; the only parallelism is an
 * OpenMP "parallel for" over independent outputs (spaxel x channel block / voxels / particles).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORC_C_KMS 299792.458     /* speed of light, km/s (SURVEY.md 8 notation) */
/* Observed wavelengths (reading R16): lambda_k = l0_obs + k dl_obs, or, while an explicit array is
 * installed with orc_set_lambda_obs, lambda_k = lambda_obs[k] / (1 + z) (arbitrary, increasing telescope grid;
 * point-sampled rule only).  The array is installed by the Python wrapper around one call and removed
 * afterwards; the OpenMP threads only read it. */
static const float *g_lambda_obs = 0;
static double g_lambda_div = 1.0;
void orc_set_lambda_obs(const float *lambda_obs, double one_plus_z)
{
    g_lambda_obs = lambda_obs;
    g_lambda_div = one_plus_z;
}
static double observed_lambda(int32_t k, double l0_obs, double dl_obs)
{
    return g_lambda_obs ? (double)g_lambda_obs[k] / g_lambda_div : l0_obs + dl_obs * (double)k;
}

#define ORC_VCAP_KMS 14989.623f  /* 0.05 c: |v_los| above this (or NaN) => particle dropped
                                    (reading R5; physical stars never reach it) */

/* ------------------------------------------------------------------------------------
 * Steps 1-2: rotate, project, bin.  SURVEY.md 8(a) rows 1-2, 8(c) rows 1-2.
 * fp32, round-to-nearest, every * and + separately rounded, in exactly this order:
 *   xr = (R00*x + R01*y) + R02*z ; yr likewise ; vl = (R20*vx + R21*vy) + R22*vz
 *   hx = (0.5f*N_x)*s ; u = (xr + hx) / s ; inside iff 0 <= u < N_x (same for y)
 *   key = floor(u)*N_y + floor(v) if inside (and |vl| <= cap) else N_x*N_y
 * Line of sight = +z' (receding positive).
 * ------------------------------------------------------------------------------------ */
void orc_rotate_bin(int64_t n, const float *pos, const float *vel, const float *R,
                    int32_t n_x, int32_t n_y, float s, int32_t *key, float *vlos)
{
    const float hx = (0.5f * (float)n_x) * s;
    const float hy = (0.5f * (float)n_y) * s;
    for (int64_t i = 0; i < n; ++i) {
        const float x = pos[3 * i], y = pos[3 * i + 1], z = pos[3 * i + 2];
        const float vx = vel[3 * i], vy = vel[3 * i + 1], vz = vel[3 * i + 2];
        const float xr = (R[0] * x + R[1] * y) + R[2] * z;
        const float yr = (R[3] * x + R[4] * y) + R[5] * z;
        const float vl = (R[6] * vx + R[7] * vy) + R[8] * vz;
        const float u = (xr + hx) / s;
        const float v = (yr + hy) / s;
        const int inside = (u >= 0.0f) && (u < (float)n_x) && (v >= 0.0f) && (v < (float)n_y)
                           && (fabsf(vl) <= ORC_VCAP_KMS);
        key[i] = inside ? (int32_t)floorf(u) * n_y + (int32_t)floorf(v) : n_x * n_y;
        vlos[i] = vl;
    }
}

/* ------------------------------------------------------------------------------------
 * Step 3: stable order by (key, original index) and segment offsets.
 * SURVEY.md 8(a) row 3, 8(c) row 3.  seg_off has n_s+2 entries: segment s is
 * perm[seg_off[s] .. seg_off[s+1]), s = n_s is the out-of-FoV segment.
 * ------------------------------------------------------------------------------------ */
void orc_sort(int64_t n, const int32_t *key, int32_t n_s, int32_t *perm, int32_t *seg_off)
{
    int64_t *cursor = (int64_t *)calloc((size_t)n_s + 2, sizeof(int64_t));
    for (int64_t i = 0; i < n; ++i) cursor[key[i] + 1] += 1;
    for (int32_t s = 0; s <= n_s; ++s) cursor[s + 1] += cursor[s];
    for (int32_t s = 0; s <= n_s + 1; ++s) seg_off[s] = (int32_t)cursor[s];
    for (int64_t i = 0; i < n; ++i) perm[cursor[key[i]]++] = (int32_t)i;  /* ascending i */
    free(cursor);
}

/* ------------------------------------------------------------------------------------
 * Step 4a: SSP cell and interpolation parameter on one axis.  SURVEY.md 8(c) row 4:
 *   i = clamp(max{j : A[j] <= q}, 0, n-2),  t = clamp((q - A[i]) / (A[i+1] - A[i]), 0, 1)
 * ------------------------------------------------------------------------------------ */
static void axis_cell(const float *A, int32_t n, float qf, int32_t *cell, double *t)
{
    const double q = (double)qf;
    int32_t i = -1;
    for (int32_t j = 0; j < n; ++j)
        if ((double)A[j] <= q) i = j;
    if (i < 0) i = 0;
    if (i > n - 2) i = n - 2;
    double tt = (q - (double)A[i]) / ((double)A[i + 1] - (double)A[i]);
    if (tt < 0.0) tt = 0.0;
    if (tt > 1.0) tt = 1.0;
    *cell = i;
    *t = tt;
}

void orc_ssp_cells(int64_t n, const float *log_age, const float *log_z, int32_t n_age,
                   int32_t n_z, const float *age_axis, const float *z_axis, int32_t *ia,
                   int32_t *iz, double *ta, double *tz)
{
    for (int64_t p = 0; p < n; ++p) {
        axis_cell(age_axis, n_age, log_age[p], &ia[p], &ta[p]);
        axis_cell(z_axis, n_z, log_z[p], &iz[p], &tz[p]);
    }
}

/* ------------------------------------------------------------------------------------
 * Steps 4b-5: one particle's observed spectrum.  SURVEY.md 8(c) rows 4-5.
 *   S(j)  = m * [ (1-ta)(1-tz) T[i][j'] + ta(1-tz) T[i+1][j'] + (1-ta)tz T[i][j'+1]
 *                 + ta tz T[i+1][j'+1] ](j)          (linear in flux, array order [age][Z][lambda])
 *   F[k]  = S evaluated by linear interpolation at rest wavelength lambda_k / (1 + beta),
 *           beta = v_los / c, 0 outside the SSP wavelength coverage
 *         = numpy.interp(lambda_obs/(1+beta), lambda_ssp, S, left=0, right=0)
 * flux: [n_age][n_z][n_lambda].  If dS (length n_c) is non-NULL it receives the slope
 * dS/dx at the sample (x in SSP-sample units), used by the analytic adjoint.
 * ------------------------------------------------------------------------------------ */
static void particle_spectrum(double mass, int32_t ia, int32_t iz, double ta, double tz,
                              double vlos, const float *flux, int32_t n_z, int32_t n_lambda,
                              double l0_ssp, double dl_ssp, int32_t k_begin, int32_t k_end,
                              double l0_obs, double dl_obs, double *F, double *dS, int32_t log_grid)
{   /* fills F[k] (and dS[k]) for channels k_begin <= k < k_end.
     * log_grid = 1 (reading R15): the SSP grid is log-sampled, lambda_j = l0_ssp * 10^(j dl_ssp)
     * (dl_ssp in dex), the sampling coordinate is x = log10(lambda_rest / l0_ssp) / dl_ssp and the
     * interpolant is linear in x between knots: numpy.interp(log10 lambda_rest, log10 lambda_ssp, S). */
    const float *T00 = flux + ((int64_t)ia * n_z + iz) * n_lambda;
    const float *T10 = flux + ((int64_t)(ia + 1) * n_z + iz) * n_lambda;
    const float *T01 = flux + ((int64_t)ia * n_z + iz + 1) * n_lambda;
    const float *T11 = flux + ((int64_t)(ia + 1) * n_z + iz + 1) * n_lambda;
    const double w00 = (1.0 - ta) * (1.0 - tz), w10 = ta * (1.0 - tz);
    const double w01 = (1.0 - ta) * tz, w11 = ta * tz;
    const double beta = vlos / ORC_C_KMS;
    const double lam_first = l0_ssp;
    const double lam_last = log_grid ? l0_ssp * pow(10.0, dl_ssp * (double)(n_lambda - 1))
                                     : l0_ssp + dl_ssp * (double)(n_lambda - 1);
    for (int32_t k = k_begin; k < k_end; ++k) {
        const double lam_obs = observed_lambda(k, l0_obs, dl_obs);
        const double lam_rest = lam_obs / (1.0 + beta);
        if (lam_rest < lam_first || lam_rest > lam_last) {
            F[k] = 0.0;
            if (dS) dS[k] = 0.0;
            continue;
        }
        double x = log_grid ? log10(lam_rest / l0_ssp) / dl_ssp : (lam_rest - l0_ssp) / dl_ssp;
        if (x < 0.0) x = 0.0;                              /* rounding at the first knot */
        int32_t j = (int32_t)floor(x);
        if (j > n_lambda - 2) j = n_lambda - 2;
        const double f = x - (double)j;
        const double s0 = mass * (w00 * T00[j] + w10 * T10[j] + w01 * T01[j] + w11 * T11[j]);
        const double s1 = mass * (w00 * T00[j + 1] + w10 * T10[j + 1] + w01 * T01[j + 1]
                                  + w11 * T11[j + 1]);
        F[k] = s0 + f * (s1 - s0);
        if (dS) dS[k] = s1 - s0;
    }
}

/* ------------------------------------------------------------------------------------
 * Step 5, flux-conserving variant ("Additional resampling is
 * performed to match the wavelength grid of the observed telescope"; reading R13).
 * Channel k is the bin [lambda_k - dl_obs/2, lambda_k + dl_obs/2]; its value is the bin AVERAGE
 * of the Doppler-shifted spectrum,
 *   F[k] = (1/dl_obs) * integral over the bin of S~(lambda / (1 + beta)) d lambda,
 * where S~ is the piecewise-linear interpolant of the blended samples S(j) on the SSP
 * coverage and 0 outside it.  In SSP-sample units x = (lambda/(1+beta) - l0_ssp)/dl_ssp the
 * bin is [x_lo, x_hi] with x_hi - x_lo = B = dl_obs / ((1+beta) dl_ssp) and
 *   F[k] = (1/B) * integral_{x_lo}^{x_hi} S~(x) dx.
 * The integral is taken exactly, one knot interval at a time (a trapezoid is exact for a
 * linear piece).  No 1/(1+beta) flux-density factor, as in the point-sampled variant.
 * ------------------------------------------------------------------------------------ */
static void particle_spectrum_flux(double mass, int32_t ia, int32_t iz, double ta, double tz,
                                   double vlos, const float *flux, int32_t n_z, int32_t n_lambda,
                                   double l0_ssp, double dl_ssp, int32_t k_begin, int32_t k_end,
                                   double l0_obs, double dl_obs, double *F)
{
    const float *T00 = flux + ((int64_t)ia * n_z + iz) * n_lambda;
    const float *T10 = flux + ((int64_t)(ia + 1) * n_z + iz) * n_lambda;
    const float *T01 = flux + ((int64_t)ia * n_z + iz + 1) * n_lambda;
    const float *T11 = flux + ((int64_t)(ia + 1) * n_z + iz + 1) * n_lambda;
    const double w00 = (1.0 - ta) * (1.0 - tz), w10 = ta * (1.0 - tz);
    const double w01 = (1.0 - ta) * tz, w11 = ta * tz;
    const double beta = vlos / ORC_C_KMS;
    const double x_last = (double)(n_lambda - 1);
    const double B = dl_obs / ((1.0 + beta) * dl_ssp);
    for (int32_t k = k_begin; k < k_end; ++k) {
        const double lam_c = l0_obs + dl_obs * (double)k;
        double x_lo = ((lam_c - 0.5 * dl_obs) / (1.0 + beta) - l0_ssp) / dl_ssp;
        double x_hi = ((lam_c + 0.5 * dl_obs) / (1.0 + beta) - l0_ssp) / dl_ssp;
        if (x_lo < 0.0) x_lo = 0.0;
        if (x_hi > x_last) x_hi = x_last;
        double total = 0.0, pos = x_lo;
        while (pos < x_hi) {
            int32_t j = (int32_t)floor(pos);
            if (j > n_lambda - 2) j = n_lambda - 2;
            double next = (double)(j + 1);
            if (next > x_hi) next = x_hi;
            const double s0 = mass * (w00 * T00[j] + w10 * T10[j] + w01 * T01[j] + w11 * T11[j]);
            const double s1 = mass * (w00 * T00[j + 1] + w10 * T10[j + 1] + w01 * T01[j + 1]
                                      + w11 * T11[j + 1]);
            const double va = s0 + (pos - (double)j) * (s1 - s0);
            const double vb = s0 + (next - (double)j) * (s1 - s0);
            total += 0.5 * (next - pos) * (va + vb);
            pos = next;
        }
        F[k] = total / B;
    }
}

/* ------------------------------------------------------------------------------------
 * Step 5 on general grids ("Additional resampling is performed to match the
 * wavelength grid of the observed telescope", L44 the experiment's library "Mastar_CB19_SLOG_1_5" is log-sampled;
 * DESIGN.md readings R20, R21).  One definition covers every combination of
 *   SSP grid       kind 0  lambda_j = l0 + j dl                 sampling coordinate x = (lambda - l0) / dl
 *                  kind 1  lambda_j = l0 10^(j dl)  (R15)       x = log10(lambda / l0) / dl
 *                  kind 2  lambda_j listed, increasing (R21)    x = j + (lambda - lambda_j) / (lambda_{j+1} - lambda_j)
 *                          on knot interval j (continued linearly with the first / last interval outside the coverage)
 *   observed grid  uniform l0_obs + k dl_obs, or listed lambda_obs[k] (R16)
 *   rule           point:  F[k] = S~(x(lambda_k / (1+beta)))
 *                  bin average (R20):  channel k is the bin [e_k, e_{k+1}] of OBSERVED wavelength -- e_k = lambda_k - dl_obs/2
 *                          on a uniform grid; on a listed grid the midpoints of neighbouring channels, the first and last
 *                          edge half a neighbouring spacing outside -- and
 *                              F[k] = (1 / (x_hi - x_lo)) * integral_{x_lo}^{x_hi} S~(x) dx,   x_lo/hi = x(e / (1+beta)),
 *                          the average of the interpolant over the bin IN THE SAMPLING COORDINATE x (S~ = 0 outside the
 *                          coverage, the bin keeps its full width).  On a linearly sampled grid x is affine in lambda and
 *                          this is R13 exactly; on a log-sampled grid it is the average per unit log lambda, which differs
 *                          from the average per unit lambda by O((dl_obs / lambda)^2).  sum_k F[k] (x_hi - x_lo)_k telescopes
 *                          to the integral of S~ over the covered part of the detector.
 * S~(x) = S_j + (x - j)(S_{j+1} - S_j), j = floor(x), is the piecewise-linear interpolant of the blended samples in x
 * for every kind (numpy.interp in lambda, in log lambda, or on the listed knots).
 * If dF (length k_end) is non-NULL it receives dF[k] / d beta (analytic; edges clipped to the coverage do not move).
 * ------------------------------------------------------------------------------------ */
static const float *g_lambda_ssp = 0;      /* kind 2: listed SSP wavelengths [n_lambda], installed around one call */
void orc_set_lambda_ssp(const float *lambda_ssp) { g_lambda_ssp = lambda_ssp; }

/* sampling coordinate of rest wavelength lam and d x / d lambda there */
static double sample_coord(double lam, int32_t kind, double l0, double dl, int32_t n_lambda, double *dxdlam)
{
    if (kind == 0) { *dxdlam = 1.0 / dl; return (lam - l0) / dl; }
    if (kind == 1) { *dxdlam = 1.0 / (lam * dl * log(10.0)); return log10(lam / l0) / dl; }
    const float *L = g_lambda_ssp;
    int32_t j = 0;
    if (lam >= (double)L[n_lambda - 1]) j = n_lambda - 2;
    else if (lam > (double)L[0]) {
        int32_t lo = 0, hi = n_lambda - 1;             /* largest j with L[j] <= lam */
        while (lo < hi) { const int32_t mid = (lo + hi + 1) / 2; if ((double)L[mid] <= lam) lo = mid; else hi = mid - 1; }
        j = lo > n_lambda - 2 ? n_lambda - 2 : lo;
    }
    const double w = (double)L[j + 1] - (double)L[j];
    *dxdlam = 1.0 / w;
    return (double)j + (lam - (double)L[j]) / w;
}

typedef struct { const float *T[4]; double w[4]; double mass; int32_t n_lambda; } blend_t;
static double blend_sample(const blend_t *b, int32_t j)
{
    return b->mass * (b->w[0] * b->T[0][j] + b->w[1] * b->T[1][j] + b->w[2] * b->T[2][j] + b->w[3] * b->T[3][j]);
}
/* S~(x), 0 outside [0, n_lambda - 1] */
static double interpolant(const blend_t *b, double x)
{
    if (x < 0.0 || x > (double)(b->n_lambda - 1)) return 0.0;
    int32_t j = (int32_t)floor(x);
    if (j > b->n_lambda - 2) j = b->n_lambda - 2;
    const double s0 = blend_sample(b, j), s1 = blend_sample(b, j + 1);
    return s0 + (x - (double)j) * (s1 - s0);
}
/* integral of S~ over [a, c] clipped to the coverage, one knot interval at a time (a trapezoid is exact) */
static double interpolant_integral(const blend_t *b, double a, double c)
{
    const double x_last = (double)(b->n_lambda - 1);
    if (a < 0.0) a = 0.0;
    if (c > x_last) c = x_last;
    double total = 0.0, pos = a;
    while (pos < c) {
        int32_t j = (int32_t)floor(pos);
        if (j > b->n_lambda - 2) j = b->n_lambda - 2;
        double next = (double)(j + 1);
        if (next > c) next = c;
        const double s0 = blend_sample(b, j), s1 = blend_sample(b, j + 1);
        const double va = s0 + (pos - (double)j) * (s1 - s0), vb = s0 + (next - (double)j) * (s1 - s0);
        total += 0.5 * (next - pos) * (va + vb);
        pos = next;
    }
    return total;
}

/* observed bin edge e (0 <= e <= n_c) of reading R20, already divided by (1 + z) like observed_lambda */
static double observed_edge(int32_t e, int32_t n_c, double l0_obs, double dl_obs)
{
    if (!g_lambda_obs) return l0_obs + dl_obs * ((double)e - 0.5);
    if (n_c < 2) return 0.0;                                       /* refused by the wrapper */
    if (e == 0) return observed_lambda(0, 0, 0) - 0.5 * (observed_lambda(1, 0, 0) - observed_lambda(0, 0, 0));
    if (e == n_c) return observed_lambda(n_c - 1, 0, 0) + 0.5 * (observed_lambda(n_c - 1, 0, 0) - observed_lambda(n_c - 2, 0, 0));
    return 0.5 * (observed_lambda(e - 1, 0, 0) + observed_lambda(e, 0, 0));
}

static void particle_spectrum_general(int32_t rule, int32_t kind, double mass, int32_t ia, int32_t iz, double ta, double tz,
                                      double vlos, const float *flux, int32_t n_z, int32_t n_lambda, double l0_ssp,
                                      double dl_ssp, int32_t k_begin, int32_t k_end, int32_t n_c, double l0_obs,
                                      double dl_obs, double *F, double *dF)
{
    blend_t b;
    b.T[0] = flux + ((int64_t)ia * n_z + iz) * n_lambda;
    b.T[1] = flux + ((int64_t)(ia + 1) * n_z + iz) * n_lambda;
    b.T[2] = flux + ((int64_t)ia * n_z + iz + 1) * n_lambda;
    b.T[3] = flux + ((int64_t)(ia + 1) * n_z + iz + 1) * n_lambda;
    b.w[0] = (1.0 - ta) * (1.0 - tz); b.w[1] = ta * (1.0 - tz); b.w[2] = (1.0 - ta) * tz; b.w[3] = ta * tz;
    b.mass = mass;
    b.n_lambda = n_lambda;
    const double opb = 1.0 + vlos / ORC_C_KMS, x_last = (double)(n_lambda - 1);
    for (int32_t k = k_begin; k < k_end; ++k) {
        if (rule == 0) {
            const double lam = observed_lambda(k, l0_obs, dl_obs) / opb;
            double dxdl;
            const double x = sample_coord(lam, kind, l0_ssp, dl_ssp, n_lambda, &dxdl);
            F[k] = interpolant(&b, x);
            if (dF) {                                              /* dF/dbeta = S~'(x) dx/dlambda dlambda/dbeta */
                double slope = 0.0;
                if (x >= 0.0 && x <= x_last) {
                    int32_t j = (int32_t)floor(x);
                    if (j > n_lambda - 2) j = n_lambda - 2;
                    slope = blend_sample(&b, j + 1) - blend_sample(&b, j);
                }
                dF[k] = slope * dxdl * (-lam / opb);
            }
        } else {
            const double lam_lo = observed_edge(k, n_c, l0_obs, dl_obs) / opb, lam_hi = observed_edge(k + 1, n_c, l0_obs, dl_obs) / opb;
            double dlo, dhi;
            const double x_lo = sample_coord(lam_lo, kind, l0_ssp, dl_ssp, n_lambda, &dlo);
            const double x_hi = sample_coord(lam_hi, kind, l0_ssp, dl_ssp, n_lambda, &dhi);
            const double W = x_hi - x_lo;
            const double I = interpolant_integral(&b, x_lo, x_hi);
            F[k] = I / W;
            if (dF) {
                /* F = I / W:  I' = S~(x_hi) x_hi' - S~(x_lo) x_lo'  (S~ = 0 at a clipped edge),  W' = x_hi' - x_lo' */
                const double xlo_b = dlo * (-lam_lo / opb), xhi_b = dhi * (-lam_hi / opb);
                const double Ip = interpolant(&b, x_hi) * xhi_b - interpolant(&b, x_lo) * xlo_b;
                dF[k] = Ip / W - F[k] * (xhi_b - xlo_b) / W;
            }
        }
    }
}

/* mode bit 0: 0 = point-sampled linear interpolation, 1 = bin average (R13 / R20);
 * mode bit 1: SSP grid log-sampled (R15);  mode bit 2: SSP wavelengths listed (R21, orc_set_lambda_ssp).
 * The combinations added by readings R20 / R21 (bin average on a log-sampled grid or on listed channel
 * wavelengths; listed SSP wavelengths) go through particle_spectrum_general, the others through the
 * functions above, whose arithmetic is unchanged. */
static int32_t general_mode(int32_t mode)
{
    return (mode & 4) != 0 || ((mode & 1) != 0 && ((mode & 2) != 0 || g_lambda_obs != 0));
}
static int32_t grid_kind(int32_t mode) { return (mode & 4) ? 2 : ((mode & 2) ? 1 : 0); }

static void particle_spectrum_mode(int32_t mode, double mass, int32_t ia, int32_t iz, double ta,
                                   double tz, double vlos, const float *flux, int32_t n_z,
                                   int32_t n_lambda, double l0_ssp, double dl_ssp, int32_t k_begin,
                                   int32_t k_end, int32_t n_c, double l0_obs, double dl_obs, double *F)
{
    if (general_mode(mode))
        particle_spectrum_general(mode & 1, grid_kind(mode), mass, ia, iz, ta, tz, vlos, flux, n_z, n_lambda, l0_ssp,
                                  dl_ssp, k_begin, k_end, n_c, l0_obs, dl_obs, F, 0);
    else if ((mode & 1) == 1)
        particle_spectrum_flux(mass, ia, iz, ta, tz, vlos, flux, n_z, n_lambda, l0_ssp, dl_ssp,
                               k_begin, k_end, l0_obs, dl_obs, F);
    else
        particle_spectrum(mass, ia, iz, ta, tz, vlos, flux, n_z, n_lambda, l0_ssp, dl_ssp, k_begin,
                          k_end, l0_obs, dl_obs, F, 0, (mode >> 1) & 1);
}

/* Cosmological redshift and flux scaling (reading R14; "Doppler shifted based
 * on the galaxy distance and line-of-sight velocity"): lambda_rest = lambda_obs / ((1+z)(1+beta)), which
 * is the z = 0 computation on the observed grid divided by (1+z) (bin edges included: the bin average is
 * unchanged by that rescaling); every spectrum is multiplied by flux_scale (passed on as a factor of the
 * mass, in which the spectrum is linear). */
void orc_particle_spectrum_mode(int32_t mode, double zc, double scale, float mass, float log_age, float log_z, float vlos,
                                int32_t n_age, int32_t n_z, int32_t n_lambda, const float *age_axis,
                                const float *z_axis, float l0_ssp, float dl_ssp, const float *flux,
                                int32_t n_c, float l0_obs, float dl_obs, double *F)
{
    int32_t ia, iz;
    double ta, tz;
    axis_cell(age_axis, n_age, log_age, &ia, &ta);
    axis_cell(z_axis, n_z, log_z, &iz, &tz);
    particle_spectrum_mode(mode, scale * (double)mass, ia, iz, ta, tz, (double)vlos, flux, n_z, n_lambda,
                           (double)l0_ssp, (double)dl_ssp, 0, n_c, n_c, (double)l0_obs / (1.0 + zc),
                           (double)dl_obs / (1.0 + zc), F);
}

void orc_particle_spectrum(float mass, float log_age, float log_z, float vlos, int32_t n_age,
                           int32_t n_z, int32_t n_lambda, const float *age_axis,
                           const float *z_axis, float l0_ssp, float dl_ssp, const float *flux,
                           int32_t n_c, float l0_obs, float dl_obs, double *F)
{
    int32_t ia, iz;
    double ta, tz;
    axis_cell(age_axis, n_age, log_age, &ia, &ta);
    axis_cell(z_axis, n_z, log_z, &iz, &tz);
    particle_spectrum((double)mass, ia, iz, ta, tz, (double)vlos, flux, n_z, n_lambda,
                      (double)l0_ssp, (double)dl_ssp, 0, n_c, (double)l0_obs, (double)dl_obs, F, 0, 0);
}

/* Same, but with the interpolation parameters given in fp64 (finite differences perturb
 * log age / log Z / v_los by steps far below fp32 resolution). */
void orc_particle_spectrum_f64_mode(int32_t mode, double zc, double scale, double mass, double log_age, double log_z,
                                    double vlos, int32_t n_age, int32_t n_z, int32_t n_lambda,
                                    const float *age_axis, const float *z_axis, float l0_ssp,
                                    float dl_ssp, const float *flux, int32_t n_c, float l0_obs,
                                    float dl_obs, int32_t ia, int32_t iz, double *F)
{
    /* cell (ia, iz) is held fixed by the caller: FD stays inside one bilinear patch */
    const double a0 = age_axis[ia], a1 = age_axis[ia + 1];
    const double z0 = z_axis[iz], z1 = z_axis[iz + 1];
    (void)n_age;
    particle_spectrum_mode(mode, scale * mass, ia, iz, (log_age - a0) / (a1 - a0), (log_z - z0) / (z1 - z0),
                           vlos, flux, n_z, n_lambda, (double)l0_ssp, (double)dl_ssp, 0, n_c, n_c,
                           (double)l0_obs / (1.0 + zc), (double)dl_obs / (1.0 + zc), F);
}

void orc_particle_spectrum_f64(double mass, double log_age, double log_z, double vlos,
                               int32_t n_age, int32_t n_z, int32_t n_lambda,
                               const float *age_axis, const float *z_axis, float l0_ssp,
                               float dl_ssp, const float *flux, int32_t n_c, float l0_obs,
                               float dl_obs, int32_t ia, int32_t iz, double *F)
{
    orc_particle_spectrum_f64_mode(0, 0.0, 1.0, mass, log_age, log_z, vlos, n_age, n_z, n_lambda, age_axis,
                                   z_axis, l0_ssp, dl_ssp, flux, n_c, l0_obs, dl_obs, ia, iz, F);
}

/* ------------------------------------------------------------------------------------
 * Step 6: cube[s][k] = sum over particles with key == s of F_p[k].  SURVEY.md 8(c) row 6.
 * If n_sel > 0 only the listed spaxels are computed and cube is [n_sel][n_c]; otherwise
 * cube is [n_s][n_c].  Particles are visited in the stable order of step 3.
 * ------------------------------------------------------------------------------------ */
void orc_build_cube_mode(int32_t mode, double zc, double scale, int64_t n, const float *pos, const float *vel, const float *mass,
                         const float *log_age, const float *log_z, const float *R, int32_t n_age,
                         int32_t n_z, int32_t n_lambda, const float *age_axis, const float *z_axis,
                         float l0_ssp, float dl_ssp, const float *flux, int32_t n_x, int32_t n_y,
                         float spaxel, int32_t n_c, float l0_obs, float dl_obs, const int32_t *sel,
                         int32_t n_sel, double *cube)
{
    const int32_t n_s = n_x * n_y;
    int32_t *key = (int32_t *)malloc(sizeof(int32_t) * (size_t)(n > 0 ? n : 1));
    int32_t *perm = (int32_t *)malloc(sizeof(int32_t) * (size_t)(n > 0 ? n : 1));
    int32_t *seg = (int32_t *)malloc(sizeof(int32_t) * ((size_t)n_s + 2));
    float *vlos = (float *)malloc(sizeof(float) * (size_t)(n > 0 ? n : 1));
    orc_rotate_bin(n, pos, vel, R, n_x, n_y, spaxel, key, vlos);
    orc_sort(n, key, n_s, perm, seg);
    const int32_t n_out = n_sel > 0 ? n_sel : n_s;
    /* Independent outputs: (spaxel, block of channels).  Splitting the channels only spreads
     * one heavy spaxel over several threads; each voxel still sums its particles in the
     * stable order of step 3. */
    enum { N_BLK = 8 };
#pragma omp parallel
    {
        double *F = (double *)malloc(sizeof(double) * (size_t)n_c);
#pragma omp for schedule(dynamic, 1) collapse(2)
        for (int32_t o = 0; o < n_out; ++o)
            for (int32_t blk = 0; blk < N_BLK; ++blk) {
                const int32_t s = n_sel > 0 ? sel[o] : o;
                const int32_t kb = (int32_t)(((int64_t)n_c * blk) / N_BLK);
                const int32_t ke = (int32_t)(((int64_t)n_c * (blk + 1)) / N_BLK);
                double *row = cube + (int64_t)o * n_c;
                for (int32_t k = kb; k < ke; ++k) row[k] = 0.0;
                for (int32_t q = seg[s]; q < seg[s + 1]; ++q) {
                    const int32_t p = perm[q];
                    int32_t ia, iz;
                    double ta, tz;
                    axis_cell(age_axis, n_age, log_age[p], &ia, &ta);
                    axis_cell(z_axis, n_z, log_z[p], &iz, &tz);
                    particle_spectrum_mode(mode, scale * (double)mass[p], ia, iz, ta, tz, (double)vlos[p], flux,
                                           n_z, n_lambda, (double)l0_ssp, (double)dl_ssp, kb, ke, n_c,
                                           (double)l0_obs / (1.0 + zc), (double)dl_obs / (1.0 + zc), F);
                    for (int32_t k = kb; k < ke; ++k) row[k] += F[k];
                }
            }
        free(F);
    }
    free(key); free(perm); free(seg); free(vlos);
}

void orc_build_cube(int64_t n, const float *pos, const float *vel, const float *mass,
                    const float *log_age, const float *log_z, const float *R, int32_t n_age,
                    int32_t n_z, int32_t n_lambda, const float *age_axis, const float *z_axis,
                    float l0_ssp, float dl_ssp, const float *flux, int32_t n_x, int32_t n_y,
                    float spaxel, int32_t n_c, float l0_obs, float dl_obs, const int32_t *sel,
                    int32_t n_sel, double *cube)
{
    orc_build_cube_mode(0, 0.0, 1.0, n, pos, vel, mass, log_age, log_z, R, n_age, n_z, n_lambda, age_axis, z_axis,
                        l0_ssp, dl_ssp, flux, n_x, n_y, spaxel, n_c, l0_obs, dl_obs, sel, n_sel, cube);
}

/* ------------------------------------------------------------------------------------
 * Steps 7-8: Gaussian taps and the PSF / LSF convolutions.  SURVEY.md 8(c) rows 7-8.
 *   taps g[i] = exp(-i^2 / (2 sigma^2)), i = -(size-1)/2 .. (size-1)/2, point-sampled,
 *   normalised to sum 1.  PSF = g (x) g over (x, y), the same for every channel; LSF = h
 *   along the channel axis; 'same' output, zero padding.  size 0 = that stage is off.
 * orc_convolve applies the LSF, then the direct (size x size)-tap 2-D PSF.
 * ------------------------------------------------------------------------------------ */
void orc_gauss_taps(int32_t size, double sigma, double *taps)
{
    const int32_t h = (size - 1) / 2;
    double sum = 0.0;
    for (int32_t i = -h; i <= h; ++i) {
        taps[i + h] = exp(-((double)i * (double)i) / (2.0 * sigma * sigma));
        sum += taps[i + h];
    }
    for (int32_t i = 0; i < size; ++i) taps[i] /= sum;
}

/* Wavelength-dependent PSF (reading R18): while an array is installed with orc_set_psf_sigma, channel k
 * uses taps of width psf_sigma_k[k] (the wrapper computes sigma_k = psf_sigma (lambda_k / lambda_ref)^alpha);
 * otherwise every channel uses psf_sigma.  Table [n_c][psf_size] of normalised taps. */
static const double *g_psf_sigma_k = 0;
void orc_set_psf_sigma(const double *sigma_k) { g_psf_sigma_k = sigma_k; }
static double *psf_taps_table(int32_t psf_size, double psf_sigma, int32_t n_c)
{
    double *t = (double *)malloc(sizeof(double) * (size_t)psf_size * (size_t)(n_c > 0 ? n_c : 1));
    for (int32_t k = 0; k < n_c; ++k)
        orc_gauss_taps(psf_size, g_psf_sigma_k ? g_psf_sigma_k[k] : psf_sigma, t + (size_t)k * psf_size);
    return t;
}

void orc_convolve(const double *in, int32_t n_x, int32_t n_y, int32_t n_c, int32_t psf_size,
                  double psf_sigma, int32_t lsf_size, double lsf_sigma, double *out)
{
    const int64_t n_vox = (int64_t)n_x * n_y * n_c;
    double *tmp = (double *)malloc(sizeof(double) * (size_t)(n_vox > 0 ? n_vox : 1));
    /* LSF along the channel, per spaxel */
    if (lsf_size > 0) {
        const int32_t h = (lsf_size - 1) / 2;
        double *taps = (double *)malloc(sizeof(double) * (size_t)lsf_size);
        orc_gauss_taps(lsf_size, lsf_sigma, taps);
#pragma omp parallel for schedule(static)
        for (int64_t s = 0; s < (int64_t)n_x * n_y; ++s)
            for (int32_t k = 0; k < n_c; ++k) {
                double acc = 0.0;
                for (int32_t d = -h; d <= h; ++d)
                    if (k + d >= 0 && k + d < n_c) acc += taps[d + h] * in[s * n_c + k + d];
                tmp[s * n_c + k] = acc;
            }
        free(taps);
    } else {
        memcpy(tmp, in, sizeof(double) * (size_t)n_vox);
    }
    /* PSF over (x, y), per channel: direct 2-D sum with the outer-product kernel */
    if (psf_size > 0) {
        const int32_t h = (psf_size - 1) / 2;
        double *taps = psf_taps_table(psf_size, psf_sigma, n_c);     /* [n_c][psf_size] */
#pragma omp parallel for schedule(static) collapse(2)
        for (int32_t x = 0; x < n_x; ++x)
            for (int32_t y = 0; y < n_y; ++y) {
                double *o = out + ((int64_t)x * n_y + y) * n_c;
                for (int32_t k = 0; k < n_c; ++k) o[k] = 0.0;
                for (int32_t dx = -h; dx <= h; ++dx)
                    for (int32_t dy = -h; dy <= h; ++dy) {
                        const int32_t xx = x + dx, yy = y + dy;
                        if (xx < 0 || xx >= n_x || yy < 0 || yy >= n_y) continue;
                        const double *r = tmp + ((int64_t)xx * n_y + yy) * n_c;
                        for (int32_t k = 0; k < n_c; ++k)
                            o[k] += taps[(size_t)k * psf_size + dx + h] * taps[(size_t)k * psf_size + dy + h] * r[k];
                    }
            }
        free(taps);
    } else {
        memcpy(out, tmp, sizeof(double) * (size_t)n_vox);
    }
    free(tmp);
}

/* Brute force on sampled output voxels of a (possibly huge) fp32 input cube: the full
 * size x size x lsf_size sum per voxel.  vox[i] = flat index ((x*n_y)+y)*n_c + k. */
void orc_convolve_voxels_f32(const float *in, int32_t n_x, int32_t n_y, int32_t n_c,
                             int32_t psf_size, double psf_sigma, int32_t lsf_size,
                             double lsf_sigma, const int64_t *vox, int64_t n_vox, double *out)
{
    const int32_t hp = psf_size > 0 ? (psf_size - 1) / 2 : 0;
    const int32_t hl = lsf_size > 0 ? (lsf_size - 1) / 2 : 0;
    const int32_t np = 2 * hp + 1;
    double *g = 0;                                         /* [n_c][np] */
    double *hh = (double *)malloc(sizeof(double) * (size_t)(2 * hl + 1));
    if (psf_size > 0) g = psf_taps_table(psf_size, psf_sigma, n_c);
    else { g = (double *)malloc(sizeof(double) * (size_t)n_c); for (int32_t k = 0; k < n_c; ++k) g[k] = 1.0; }
    if (lsf_size > 0) orc_gauss_taps(lsf_size, lsf_sigma, hh); else hh[0] = 1.0;
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n_vox; ++i) {
        const int64_t v = vox[i];
        const int32_t k = (int32_t)(v % n_c);
        const int32_t y = (int32_t)((v / n_c) % n_y);
        const int32_t x = (int32_t)(v / ((int64_t)n_c * n_y));
        double acc = 0.0;
        for (int32_t dx = -hp; dx <= hp; ++dx)
            for (int32_t dy = -hp; dy <= hp; ++dy) {
                const int32_t xx = x + dx, yy = y + dy;
                if (xx < 0 || xx >= n_x || yy < 0 || yy >= n_y) continue;
                for (int32_t dc = -hl; dc <= hl; ++dc) {
                    const int32_t kk = k + dc;
                    if (kk < 0 || kk >= n_c) continue;
                    /* LSF first, then the PSF of the OUTPUT channel k (the PSF acts per channel after the LSF) */
                    acc += g[(size_t)k * np + dx + hp] * g[(size_t)k * np + dy + hp] * hh[dc + hl]
                           * (double)in[((int64_t)xx * n_y + yy) * n_c + kk];
                }
            }
        out[i] = acc;
    }
    free(g); free(hh);
}

/* Transpose of orc_convolve (true scatter form, not assuming symmetry):
 * in_grad = LSF^T PSF^T out_grad.  Used by the adjoint and by the dot-product pin. */
void orc_convolve_transpose(const double *gout, int32_t n_x, int32_t n_y, int32_t n_c,
                            int32_t psf_size, double psf_sigma, int32_t lsf_size,
                            double lsf_sigma, double *gin)
{
    const int64_t n_vox = (int64_t)n_x * n_y * n_c;
    double *tmp = (double *)calloc((size_t)(n_vox > 0 ? n_vox : 1), sizeof(double));
    if (psf_size > 0) {
        const int32_t h = (psf_size - 1) / 2;
        double *taps = psf_taps_table(psf_size, psf_sigma, n_c);
        for (int32_t x = 0; x < n_x; ++x)          /* scatter: serial, small cubes only */
            for (int32_t y = 0; y < n_y; ++y)
                for (int32_t dx = -h; dx <= h; ++dx)
                    for (int32_t dy = -h; dy <= h; ++dy) {
                        const int32_t xx = x + dx, yy = y + dy;
                        if (xx < 0 || xx >= n_x || yy < 0 || yy >= n_y) continue;
                        const double *o = gout + ((int64_t)x * n_y + y) * n_c;
                        double *t = tmp + ((int64_t)xx * n_y + yy) * n_c;
                        for (int32_t k = 0; k < n_c; ++k)
                            t[k] += taps[(size_t)k * psf_size + dx + h] * taps[(size_t)k * psf_size + dy + h] * o[k];
                    }
        free(taps);
    } else {
        memcpy(tmp, gout, sizeof(double) * (size_t)n_vox);
    }
    if (lsf_size > 0) {
        const int32_t h = (lsf_size - 1) / 2;
        double *taps = (double *)malloc(sizeof(double) * (size_t)lsf_size);
        orc_gauss_taps(lsf_size, lsf_sigma, taps);
        for (int64_t i = 0; i < n_vox; ++i) gin[i] = 0.0;
        for (int64_t s = 0; s < (int64_t)n_x * n_y; ++s)
            for (int32_t k = 0; k < n_c; ++k)
                for (int32_t d = -h; d <= h; ++d)
                    if (k + d >= 0 && k + d < n_c)
                        gin[s * n_c + k + d] += taps[d + h] * tmp[s * n_c + k];
        free(taps);
    } else {
        memcpy(gin, tmp, sizeof(double) * (size_t)n_vox);
    }
    free(tmp);
}

/* ------------------------------------------------------------------------------------
 * Step 9: analytic adjoint.  SURVEY.md 8(a) row 9, 8(c) row 9.  Given G = dL/d(final cube):
 *   G' = LSF^T PSF^T G ; for particle p in spaxel s, with x_k its rest position (in SSP
 *   samples) at channel k, cell corners c with weights w_c(ta, tz):
 *     D_c    = sum_k G'[s][k] * lerp(T_c; x_k)
 *     E      = sum_k G'[s][k] * lambda_k * sum_c w_c * (T_c[j+1] - T_c[j]) / dl_ssp
 *     dL/dm      = sum_c w_c D_c
 *     dL/dlogA   = m * sum_c (dw_c/dta) D_c / (A[i+1] - A[i])    (0 if ta is clamped)
 *     dL/dlogZ   likewise
 *     dL/dv_los  = -m E / (c (1+beta)^2)
 *   out-of-FoV particles get 0.  Output in ORIGINAL particle order, fp64.
 * ------------------------------------------------------------------------------------ */
void orc_adjoint_mode(int32_t mode, double zc, double scale, int64_t n, const float *pos, const float *vel, const float *mass,
                 const float *log_age, const float *log_z, const float *R, int32_t n_age,
                 int32_t n_z, int32_t n_lambda, const float *age_axis, const float *z_axis,
                 float l0_ssp, float dl_ssp, const float *flux, int32_t n_x, int32_t n_y,
                 float spaxel, int32_t n_c, float l0_obs_f, float dl_obs_f, int32_t psf_size,
                 double psf_sigma, int32_t lsf_size, double lsf_sigma, const double *grad_cube,
                 double *g_mass, double *g_log_age, double *g_log_z, double *g_vlos)
{
    const int32_t n_s = n_x * n_y;
    /* observed grid divided by (1 + z): see orc_particle_spectrum_mode */
    const double l0_obs = (double)l0_obs_f / (1.0 + zc), dl_obs = (double)dl_obs_f / (1.0 + zc);
    const int64_t n_vox = (int64_t)n_s * n_c;
    double *gp = (double *)malloc(sizeof(double) * (size_t)(n_vox > 0 ? n_vox : 1));
    orc_convolve_transpose(grad_cube, n_x, n_y, n_c, psf_size, psf_sigma, lsf_size, lsf_sigma, gp);
    int32_t *key = (int32_t *)malloc(sizeof(int32_t) * (size_t)(n > 0 ? n : 1));
    float *vlos = (float *)malloc(sizeof(float) * (size_t)(n > 0 ? n : 1));
    orc_rotate_bin(n, pos, vel, R, n_x, n_y, spaxel, key, vlos);
#pragma omp parallel
    {
        double *F = (double *)malloc(sizeof(double) * (size_t)(n_c + 1));
        double *dS = (double *)malloc(sizeof(double) * (size_t)(n_c + 1));
#pragma omp for schedule(static)
        for (int64_t p = 0; p < n; ++p) {
            g_mass[p] = g_log_age[p] = g_log_z[p] = g_vlos[p] = 0.0;
            if (key[p] >= n_s) continue;
            const double *g = gp + (int64_t)key[p] * n_c;
            int32_t ia, iz;
            double ta, tz;
            axis_cell(age_axis, n_age, log_age[p], &ia, &ta);
            axis_cell(z_axis, n_z, log_z[p], &iz, &tz);
            /* D_c: dot of G' with the resampled corner template (unit mass, weight 1) */
            double D[4];
            for (int32_t c = 0; c < 4; ++c) {
                const double cta = (c & 1) ? 1.0 : 0.0, ctz = (c & 2) ? 1.0 : 0.0;
                particle_spectrum_mode(mode, 1.0, ia, iz, cta, ctz, (double)vlos[p], flux, n_z, n_lambda,
                                       (double)l0_ssp, (double)dl_ssp, 0, n_c, n_c, (double)l0_obs,
                                       (double)dl_obs, F);
                double acc = 0.0;
                for (int32_t k = 0; k < n_c; ++k) acc += g[k] * F[k];
                D[c] = acc;  /* c = 0:(i,j) 1:(i+1,j) 2:(i,j+1) 3:(i+1,j+1) */
            }
            double E = 0.0;
            if (general_mode(mode)) {
                /* readings R20 / R21: sum_k g[k] dF[k]/dbeta of the blended unit-mass spectrum, analytic */
                particle_spectrum_general(mode & 1, grid_kind(mode), 1.0, ia, iz, ta, tz, (double)vlos[p], flux, n_z,
                                          n_lambda, (double)l0_ssp, (double)dl_ssp, 0, n_c, n_c, (double)l0_obs,
                                          (double)dl_obs, F, dS);
                for (int32_t k = 0; k < n_c; ++k) E += g[k] * dS[k];
            } else if ((mode & 1) == 1) {
                /* Flux-conserving rule.  F[k] = (C(x_hi) - C(x_lo)) / B with C' = S~, the bin edges
                 * x(lambda_e) = (lambda_e/(1+beta) - l0_ssp)/dl_ssp and B = dl_obs/((1+beta) dl_ssp):
                 *   dF[k]/dbeta = F[k]/(1+beta) - (lambda_hi S~(x_hi) - lambda_lo S~(x_lo)) / (dl_obs (1+beta)),
                 * an edge clipped to the coverage does not move (S~ = 0 outside the coverage gives
                 * exactly that).  E = sum_k g[k] (lambda_hi S~(x_hi) - lambda_lo S~(x_lo)) for the blended
                 * unit-mass spectrum, point-evaluated at the n_c + 1 bin edges. */
                particle_spectrum(1.0, ia, iz, ta, tz, (double)vlos[p], flux, n_z, n_lambda,
                                  (double)l0_ssp, (double)dl_ssp, 0, n_c + 1,
                                  (double)l0_obs - 0.5 * (double)dl_obs, (double)dl_obs, F, 0, 0);
                for (int32_t k = 0; k < n_c; ++k) {
                    const double lam_lo = (double)l0_obs + (double)dl_obs * ((double)k - 0.5);
                    const double lam_hi = lam_lo + (double)dl_obs;
                    E += g[k] * (lam_hi * F[k + 1] - lam_lo * F[k]);
                }
            } else {
                /* E: needs the slope of the blended unit-mass spectrum */
                particle_spectrum(1.0, ia, iz, ta, tz, (double)vlos[p], flux, n_z, n_lambda,
                                  (double)l0_ssp, (double)dl_ssp, 0, n_c, (double)l0_obs,
                                  (double)dl_obs, F, dS, (mode >> 1) & 1);
                /* dF/dbeta = dS/dx * dx/dbeta;  linear grid: dx/dbeta = -lambda_k / ((1+beta)^2 dl_ssp);
                 * log grid: x = log10(lambda_k / ((1+beta) l0_ssp)) / dl_ssp, dx/dbeta = -1 / ((1+beta) dl_ssp ln 10),
                 * written as the same expression with lambda_k replaced by (1+beta) / ln 10 */
                for (int32_t k = 0; k < n_c; ++k) {
                    const double lam_eff = ((mode >> 1) & 1) ? (1.0 + (double)vlos[p] / ORC_C_KMS) / log(10.0)
                                                             : observed_lambda(k, (double)l0_obs, (double)dl_obs);
                    E += g[k] * lam_eff * dS[k] / (double)dl_ssp;
                }
            }
            const double m = scale * (double)mass[p];
            const double beta = (double)vlos[p] / ORC_C_KMS;
            /* unit-mass, unit-scale sum_k g_k F_k; scaled after g_vlos below has used it */
            g_mass[p] = (1 - ta) * (1 - tz) * D[0] + ta * (1 - tz) * D[1] + (1 - ta) * tz * D[2]
                        + ta * tz * D[3];
            const double dA = (double)age_axis[ia + 1] - (double)age_axis[ia];
            const double dZ = (double)z_axis[iz + 1] - (double)z_axis[iz];
            const int a_free = ((double)log_age[p] > (double)age_axis[0])
                               && ((double)log_age[p] < (double)age_axis[n_age - 1]);
            const int z_free = ((double)log_z[p] > (double)z_axis[0])
                               && ((double)log_z[p] < (double)z_axis[n_z - 1]);
            g_log_age[p] = a_free ? m * (-(1 - tz) * D[0] + (1 - tz) * D[1] - tz * D[2] + tz * D[3]) / dA
                                  : 0.0;
            g_log_z[p] = z_free ? m * (-(1 - ta) * D[0] - ta * D[1] + (1 - ta) * D[2] + ta * D[3]) / dZ
                                : 0.0;
            if (general_mode(mode))
                g_vlos[p] = m * E / ORC_C_KMS;                     /* d/dv_los = (1/c) d/dbeta */
            else if ((mode & 1) == 1)
                g_vlos[p] = m * (g_mass[p] - E / (double)dl_obs) / (ORC_C_KMS * (1.0 + beta));
            else
                g_vlos[p] = -m * E / (ORC_C_KMS * (1.0 + beta) * (1.0 + beta));
            g_mass[p] *= scale;
        }
        free(F); free(dS);
    }
    free(gp); free(key); free(vlos);
}

void orc_adjoint(int64_t n, const float *pos, const float *vel, const float *mass,
                 const float *log_age, const float *log_z, const float *R, int32_t n_age,
                 int32_t n_z, int32_t n_lambda, const float *age_axis, const float *z_axis,
                 float l0_ssp, float dl_ssp, const float *flux, int32_t n_x, int32_t n_y,
                 float spaxel, int32_t n_c, float l0_obs, float dl_obs, int32_t psf_size,
                 double psf_sigma, int32_t lsf_size, double lsf_sigma, const double *grad_cube,
                 double *g_mass, double *g_log_age, double *g_log_z, double *g_vlos)
{
    orc_adjoint_mode(0, 0.0, 1.0, n, pos, vel, mass, log_age, log_z, R, n_age, n_z, n_lambda, age_axis, z_axis,
                     l0_ssp, dl_ssp, flux, n_x, n_y, spaxel, n_c, l0_obs, dl_obs, psf_size, psf_sigma,
                     lsf_size, lsf_sigma, grad_cube, g_mass, g_log_age, g_log_z, g_vlos);
}

/* ------------------------------------------------------------------------------------
 * Noise stage ("add realistic noise"; reading R17 -- the paper
 * names no model).  cube_noisy[v] = cube[v] + sigma_v n_v,
 *   sigma_v = sqrt(sigma_read^2 + gain * max(cube[v], 0))      (read noise + shot noise, flux units)
 *   n_v ~ N(0, 1), independent, from a COUNTER-BASED generator so that both implementations draw the
 *   same numbers: Philox4x32-10 (Salmon et al. 2011) with key = (seed low, seed high) and counter
 *   (q low, q high, 0, 0), q = v / 4, gives four 32-bit words r0..r3 for voxels 4q .. 4q+3;
 *   u_i = ((r_i >> 9) + 0.5) 2^-23 in (0, 1)  (exact in fp32);  Box-Muller:
 *   n_{4q} = R0 cos(2 pi u1), n_{4q+1} = R0 sin(2 pi u1), R0 = sqrt(-2 ln u0); voxels 4q+2, 4q+3 from (u2, u3).
 * ------------------------------------------------------------------------------------ */
static uint32_t mulhilo32(uint32_t a, uint32_t b, uint32_t *hi)
{
    const uint64_t p = (uint64_t)a * (uint64_t)b;
    *hi = (uint32_t)(p >> 32);
    return (uint32_t)p;
}

void orc_philox4x32_10(const uint32_t ctr_in[4], const uint32_t key_in[2], uint32_t out[4])
{
    uint32_t c0 = ctr_in[0], c1 = ctr_in[1], c2 = ctr_in[2], c3 = ctr_in[3];
    uint32_t k0 = key_in[0], k1 = key_in[1];
    for (int r = 0; r < 10; ++r) {
        uint32_t hi0, hi1;
        const uint32_t lo0 = mulhilo32(0xD2511F53u, c0, &hi0);
        const uint32_t lo1 = mulhilo32(0xCD9E8D57u, c2, &hi1);
        const uint32_t n0 = hi1 ^ c1 ^ k0, n1 = lo1, n2 = hi0 ^ c3 ^ k1, n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;                              /* Weyl sequence of the key schedule */
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

void orc_noise_normals(int64_t n, uint64_t seed, double *normals)
{   /* the standard normal deviates n_v alone (pinned on their own) */
    const double two_pi = 6.283185307179586476925286766559;
    const uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
    for (int64_t q = 0; 4 * q < n; ++q) {
        const uint32_t ctr[4] = {(uint32_t)(uint64_t)q, (uint32_t)((uint64_t)q >> 32), 0u, 0u};
        uint32_t r[4];
        orc_philox4x32_10(ctr, key, r);
        double u[4], z[4];
        for (int i = 0; i < 4; ++i) u[i] = ((double)(r[i] >> 9) + 0.5) * (1.0 / 8388608.0);
        const double R0 = sqrt(-2.0 * log(u[0])), R1 = sqrt(-2.0 * log(u[2]));
        z[0] = R0 * cos(two_pi * u[1]); z[1] = R0 * sin(two_pi * u[1]);
        z[2] = R1 * cos(two_pi * u[3]); z[3] = R1 * sin(two_pi * u[3]);
        for (int i = 0; i < 4 && 4 * q + i < n; ++i) normals[4 * q + i] = z[i];
    }
}

void orc_add_noise(const double *cube, int64_t n, double sigma_read, double gain, uint64_t seed, double *out)
{
    double *z = (double *)malloc(sizeof(double) * (size_t)(n > 0 ? n : 1));
    orc_noise_normals(n, seed, z);
    for (int64_t v = 0; v < n; ++v) {
        const double f = cube[v] > 0.0 ? cube[v] : 0.0;
        out[v] = cube[v] + sqrt(sigma_read * sigma_read + gain * f) * z[v];
    }
    free(z);
}

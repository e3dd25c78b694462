// General-grid mode of step 5 (readings R20, R21): the combinations the fixed-point
// resamplers do not take -- the bin average on a log-sampled SSP grid or on listed channel wavelengths, and listed
// (irregular) SSP wavelengths under either rule.  Positions are evaluated per sample in fp64:
//     x = X(tab[e], g)        tab: per-launch table over the channel centres (point rule) or the n_c + 1 bin edges
//                             (bin average); g: one fp64 value per particle (Rec::a_fx holds its bits)
//   kind 0  lambda_j = l0 + j dl      tab = lambda / ((1+z) dl),             g = 1/(1+beta),            x = tab g - l0/dl
//   kind 1  lambda_j = l0 10^(j dl)   tab = log10(lambda / ((1+z) l0)) / dl, g = -log10(1+beta) / dl,   x = tab + g
//   kind 2  lambda_j listed           tab = lambda / (1+z),                  g = 1/(1+beta),            x = j + (tab g - lambda_j) / (lambda_{j+1} - lambda_j)
//           on the knot interval j that holds tab g (first / last interval continued outside the coverage), found through
//           a uniform look-up table over the covered wavelengths (cell -> knot interval at the cell's start) and a short walk.
#pragma once
#include <stdint.h>

namespace rubix {

constexpr int kGenLutPerKnot = 8;           // look-up cells per SSP sample (cells of (coverage) / (8 N_l))

struct GenGrid {
    int32_t kind, n_lambda, lut_n, flux;    // flux: tab holds bin edges (n_c + 1 entries), else channel centres (n_c)
    double a0;                              // kind 0: -l0 / dl
    double lut_l0, lut_inv_h;               // kind 2: cell m covers [lut_l0 + m h, lut_l0 + (m + 1) h)
    double log_scale;                       // kind 1: 1 / dl  (g = -log10(1 + beta) * log_scale)
    const double *tab;
    const double *knots;                    // kind 2: [n_lambda] listed wavelengths
    const double *inv_w;                    // kind 2: [n_lambda - 1] 1 / (lambda_{j+1} - lambda_j)
    const int32_t *lut;
};

// Sampling coordinate of table value t for a particle with Doppler value g.  *slope = d x / d (t g) for kind 2 (else unused).
__device__ __forceinline__ double gen_coord(const GenGrid &G, double t, double g, double *slope = nullptr)
{
    if (G.kind == 0) return fma(t, g, G.a0);
    if (G.kind == 1) return t + g;
    const double lam = t * g;
    int m = (int)((lam - G.lut_l0) * G.lut_inv_h);
    m = m < 0 ? 0 : (m >= G.lut_n ? G.lut_n - 1 : m);
    int j = __ldg(G.lut + m);
    while (j < G.n_lambda - 2 && lam >= __ldg(G.knots + j + 1)) ++j;
    const double w = __ldg(G.inv_w + j);
    if (slope) *slope = w;
    return (double)j + (lam - __ldg(G.knots + j)) * w;
}

// per-particle Doppler value g of the header (beta = v_los / c)
__device__ __forceinline__ double gen_doppler(const GenGrid &G, double opb)
{
    return G.kind == 1 ? -log10(opb) * G.log_scale : 1.0 / opb;
}

}  // namespace rubix

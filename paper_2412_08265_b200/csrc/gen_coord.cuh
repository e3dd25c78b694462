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

constexpr int kGenLutPerKnot = 1;           // look-up cells per SSP sample, at least (cells of (coverage) / N_l) ...
constexpr int kGenLutMaxPerKnot = 64;       // ... and as many as it takes to make a cell narrower than TWO of the narrowest knot
                                            // intervals (then two conditional steps find the interval), up to this many.  The
                                            // table stays small on purpose: it has to live in L1 next to the knots.

struct GenGrid {
    int32_t kind, n_lambda, lut_n, flux;    // flux: tab holds bin edges (n_c + 1 entries), else channel centres (n_c)
    double a0;                              // kind 0: -l0 / dl
    double lut_l0, lut_inv_h;               // kind 2: cell m covers [lut_l0 + m h, lut_l0 + (m + 1) h)
    double log_scale;                       // kind 1: 1 / dl  (g = -log10(1 + beta) * log_scale)
    const double *tab;
    const double2 *kw;                      // kind 2: [n_lambda] (lambda_j, 1 / (lambda_{j+1} - lambda_j)); the last entry repeats
                                            // the last interval's width
    const int32_t *lut;
    int32_t walk;                           // kind 2: 1 = a cell may hold more than two knots (walk), 0 = at most two (two steps)
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
    // the cell starts in knot interval j; with cells narrower than two of the narrowest intervals the position is in
    // j, j + 1 or j + 2
    double2 a = __ldg(G.kw + j), b = __ldg(G.kw + j + 1);
    while (j < G.n_lambda - 2 && lam >= b.x) { ++j; a = b; b = __ldg(G.kw + j + 1); }
    if (slope) *slope = a.y;
    return (double)j + (lam - a.x) * a.y;
}

// The same with the kind fixed at compile time (the accumulate kernel evaluates it 29-58 times per thread and particle:
// only one of the three paths is compiled in, which keeps the unrolled loop inside the instruction cache).
template <int KIND>
__device__ __forceinline__ double gen_coord_k(const GenGrid &G, double t, double g)
{
    if (KIND == 0) return fma(t, g, G.a0);
    if (KIND == 1) return t + g;
    const double lam = t * g;
    int m = (int)((lam - G.lut_l0) * G.lut_inv_h);
    m = m < 0 ? 0 : (m >= G.lut_n ? G.lut_n - 1 : m);
    int j = __ldg(G.lut + m);
    const int jt = G.n_lambda - 2;
    double2 a = __ldg(G.kw + j), b = __ldg(G.kw + j + 1);
    if (G.walk) {
        while (j < jt && lam >= b.x) { ++j; a = b; b = __ldg(G.kw + j + 1); }
    } else {                                                 // two conditional steps, no branch
        const double2 c = __ldg(G.kw + min(j + 2, jt + 1));
        const bool s1 = j < jt && lam >= b.x;
        const bool s2 = s1 && j + 1 < jt && lam >= c.x;
        j += (s1 ? 1 : 0) + (s2 ? 1 : 0);
        a.x = s2 ? c.x : (s1 ? b.x : a.x);
        a.y = s2 ? c.y : (s1 ? b.y : a.y);
    }
    return (double)j + (lam - a.x) * a.y;
}

// per-particle Doppler value g of the header (beta = v_los / c)
__device__ __forceinline__ double gen_doppler(const GenGrid &G, double opb)
{
    return G.kind == 1 ? -log10(opb) * G.log_scale : 1.0 / opb;
}

}  // namespace rubix

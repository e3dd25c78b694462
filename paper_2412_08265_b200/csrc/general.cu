// General-grid mode of step 5 (gen_coord.cuh; readings R20, R21): per-launch tables and the adjoint kernel.
//   k_gen_knots / k_gen_lut   listed SSP wavelengths -> fp64 knots, inverse interval widths, look-up table
//   k_gen_tab                 observed channel centres or bin edges -> the table `tab` of gen_coord.cuh
//   k_adjoint_general         step 9 for these modes: one warp per particle, lanes over the channels, fp64 positions
#include <math.h>

#include <vector>

#include "common.cuh"
#include "gen_coord.cuh"

namespace rubix {

__global__ void __launch_bounds__(256)
k_gen_knots(int32_t n_lambda, const float *__restrict__ lam, double2 *__restrict__ kw)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n_lambda) return;
    const int i = j + 1 < n_lambda ? j : n_lambda - 2;      // the last entry repeats the last interval's width
    kw[j] = make_double2((double)lam[j], 1.0 / ((double)lam[i + 1] - (double)lam[i]));
}

// lut[m] = largest j <= n_lambda - 2 with knots[j] <= start of cell m (0 for cells that start below the first knot)
__global__ void __launch_bounds__(256)
k_gen_lut(int32_t lut_n, double l0, double h, const double2 *__restrict__ kw, int32_t n_lambda, int32_t *__restrict__ lut)
{
    const int m = blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= lut_n) return;
    const double start = l0 + h * (double)m;
    int lo = 0, hi = n_lambda - 2;
    while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (kw[mid].x <= start) lo = mid; else hi = mid - 1;
    }
    lut[m] = lo;
}

// Observed wavelength of table entry e: channel centre (point rule) or bin edge (bin average, reading R20: on a uniform
// grid lambda_e = l0 + (e - 1/2) dl; on a listed grid the midpoints of neighbouring channels, the outer edges half a
// neighbouring spacing outside), divided by (1 + z), mapped to the table value of gen_coord.cuh.
__global__ void __launch_bounds__(256)
k_gen_tab(int32_t n_e, int32_t n_c, int32_t flux, const float *__restrict__ lam, double l0_obs, double dl_obs, double zp1,
          int32_t kind, double l0_ssp, double dl_ssp, double *__restrict__ tab)
{
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n_e) return;
    double l;
    if (!flux) {
        l = lam ? (double)lam[e] : l0_obs + dl_obs * (double)e;
    } else if (!lam) {
        l = l0_obs + dl_obs * ((double)e - 0.5);
    } else if (e == 0) {
        l = (double)lam[0] - 0.5 * ((double)lam[1] - (double)lam[0]);
    } else if (e == n_c) {
        l = (double)lam[n_c - 1] + 0.5 * ((double)lam[n_c - 1] - (double)lam[n_c - 2]);
    } else {
        l = 0.5 * ((double)lam[e - 1] + (double)lam[e]);
    }
    l /= zp1;
    tab[e] = kind == 0 ? l / dl_ssp : (kind == 1 ? log10(l / l0_ssp) / dl_ssp : l);
}

int gen_kind(const rubix_ssp *s) { return s->lambda_grid ? 2 : (s->log_lambda ? 1 : 0); }

// ---- host: the same coordinate map in fp64, for the window capacity (largest span of one channel, in samples)
static double host_coord(const rubix_ssp *s, double lam_rest)
{
    if (!s->lambda_grid) {
        return s->log_lambda ? log10(lam_rest / (double)s->lambda0) / (double)s->dlambda
                             : (lam_rest - (double)s->lambda0) / (double)s->dlambda;
    }
    const float *L = s->lambda_grid;
    const int n = s->n_lambda;
    int j = 0;
    if (lam_rest >= (double)L[n - 1]) j = n - 2;
    else if (lam_rest > (double)L[0]) {
        int lo = 0, hi = n - 1;
        while (lo < hi) { const int mid = (lo + hi + 1) / 2; if ((double)L[mid] <= lam_rest) lo = mid; else hi = mid - 1; }
        j = lo > n - 2 ? n - 2 : lo;
    }
    return (double)j + (lam_rest - (double)L[j]) / ((double)L[j + 1] - (double)L[j]);
}

static double host_edge(const rubix_telescope *t, int e, bool flux)
{
    const float *lam = t->lambda_obs;
    const int n_c = t->n_channels;
    double l;
    if (!flux) l = lam ? (double)lam[e < n_c ? e : n_c - 1] : (double)t->lambda0 + (double)t->dlambda * e;
    else if (!lam) l = (double)t->lambda0 + (double)t->dlambda * ((double)e - 0.5);
    else if (e == 0) l = (double)lam[0] - 0.5 * ((double)lam[1] - (double)lam[0]);
    else if (e >= n_c) l = (double)lam[n_c - 1] + 0.5 * ((double)lam[n_c - 1] - (double)lam[n_c - 2]);
    else l = 0.5 * ((double)lam[e - 1] + (double)lam[e]);
    return l / (1.0 + (double)t->redshift);
}

double gen_step_max(const rubix_ssp *s, const rubix_telescope *t)
{
    const bool flux = t->resample == RUBIX_RESAMPLE_FLUX;
    const double betas[3] = {-kBetaCap, 0.0, kBetaCap};
    const double x_top = (double)(s->n_lambda - 1);
    double m = 0.0;
    for (int b = 0; b < 3; ++b) {
        const double c = 1.0 / (1.0 + betas[b]);
        double prev = host_coord(s, host_edge(t, 0, flux) * c);
        for (int e = 1; e <= t->n_channels - (flux ? 0 : 1); ++e) {
            const double x = host_coord(s, host_edge(t, e, flux) * c);
            // only the part of the span inside the coverage needs table samples
            const double lo = fmin(fmax(prev, 0.0), x_top), hi = fmin(fmax(x, 0.0), x_top);
            m = fmax(m, hi - lo);
            prev = x;
        }
    }
    return m * 1.001 + 1e-6;
}

// Largest number of SSP samples spanned by `tc` consecutive channels (point rule: channel k .. k + tc - 1; bin average:
// edges k .. k + tc), inside the coverage, over the three Doppler factors that bound the velocity cap: what one channel
// tile's table has to hold.  (gen_step_max x tc would charge the densest stretch of a listed grid to the whole tile.)
double gen_window_max(const rubix_ssp *s, const rubix_telescope *t, int tc)
{
    const bool flux = t->resample == RUBIX_RESAMPLE_FLUX;
    const int n_e = t->n_channels + (flux ? 1 : 0);
    const int reach = flux ? tc : tc - 1;
    const double betas[3] = {-kBetaCap, 0.0, kBetaCap};
    const double x_top = (double)(s->n_lambda - 1);
    std::vector<double> x((size_t)n_e);
    double m = 0.0;
    for (int b = 0; b < 3; ++b) {
        const double c = 1.0 / (1.0 + betas[b]);
        for (int e = 0; e < n_e; ++e) x[e] = fmin(fmax(host_coord(s, host_edge(t, e, flux) * c), 0.0), x_top);
        for (int e = 0; e < n_e; ++e) {
            const int hi = e + reach < n_e ? e + reach : n_e - 1;
            m = fmax(m, x[hi] - x[e]);
        }
    }
    return m * 1.001 + 1e-3;
}

// the GenGrid of a launch: pointers into the workspace and constants (host only, no launch)
void gen_grid_params(const PassInputs &in, const Layout &L, char *ws, GenGrid *G)
{
    const rubix_ssp *s = in.ssp;
    G->kind = gen_kind(s);
    G->n_lambda = s->n_lambda;
    G->flux = in.tel->resample == RUBIX_RESAMPLE_FLUX ? 1 : 0;
    G->a0 = -(double)s->lambda0 / (double)s->dlambda;
    G->log_scale = 1.0 / (double)s->dlambda;
    G->tab = (const double *)(ws + L.off_gtab);
    G->kw = (const double2 *)(ws + L.off_gknots);
    G->lut = (const int32_t *)(ws + L.off_glut);
    G->lut_n = kGenLutPerKnot * s->n_lambda;
    G->lut_l0 = 0.0;
    G->lut_inv_h = 0.0;
    G->walk = 0;
    if (G->kind == 2) {
        const double first = (double)s->lambda_grid[0], last = (double)s->lambda_grid[s->n_lambda - 1];
        double narrowest = last - first;
        for (int j = 1; j < s->n_lambda; ++j)
            narrowest = fmin(narrowest, (double)s->lambda_grid[j] - (double)s->lambda_grid[j - 1]);
        // cells narrower than two of the narrowest intervals => the interval is the cell's or one of the next two
        const double want = ceil((last - first) / (2.0 * narrowest) * (1.0 + 1e-6)) + 1.0;
        const double cap = (double)kGenLutMaxPerKnot * s->n_lambda;
        if (want > (double)G->lut_n) G->lut_n = (int32_t)(want < cap ? want : cap);
        G->walk = want > cap ? 1 : 0;
        G->lut_l0 = first;
        G->lut_inv_h = (double)G->lut_n / (last - first);
    }
}

cudaError_t launch_gen_setup(const PassInputs &in, const Layout &L, char *ws, cudaStream_t st, GenGrid *G)
{
    const rubix_ssp *s = in.ssp;
    const rubix_telescope *t = in.tel;
    gen_grid_params(in, L, ws, G);
    cudaError_t e;
    if (G->kind == 2) {
        float *lam_dev = (float *)(ws + L.off_glam);
        e = cudaMemcpyAsync(lam_dev, s->lambda_grid, (size_t)s->n_lambda * 4, cudaMemcpyHostToDevice, st);
        if (e != cudaSuccess) return e;
        k_gen_knots<<<(unsigned)((s->n_lambda + 255) / 256), 256, 0, st>>>(s->n_lambda, lam_dev, (double2 *)(ws + L.off_gknots));
        RUBIX_LAUNCH_CHECK();
        const double first = G->lut_l0, h = 1.0 / G->lut_inv_h;
        k_gen_lut<<<(unsigned)((G->lut_n + 255) / 256), 256, 0, st>>>(G->lut_n, first, h, G->kw, s->n_lambda,
                                                                      (int32_t *)(ws + L.off_glut));
        RUBIX_LAUNCH_CHECK();
    }
    const float *lam_obs_dev = nullptr;
    if (t->lambda_obs) {
        lam_obs_dev = (const float *)(ws + L.off_lamobs);
        e = cudaMemcpyAsync(ws + L.off_lamobs, t->lambda_obs, (size_t)L.n_c * 4, cudaMemcpyHostToDevice, st);
        if (e != cudaSuccess) return e;
    }
    const int n_e = L.n_c + (G->flux ? 1 : 0);
    k_gen_tab<<<(unsigned)((n_e + 255) / 256), 256, 0, st>>>(n_e, L.n_c, G->flux, lam_obs_dev, (double)t->lambda0, (double)t->dlambda,
                                                             1.0 + (double)t->redshift, G->kind, (double)s->lambda0,
                                                             (double)s->dlambda, (double *)(ws + L.off_gtab));
    RUBIX_LAUNCH_CHECK();
    return cudaSuccess;
}

// ------------------------------------------------------------------------------------------
// k_adjoint_general: step 9 in the general-grid mode.  One warp per in-FoV particle (sorted
// order), lanes stride over its covered channels / bins.  With x the fp64 position and u_c the bilinear weights:
//   point rule   v_c = lerp(T_c; x_k);  d F_k / d beta = (sum_c u_c (T_c[j+1] - T_c[j])) x_k'
//   bin average  F_c[k] = (1/W_k) sum_j w_j T_c[j],  w_j = H(x_hi - j) - H(x_lo - j) (edges clipped to the coverage, H the
//                integral of the hat function), W_k = x_hi - x_lo the FULL width;
//                d F_k / d beta = [S~(x_hi) x_hi' - S~(x_lo) x_lo'] / W_k - F_k (x_hi' - x_lo') / W_k   (S~ = 0 at a clipped edge)
//   x' = d x / d beta:  kind 0  -(x - a0) / (1+beta);  kind 1  -1 / ((1+beta) dl ln 10);  kind 2  -lambda_rest / ((1+beta) w_j)
// The sums over channels use the difference basis of k_adjoint (P0, Pa, Pz, Pq) in fp32 per channel and fp64 across
// channels; the velocity sum is fp64 throughout (x' ~ 3000 multiplies a slope).  No atomics; ORIGINAL particle order.
// ------------------------------------------------------------------------------------------
struct AdjGenParams {
    const int32_t *perm, *seg_off, *key;
    const float *vlos, *mass, *flux, *gconv;
    const Rec *rec;
    const AdjAux *aux;
    float *g_mass, *g_age, *g_z, *g_v;
    int32_t n_lambda, pitch, n_z, n_c, n_s;
    float flux_scale;
    int64_t n;
    GenGrid gen;
};

__device__ __forceinline__ double gen_hat_integral(double t)
{
    const double a = fmin(fmax(t, -1.0), 1.0);
    const double lo = 0.5 * (1.0 + a) * (1.0 + a);
    const double hi = 1.0 - 0.5 * (1.0 - a) * (1.0 - a);
    return a <= 0.0 ? lo : hi;
}

template <bool FLUX>
__global__ void __launch_bounds__(256)
k_adjoint_general(const __grid_constant__ AdjGenParams P)
{
    const int64_t i = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;   // sorted position
    const int lane = threadIdx.x & 31;
    if (i >= P.n) return;
    const int p = P.perm[i];
    if (i >= P.seg_off[P.n_s]) {                            // dropped particle: zero gradient
        if (lane == 0) P.g_mass[p] = P.g_age[p] = P.g_z[p] = P.g_v[p] = 0.0f;
        return;
    }
    const Rec r = P.rec[i];
    const AdjAux ax = P.aux[i];
    const GenGrid &G = P.gen;
    const double opb = 1.0 + (double)P.vlos[p] / kCkms, inv_opb = 1.0 / opb;
    const double g = gen_doppler(G, opb);                   // (the table mode's records carry fixed-point values instead)
    const float *gr = P.gconv + (size_t)P.key[p] * P.n_c;
    const float *T0 = P.flux + r.cell;
    const float *T1 = T0 + (size_t)P.n_z * P.pitch, *T2 = T0 + P.pitch, *T3 = T1 + P.pitch;
    const double ta = (double)ax.ta, tz = (double)ax.tz;
    const float u0 = (float)((1.0 - ta) * (1.0 - tz)), u1 = (float)(ta * (1.0 - tz));
    const float u2 = (float)((1.0 - ta) * tz), u3 = (float)(ta * tz);
    const double x_top = (double)(P.n_lambda - 1);
    const int jmax = P.n_lambda - 2;
    const double xp_log = -G.log_scale * inv_opb * 0.43429448190325182765;      // kind 1: the same for every channel
    // d x / d beta at table value t (x = gen_coord(t), slope = d x / d lambda_rest for kind 2)
    auto xprime = [&](double x, double t, double slope) -> double {
        if (G.kind == 0) return -(x - G.a0) * inv_opb;
        if (G.kind == 1) return xp_log;
        return -slope * t * g * inv_opb;
    };
    // blended unit-mass interpolant at x inside the coverage, in the difference basis with the SAME fp64 (ta, tz) as the
    // bin average F below: the edge terms and F W'/W cancel to the derivative, so their weights must agree exactly
    auto blended = [&](double x) -> double {
        const int j = min((int)x, jmax);
        const double f = x - (double)j;
        const uint32_t ju = (uint32_t)j;
        auto mix = [&](uint32_t q) -> double {
            const float t0 = __ldg(T0 + q), t1 = __ldg(T1 + q), t2 = __ldg(T2 + q), t3 = __ldg(T3 + q);
            // promoted BEFORE subtracting: corners may differ by far more than a factor of two, where an fp32 difference
            // rounds at the level of the larger sample -- and the derivative below is a difference of such blends
            const double d0 = t0, d1 = t1, d2 = t2, d3 = t3;
            return d0 + ta * (d1 - d0) + tz * (d2 - d0) + ta * tz * ((d3 - d2) - (d1 - d0));
        };
        const double a = mix(ju), b = mix(ju + 1);
        return a + f * (b - a);
    };
    double P0 = 0, Pa = 0, Pz = 0, Pq = 0, E = 0;
    for (int k = r.k_lo + lane; k <= r.k_hi; k += 32) {
        const float gk = __ldg(gr + k);
        if (!FLUX) {
            double slope = 0.0;
            const double t = __ldg(G.tab + k);
            const double x = gen_coord(G, t, g, &slope);
            if (!(x >= 0.0 && x <= x_top)) continue;
            const int j = min((int)x, jmax);
            const float f = (float)(x - (double)j);
            const uint32_t ju = (uint32_t)j;
            const float a0 = __ldg(T0 + ju), b0 = __ldg(T0 + ju + 1) - a0;
            const float a1 = __ldg(T1 + ju), b1 = __ldg(T1 + ju + 1) - a1;
            const float a2 = __ldg(T2 + ju), b2 = __ldg(T2 + ju + 1) - a2;
            const float a3 = __ldg(T3 + ju), b3 = __ldg(T3 + ju + 1) - a3;
            const float v0 = fmaf(f, b0, a0);
            const float da = fmaf(f, b1 - b0, a1 - a0), dz = fmaf(f, b2 - b0, a2 - a0);
            const float dq = fmaf(f, (b3 - b2) - (b1 - b0), (a3 - a2) - (a1 - a0));
            P0 += (double)(gk * v0); Pa += (double)(gk * da); Pz += (double)(gk * dz); Pq += (double)(gk * dq);
            const float sl = fmaf(u3, b3, fmaf(u2, b2, fmaf(u1, b1, u0 * b0)));
            E += (double)(gk * sl) * xprime(x, t, slope);
        } else {
            double sl_lo = 0.0, sl_hi = 0.0;
            const double t_lo = __ldg(G.tab + k), t_hi = __ldg(G.tab + k + 1);
            const double xlo = gen_coord(G, t_lo, g, &sl_lo), xhi = gen_coord(G, t_hi, g, &sl_hi);
            const double cl = fmax(xlo, 0.0), ch = fmin(xhi, x_top);
            if (!(ch > cl)) continue;
            const double inv_w = 1.0 / (xhi - xlo);
            const int jl = (int)cl, ju_ = min((int)ch + 1, P.n_lambda - 1);
            // fp64 throughout: on listed knots x' jumps from one interval to the next, so F_k W_k' / W_k and the edge terms
            // cancel to the derivative only if the bin average itself is accurate far beyond fp32
            double v0 = 0.0, da = 0.0, dz = 0.0, dq = 0.0;
            for (int j = jl; j <= ju_; ++j) {
                const double w = gen_hat_integral(ch - (double)j) - gen_hat_integral(cl - (double)j);
                const uint32_t j32 = (uint32_t)j;
                const double t0 = __ldg(T0 + j32), t1 = __ldg(T1 + j32), t2 = __ldg(T2 + j32), t3 = __ldg(T3 + j32);
                v0 += w * t0;
                da += w * (t1 - t0);
                dz += w * (t2 - t0);
                dq += w * ((t3 - t2) - (t1 - t0));
            }
            const double gw = (double)gk * inv_w;
            P0 += gw * v0; Pa += gw * da; Pz += gw * dz; Pq += gw * dq;
            const double F = (v0 + ta * da + tz * dz + ta * tz * dq) * inv_w;     // blended unit-mass bin average
            const double xlo_p = xprime(xlo, t_lo, sl_lo), xhi_p = xprime(xhi, t_hi, sl_hi);
            double Ip = 0.0;
            if (xhi <= x_top) Ip += blended(xhi) * xhi_p;     // an edge clipped to the coverage does not move
            if (xlo >= 0.0) Ip -= blended(xlo) * xlo_p;
            E += (double)gk * (Ip * inv_w - F * (xhi_p - xlo_p) * inv_w);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        P0 += __shfl_xor_sync(0xffffffffu, P0, o);
        Pa += __shfl_xor_sync(0xffffffffu, Pa, o);
        Pz += __shfl_xor_sync(0xffffffffu, Pz, o);
        Pq += __shfl_xor_sync(0xffffffffu, Pq, o);
        E += __shfl_xor_sync(0xffffffffu, E, o);
    }
    if (lane == 0) {
        const double m = (double)P.mass[p] * (double)P.flux_scale;
        P.g_mass[p] = (float)((double)P.flux_scale * (P0 + ta * Pa + tz * Pz + ta * tz * Pq));
        P.g_age[p] = (float)(m * (Pa + tz * Pq) * (double)ax.inv_wa);
        P.g_z[p] = (float)(m * (Pz + ta * Pq) * (double)ax.inv_wz);
        P.g_v[p] = (float)(m * E / kCkms);                  // d / d v_los = (1 / c) d / d beta
    }
}

cudaError_t launch_adjoint_general(const PassInputs &in, const Layout &L, char *ws, const float *gconv, float *g_mass,
                                   float *g_age, float *g_z, float *g_v, cudaStream_t st)
{
    AdjGenParams P;
    P.perm = (const int32_t *)(ws + L.off_permbuf[L.final_buf]);
    P.seg_off = (const int32_t *)(ws + L.off_seg);
    P.key = (const int32_t *)(ws + L.off_key);
    P.vlos = (const float *)(ws + L.off_vlos);
    P.mass = in.p->mass;
    P.flux = (const float *)(ws + L.off_flux);
    P.gconv = gconv;
    P.rec = (const Rec *)(ws + L.off_rec);
    P.aux = (const AdjAux *)(ws + L.off_aux);
    P.g_mass = g_mass; P.g_age = g_age; P.g_z = g_z; P.g_v = g_v;
    P.n_lambda = in.ssp->n_lambda; P.pitch = L.pitch; P.n_z = in.ssp->n_z; P.n_c = L.n_c; P.n_s = L.n_s;
    P.flux_scale = in.tel->flux_scale;
    P.n = L.n;
    gen_grid_params(in, L, ws, &P.gen);
    const int64_t threads = L.n * 32;
    const unsigned grid = (unsigned)((threads + 255) / 256);
    if (in.tel->resample == RUBIX_RESAMPLE_FLUX) k_adjoint_general<true><<<grid, 256, 0, st>>>(P);
    else k_adjoint_general<false><<<grid, 256, 0, st>>>(P);
    RUBIX_LAUNCH_CHECK();
    return cudaSuccess;
}

}  // namespace rubix

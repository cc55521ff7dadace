/*
 * wcsim_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, fp64 CPU statement of what the Wire-Cell signal-simulation hot
 * path computes on one wire plane:  M(t,x) = (R (*) S)(t,x) + N(t,x)
 * (Section 2.1, Eq. 1), with S built by the Raster and
 * Scatter-add tasks of PAPER.md:54-58 (Section 2.2) and the convolution done
 * either by its plain definition or by the FFT route of PAPER.md:46-52 (Eq. 2).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call this file.  It shares no code,
 * header, table or constant generator with the CUDA path under
 * paper_2203_02479_b200/csrc/ and neither includes the other.
 *
 * Where the paper is silent the readings A1-A20 listed in DESIGN.md
 * ("Readings of the paper") are followed; each function names the ones it uses.
 *
 * Pins (tests/test_oracle_*.py, all run with -m "not gpu"):
 *   axis weights .......... Gauss-Legendre quadrature of the Gaussian pdf, telescoping
 *                           sum, moments, sigma->0 limit, bin-edge symmetry
 *   scatter ............... brute force on tiny grids, charge conservation
 *   convolve_direct ....... delta input reproduces R, linearity, numpy brute force
 *   convolve_fft .......... agrees with convolve_direct and numpy; pad-one-short fails
 *   philox ................ published known-answer vectors (tests/golden/)
 *   norm_ppf .............. published normal quantiles (tests/golden/), scipy ndtri
 *   binomial .............. exact binomial CDF break points, mirror identity, moments
 *   digitize .............. hand-worked codes (ties, clamps), monotone, numpy restatement
 *   drift ................. the widths BASELINE.json configs[1] states for td = 2.25 ms, closed forms
 *   normal_draw ........... its formula restated with scipy's ndtri, moments, the paper's
 *                           0.01 % agreement with the binomial waveforms
 *   noise ................. Parseval closed form, spectrum round trip, direct vs FFT
 *   convolve_impact ....... K = 1 is convolve_direct; a delta at impact position k reproduces R_k;
 *                           linearity; pure-python brute force; sum over the K sub-grids of convolve_direct
 * PARITY UNPINNED (conventions of this build that nothing in the paper fixes;
 * DESIGN.md readings A3, A6, A8, A15): no patch renormalisation; the mu<16
 * inversion / mu>=16 rounded-normal split of the binomial sampler and its use of
 * AS 241; the Philox counter layout; the orthonormal noise scaling; and, of the
 * steps around the hot path, the conventions of readings A21-A25 (clamp and
 * rounding of the normal draw, drift coordinates and units, the ideal ADC, the
 * patch renormalisation, the layout of the impact-position grid and response).
 *
 * Build: gcc -O2 -std=c11 -fopenmp -ffp-contract=off -shared -fPIC
 *        (-ffp-contract=off: every product and sum is rounded separately, so the
 *        arithmetic is exactly what is written here.)
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif

/* ------------------------------------------------------------------------- */
/* Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11).  Used for the binomial    */
/* charge fluctuation the CPU reference of the paper draws (PAPER.md:82,       */
/* Section 3.1) and for the noise phases (BASELINE.json configs[3]).           */
/* ------------------------------------------------------------------------- */
void wco_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        if (round > 0) { k0 += 0x9E3779B9u; k1 += 0xBB67AE85u; }
        uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* uniform in (0,1) from one 32-bit word: u = (w + 1/2) 2^-32, exact in fp64 */
static double u01(uint32_t w) { return ((double)w + 0.5) * (1.0 / 4294967296.0); }

#define WCO_TAG_FLUCT 0x464C5543u /* "FLUC" */
#define WCO_TAG_NOISE 0x4E4F4953u /* "NOIS" */

/* The 32-bit word that decides the draw of absolute grid bin g of depo `id`
 * (reading A8): counter (id lo, id hi, g>>2, tag), key (seed lo, seed hi), word g&3. */
uint32_t wco_fluct_word(uint64_t seed, uint64_t depo_id, uint64_t g)
{
    uint32_t ctr[4] = { (uint32_t)depo_id, (uint32_t)(depo_id >> 32), (uint32_t)(g >> 2), WCO_TAG_FLUCT };
    uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    uint32_t out[4];
    wco_philox4x32_10(ctr, key, out);
    return out[g & 3u];
}

/* The word that fixes the noise phase of frequency bin k on `wire`. */
uint32_t wco_noise_word(uint64_t seed, uint32_t wire, uint32_t k)
{
    uint32_t ctr[4] = { k >> 2, wire, 0u, WCO_TAG_NOISE };
    uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    uint32_t out[4];
    wco_philox4x32_10(ctr, key, out);
    return out[k & 3u];
}

/* ------------------------------------------------------------------------- */
/* Normal quantile: Wichura, Algorithm AS 241 (Appl. Statist. 37, 1988),       */
/* routine PPND16, restated.  Used only by the mu >= 16 branch of the sampler. */
/* ------------------------------------------------------------------------- */
double wco_norm_ppf(double p)
{
    static const double a[8] = { 3.3871328727963666080e0, 1.3314166789178437745e+2, 1.9715909503065514427e+3,
                                 1.3731693765509461125e+4, 4.5921953931549871457e+4, 6.7265770927008700853e+4,
                                 3.3430575583588128105e+4, 2.5090809287301226727e+3 };
    static const double b[8] = { 1.0, 4.2313330701600911252e+1, 6.8718700749205790830e+2, 5.3941960214247511077e+3,
                                 2.1213794301586595867e+4, 3.9307895800092710610e+4, 2.8729085735721942674e+4,
                                 5.2264952788528545610e+3 };
    static const double c[8] = { 1.42343711074968357734e0, 4.63033784615654529590e0, 5.76949722146069140550e0,
                                 3.64784832476320460504e0, 1.27045825245236838258e0, 2.41780725177450611770e-1,
                                 2.27238449892691845833e-2, 7.74545014278341407640e-4 };
    static const double d[8] = { 1.0, 2.05319162663775882187e0, 1.67638483018380384940e0, 6.89767334985100004550e-1,
                                 1.48103976427480074590e-1, 1.51986665636164571966e-2, 5.47593808499534494600e-4,
                                 1.05075007164441684324e-9 };
    static const double e[8] = { 6.65790464350110377720e0, 5.46378491116411436990e0, 1.78482653991729133580e0,
                                 2.96560571828504891230e-1, 2.65321895265761230930e-2, 1.24266094738807843860e-3,
                                 2.71155556874348757815e-5, 2.01033439929228813265e-7 };
    static const double f[8] = { 1.0, 5.99832206555887937690e-1, 1.36929880922735805310e-1, 1.48753612908506148525e-2,
                                 7.86869131145613259100e-4, 1.84631831751005468180e-5, 1.42151175831644588870e-7,
                                 2.04426310338993978564e-15 };
    double q = p - 0.5, r, num, den;
    const double *nu, *de;
    if (fabs(q) <= 0.425) {
        r = 0.180625 - q * q;
        num = a[7]; den = b[7];
        for (int i = 6; i >= 0; --i) { num = num * r + a[i]; den = den * r + b[i]; }
        return q * num / den;
    }
    r = (q < 0.0) ? p : 1.0 - p;
    r = sqrt(-log(r));
    if (r <= 5.0) { r = r - 1.6; nu = c; de = d; }
    else          { r = r - 5.0; nu = e; de = f; }
    num = nu[7]; den = de[7];
    for (int i = 6; i >= 0; --i) { num = num * r + nu[i]; den = den * r + de[i]; }
    double val = num / den;
    return (q < 0.0) ? -val : val;
}

/* ------------------------------------------------------------------------- */
/* Binomial draw B(N, p, w): a pure function of the trial count N (integer-     */
/* valued double), the success probability p and one 32-bit word w.            */
/* PAPER.md:82 (Section 3.1): the CPU reference "uses binomial distribution";  */
/* reading A6 fixes the sampler:                                               */
/*   N = 0 or p <= 0 -> 0;  p >= 1 -> N;  p > 1/2 -> N - B(N, 1-p, ~w);         */
/*   mu = N p < 16: CDF inversion from k = 0;                                  */
/*   else: clamp(rint(mu + sqrt(mu (1-p)) Phi^-1(u)), 0, N), round-half-even.   */
/* ------------------------------------------------------------------------- */
double wco_binomial(double N, double p, uint32_t w)
{
    if (!(N > 0.0) || !(p > 0.0)) return 0.0;
    if (p >= 1.0) return N;
    if (p > 0.5) return N - wco_binomial(N, 1.0 - p, ~w);
    double u = u01(w);
    double mu = N * p;
    if (mu < 16.0) {
        double f = exp(N * log1p(-p));
        double c = f;
        double k = 0.0;
        double r = p / (1.0 - p);
        while (u > c && k < N) {
            k += 1.0;
            f = f * ((r * (N - k + 1.0)) / k);
            c = c + f;
        }
        return k;
    }
    double sd = sqrt(mu * (1.0 - p));
    double x = mu + sd * wco_norm_ppf(u);
    double k = rint(x); /* default rounding mode: half to even */
    if (k < 0.0) k = 0.0;
    if (k > N) k = N;
    return k;
}

/* ------------------------------------------------------------------------- */
/* Raster (Section 2.2: each diffused electron group is binned     */
/* "as a patch").  Readings A1 (bin k covers [k,k+1)), A2 (extent snapped      */
/* outward), A3 (no renormalisation), A4 (sigma -> 0).                         */
/* ------------------------------------------------------------------------- */
/* Sum of the axis weights over the whole extent [i0, i1) of reading A2, from its two outer edges (the sum of
 * differences of erf telescopes; the pin O2 of the tests checks that identity): the norm of reading A24. */
double wco_axis_norm(int64_t i0, int64_t i1, double centre, double sigma)
{
    if (sigma < 1e-6) return 1.0;
    double s = sqrt(2.0) * sigma;
    double hi = erf(((double)i1 - centre) / s);
    double lo = erf(((double)i0 - centre) / s);
    return 0.5 * (hi - lo);
}

void wco_axis_extent(double centre, double sigma, double nsigma, int64_t *i0, int64_t *i1)
{
    *i0 = (int64_t)floor(centre - nsigma * sigma);
    *i1 = (int64_t)floor(centre + nsigma * sigma) + 1;
}

/* probability content of bin i = [i, i+1) of a Gaussian N(centre, sigma^2):
 * 1/2 [erf((i+1-c)/(sqrt2 sigma)) - erf((i-c)/(sqrt2 sigma))] */
double wco_axis_weight(int64_t i, double centre, double sigma)
{
    if (sigma < 1e-6) return ((int64_t)floor(centre) == i) ? 1.0 : 0.0;
    double s = sqrt(2.0) * sigma;
    double hi = erf(((double)(i + 1) - centre) / s);
    double lo = erf(((double)i - centre) / s);
    return 0.5 * (hi - lo);
}

static int depo_ok(double t0, double x0, double st, double sx, double q)
{
    return isfinite(t0) && isfinite(x0) && isfinite(st) && isfinite(sx) && isfinite(q) && st >= 0.0 && sx >= 0.0;
}

/* One depo's patch: extents and per-axis weights (for the pins and for the
 * sampled full-size parity checks).  wt has room for max_t entries, wx for max_x.
 * Returns 0, or -1 if the depo is invalid, -2 if the buffers are too small. */
int wco_patch_axes(float t0, float x0, float sigma_t, float sigma_x, double nsigma,
                   int64_t *it0, int64_t *it1, int64_t *ix0, int64_t *ix1,
                   double *wt, int max_t, double *wx, int max_x)
{
    double T0 = t0, X0 = x0, ST = sigma_t, SX = sigma_x;
    if (!depo_ok(T0, X0, ST, SX, 0.0)) return -1;
    wco_axis_extent(T0, ST, nsigma, it0, it1);
    wco_axis_extent(X0, SX, nsigma, ix0, ix1);
    if (*it1 - *it0 > max_t || *ix1 - *ix0 > max_x) return -2;
    for (int64_t i = *it0; i < *it1; ++i) wt[i - *it0] = wco_axis_weight(i, T0, ST);
    for (int64_t j = *ix0; j < *ix1; ++j) wx[j - *ix0] = wco_axis_weight(j, X0, SX);
    return 0;
}

/* ------------------------------------------------------------------------- */
/* Normal-approximation draw G(N, p, w) -- the sampler of the paper's Kokkos    */
/* port: "the Kokkos version uses normal distribution to approximate the       */
/* binomial distribution", PAPER.md:82 (Section 3.1).  Reading A21:            */
/*   N = 0 or p <= 0 -> 0;  p >= 1 -> N;                                       */
/*   else clamp(rint(N p + sqrt(N p (1-p)) Phi^-1(u)), 0, N) for EVERY mu       */
/*   (no inversion branch, no mirror), u = (w + 1/2) 2^-32, Phi^-1 = AS 241.    */
/* ------------------------------------------------------------------------- */
double wco_normal_draw(double N, double p, uint32_t w)
{
    if (!(N > 0.0) || !(p > 0.0)) return 0.0;
    if (p >= 1.0) return N;
    double u = u01(w);
    double mu = N * p;
    double sd = sqrt(mu * (1.0 - p));
    double x = mu + sd * wco_norm_ppf(u);
    double k = rint(x);
    if (k < 0.0) k = 0.0;
    if (k > N) k = N;
    return k;
}

/* ------------------------------------------------------------------------- */
/* Digitisation (downstream of M).  PAPER.md:40: "M(t,x) is the  */
/* 'measured' value such as what is input to an analog-to-digital converter    */
/* (ADC) channel x at time t".  Reading A23: an ideal ADC of `bits` bits,       */
/*   code = clamp(rint(M gain + baseline), 0, 2^bits - 1),  round half to even, */
/* the product and the sum each rounded to fp32 (M is an fp32 array; this is   */
/* integer work decided in the kernel's precision).  NaN -> 0.                 */
/* ------------------------------------------------------------------------- */
int wco_digitize(const float *M, int64_t n, float gain, float baseline, int bits, int16_t *adc)
{
    if (n < 0 || bits < 1 || bits > 15) return -1;
    const float top = (float)((1 << bits) - 1);
    for (int64_t i = 0; i < n; ++i) {
        float prod = M[i] * gain;
        float v = prod + baseline;
        float c = rintf(v);
        if (!(c > 0.0f)) c = 0.0f; /* also NaN */
        if (c > top) c = top;
        adc[i] = (int16_t)c;
    }
    return 0;
}

/* ------------------------------------------------------------------------- */
/* Drift (upstream of Raster).  PAPER.md:54: "After simulating   */
/* the diffusion process along the drifting, each ionization electron group is */
/* diffused into a 2D distribution along the drifting and wire pitch           */
/* directions."  Reading A22, with BASELINE.json configs[1]'s width formulas:   */
/*   td      = (x - x_plane) / v_drift                     [us]; td < 0 -> NaN  */
/*   t0      = (t + td - t_origin) / tick                   [ticks]             */
/*   x0      = (y cos(theta) + z sin(theta) - pitch_origin) / pitch  [pitches]  */
/*   sigma_t = sqrt(2 D_L td) / v_drift / tick,  sigma_x = sqrt(2 D_T td)/pitch */
/*   Q       = q exp(-td / lifetime)   (lifetime <= 0: no attenuation)          */
/* Units: cm, us, D in cm^2/s (so 2 D td carries a factor 1e-6).  Everything    */
/* in fp64, results rounded once to fp32.  A group behind the plane (td < 0)    */
/* gets NaN in all five fields, which the raster skips and counts.             */
/* ------------------------------------------------------------------------- */
int wco_drift(const float *x, const float *y, const float *z, const float *t, const float *q, int64_t n,
              double v_drift, double D_L, double D_T, double tick, double t_origin, double lifetime,
              double x_plane, double cos_theta, double sin_theta, double pitch_origin, double pitch,
              float *t0, float *x0, float *sigma_t, float *sigma_x, float *Q)
{
    if (n < 0 || !(v_drift > 0.0) || !(tick > 0.0) || !(pitch > 0.0) || D_L < 0.0 || D_T < 0.0) return -1;
    for (int64_t i = 0; i < n; ++i) {
        double td = ((double)x[i] - x_plane) / v_drift;
        if (!(td >= 0.0)) {
            t0[i] = x0[i] = sigma_t[i] = sigma_x[i] = Q[i] = (float)NAN;
            continue;
        }
        t0[i] = (float)((((double)t[i] + td) - t_origin) / tick);
        x0[i] = (float)((((double)y[i] * cos_theta + (double)z[i] * sin_theta) - pitch_origin) / pitch);
        sigma_t[i] = (float)((sqrt((2.0 * D_L * 1e-6) * td) / v_drift) / tick);
        sigma_x[i] = (float)(sqrt((2.0 * D_T * 1e-6) * td) / pitch);
        Q[i] = (float)((lifetime > 0.0) ? (double)q[i] * exp(-td / lifetime) : (double)q[i]);
    }
    return 0;
}

/* ------------------------------------------------------------------------- */
/* Raster + Scatter-add: patches "stacked and summed over a    */
/* larger grid"; dense grid as in PAPER.md:75.  Serial, in depo order.          */
/*                                                                            */
/* Grid: n_wires x n_ticks, S[wire][tick], tick fastest.  Only bins inside the */
/* window [w0,w1) x [k0,k1) are accumulated, into Swin[(w-w0)*(k1-k0)+(k-k0)]  */
/* (pass the whole grid as the window for the full S).  Bins outside the grid  */
/* are dropped and, with fluctuation, not drawn (reading A5).  Because every   */
/* draw is keyed by the absolute bin (A8), a window sees exactly the values    */
/* the full grid would.                                                       */
/*                                                                            */
/* fluctuate = 0: c = Q p.   fluctuate = 1: Ntr = floor(|Q| + 1/2),             */
/* c = sign(Q) B(Ntr, p, word(seed, id, g)), g = wire*n_ticks + tick (A6-A9).   */
/* fluctuate = 2: the same with the normal-approximation draw G (A21).          */
/* normalize != 0 (reading A24): p_ij = (wt_i wx_j) / (W_t W_x)  */
/* with W the sum of the axis weights over the whole +-n sigma extent, so that */
/* a patch inside the grid carries exactly Q (fluctuation off).                */
/* ids == NULL means depo i has id id_base + i.                                */
/* totals (optional, n entries): signed sum of the draws over all in-grid bins */
/* of each depo (forces drawing outside the window too).                       */
/* stats[0] = depos skipped as invalid, stats[1] = bins drawn or deposited.    */
/* ------------------------------------------------------------------------- */
int wco_raster_scatter(int n_wires, int n_ticks,
                       const float *t0, const float *x0, const float *sigma_t, const float *sigma_x, const float *q,
                       int64_t n, const uint64_t *ids, uint64_t id_base, uint64_t seed, int fluctuate, double nsigma,
                       int w0, int w1, int k0, int k1, double *Swin, int32_t *totals, int64_t *stats, int normalize)
{
    if (n_wires <= 0 || n_ticks <= 0 || n < 0 || !(nsigma > 0.0)) return -1;
    if (w0 < 0 || w1 > n_wires || k0 < 0 || k1 > n_ticks || w0 > w1 || k0 > k1) return -1;
    int64_t skipped = 0, drawn = 0;
    const int64_t wk = (int64_t)k1 - k0;
    for (int64_t d = 0; d < n; ++d) {
        double T0 = t0[d], X0 = x0[d], ST = sigma_t[d], SX = sigma_x[d], Q = q[d];
        if (totals) totals[d] = 0;
        if (!depo_ok(T0, X0, ST, SX, Q)) { ++skipped; continue; }
        uint64_t id = ids ? ids[d] : id_base + (uint64_t)d;
        int64_t it0, it1, ix0, ix1;
        wco_axis_extent(T0, ST, nsigma, &it0, &it1);
        wco_axis_extent(X0, SX, nsigma, &ix0, &ix1);
        double Ntr = floor(fabs(Q) + 0.5);
        double sgn = (Q < 0.0) ? -1.0 : 1.0;
        double norm = normalize ? wco_axis_norm(it0, it1, T0, ST) * wco_axis_norm(ix0, ix1, X0, SX) : 1.0;
        int64_t tot = 0;
        for (int64_t j = ix0; j < ix1; ++j) {
            if (j < 0 || j >= n_wires) continue;
            int in_w = (j >= w0 && j < w1);
            if (!in_w && !totals) continue;
            double wxj = wco_axis_weight(j, X0, SX);
            for (int64_t i = it0; i < it1; ++i) {
                if (i < 0 || i >= n_ticks) continue;
                int in_win = in_w && i >= k0 && i < k1;
                if (!in_win && !totals) continue;
                double wti = wco_axis_weight(i, T0, ST);
                double p = wti * wxj;
                if (normalize) p = p / norm;
                double c;
                if (fluctuate) {
                    uint64_t g = (uint64_t)j * (uint64_t)n_ticks + (uint64_t)i;
                    uint32_t word = wco_fluct_word(seed, id, g);
                    double k = (fluctuate == 2) ? wco_normal_draw(Ntr, p, word) : wco_binomial(Ntr, p, word);
                    tot += (int64_t)(sgn * k);
                    c = sgn * k;
                } else {
                    c = Q * p;
                }
                ++drawn;
                if (in_win) Swin[(j - w0) * wk + (i - k0)] += c;
            }
        }
        if (totals) totals[d] = (int32_t)tot;
    }
    if (stats) { stats[0] = skipped; stats[1] = drawn; }
    return 0;
}

/* ------------------------------------------------------------------------- */
/* Convolution, plain definition (Eq. 1, discretised: A10-A12):   */
/*   M[x][t] = sum_{dx=-c..c} sum_{dt=0..n_rt-1} R[dx+c][dt] S[x-dx][t-dt],     */
/* S = 0 outside the grid, c = (n_rw-1)/2.  Output rows are independent, so    */
/* the loop over x may run in parallel; inside a row the order is fixed.       */
/* Zero bins of S are skipped (they add exact zeros).                          */
/* ------------------------------------------------------------------------- */
int wco_convolve_direct(int n_wires, int n_ticks, const double *S, const double *R, int n_rw, int n_rt, double *M)
{
    if (n_wires <= 0 || n_ticks <= 0 || n_rw <= 0 || n_rt <= 0 || (n_rw % 2) == 0) return -1;
    const int c = (n_rw - 1) / 2;
#pragma omp parallel for schedule(dynamic, 4)
    for (int x = 0; x < n_wires; ++x) {
        double *Mx = M + (size_t)x * n_ticks;
        for (int t = 0; t < n_ticks; ++t) Mx[t] = 0.0;
        for (int dx = -c; dx <= c; ++dx) {
            int xs = x - dx;
            if (xs < 0 || xs >= n_wires) continue;
            const double *Sx = S + (size_t)xs * n_ticks;
            const double *Rd = R + (size_t)(dx + c) * n_rt;
            for (int ts = 0; ts < n_ticks; ++ts) {
                double s = Sx[ts];
                if (s == 0.0) continue;
                int lim = n_ticks - ts < n_rt ? n_ticks - ts : n_rt;
                for (int dt = 0; dt < lim; ++dt) Mx[ts + dt] += Rd[dt] * s;
            }
        }
    }
    return 0;
}

/* ------------------------------------------------------------------------- */
/* Sub-wire ("impact position") response binning (reading A25 of DESIGN.md;    */
/* patches are "typically O(20x20) elements", which a raster on    */
/* whole wires does not give -- SURVEY 8(f)-4).  The charge grid is K times     */
/* finer along the wire axis: fine row xf = x*K + k holds the charge that       */
/* arrives at impact position k (0..K-1) of wire x, i.e. at pitch coordinate    */
/* [xf/K, (xf+1)/K).  The response is given per impact position, R[k][dx+c][dt],*/
/* and the measured waveform of wire x sums over the impact positions:          */
/*   M[x][t] = sum_{k=0..K-1} sum_{dx=-c..c} sum_{dt=0..n_rt-1}                 */
/*                 R[k][dx+c][dt] Sf[(x-dx)*K + k][t-dt],   Sf = 0 outside.     */
/* K = 1 is wco_convolve_direct.  Plain loops in the order written; output rows */
/* are independent.                                                            */
/* ------------------------------------------------------------------------- */
int wco_convolve_impact(int n_wires, int n_ticks, int K, const double *Sf, const double *R, int n_rw, int n_rt,
                        double *M)
{
    if (n_wires <= 0 || n_ticks <= 0 || K <= 0 || n_rw <= 0 || n_rt <= 0 || (n_rw % 2) == 0) return -1;
    const int c = (n_rw - 1) / 2;
#pragma omp parallel for schedule(dynamic, 4)
    for (int x = 0; x < n_wires; ++x) {
        double *Mx = M + (size_t)x * n_ticks;
        for (int t = 0; t < n_ticks; ++t) Mx[t] = 0.0;
        for (int k = 0; k < K; ++k) {
            for (int dx = -c; dx <= c; ++dx) {
                int xs = x - dx;
                if (xs < 0 || xs >= n_wires) continue;
                const double *Sx = Sf + ((size_t)xs * K + k) * n_ticks;
                const double *Rd = R + ((size_t)k * n_rw + (size_t)(dx + c)) * n_rt;
                for (int ts = 0; ts < n_ticks; ++ts) {
                    double s = Sx[ts];
                    if (s == 0.0) continue;
                    int lim = n_ticks - ts < n_rt ? n_ticks - ts : n_rt;
                    for (int dt = 0; dt < lim; ++dt) Mx[ts + dt] += Rd[dt] * s;
                }
            }
        }
    }
    return 0;
}

/* M at listed points only, each by the definition (for sampled full-size checks). */
int wco_convolve_points(int n_wires, int n_ticks, const double *S, const double *R, int n_rw, int n_rt,
                        int64_t npts, const int *px, const int *pt, double *out)
{
    if ((n_rw % 2) == 0) return -1;
    const int c = (n_rw - 1) / 2;
    for (int64_t i = 0; i < npts; ++i) {
        int x = px[i], t = pt[i];
        double acc = 0.0;
        for (int dx = -c; dx <= c; ++dx) {
            int xs = x - dx;
            if (xs < 0 || xs >= n_wires) continue;
            for (int dt = 0; dt < n_rt; ++dt) {
                int ts = t - dt;
                if (ts < 0 || ts >= n_ticks) continue;
                acc += R[(size_t)(dx + c) * n_rt + dt] * S[(size_t)xs * n_ticks + ts];
            }
        }
        out[i] = acc;
    }
    return 0;
}

/* ------------------------------------------------------------------------- */
/* Convolution by the FFT route of Eq. 2: own iterative       */
/* radix-2 complex FFT in fp64, rows then columns, on the zero-padded grid     */
/* pad_w x pad_t (powers of two; A13: pad_t >= n_ticks+n_rt-1,                 */
/* pad_w >= n_wires+c).  R is embedded tick-causal and wire-centred with       */
/* wrap-around on the wire axis (A11).  This is the "same algorithm" CPU      */
/* baseline that bench.py times.                                               */
/* ------------------------------------------------------------------------- */
static int is_pow2(int n) { return n > 0 && (n & (n - 1)) == 0; }

/* in-place radix-2 decimation-in-time FFT of n complex numbers with stride;
 * sign = -1 forward, +1 inverse (unnormalised) */
static void fft_radix2(double *re, double *im, int n, ptrdiff_t stride, int sign)
{
    for (int i = 1, j = 0; i < n; ++i) {
        int bit = n >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) {
            double tr = re[i * stride]; re[i * stride] = re[j * stride]; re[j * stride] = tr;
            double ti = im[i * stride]; im[i * stride] = im[j * stride]; im[j * stride] = ti;
        }
    }
    for (int len = 2; len <= n; len <<= 1) {
        int half = len >> 1;
        for (int k = 0; k < half; ++k) {
            double ang = sign * 2.0 * M_PI * (double)k / (double)len;
            double wr = cos(ang), wi = sin(ang);
            for (int s = 0; s < n; s += len) {
                ptrdiff_t a = (ptrdiff_t)(s + k) * stride, b = (ptrdiff_t)(s + k + half) * stride;
                double xr = re[b] * wr - im[b] * wi;
                double xi = re[b] * wi + im[b] * wr;
                re[b] = re[a] - xr; im[b] = im[a] - xi;
                re[a] = re[a] + xr; im[a] = im[a] + xi;
            }
        }
    }
}

static void fft2d(double *re, double *im, int rows, int cols, int sign)
{
#pragma omp parallel for schedule(static)
    for (int r = 0; r < rows; ++r) fft_radix2(re + (size_t)r * cols, im + (size_t)r * cols, cols, 1, sign);
#pragma omp parallel for schedule(static)
    for (int c = 0; c < cols; ++c) fft_radix2(re + c, im + c, rows, cols, sign);
}

int wco_convolve_fft(int n_wires, int n_ticks, const double *S, const double *R, int n_rw, int n_rt,
                     int pad_w, int pad_t, double *M)
{
    if (!is_pow2(pad_w) || !is_pow2(pad_t) || (n_rw % 2) == 0) return -1;
    const int c = (n_rw - 1) / 2;
    if (pad_w < n_wires || pad_t < n_ticks || pad_w < n_rw || pad_t < n_rt) return -1;
    size_t tot = (size_t)pad_w * pad_t;
    double *sr = calloc(tot, sizeof(double)), *si = calloc(tot, sizeof(double));
    double *rr = calloc(tot, sizeof(double)), *ri = calloc(tot, sizeof(double));
    if (!sr || !si || !rr || !ri) { free(sr); free(si); free(rr); free(ri); return -2; }
    for (int x = 0; x < n_wires; ++x)
        memcpy(sr + (size_t)x * pad_t, S + (size_t)x * n_ticks, sizeof(double) * n_ticks);
    for (int dx = -c; dx <= c; ++dx) {
        int row = ((dx % pad_w) + pad_w) % pad_w;
        for (int dt = 0; dt < n_rt; ++dt) rr[(size_t)row * pad_t + dt] += R[(size_t)(dx + c) * n_rt + dt];
    }
    fft2d(sr, si, pad_w, pad_t, -1);
    fft2d(rr, ri, pad_w, pad_t, -1);
    for (size_t i = 0; i < tot; ++i) {
        double a = sr[i] * rr[i] - si[i] * ri[i];
        double b = sr[i] * ri[i] + si[i] * rr[i];
        sr[i] = a; si[i] = b;
    }
    fft2d(sr, si, pad_w, pad_t, +1);
    const double norm = 1.0 / ((double)pad_w * (double)pad_t);
    for (int x = 0; x < n_wires; ++x)
        for (int t = 0; t < n_ticks; ++t) M[(size_t)x * n_ticks + t] = sr[(size_t)x * pad_t + t] * norm;
    free(sr); free(si); free(rr); free(ri);
    return 0;
}

/* ------------------------------------------------------------------------- */
/* Noise N(t,x) ("voltage level output of various electronics and */
/* coherent noise models"; model from BASELINE.json configs[3]; readings       */
/* A15-A17).  On the padded tick length P, per wire, k = 0..P/2:               */
/*   f_k = k/P, f0 = 0.1 * 1/2, A_k = 3 (f_k/f0) exp(-f_k/f0) unless `amp`      */
/*   is given; phi = 2 pi u(seed, wire, k); Z_k = A_k e^{i phi};                */
/*   N[t] = P^-1/2 [Re Z_0 + 2 sum_{k=1}^{P/2-1} Re(Z_k e^{2 pi i k t/P})       */
/*                  + Re(Z_{P/2}) (-1)^t].                                      */
/* ------------------------------------------------------------------------- */
void wco_noise_amp(int P, double *amp)
{
    const double f0 = 0.1 * 0.5;
    for (int k = 0; k <= P / 2; ++k) {
        double f = (double)k / (double)P;
        amp[k] = 3.0 * (f / f0) * exp(-(f / f0));
    }
}

void wco_noise_spectrum(int P, uint64_t seed, uint32_t wire, const double *amp, double *zre, double *zim)
{
    for (int k = 0; k <= P / 2; ++k) {
        double phi = 2.0 * M_PI * u01(wco_noise_word(seed, wire, (uint32_t)k));
        zre[k] = amp[k] * cos(phi);
        zim[k] = amp[k] * sin(phi);
    }
}

/* the definition, one output sample at a time: O(P) per sample */
int wco_noise_points(int P, uint64_t seed, const double *amp_or_null, int64_t npts, const int *pwire, const int *ptick,
                     double *out)
{
    if (!is_pow2(P) || P < 2) return -1;
    double *amp = malloc(sizeof(double) * (P / 2 + 1));
    double *zre = malloc(sizeof(double) * (P / 2 + 1)), *zim = malloc(sizeof(double) * (P / 2 + 1));
    if (!amp || !zre || !zim) { free(amp); free(zre); free(zim); return -2; }
    if (amp_or_null) memcpy(amp, amp_or_null, sizeof(double) * (P / 2 + 1)); else wco_noise_amp(P, amp);
    int last_wire = -1;
    for (int64_t i = 0; i < npts; ++i) {
        if (pwire[i] != last_wire) { wco_noise_spectrum(P, seed, (uint32_t)pwire[i], amp, zre, zim); last_wire = pwire[i]; }
        int t = ptick[i];
        double acc = zre[0];
        for (int k = 1; k < P / 2; ++k) {
            /* reduce k*t mod P in integers so the angle stays accurate */
            int64_t m = ((int64_t)k * (int64_t)t) % (int64_t)P;
            double ang = 2.0 * M_PI * (double)m / (double)P;
            acc += 2.0 * (zre[k] * cos(ang) - zim[k] * sin(ang));
        }
        acc += zre[P / 2] * ((t & 1) ? -1.0 : 1.0);
        out[i] = acc / sqrt((double)P);
    }
    free(amp); free(zre); free(zim);
    return 0;
}

/* the same numbers for whole wires through an inverse complex FFT of the
 * Hermitian-extended spectrum (library-primitive step); M[wire][t] += N, t < n_ticks */
int wco_noise_add(int P, int n_wires, int n_ticks, uint64_t seed, const double *amp_or_null, double *M)
{
    if (!is_pow2(P) || P < 2 || n_ticks > P) return -1;
    double *amp = malloc(sizeof(double) * (P / 2 + 1));
    if (!amp) return -2;
    if (amp_or_null) memcpy(amp, amp_or_null, sizeof(double) * (P / 2 + 1)); else wco_noise_amp(P, amp);
    int err = 0;
#pragma omp parallel
    {
        double *zre = malloc(sizeof(double) * (P / 2 + 1)), *zim = malloc(sizeof(double) * (P / 2 + 1));
        double *re = malloc(sizeof(double) * P), *im = malloc(sizeof(double) * P);
        if (!zre || !zim || !re || !im) {
#pragma omp atomic write
            err = 1;
        } else {
#pragma omp for schedule(static)
            for (int x = 0; x < n_wires; ++x) {
                wco_noise_spectrum(P, seed, (uint32_t)x, amp, zre, zim);
                re[0] = zre[0]; im[0] = 0.0;
                re[P / 2] = zre[P / 2]; im[P / 2] = 0.0;
                for (int k = 1; k < P / 2; ++k) {
                    re[k] = zre[k]; im[k] = zim[k];
                    re[P - k] = zre[k]; im[P - k] = -zim[k];
                }
                fft_radix2(re, im, P, 1, +1);
                double s = 1.0 / sqrt((double)P);
                for (int t = 0; t < n_ticks; ++t) M[(size_t)x * n_ticks + t] += re[t] * s;
            }
        }
        free(zre); free(zim); free(re); free(im);
    }
    free(amp);
    return err ? -2 : 0;
}

/* plain complex FFT exposed for the pins (compared with an O(N^2) DFT) */
int wco_fft(double *re, double *im, int n, int sign)
{
    if (!is_pow2(n)) return -1;
    fft_radix2(re, im, n, 1, sign < 0 ? -1 : +1);
    return 0;
}

/* threads used by the parallel loops over independent rows (timing only; no arithmetic depends on it) */
void wco_set_num_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

int wco_num_threads(void)
{
    int n = 1;
#ifdef _OPENMP
#pragma omp parallel
    {
#pragma omp single
        n = omp_get_num_threads();
    }
#endif
    return n;
}

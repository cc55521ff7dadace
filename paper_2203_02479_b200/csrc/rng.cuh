// rng.cuh -- device-side counter-based random numbers for the charge fluctuation (Section 3.1: the
// CPU reference draws per-bin binomials) and the noise phases (BASELINE.json configs[3]).
//
// Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11) restated for CUDA, the counter layouts of DESIGN.md reading A8,
// the AS 241 (PPND16) normal quantile and the hybrid binomial sampler of reading A6.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace wcsim {

constexpr uint32_t kTagFluct = 0x464C5543u; // "FLUC"
constexpr uint32_t kTagNoise = 0x4E4F4953u; // "NOIS"

__device__ __forceinline__ uint4 philox4x32_10(uint4 c, uint2 k)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c.x), lo0 = 0xD2511F53u * c.x;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c.z), lo1 = 0xCD9E8D57u * c.z;
        c = make_uint4(hi1 ^ c.y ^ k.x, lo1, hi0 ^ c.w ^ k.y, lo0);
        k.x += 0x9E3779B9u;
        k.y += 0xBB67AE85u;
    }
    return c;
}

__device__ __forceinline__ uint32_t pick_word(uint4 v, uint32_t j)
{
    return j == 0 ? v.x : j == 1 ? v.y : j == 2 ? v.z : v.w;
}

// the four words that decide absolute grid bins 4*(g>>2) .. 4*(g>>2)+3 of depo `id` (A8)
__device__ __forceinline__ uint4 fluct_words(uint64_t seed, uint64_t id, uint64_t g4)
{
    return philox4x32_10(make_uint4((uint32_t)id, (uint32_t)(id >> 32), (uint32_t)g4, kTagFluct),
                         make_uint2((uint32_t)seed, (uint32_t)(seed >> 32)));
}

// the four words that fix the noise phases of frequency bins 4*k4 .. 4*k4+3 on `wire`
__device__ __forceinline__ uint4 noise_words(uint64_t seed, uint32_t wire, uint32_t k4)
{
    return philox4x32_10(make_uint4(k4, wire, 0u, kTagNoise), make_uint2((uint32_t)seed, (uint32_t)(seed >> 32)));
}

// ------------------------------------------------------------------------------------------------------------------
// B(N, p; w): N an integer-valued double >= 0, p a probability, w one 32-bit word (A6).
//   N = 0 or p <= 0 -> 0;  p >= 1 -> N;  p > 1/2 -> N - B(N, 1-p; ~w);
//   mu = N p < 16: inversion of the CDF from k = 0;  else clamp(rint(mu + sqrt(mu (1-p)) Phi^-1(u)), 0, N).
// The sampler is split into a classification and three straight-line draw routines so that the raster kernel can
// sort the bins of a warp by routine before drawing (no divergence between the inversion loop, the central and
// the tail branch of AS 241).  The draws are plain fp64 (FMA contraction allowed, Newton reciprocals instead of IEEE
// division, own exp/log1p series): against the oracle's separately rounded operations this moves a CDF break point
// or a rounding boundary by ~1e-15 relative, i.e. it flips a draw with probability ~1e-12, far inside the 1e-6
// budget of BASELINE.json north_star.
// ------------------------------------------------------------------------------------------------------------------
enum DrawClass : int {
    kDrawZero = -2,        // k = 0 without a draw
    kDrawAll = -1,         // p >= 1: k = N
    kDrawInversion0 = 0,   // inversion, mu < 2
    kDrawInversion1 = 1,   // inversion, 2 <= mu < 6
    kDrawInversion2 = 2,   // inversion, 6 <= mu < 16
    kDrawNormalCentral = 3,
    kDrawNormalTail = 4
};
constexpr int kNumDrawQueues = 5;

// 1/k for the inversion recurrence (k is the trip count, the same in every lane that is still in the loop)
constexpr int kInvTable = 64;
static __constant__ double c_inv_k[kInvTable] = {0.0, 1.0 / 1.0, 1.0 / 2.0, 1.0 / 3.0, 1.0 / 4.0, 1.0 / 5.0, 1.0 / 6.0, 1.0 / 7.0, 1.0 / 8.0, 1.0 / 9.0, 1.0 / 10.0, 1.0 / 11.0, 1.0 / 12.0, 1.0 / 13.0, 1.0 / 14.0, 1.0 / 15.0, 1.0 / 16.0, 1.0 / 17.0, 1.0 / 18.0, 1.0 / 19.0, 1.0 / 20.0, 1.0 / 21.0, 1.0 / 22.0, 1.0 / 23.0, 1.0 / 24.0, 1.0 / 25.0, 1.0 / 26.0, 1.0 / 27.0, 1.0 / 28.0, 1.0 / 29.0, 1.0 / 30.0, 1.0 / 31.0, 1.0 / 32.0, 1.0 / 33.0, 1.0 / 34.0, 1.0 / 35.0, 1.0 / 36.0, 1.0 / 37.0, 1.0 / 38.0, 1.0 / 39.0, 1.0 / 40.0, 1.0 / 41.0, 1.0 / 42.0, 1.0 / 43.0, 1.0 / 44.0, 1.0 / 45.0, 1.0 / 46.0, 1.0 / 47.0, 1.0 / 48.0, 1.0 / 49.0, 1.0 / 50.0, 1.0 / 51.0, 1.0 / 52.0, 1.0 / 53.0, 1.0 / 54.0, 1.0 / 55.0, 1.0 / 56.0, 1.0 / 57.0, 1.0 / 58.0, 1.0 / 59.0, 1.0 / 60.0, 1.0 / 61.0, 1.0 / 62.0, 1.0 / 63.0};

// AS 241 PPND16 coefficients: central region a0..a7 / b1..b7 and first tail region c0..c7 / d1..d7 (highest first)
static __constant__ double c_as241_a[8] = {2.5090809287301226727e+3, 3.3430575583588128105e+4, 6.7265770927008700853e+4,
                                           4.5921953931549871457e+4, 1.3731693765509461125e+4, 1.9715909503065514427e+3,
                                           1.3314166789178437745e+2, 3.3871328727963666080e0};
static __constant__ double c_as241_b[8] = {5.2264952788528545610e+3, 2.8729085735721942674e+4, 3.9307895800092710610e+4,
                                           2.1213794301586595867e+4, 5.3941960214247511077e+3, 6.8718700749205790830e+2,
                                           4.2313330701600911252e+1, 1.0};
static __constant__ double c_as241_c[8] = {7.74545014278341407640e-4, 2.27238449892691845833e-2, 2.41780725177450611770e-1,
                                           1.27045825245236838258e0,  3.64784832476320460504e0,  5.76949722146069140550e0,
                                           4.63033784615654529590e0,  1.42343711074968357734e0};
static __constant__ double c_as241_d[8] = {1.05075007164441684324e-9, 5.47593808499534494600e-4, 1.51986665636164571966e-2,
                                           1.48103976427480074590e-1, 6.89767334985100004550e-1, 1.67638483018380384940e0,
                                           2.05319162663775882187e0,  1.0};

__device__ __forceinline__ double word_to_u01(uint32_t w)
{
    return __dmul_rn(__dadd_rn((double)w, 0.5), 1.0 / 4294967296.0); // exact
}

// |u - 1/2| <= 0.425 (the double nearest 0.425) for u = (w + 1/2) 2^-32, decided on the integer word:
// 0.075 2^32 = 322122547.2 and 0.925 2^32 = 3972844748.8, so the central region is 322122547 <= w <= 3972844748.
__device__ __forceinline__ bool word_is_central(uint32_t w) { return w - 322122547u <= 3972844748u - 322122547u; }

// Folds the p > 1/2 mirror into (p, w) and says which routine draws k.  On return p <= 1/2.
// Shortcut: (1-p)^N >= 1 - N p (Bernoulli), so u <= 1 - mu already implies u <= F(0), i.e. k = 0, without exp/log.
// normal_only: the normal-approximation sampler of the paper's Kokkos port (reading A21): the rounded normal
// for every mu, no inversion branch and no mirror -- only the two AS 241 routines are ever queued.
__device__ __forceinline__ int classify_draw(double N, double &p, uint32_t &w, bool &mirror, bool normal_only = false)
{
    mirror = false;
    if (!(N > 0.0) || !(p > 0.0)) return kDrawZero;
    if (p >= 1.0) return kDrawAll;
    if (normal_only) return word_is_central(w) ? kDrawNormalCentral : kDrawNormalTail;
    mirror = p > 0.5;
    if (mirror) {
        p = __dsub_rn(1.0, p);
        w = ~w;
    }
    const double mu = __dmul_rn(N, p);
    if (mu < 16.0) {
        if (mu < 1.0 && word_to_u01(w) <= 1.0 - mu) return mirror ? kDrawAll : kDrawZero;
        return mu < 2.0 ? kDrawInversion0 : mu < 6.0 ? kDrawInversion1 : kDrawInversion2;
    }
    return word_is_central(w) ? kDrawNormalCentral : kDrawNormalTail;
}

// ---- fp64 helpers of the draw routines.  They replace the CUDA math library's division, log1p and exp by straight-line
// code whose constants sit in constant memory (DFMA reads them as c[][] operands; literals cost two UMOVs each).  All are
// accurate to ~1e-15 relative, which moves a CDF break point or a rounding boundary by that much: see the note above.
__device__ __forceinline__ double fast_rcp(double b) // b normal, |b| in [1e-290, 1e290]
{
    double x;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(x) : "d"(b)); // ~20 bits
    double e = fma(-b, x, 1.0);
    x = fma(x, e, x);
    e = fma(-b, x, 1.0);
    return fma(x, e, x);
}
__device__ __forceinline__ double fast_div(double a, double b)
{
    const double x = fast_rcp(b);
    const double q = a * x;
    return fma(fma(-b, q, a), x, q);
}

// g(p) = sum_{j=0}^{10} p^j / (j+1):  log1p(-p) = -p g(p) for p < 2^-5 (truncation p^11/12 < 2^-58 relative)
static __constant__ double c_log1m[11] = {1.0 / 11.0, 1.0 / 10.0, 1.0 / 9.0, 1.0 / 8.0, 1.0 / 7.0, 1.0 / 6.0,
                                          1.0 / 5.0,  1.0 / 4.0,  1.0 / 3.0, 1.0 / 2.0, 1.0};
// 1/j!, j = 13 .. 0: exp(r) on |r| <= ln2/2 (truncation r^14/14! < 5e-18)
static __constant__ double c_exp[14] = {1.0 / 6227020800.0, 1.0 / 479001600.0, 1.0 / 39916800.0, 1.0 / 3628800.0,
                                        1.0 / 362880.0,     1.0 / 40320.0,     1.0 / 5040.0,     1.0 / 720.0,
                                        1.0 / 120.0,        1.0 / 24.0,        1.0 / 6.0,        0.5,
                                        1.0,                1.0};
static __constant__ double c_exp_red[4] = {1.4426950408889634074, 6.93147180369123816490e-01, 1.90821492927058770002e-10,
                                           6755399441055744.0}; // log2 e, ln2 hi, ln2 lo, 1.5 2^52

// exp(y) for -700 < y <= 0
__device__ __forceinline__ double exp_neg(double y)
{
    const double sh = fma(y, c_exp_red[0], c_exp_red[3]); // low word of sh = rint(y log2 e) (two's complement)
    const double kd = sh - c_exp_red[3];
    double r = fma(kd, -c_exp_red[1], y);
    r = fma(kd, -c_exp_red[2], r);
    double e = c_exp[0];
#pragma unroll
    for (int j = 1; j < 14; ++j) e = fma(e, r, c_exp[j]);
    const int k = __double2loint(sh);
    return __hiloint2double(__double2hiint(e) + (k << 20), __double2loint(e)); // e in [0.7, 1.42), k >= -1010
}

// log(1 - p) for 2^-5 <= p <= 1/2: rare (N < 512 for mu < 16), kept out of line so that the library routine is
// instantiated once per kernel
static __device__ __noinline__ double log1m_large(double p) { return log1p(-p); }

// (1 - p)^N for 0 < p <= 1/2
__device__ __forceinline__ double pow_one_minus(double N, double p)
{
    double L;
    if (p < 0.03125) {
        double g = c_log1m[0];
#pragma unroll
        for (int j = 1; j < 11; ++j) g = fma(g, p, c_log1m[j]);
        L = -p * g;
    } else {
        L = log1m_large(p);
    }
    return exp_neg(N * L);
}

__device__ __forceinline__ double draw_inversion(double N, double p, uint32_t w)
{
    const double u = word_to_u01(w);
    double f = pow_one_minus(N, p);
    double c = f;
    // f_k = f_{k-1} r (N - k + 1) / k with r = p / (1 - p), written as f_{k-1} (r (N+1) / k - r).  The trip count is kept
    // uniform over the warp (lanes that are done stop updating), so 1/k is a uniform constant-bank operand.
    const double r = fast_div(p, 1.0 - p), rN1 = r * (N + 1.0);
    double kd = 0.0;
    bool go = u > c && kd < N;
    auto step = [&](int k) {
        const double rk = k < kInvTable ? c_inv_k[k] : 1.0 / (double)k;
        if (go) {
            kd += 1.0;
            f *= fma(rN1, rk, -r);
            c += f;
            go = u > c && kd < N;
        }
    };
    for (int k = 1; __any_sync(__activemask(), go); k += 2) { // two terms per vote (four: slower, 73.4 -> 75.7 us)
        step(k);
        step(k + 1);
    }
    return kd;
}

__device__ __forceinline__ double finish_normal(double N, double p, double z)
{
    const double mu = N * p;
    const double sd = sqrt(mu * (1.0 - p));
    double k = rint(fma(sd, z, mu));
    k = k < 0.0 ? 0.0 : k;
    return k > N ? N : k;
}

// AS 241 PPND16, |u - 1/2| <= 0.425: the quantile z
__device__ __forceinline__ double as241_central(uint32_t w)
{
    const double q = word_to_u01(w) - 0.5;
    const double r = 0.180625 - q * q;
    double num = c_as241_a[0], den = c_as241_b[0];
#pragma unroll
    for (int j = 1; j < 8; ++j) {
        num = fma(num, r, c_as241_a[j]);
        den = fma(den, r, c_as241_b[j]);
    }
    return fast_div(q * num, den);
}
__device__ __forceinline__ double draw_normal_central(double N, double p, uint32_t w)
{
    return finish_normal(N, p, as241_central(w));
}

// AS 241 PPND16, |u - 1/2| > 0.425.  r = sqrt(-log(min(u, 1-u))) <= sqrt(33 log 2) = 4.79 for a 32-bit word, so the
// routine's third region (r > 5) cannot be reached from a 32-bit word and is not coded.
__device__ __forceinline__ double as241_tail(uint32_t w)
{
    const double u = word_to_u01(w);
    const double q = u - 0.5;
    const double r = sqrt(-log(q < 0.0 ? u : 1.0 - u)) - 1.6;
    double num = c_as241_c[0], den = c_as241_d[0];
#pragma unroll
    for (int j = 1; j < 8; ++j) {
        num = fma(num, r, c_as241_c[j]);
        den = fma(den, r, c_as241_d[j]);
    }
    const double val = fast_div(num, den);
    return q < 0.0 ? -val : val;
}
__device__ __forceinline__ double draw_normal_tail(double N, double p, uint32_t w)
{
    return finish_normal(N, p, as241_tail(w));
}

// the draw of an already classified bin (cls >= 0), mirror undone
__device__ __forceinline__ double draw_classified(int cls, double N, double p, uint32_t w, bool mirror)
{
    const double k = cls <= kDrawInversion2       ? draw_inversion(N, p, w)
                     : cls == kDrawNormalCentral ? draw_normal_central(N, p, w)
                                                 : draw_normal_tail(N, p, w);
    return mirror ? N - k : k;
}

// ------------------------------------------------------------------------------------------------------------------
// Guarded fp32 fast path of the rounded-normal branch (mu >= 16, or every mu with the normal-approximation sampler).
// k = clamp(rint(mu + sd z), 0, N) is an integer decision: if an fp32 estimate x32 of x = mu + sd z is farther from the
// nearest half-integer than a bound E on |x32 - x|, then rint(x32) = rint(x) and the fp64 evaluation is not needed.
// Bins that fail the test are drawn again by the fp64 routines above (the raster queues them), so the result is the
// exact sampler's for every bin; only the cost differs.
//
// z32: Phi^-1(u) = x g(wl), x = 2u - 1, wl = -ln(1 - x^2) = -ln(4 t (1 - t)), t = min(u, 1 - u) taken from the integer
// word so that the tails keep their relative accuracy; g is a degree-8 polynomial in (wl - 2.5) on wl < 5
// (csrc/z32_fit.py; |u - 1/2| < 0.4983, 99.66 % of the words; the rest are not accepted).  Its error against the fp64
// AS 241 routine is MEASURED over all 2^32 words by wcsim_debug_z32_scan (tests/test_gpu_fastpath.py): kZ32Err below is
// asserted there to be at least twice the measured maximum of |z32 - z64|.
// ------------------------------------------------------------------------------------------------------------------
static __constant__ float c_z32[9] = {4.035463519e-08f, 4.861039429e-07f, -4.990565230e-06f, -6.217992905e-06f,
                                      3.091502003e-04f, -1.773010124e-03f, -5.908171181e-03f, 3.488026559e-01f,
                                      2.123313665e+00f}; // highest power first
constexpr float kZ32Err = 4.0e-6f; // bound on |z32(w) - z_AS241(w)| for the accepted words (|z| < 2.93)

__device__ __forceinline__ bool z32_from_word(uint32_t w, float &z)
{
    const float x = fmaf((float)(int)(w ^ 0x80000000u), 4.656612873077393e-10f, 2.3283064365386963e-10f); // 2u - 1
    const uint32_t m = min(w, ~w);
    const float t = fmaf((float)m, 2.3283064365386963e-10f, 1.1641532182693481e-10f); // min(u, 1-u)
    const float wl = -0.6931471805599453f * __log2f(4.0f * t * (1.0f - t));
    const float d = wl - 2.5f;
    float g = c_z32[0];
#pragma unroll
    for (int j = 1; j < 9; ++j) g = fmaf(g, d, c_z32[j]);
    z = x * g;
    return wl < 5.0f;
}

// Error budget of x32 = fmaf(sd32, z32, mu32) against x = fma(sd, z, mu) of finish_normal, for 0 < p <= 1/2 (u = 2^-24):
//   mu32 = fp32(mu):                      |d mu| <= u mu
//   q32 = fp32(1 - fp32(p)):              relative 2u (1 - p >= 1/2)
//   v32 = fp32(mu32 q32):                 relative 4u;   sd32 = sqrt.approx(v32): relative 2u + 2^-22 = 6u
//   z32:                                  |d z| <= kZ32Err, |z| < 2.93
//   fmaf rounding:                        u (mu + 2.93 sd)
//   => |x32 - x| <= 2u mu + (7u 2.93 + kZ32Err) sd + second order  <  1.2e-7 mu + 5.3e-6 sd.
// The guard uses 2.5e-7 mu + 8e-6 sd + 1e-6 (the constant also covers x64's own rounding and the bound's evaluation).
constexpr float kGuardMu = 2.5e-7f, kGuardSd = 8.0e-6f, kGuardAbs = 1.0e-6f;

// true: k is the exact sampler's rounded-normal draw for (N, p; w), p <= 1/2, mu = N p (fp64).  false: not decided.
__device__ __forceinline__ bool fast_normal_draw(float N, double p, double mu, uint32_t w, float &k)
{
    float z;
    bool ok = z32_from_word(w, z);
    const float muf = (float)mu, pf = (float)p;
    float sd;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(sd) : "f"(muf * (1.0f - pf))); // MUFU.SQRT: relative error <= 2^-22
    const float x = fmaf(sd, z, muf);
    const float kf = rintf(x);
    const float E = fmaf(kGuardMu, muf, fmaf(kGuardSd, sd, kGuardAbs));
    ok = ok && (fabsf(x - kf) < 0.5f - E); // false for NaN, and for every x once E >= 1/2 (mu > 2e6)
    k = fminf(fmaxf(kf, 0.0f), N);
    return ok;
}

// ------------------------------------------------------------------------------------------------------------------
// Guarded fp32 inversion (mu < 16).  k is the number of CDF values F(0), F(1), ... below u.  The fp32 routine sums a FIXED
// number T of terms of the same recurrence (straight-line code, every lane busy; the raster queues bins by mu so that
// T = 8, 16 or 32 is enough: P(k >= T) < 1.2e-3 at the top of each band) and counts the F(j) below u.  The count is the
// fp64 routine's whenever u is farther from every F(j), j < T, than a bound on their fp32 error, and u <= F(T-1).
// Taken for N >= 128 and p < 2^-5 (every bin of BASELINE.json's workloads with mu < 16); bins that fail the guard are drawn
// again by draw_inversion in fp64.
// Error budget (u = 2^-24; quantities marked ' are the fp32 ones):
//   p' = fp32(p): relative u.   s' = p' (1 + p'/2 + ... + p'^5/6) = -log(1 - p): truncation p^6/7 < 2^-32, Horner
//   roundings 4u, the rounding of p another 1.04u;  L' = N s': relative 6.1u, L < 16.3, so |dL| < 5.9e-6;
//   f0' = ex2(-L' log2 e): the product adds 1.5e-6, ex2.approx is accurate to 2^-22 relative  =>  f0 relative 7.7e-6.
//   r' = p' rcp(1 - p'): relative 5u;  a' = r' (N + 1): relative 6u.
//   term j: f_j = f_{j-1} (a'/j - r'), one fma with the constant fp32(1/j): relative to the true factor r (N+1-j)/j the
//   error is u + 7u (N+1)/(N+1-j) + 5u j/(N+1-j) <= 14.3u for N >= 128, j < 32; with the product and the running sum
//   c_j = c_{j-1} + f_j: at most 17u = 1.0e-6 per term.
//   u' = fma(fp32(w), 2^-32, 2^-33): |u' - u| <= 2u = 1.2e-7.
//   =>  |c_j' - c_j| <= (7.7e-6 + 1.0e-6 j) c_j, c_j <= 1.  Guard G(T) = 8.2e-6 + 1.3e-6 T (absolute, for every j < T).
// ------------------------------------------------------------------------------------------------------------------
constexpr float kInvFastMinN = 128.0f, kInvFastMaxP = 0.03125f;
constexpr float kInvGuard0 = 8.2e-6f, kInvGuardK = 1.3e-6f;

__device__ __forceinline__ bool inv_fast_eligible(float N, double p) { return N >= kInvFastMinN && p < (double)kInvFastMaxP; }

// true: k is the fp64 inversion's draw for (N, p; w); false: not decided
template <int T>
__device__ __forceinline__ bool inv_fast_draw(float N, double p, uint32_t w, float &k)
{
    const float pf = (float)p;
    float g = 1.0f / 6.0f;
    g = fmaf(g, pf, 0.2f);
    g = fmaf(g, pf, 0.25f);
    g = fmaf(g, pf, 1.0f / 3.0f);
    g = fmaf(g, pf, 0.5f);
    g = fmaf(g, pf, 1.0f);
    const float L = N * (pf * g); // -N log(1 - p)
    float f, rc;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(f) : "f"(L * -1.4426950408889634f));
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(rc) : "f"(1.0f - pf));
    const float r = pf * rc, a = r * (N + 1.0f);
    const float u = fmaf((float)w, 2.3283064365386963e-10f, 1.1641532182693481e-10f);
    float c = f, dmin = fabsf(u - c);
    k = u > c ? 1.0f : 0.0f;
#pragma unroll
    for (int j = 1; j < T; ++j) {
        f *= fmaf(a, 1.0f / (float)j, -r);
        c += f;
        dmin = fminf(dmin, fabsf(u - c));
        k += u > c ? 1.0f : 0.0f;
    }
    return dmin >= kInvGuard0 + kInvGuardK * (float)T && !(u > c);
}

// the whole sampler for one bin (debug hook, big-patch and tiled paths)
__device__ __forceinline__ double binomial_draw(double N, double p, uint32_t w, bool normal_only = false)
{
    bool mirror;
    const int cls = classify_draw(N, p, w, mirror, normal_only);
    if (cls == kDrawZero) return 0.0;
    if (cls == kDrawAll) return N;
    return draw_classified(cls, N, p, w, mirror);
}

} // namespace wcsim

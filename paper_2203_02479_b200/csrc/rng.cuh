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
// the tail branch of AS 241).  The draws are plain fp64 (FMA contraction allowed, reciprocal instead of division
// in the inversion recurrence): against the oracle's separately rounded operations this moves a CDF break point
// or a rounding boundary by ~1e-16 relative, i.e. it flips a draw with probability ~1e-13, far inside the 1e-6
// budget of BASELINE.json north_star.
// ------------------------------------------------------------------------------------------------------------------
enum DrawClass : int { kDrawZero = -2, kDrawAll = -1, kDrawInversion = 0, kDrawNormalCentral = 1, kDrawNormalTail = 2 };
constexpr int kNumDrawQueues = 3;

__device__ __forceinline__ double word_to_u01(uint32_t w)
{
    return __dmul_rn(__dadd_rn((double)w, 0.5), 1.0 / 4294967296.0); // exact
}

// Folds the p > 1/2 mirror into (p, w) and says which routine draws k.  On return p <= 1/2.
__device__ __forceinline__ int classify_draw(double N, double &p, uint32_t &w, bool &mirror)
{
    mirror = false;
    if (!(N > 0.0) || !(p > 0.0)) return kDrawZero;
    if (p >= 1.0) return kDrawAll;
    mirror = p > 0.5;
    if (mirror) {
        p = __dsub_rn(1.0, p);
        w = ~w;
    }
    if (__dmul_rn(N, p) < 16.0) return kDrawInversion;
    return fabs(__dsub_rn(word_to_u01(w), 0.5)) <= 0.425 ? kDrawNormalCentral : kDrawNormalTail;
}

__device__ __forceinline__ double draw_inversion(double N, double p, uint32_t w)
{
    const double u = word_to_u01(w);
    double f = exp(N * log1p(-p));
    double c = f, k = 0.0;
    const double r = p / (1.0 - p);
    while (u > c && k < N) {
        k += 1.0;
        f *= (r * (N - k + 1.0)) * __drcp_rn(k);
        c += f;
    }
    return k;
}

__device__ __forceinline__ double finish_normal(double N, double p, double z)
{
    const double mu = N * p;
    const double sd = sqrt(mu * (1.0 - p));
    double k = rint(fma(sd, z, mu));
    k = k < 0.0 ? 0.0 : k;
    return k > N ? N : k;
}

// AS 241 PPND16, |u - 1/2| <= 0.425
__device__ __forceinline__ double draw_normal_central(double N, double p, uint32_t w)
{
    const double q = word_to_u01(w) - 0.5;
    const double r = 0.180625 - q * q;
    double num = 2.5090809287301226727e+3, den = 5.2264952788528545610e+3;
    num = fma(num, r, 3.3430575583588128105e+4); den = fma(den, r, 2.8729085735721942674e+4);
    num = fma(num, r, 6.7265770927008700853e+4); den = fma(den, r, 3.9307895800092710610e+4);
    num = fma(num, r, 4.5921953931549871457e+4); den = fma(den, r, 2.1213794301586595867e+4);
    num = fma(num, r, 1.3731693765509461125e+4); den = fma(den, r, 5.3941960214247511077e+3);
    num = fma(num, r, 1.9715909503065514427e+3); den = fma(den, r, 6.8718700749205790830e+2);
    num = fma(num, r, 1.3314166789178437745e+2); den = fma(den, r, 4.2313330701600911252e+1);
    num = fma(num, r, 3.3871328727963666080e0);  den = fma(den, r, 1.0);
    return finish_normal(N, p, q * num / den);
}

// AS 241 PPND16, |u - 1/2| > 0.425.  r = sqrt(-log(min(u, 1-u))) <= sqrt(33 log 2) = 4.79 for a 32-bit word, so the
// r > 5 branch of the routine is unreachable here; it is kept (one predicated select) for the debug hook's sake.
__device__ __forceinline__ double draw_normal_tail(double N, double p, uint32_t w)
{
    const double u = word_to_u01(w);
    const double q = u - 0.5;
    double r = sqrt(-log(q < 0.0 ? u : 1.0 - u));
    double num, den;
    if (r <= 5.0) {
        r -= 1.6;
        num = 7.74545014278341407640e-4; den = 1.05075007164441684324e-9;
        num = fma(num, r, 2.27238449892691845833e-2); den = fma(den, r, 5.47593808499534494600e-4);
        num = fma(num, r, 2.41780725177450611770e-1); den = fma(den, r, 1.51986665636164571966e-2);
        num = fma(num, r, 1.27045825245236838258e0);  den = fma(den, r, 1.48103976427480074590e-1);
        num = fma(num, r, 3.64784832476320460504e0);  den = fma(den, r, 6.89767334985100004550e-1);
        num = fma(num, r, 5.76949722146069140550e0);  den = fma(den, r, 1.67638483018380384940e0);
        num = fma(num, r, 4.63033784615654529590e0);  den = fma(den, r, 2.05319162663775882187e0);
        num = fma(num, r, 1.42343711074968357734e0);  den = fma(den, r, 1.0);
    } else {
        r -= 5.0;
        num = 2.01033439929228813265e-7; den = 2.04426310338993978564e-15;
        num = fma(num, r, 2.71155556874348757815e-5); den = fma(den, r, 1.42151175831644588870e-7);
        num = fma(num, r, 1.24266094738807843860e-3); den = fma(den, r, 1.84631831751005468180e-5);
        num = fma(num, r, 2.65321895265761230930e-2); den = fma(den, r, 7.86869131145613259100e-4);
        num = fma(num, r, 2.96560571828504891230e-1); den = fma(den, r, 1.48753612908506148525e-2);
        num = fma(num, r, 1.78482653991729133580e0);  den = fma(den, r, 1.36929880922735805310e-1);
        num = fma(num, r, 5.46378491116411436990e0);  den = fma(den, r, 5.99832206555887937690e-1);
        num = fma(num, r, 6.65790464350110377720e0);  den = fma(den, r, 1.0);
    }
    const double val = num / den;
    return finish_normal(N, p, q < 0.0 ? -val : val);
}

// the draw of an already classified bin (cls >= 0), mirror undone
__device__ __forceinline__ double draw_classified(int cls, double N, double p, uint32_t w, bool mirror)
{
    const double k = cls == kDrawInversion       ? draw_inversion(N, p, w)
                     : cls == kDrawNormalCentral ? draw_normal_central(N, p, w)
                                                 : draw_normal_tail(N, p, w);
    return mirror ? N - k : k;
}

// the whole sampler for one bin (debug hook, big-patch and tiled paths)
__device__ __forceinline__ double binomial_draw(double N, double p, uint32_t w)
{
    bool mirror;
    const int cls = classify_draw(N, p, w, mirror);
    if (cls == kDrawZero) return 0.0;
    if (cls == kDrawAll) return N;
    return draw_classified(cls, N, p, w, mirror);
}

} // namespace wcsim

// erf_table.cuh -- fp64 erf for the bin-edge weights of the fluctuated raster (reading A2: weights are
// 1/2 [erf((i+1-c)/(sqrt2 s)) - erf((i-c)/(sqrt2 s))], "bins each ... distribution into a patch").
//
// The CUDA math library's erf costs ~125 instructions per call (two branches, an exp, literals materialised by UMOV
// pairs) and is 9-12 % of the raster kernel.  Here |z| < 6 is cut into 48 intervals of width 1/8 and erf is the
// degree-12 Taylor polynomial about the interval's centre: |t| <= 1/16, remainder (sqrt2/16)^13 / sqrt(13!) ~ 2e-19.
// Coefficients come from erf's own ODE, f'' = -2 x f':
//     a_0 = erf(c),  a_1 = 2/sqrt(pi) exp(-c^2),  a_{n+1} = -2 c a_n / (n+1) - 2 (n-1) a_{n-1} / (n (n+1)),
// evaluated once per process in long double on the host and rounded to double.  For |z| >= 6, erf = +-1 to 2e-17.
// Layout [coefficient][interval] so that one load instruction of a warp touches at most 384 contiguous bytes.
#pragma once
#include <cuda_runtime.h>
#include <math.h>

namespace wcsim {

constexpr int kErfIntervals = 48, kErfDegree = 12;
constexpr double kErfWidth = 0.125;

// host: fills tab[(kErfDegree + 1) * kErfIntervals]
inline void build_erf_table(double *tab)
{
    for (int i = 0; i < kErfIntervals; ++i) {
        const long double c = ((long double)i + 0.5L) * (long double)kErfWidth;
        long double a[kErfDegree + 1];
        a[0] = erfl(c);
        a[1] = 1.128379167095512573896158903121545172L * expl(-c * c);
        for (int n = 1; n < kErfDegree; ++n)
            a[n + 1] = -2.0L * c * a[n] / (long double)(n + 1) - 2.0L * (long double)(n - 1) * a[n - 1] / ((long double)n * (long double)(n + 1));
        for (int n = 0; n <= kErfDegree; ++n) tab[n * kErfIntervals + i] = (double)a[n];
    }
}

// erf(z) from the table (host and device: the host copy backs wcsim_debug_erf and its CPU test)
__host__ __device__ __forceinline__ double erf_from_table(const double *__restrict__ tab, double z)
{
    double a = fabs(z);
    a = a < 5.99999 ? a : 5.99999; // erf(5.99999) rounds to 1
    const int i = (int)(a * (1.0 / kErfWidth));
    const double t = a - ((double)i * kErfWidth + 0.5 * kErfWidth);
    const double *c = tab + i;
    double r = c[kErfDegree * kErfIntervals];
#pragma unroll
    for (int n = kErfDegree - 1; n >= 0; --n) r = fma(r, t, c[n * kErfIntervals]);
    return z < 0.0 ? -r : r;
}

} // namespace wcsim

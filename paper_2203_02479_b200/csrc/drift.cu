// drift.cu -- the step upstream of the Raster ("After simulating the diffusion process along the drifting,
// each ionization electron group is diffused into a 2D distribution along the drifting and wire pitch directions";
// SURVEY 8(f)-2, reading A22).  One pass over the electron groups writes the depo arrays of ALL planes, so the groups
// are read once per event instead of once per plane:
//     td = (x - x_plane)/v,  t0 = (t + td - t_origin)/tick,  x0 = (y cos(theta) + z sin(theta) - origin)/pitch,
//     sigma_t = sqrt(2 D_L td)/v/tick,  sigma_x = sqrt(2 D_T td)/pitch,  Q = q exp(-td/lifetime)
// in fp64, rounded once to fp32 (units: cm, us, D in cm^2/s).  A group behind a plane gets NaN fields there, which the
// raster skips and counts.  HBM bound: 20 B in, 20 B out per group and plane.
#include "internal.h"
#include "pdl.cuh"

namespace wcsim {

namespace {

__global__ void __launch_bounds__(256) drift_kernel(DriftInputs in, long long n, DriftParams prm, DriftPlanes planes)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double x = in.x[i], y = in.y[i], z = in.z[i], t = in.t[i], q = in.q[i];
    const float nan = __int_as_float(0x7fc00000);
#pragma unroll 1
    for (int p = 0; p < planes.n; ++p) {
        const DriftPlane pl = planes.plane[p];
        const double td = __ddiv_rn(__dsub_rn(x, pl.x_plane), prm.v_drift);
        float t0 = nan, x0 = nan, st = nan, sx = nan, Q = nan;
        if (td >= 0.0) {
            t0 = (float)__ddiv_rn(__dsub_rn(__dadd_rn(t, td), prm.t_origin), prm.tick);
            const double u = __dadd_rn(__dmul_rn(y, pl.cos_theta), __dmul_rn(z, pl.sin_theta));
            x0 = (float)__ddiv_rn(__dsub_rn(u, pl.pitch_origin), pl.pitch);
            st = (float)__ddiv_rn(__ddiv_rn(__dsqrt_rn(__dmul_rn(prm.two_DL, td)), prm.v_drift), prm.tick);
            sx = (float)__ddiv_rn(__dsqrt_rn(__dmul_rn(prm.two_DT, td)), pl.pitch);
            Q = (float)(prm.lifetime > 0.0 ? __dmul_rn(q, exp(-td / prm.lifetime)) : q);
        }
        pl.out.t0[i] = t0, pl.out.x0[i] = x0, pl.out.sigma_t[i] = st, pl.out.sigma_x[i] = sx, pl.out.q[i] = Q;
    }
}

// Digitisation downstream of M (M is "what is input to an analog-to-digital converter (ADC) channel x at
// time t"; reading A23): code = clamp(rint(M gain + baseline), 0, 2^bits - 1), product and sum each
// rounded to fp32, NaN -> 0.  HBM bound: 4 B in, 2 B out per sample; four samples per thread (16-byte loads).
__device__ __forceinline__ short adc_code(float m, float gain, float baseline, float top)
{
    float c = rintf(__fadd_rn(__fmul_rn(m, gain), baseline));
    c = (c > 0.0f) ? c : 0.0f; // also NaN
    c = (c > top) ? top : c;
    return (short)c;
}

__global__ void __launch_bounds__(256) digitize_kernel(const float *__restrict__ M, long long n, float gain, float baseline,
                                                       float top, short *__restrict__ adc)
{
    const long long i4 = ((long long)blockIdx.x * blockDim.x + threadIdx.x) * 4;
    if (i4 + 3 < n) {
        const float4 m = *reinterpret_cast<const float4 *>(M + i4);
        short4 o;
        o.x = adc_code(m.x, gain, baseline, top), o.y = adc_code(m.y, gain, baseline, top);
        o.z = adc_code(m.z, gain, baseline, top), o.w = adc_code(m.w, gain, baseline, top);
        *reinterpret_cast<short4 *>(adc + i4) = o;
    } else {
        for (long long i = i4; i < n; ++i) adc[i] = adc_code(M[i], gain, baseline, top);
    }
}

// S = 0 as a kernel (not a memset node), so that the raster that follows is its programmatic dependent: the raster's CTAs
// are resident and through their prologue when the last stores of the clear land.  Persistent: a few CTAs per SM stride
// over the grid with 16-byte stores.
__global__ void __launch_bounds__(256) clear_kernel(float4 *__restrict__ p, long long n4, float *__restrict__ tail, int n_tail)
{
    pdl_trigger();
    pdl_wait(); // whoever used the grid before (the previous plane-event's forward rows) is done with it
    const float4 z = make_float4(0.f, 0.f, 0.f, 0.f);
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += (long long)gridDim.x * blockDim.x) p[i] = z;
    if (blockIdx.x == 0 && (int)threadIdx.x < n_tail) tail[threadIdx.x] = 0.f;
}

} // namespace

cudaError_t launch_clear(float *p, long long n, int sm_count, cudaStream_t st)
{
    if (n <= 0) return cudaSuccess;
    const long long n4 = n / 4; // cudaMalloc'ed: 16-byte aligned
    long long ctas = (n4 + 255) / 256;
    const long long cap = (long long)sm_count * 8;
    if (ctas > cap) ctas = cap;
    if (ctas < 1) ctas = 1;
    return launch_pdl(clear_kernel, (unsigned)ctas, 256, 0, st, reinterpret_cast<float4 *>(p), n4, p + 4 * n4, (int)(n - 4 * n4));
}

cudaError_t launch_digitize(const float *M, long long n, float gain, float baseline, int bits, short *adc, cudaStream_t st)
{
    if (n <= 0) return cudaSuccess;
    const long long threads = (n + 3) / 4;
    digitize_kernel<<<(unsigned)((threads + 255) / 256), 256, 0, st>>>(M, n, gain, baseline, (float)((1 << bits) - 1), adc);
    return cudaGetLastError();
}

cudaError_t launch_drift(DriftInputs in, long long n, DriftParams prm, DriftPlanes planes, cudaStream_t st)
{
    if (n <= 0 || planes.n <= 0) return cudaSuccess;
    drift_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(in, n, prm, planes);
    return cudaGetLastError();
}

} // namespace wcsim

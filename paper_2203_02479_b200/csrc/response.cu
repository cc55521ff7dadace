// response.cu -- step p0: the "similarly transformed 2D detector response array R(w_t, w_x)" of PAPER.md:44, built
// once per plan.  R (n_rw x n_rt, wire-centred, tick-causal: A11) is embedded in the pad_w x pad_t grid with
// wrap-around on the wire axis and transformed by the definition of the DFT in fp64 -- R has only n_rw * n_rt
// non-zero samples, so the two separable sums below are cheap -- then scaled by 1/(pad_w pad_t) (A14) and rounded
// to fp32 once.  Also holds the small diagnostic kernels behind wcsim_debug_*.
#include "internal.h"
#include "rng.cuh"

namespace wcsim {

namespace {

// exp(-2 pi i m / n) for integers 0 <= m < n, n a power of two: sincospi of an exactly representable argument
__device__ __forceinline__ double2 unit_root(long long m, int n)
{
    double s, c;
    sincospi(-2.0 * (double)m / (double)n, &s, &c);
    return make_double2(c, s);
}

// tmp[r][kt] = sum_dt R[r][dt] exp(-2 pi i kt dt / pad_t),  kt = 0 .. pad_t/2
__global__ void response_ticks_kernel(const float *__restrict__ R, int n_rw, int n_rt, int pad_t,
                                      double2 *__restrict__ tmp)
{
    const int kt = blockIdx.x * blockDim.x + threadIdx.x;
    const int r = blockIdx.y;
    if (kt > pad_t / 2) return;
    double re = 0.0, im = 0.0;
    for (int dt = 0; dt < n_rt; ++dt) {
        const double v = (double)R[(size_t)r * n_rt + dt];
        const double2 w = unit_root(((long long)kt * dt) & (pad_t - 1), pad_t);
        re += v * w.x;
        im += v * w.y;
    }
    tmp[(size_t)r * (pad_t / 2 + 1) + kt] = make_double2(re, im);
}

// Rhat[kx][kt] = scale * sum_dx tmp[dx + c][kt] exp(-2 pi i kx dx / pad_w),  dx = -c .. c
__global__ void response_wires_kernel(const double2 *__restrict__ tmp, int n_rw, int pad_w, int pad_t, int spec_stride,
                                      float2 *__restrict__ Rhat)
{
    const int kt = blockIdx.x * blockDim.x + threadIdx.x;
    const int kx = blockIdx.y;
    if (kt >= spec_stride) return;
    float2 out = make_float2(0.f, 0.f);
    if (kt <= pad_t / 2) {
        const int c = (n_rw - 1) / 2;
        double re = 0.0, im = 0.0;
        for (int r = 0; r < n_rw; ++r) {
            const long long dx = r - c;
            const long long m = ((long long)kx * dx) & (long long)(pad_w - 1); // two's complement: mod pad_w
            const double2 w = unit_root(m, pad_w);
            const double2 v = tmp[(size_t)r * (pad_t / 2 + 1) + kt];
            re += v.x * w.x - v.y * w.y;
            im += v.x * w.y + v.y * w.x;
        }
        const double scale = 1.0 / ((double)pad_w * (double)pad_t);
        out = make_float2((float)(re * scale), (float)(im * scale));
    }
    Rhat[(size_t)kx * spec_stride + kt] = out;
}

// Rt[d][kt] = tmp[d][kt] / pad_t: the tick-axis spectrum of each wire offset of the response (direct wire mode)
__global__ void response_rows_kernel(const double2 *__restrict__ tmp, int n_rw, int pad_t, int spec_stride,
                                     float2 *__restrict__ Rt)
{
    const int kt = blockIdx.x * blockDim.x + threadIdx.x;
    const int d = blockIdx.y;
    if (kt >= spec_stride) return;
    float2 out = make_float2(0.f, 0.f);
    if (d < n_rw && kt <= pad_t / 2) {
        const double2 v = tmp[(size_t)d * (pad_t / 2 + 1) + kt];
        const double scale = 1.0 / (double)pad_t;
        out = make_float2((float)(v.x * scale), (float)(v.y * scale));
    }
    Rt[(size_t)d * spec_stride + kt] = out;
}

__global__ void debug_philox_kernel(const unsigned int *ctr, const unsigned int *key, unsigned int *out, long long n)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const uint4 r = philox4x32_10(make_uint4(ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3]),
                                  make_uint2(key[2 * i], key[2 * i + 1]));
    out[4 * i] = r.x;
    out[4 * i + 1] = r.y;
    out[4 * i + 2] = r.z;
    out[4 * i + 3] = r.w;
}

__global__ void debug_binomial_kernel(const double *N, const double *p, const unsigned int *w, double *k, long long n,
                                      bool normal_only)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    k[i] = binomial_draw(N[i], p[i], w[i], normal_only);
}

// fast path of the rounded-normal draw (rng.cuh): k and whether the fp32 guard accepted it
__global__ void debug_fast_normal_kernel(const double *N, const double *p, const unsigned int *w, double *k, int *ok,
                                         long long n)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    float kf = 0.f;
    const bool a = p[i] > 0.0 && p[i] <= 0.5 && fast_normal_draw((float)N[i], p[i], __dmul_rn(N[i], p[i]), w[i], kf);
    k[i] = (double)kf;
    ok[i] = a ? 1 : 0;
}

// z32_from_word against the fp64 AS 241 quantile over the words first .. first + count - 1:
// out[0] = max |z32 - z64| over the accepted words, out[1] = max |z64| over them, out[2] = number accepted (as a double),
// out[3] = max |z32 - z64| / max(1, |z64|)
__global__ void debug_z32_scan_kernel(unsigned long long first, unsigned long long count, unsigned long long *out)
{
    double e_abs = 0.0, z_max = 0.0, e_rel = 0.0;
    unsigned long long accepted = 0;
    for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < count;
         i += (unsigned long long)gridDim.x * blockDim.x) {
        const uint32_t w = (uint32_t)(first + i);
        float z32;
        if (!z32_from_word(w, z32)) continue;
        const double z64 = word_is_central(w) ? as241_central(w) : as241_tail(w);
        const double e = fabs((double)z32 - z64), az = fabs(z64);
        e_abs = fmax(e_abs, e);
        z_max = fmax(z_max, az);
        e_rel = fmax(e_rel, e / fmax(1.0, az));
        ++accepted;
    }
    // non-negative doubles order like their bit patterns
    atomicMax(out + 0, (unsigned long long)__double_as_longlong(e_abs));
    atomicMax(out + 1, (unsigned long long)__double_as_longlong(z_max));
    atomicAdd(out + 2, accepted);
    atomicMax(out + 3, (unsigned long long)__double_as_longlong(e_rel));
}

} // namespace

cudaError_t build_response_spectrum(const float *dev_R, int n_rw, int n_rt, int pad_w, int pad_t, int spec_stride,
                                    double2 *dev_tmp, float2 *dev_Rhat, cudaStream_t st)
{
    const int threads = 128;
    dim3 g1((pad_t / 2 + 1 + threads - 1) / threads, n_rw);
    response_ticks_kernel<<<g1, threads, 0, st>>>(dev_R, n_rw, n_rt, pad_t, dev_tmp);
    cudaError_t err = cudaGetLastError();
    if (err != cudaSuccess || dev_Rhat == nullptr) return err; // no Rhat: only the tick-axis spectra are wanted
    dim3 g2((spec_stride + threads - 1) / threads, pad_w);
    response_wires_kernel<<<g2, threads, 0, st>>>(dev_tmp, n_rw, pad_w, pad_t, spec_stride, dev_Rhat);
    return cudaGetLastError();
}

cudaError_t build_response_rows(const double2 *dev_tmp, int n_rw, int rt_rows, int pad_t, int spec_stride,
                                float2 *dev_Rt, cudaStream_t st)
{
    const int threads = 128;
    dim3 grid((spec_stride + threads - 1) / threads, rt_rows);
    response_rows_kernel<<<grid, threads, 0, st>>>(dev_tmp, n_rw, pad_t, spec_stride, dev_Rt);
    return cudaGetLastError();
}

cudaError_t launch_debug_philox(const unsigned int *ctr, const unsigned int *key, unsigned int *out, long long n,
                                cudaStream_t st)
{
    if (n <= 0) return cudaSuccess;
    debug_philox_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(ctr, key, out, n);
    return cudaGetLastError();
}

cudaError_t launch_debug_binomial(const double *N, const double *p, const unsigned int *w, double *k, long long n,
                                  bool normal_only, cudaStream_t st)
{
    if (n <= 0) return cudaSuccess;
    debug_binomial_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(N, p, w, k, n, normal_only);
    return cudaGetLastError();
}

cudaError_t launch_debug_fast_normal(const double *N, const double *p, const unsigned int *w, double *k, int *ok,
                                     long long n, cudaStream_t st)
{
    if (n <= 0) return cudaSuccess;
    debug_fast_normal_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(N, p, w, k, ok, n);
    return cudaGetLastError();
}

cudaError_t launch_debug_z32_scan(unsigned long long first, unsigned long long count, unsigned long long *out4,
                                  cudaStream_t st)
{
    cudaError_t err = cudaMemsetAsync(out4, 0, 4 * sizeof(unsigned long long), st);
    if (err != cudaSuccess || count == 0) return err;
    debug_z32_scan_kernel<<<148 * 8, 256, 0, st>>>(first, count, out4);
    return cudaGetLastError();
}

} // namespace wcsim

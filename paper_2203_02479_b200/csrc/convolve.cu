// convolve.cu -- steps a4-a6 (and a7 fused) of the hot path: the FFT convolution of Eq. (2), PAPER.md:46-52:
//     S(t,x) -> S(w_t, w_x),   M(w_t, w_x) = R(w_t, w_x) S(w_t, w_x),   M(w_t, w_x) -> M(t,x)
// as three kernels over the zero-padded pad_w x pad_t grid (A13), none of which touches a padded element in HBM:
//
//   rows_forward : one CTA per populated wire row.  The real row of pad_t samples is packed as pad_t/2 complex
//                  points (even + i odd), transformed in shared memory, and split into the half spectrum
//                  k = 0 .. pad_t/2.  Samples beyond n_ticks are zeros made in registers.
//   wires        : (default up to the measured crossover width, wcsim.cu wires_direct) the wire-axis transform / multiply / inverse done
//                  directly as an n_rw-tap convolution over wires for every tick frequency; see wires_kernel.
//   cols         : (otherwise, or on request) one CTA per tile of C adjacent tick-frequencies.  Forward transform over
//                  the wire axis (rows beyond n_wires are zeros made in registers), multiply by the response spectrum
//                  while the data is still in registers, inverse transform, store only the n_wires rows that are kept.
//   rows_inverse : one CTA per kept wire row (rows_inverse_tma_kernel: persistent CTAs, next row staged by a TMA bulk
//                  copy).  Half spectrum -> packed complex -> inverse transform -> the first n_ticks real samples.
//                  The noise spectrum of step a7 is added to the row spectrum here, so noise costs no pass over M.
//
// The 1/(pad_w pad_t) of the inverse transform is folded into Rhat / Rt (A14).  The FFT engine is csrc/fft.cuh.  The
// kernels of one plane-event are programmatic dependents of one another (csrc/pdl.cuh).
#include "fft.cuh"
#include "internal.h"
#include "rng.cuh"
#include "pdl.cuh"
#include "tma.cuh"

namespace wcsim {

namespace {

template <int N, bool FORWARD = true>
struct RowCfg {
    // 8192-point FORWARD rows (pad_t = 16384, configs[4]): 32 points per thread and a radix-32 first pass, 32.16.16: two
    // shared-memory exchanges instead of the three of 2.16.16.16 (the row transforms are bound by the load/store path):
    // 84.8 -> 74.1 us.  The inverse rows lose with it (92.5 -> 100.6 us: their staging of the partner bins doubles per
    // thread too) and keep 16 points per thread.
#ifdef WCSIM_ROWS_NO_R32
    static constexpr bool r32 = false;
#else
    static constexpr bool r32 = FORWARD && N == 8192;
#endif
    static constexpr int E = r32 ? 32 : 16;
    static constexpr int threads = N / E;
    static constexpr int smem_bytes = SmemSize<N, 1>::float2s * (int)sizeof(float2);
    // 64 registers per thread (E = 16): 1024 threads of row transforms resident per SM whatever the row length;
    // 128 registers with 32 points per thread: 512 threads
    static constexpr int per_sm_threads = r32 ? 512 : 1024;
    static constexpr int min_ctas = threads >= per_sm_threads ? 1 : (per_sm_threads / threads > 8 ? 8 : per_sm_threads / threads);
};
template <int N>
struct ColCfg {
    static constexpr int C = N <= 1024 ? 8 : (N <= 4096 ? 4 : 2);
    static constexpr int E = N <= 1024 ? 16 : 32;
    static constexpr int threads = (N / E) * C;
    static constexpr int smem_bytes = SmemSize<N, C>::float2s * (int)sizeof(float2);
};

// ------------------------------------------------------------------------------------------------------------------
// a4, tick axis: real row -> half spectrum
// ------------------------------------------------------------------------------------------------------------------
template <int N, bool VEC>
__global__ void __launch_bounds__(RowCfg<N>::threads, RowCfg<N>::min_ctas) rows_forward_kernel(GridDims g, ConvBuffers b,
                                                                                                    int tail_from)
{
    constexpr int E = RowCfg<N>::E, NT = N / E;
    extern __shared__ float2 smem[];
    const int row = blockIdx.x, i = threadIdx.x;
    if ((int)blockIdx.x >= tail_from) pdl_trigger();
    pdl_wait(); // S is the raster's
    const float *src = b.S + (size_t)row * g.n_ticks;
    float2 v[E];
#pragma unroll
    for (int e = 0; e < E; ++e) {
        const int pt = i + e * NT;
        if constexpr (VEC) {
            v[e] = (2 * pt < g.n_ticks) ? reinterpret_cast<const float2 *>(src)[pt] : make_float2(0.f, 0.f);
        } else {
            v[e].x = (2 * pt < g.n_ticks) ? src[2 * pt] : 0.f;
            v[e].y = (2 * pt + 1 < g.n_ticks) ? src[2 * pt + 1] : 0.f;
        }
    }
    fft_block<N, 1, E, -1, 1, RowCfg<N>::r32>(v, smem, i, 0, b.tw_row, false);
    // split Z = FFT(even + i odd) into the spectrum of the real row:
    //   A = (Z_k + conj Z_{N-k})/2, B = (Z_k - conj Z_{N-k})/(2i), X_k = A + exp(-2 pi i k / 2N) B
    __syncthreads();
#pragma unroll
    for (int e = 0; e < E; ++e) smem[smem_index<1>(i + e * NT, 0)] = v[e];
    __syncthreads();
    const int pl = plane_of_row(b.planes, row);
    float2 *dst = b.spec + (size_t)(b.planes.srow0[pl] + row - b.planes.row0[pl]) * b.spec_stride;
    float2 tws[E];
    split_twiddles<E>(tws, load_tw(b.tw_real, i)); // exp(-2 pi i k / 2N) at k = i + e NT: one load, 15 constant rotations
#pragma unroll
    for (int e = 0; e < E; ++e) {
        const int k = i + e * NT;
        const float2 zk = v[e];
        const float2 zn = smem[smem_index<1>((N - k) & (N - 1), 0)];
        const float2 A = make_float2(0.5f * (zk.x + zn.x), 0.5f * (zk.y - zn.y));
        const float2 B = make_float2(0.5f * (zk.y + zn.y), -0.5f * (zk.x - zn.x));
        const float2 w = tws[e];
        dst[k] = cadd(A, cmul(w, B));
        if (k == 0) dst[N] = make_float2(zk.x - zk.y, 0.f);
    }
}

// Persistent, TMA-staged variant of the inverse row kernel (512 <= pad_t/2 <= 4096: configs[0..3]).  A CTA walks rows
// blockIdx.x, blockIdx.x + gridDim.x, ...; one thread issues a single bulk copy (cp.async.bulk, mbarrier-tracked) of
// the NEXT row into the staging buffer as soon as every thread has lifted the current row into registers, so the copy
// runs under the butterflies and the rows are no longer load -> wait -> compute one after the other.
// Shared memory per CTA: FFT exchange buffer + one staged row + the mbarrier, three CTAs per SM.
// (The same staging was tried for the forward rows and lost 1.5 us on configs[1]: there the plain kernel already reads
// its row straight into registers, and four 64-register CTAs per SM beat three 80-register ones.)
template <int N>
struct RowTma {
    static constexpr int threads = RowCfg<N, false>::threads;
    static constexpr int min_ctas = threads <= 256 ? 3 : (threads <= 512 ? 2 : 1);
    static constexpr int work_bytes = (RowCfg<N, false>::smem_bytes + 127) / 128 * 128;
    static constexpr bool enabled = N <= 4096 && N >= 512;
    static int smem_bytes(int stage_bytes) { return work_bytes + (stage_bytes + 127) / 128 * 128 + 16; }
    static int grid(int rows, int stage_bytes, int sm_count)
    {
        int per_sm = (227 * 1024) / (smem_bytes(stage_bytes) + 1024);
        per_sm = per_sm > min_ctas ? min_ctas : per_sm;
        const int slots = sm_count * (per_sm > 0 ? per_sm : 1);
        // equal rows per CTA where the count allows it: ceil(rows / ceil(rows / slots))
        const int rounds = (rows + slots - 1) / slots;
        return (rows + rounds - 1) / rounds;
    }
};

// ------------------------------------------------------------------------------------------------------------------
// a4 wire axis, a5 multiply, a6 wire axis
// ------------------------------------------------------------------------------------------------------------------
template <int N>
__global__ void __launch_bounds__(ColCfg<N>::threads) cols_kernel(GridDims g, ConvBuffers b)
{
    constexpr int C = ColCfg<N>::C, E = ColCfg<N>::E, NT = N / E;
    extern __shared__ float2 smem[];
    const int c = threadIdx.x % C, i = threadIdx.x / C;
    const int col = blockIdx.x * C + c;
    pdl_wait();
    float2 *spec = b.spec + col;
    const float2 *rh = b.Rhat + col;
    float2 v[E];
#pragma unroll
    for (int e = 0; e < E; ++e) {
        const int x = i + e * NT;
        v[e] = (x < g.n_wires) ? spec[(size_t)x * b.spec_stride] : make_float2(0.f, 0.f);
    }
    fft_block<N, C, E, -1>(v, smem, i, c, b.tw_col, false);
#pragma unroll
    for (int e = 0; e < E; ++e) {
        const int x = i + e * NT;
        v[e] = cmul(v[e], __ldg(rh + (size_t)x * b.spec_stride));
    }
    fft_block<N, C, E, +1>(v, smem, i, c, b.tw_col, true);
#pragma unroll
    for (int e = 0; e < E; ++e) {
        const int x = i + e * NT;
        if (x < g.n_wires) spec[(size_t)x * b.spec_stride] = v[e];
    }
}

// ------------------------------------------------------------------------------------------------------------------
// a4 wire axis, a5 multiply, a6 wire axis, direct form.  With the tick axis transformed, Eq. (2)'s wire-axis
// transform / multiply / inverse transform is, for every tick frequency k, the linear convolution
//     Mhat[x][k] = sum_{d=0}^{n_rw-1} Rt[d][k] Shat[x + c - d][k],      Rt[d][.] = rfft_t(R[d][.]) / pad_t,
// over the n_rw wire offsets of the response (Shat = 0 outside [0, n_wires)).  For the 21- and 41-wire responses of
// BASELINE.json's configs that is 4 n_rw FMAs per output against the ~2 x 4.3 log2(pad_w) adds and multiplies of the
// FFT route, needs no zero-padded wire rows, no shared memory, and reads n_rw rows of Rt (0.7 MB for configs[1])
// instead of the pad_w rows of Rhat (33.6 MB).  One thread owns one k and O consecutive output wires; lanes run
// along k (coalesced 256-byte rows); the response is walked in chunks of D offsets held in registers, so every
// register index below is static.  The spectrum buffer carries zero halo rows below wire 0 and above wire
// n_wires-1 (wires_halo(), written once at plan time), so no load is predicated, and with the row stride a template
// argument every load of a chunk is one instruction off a single pointer (immediate offsets): the inner loop is
// 4 O D FFMAs against O + 2 D - 1 loads.  Neighbouring row groups of a CTA share their halo rows through L1.
// ------------------------------------------------------------------------------------------------------------------
#ifndef WCSIM_WIRES_CTAS
#define WCSIM_WIRES_CTAS 3
#endif
#ifndef WCSIM_WIRES_RG
#define WCSIM_WIRES_RG 8
#endif
#ifndef WCSIM_WIRES_D
#define WCSIM_WIRES_D 7
#endif
constexpr int kWiresD = WCSIM_WIRES_D, kWiresRG = WCSIM_WIRES_RG, kWiresO = 8;
constexpr int kWiresNch21 = (21 + kWiresD - 1) / kWiresD, kWiresNch41 = (41 + kWiresD - 1) / kWiresD; // chunks of BASELINE.json's widths
constexpr int kWiresCtas = WCSIM_WIRES_CTAS; // resident CTAs per SM the register budget is set for

// STRIDE = 0: row stride read from the buffers (any pad_t); NCH = 0: chunk count read from the buffers (any n_rw),
// else the chunk loop is unrolled so that the loads of the next chunk are in flight under the FFMAs of this one
template <int O, int D, int NCH, int STRIDE>
__global__ void __launch_bounds__(32 * kWiresRG, kWiresCtas) wires_kernel(GridDims g, ConvBuffers b, int nk, int tail_from)
{
    if ((int)(blockIdx.y * gridDim.x + blockIdx.x) >= tail_from) pdl_trigger();
    pdl_wait(); // the row spectra are rows_forward's
    const int k = blockIdx.x * 32 + threadIdx.x;
    int pl = 0; // the plane of this row group (uniform over the CTA)
    while (pl + 1 < b.planes.n && (int)blockIdx.y >= b.planes.grp0[pl + 1]) ++pl;
    const int x0 = ((blockIdx.y - b.planes.grp0[pl]) * kWiresRG + threadIdx.y) * O; // first output wire, in the plane
    const int n_wires = b.planes.row0[pl + 1] - b.planes.row0[pl];
    if (k >= nk || x0 >= n_wires) return;
    const ptrdiff_t stride = STRIDE ? (ptrdiff_t)STRIDE : (ptrdiff_t)b.spec_stride;
    // impact positions (reading A25): position kk of wire x is fine row x K + kk of the row spectra, so the inputs of one
    // position are K rows apart and the taps of every position accumulate into the same outputs.  The instances with a
    // compile-time stride are only launched for K = 1.
    const int K = STRIDE ? 1 : b.impact_K;
    const ptrdiff_t rstep = STRIDE ? (ptrdiff_t)STRIDE : stride * K;
    const int c = (b.n_rw - 1) / 2;
    float2 acc[O];
#pragma unroll
    for (int o = 0; o < O; ++o) acc[o] = make_float2(0.f, 0.f);
    const int n_chunks = NCH ? NCH : b.rt_rows / D;
    for (int kk = 0; kk < K; ++kk) {
        // chunk d0 uses wire rows x0 + c - d0 - (D-1) .. x0 + c - d0 + O - 1 (halo rows included) and Rt rows d0 .. d0+D-1
        const float2 *in = b.spec + k + ((ptrdiff_t)b.planes.srow0[pl] + ((ptrdiff_t)x0 + c - (D - 1)) * K + kk) * stride; // plain loads: see pdl.cuh
        const float2 *__restrict__ rt = b.Rt + k + ((ptrdiff_t)pl * K + kk) * b.rt_rows * stride;
#pragma unroll
        for (int ch = 0; ch < n_chunks; ++ch) {
            float2 coef[D], s[O + D - 1];
#pragma unroll
            for (int j = 0; j < D; ++j) coef[j] = __ldg(rt + j * stride);
#pragma unroll
            for (int q = 0; q < O + D - 1; ++q) s[q] = in[q * rstep];
#pragma unroll
            for (int o = 0; o < O; ++o)
#pragma unroll
                for (int j = 0; j < D; ++j) {
                    const float2 v = s[o - j + D - 1], w = coef[j];
                    acc[o].x = fmaf(w.x, v.x, acc[o].x);
                    acc[o].x = fmaf(-w.y, v.y, acc[o].x);
                    acc[o].y = fmaf(w.x, v.y, acc[o].y);
                    acc[o].y = fmaf(w.y, v.x, acc[o].y);
                }
            in -= D * rstep;
            rt += D * stride;
        }
    }
    float2 *__restrict__ out = b.spec2 + k + (ptrdiff_t)(b.planes.row0[pl] + x0) * stride;
#pragma unroll
    for (int o = 0; o < O; ++o)
        if (x0 + o < n_wires) out[o * stride] = acc[o];
}

// ------------------------------------------------------------------------------------------------------------------
// a6 tick axis (+ a7 noise): half spectrum -> real row
// ------------------------------------------------------------------------------------------------------------------
// noise spectrum of bin k on `wire`: amp[k] exp(2 pi i u), u = (word + 1/2) 2^-32 (A15-A17); amp is pre-scaled
__device__ __forceinline__ float noise_phase(uint32_t w) // 2u = w 2^-31 + 2^-32, the argument of sincospi
{
    return (float)w * 4.656612873077393e-10f + 2.3283064365386963e-10f;
}
// sin and cos of pi x for x = 2u in (0, 2).  Default: the special-function unit on pi (x - 1) in [-pi, pi) with the sign
// flipped (sin pi x = -sin pi (x - 1)); MUFU.SIN / MUFU.COS are accurate to 2^-21.4 absolute there and the product pi (x - 1)
// to 4e-7, so a noise sample is off by ~5e-7 of its amplitude (measured: rel-L2 of N against the oracle 2.4e-7 - 2.7e-7, with sincospif 1.3e-7 - 1.7e-7; bound 1e-5)
// for 5 instructions instead of the ~35 of sincospif, which cost 8 us per 800-row plane inside the inverse row transform (now 4 us).
__device__ __forceinline__ void noise_sincos(float x, float *s, float *c)
{
#ifdef WCSIM_NOISE_SINCOSPI
    sincospif(x, s, c);
#else
    const float a = 3.14159265358979f * (x - 1.0f);
    *s = -__sinf(a);
    *c = -__cosf(a);
#endif
}
__device__ __forceinline__ float2 noise_bin(const NoiseArgs &nz, uint64_t seed, uint32_t wire, uint32_t k)
{
    const uint4 words = noise_words(seed, wire, k >> 2);
    const uint32_t w = pick_word(words, k & 3u);
    float s, c;
    noise_sincos(noise_phase(w), &s, &c);
    const float a = __ldg(nz.amp + k);
    return make_float2(a * c, a * s);
}

template <int N, bool VEC>
__global__ void __launch_bounds__(RowCfg<N, false>::threads, RowCfg<N, false>::min_ctas) rows_inverse_kernel(GridDims g, ConvBuffers b, NoiseArgs nz,
                                                                           bool use_spec, bool accumulate)
{
    constexpr int E = RowCfg<N, false>::E, NT = N / E;
    extern __shared__ float2 smem[];
    const int row = blockIdx.x, i = threadIdx.x;
    pdl_wait(); // a no-op unless launched as a programmatic dependent
    const float2 *src = b.spec_inv + (size_t)row * b.spec_stride;
    const bool noisy = nz.amp != nullptr;
    const int noise_plane = plane_of_row(b.planes, row);
    const uint32_t wire = (uint32_t)(row - b.planes.row0[noise_plane]); // the noise is keyed by the plane's own wire ...
    const uint64_t noise_seed = nz.seed[noise_plane];                  // ... and the plane's own seed (A26)
    float2 v[E];
    float2 tws[E];
    split_twiddles<E>(tws, load_tw(b.tw_real, i)); // exp(-2 pi i k / 2N) at k = i + e NT: one load, 15 constant rotations
    if (use_spec && !noisy) {
        // plain convolution: the partner bin X_{N-k} is read straight from the spectrum row (descending, still
        // coalesced; L1 / L2 hits), which saves the staging stores and a barrier
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const int k = i + e * NT;
            float2 xk = src[k], xn = src[N - k];
            if (k == 0) xk.y = 0.f, xn.y = 0.f; // imaginary parts of the DC and Nyquist bins do not reach a real output
            const float2 s = make_float2(xk.x + xn.x, xk.y - xn.y);
            const float2 d = make_float2(xk.x - xn.x, xk.y + xn.y);
            const float2 w = tws[e]; // (cos, -sin)
            const float2 t = make_float2(w.x * d.x + w.y * d.y, w.x * d.y - w.y * d.x);
            v[e] = make_float2(s.x - t.y, s.y + t.x);
        }
        fft_block<N, 1, E, +1, 1, RowCfg<N, false>::r32>(v, smem, i, 0, b.tw_row, false);
    } else {
        // stage X_k (+ noise) in shared memory so that every thread can reach the partner X_{N-k}
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const int k = i + e * NT;
            float2 x = use_spec ? src[k] : make_float2(0.f, 0.f);
            if (noisy) x = cadd(x, noise_bin(nz, noise_seed, wire, (uint32_t)k));
            if (k == 0) {
                x.y = 0.f; // the imaginary parts of the DC and Nyquist bins do not reach a real output
                float2 xn = use_spec ? src[N] : make_float2(0.f, 0.f);
                if (noisy) xn = cadd(xn, noise_bin(nz, noise_seed, wire, (uint32_t)N));
                xn.y = 0.f;
                smem[smem_index<1>(N, 0)] = xn;
            }
            smem[smem_index<1>(k, 0)] = x;
        }
        __syncthreads();
        // Z_k = (X_k + conj X_{N-k}) + i exp(+2 pi i k / 2N) (X_k - conj X_{N-k});  inverse FFT of Z = even + i odd
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const int k = i + e * NT;
            const float2 xk = smem[smem_index<1>(k, 0)];
            const float2 xn = smem[smem_index<1>(N - k, 0)];
            const float2 s = make_float2(xk.x + xn.x, xk.y - xn.y);
            const float2 d = make_float2(xk.x - xn.x, xk.y + xn.y);
            const float2 w = tws[e]; // (cos, -sin)
            const float2 t = make_float2(w.x * d.x + w.y * d.y, w.x * d.y - w.y * d.x);
            v[e] = make_float2(s.x - t.y, s.y + t.x);
        }
        fft_block<N, 1, E, +1, 1, RowCfg<N, false>::r32>(v, smem, i, 0, b.tw_row, true);
    }
    float *dst = b.M + (size_t)row * g.n_ticks;
#pragma unroll
    for (int e = 0; e < E; ++e) {
        const int pt = i + e * NT;
        if constexpr (VEC) {
            if (2 * pt < g.n_ticks) {
                float2 *p = reinterpret_cast<float2 *>(dst) + pt;
                float2 o = v[e];
                if (accumulate) o = cadd(o, *p);
                *p = o;
            }
        } else {
            if (2 * pt < g.n_ticks) dst[2 * pt] = v[e].x + (accumulate ? dst[2 * pt] : 0.f);
            if (2 * pt + 1 < g.n_ticks) dst[2 * pt + 1] = v[e].y + (accumulate ? dst[2 * pt + 1] : 0.f);
        }
    }
}

// a6 tick axis (+ a7 noise), TMA-staged: the row spectrum lands in shared memory by one bulk copy, so the partner bin
// X_{N-k} is read where the copy put it (no staging stores); the noise spectrum is added to the staged row in place.
template <int N>
__global__ void __launch_bounds__(RowTma<N>::threads, RowTma<N>::min_ctas) rows_inverse_tma_kernel(GridDims g, ConvBuffers b,
                                                                                                   NoiseArgs nz)
{
    constexpr int E = RowCfg<N, false>::E, NT = N / E;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float2 *smem = reinterpret_cast<float2 *>(smem_raw);
    const uint32_t row_bytes = (uint32_t)b.spec_stride * 8u; // whole stride: a multiple of 64
    float2 *stage = reinterpret_cast<float2 *>(smem_raw + RowTma<N>::work_bytes);
    uint64_t *bar = reinterpret_cast<uint64_t *>(smem_raw + RowTma<N>::work_bytes + (row_bytes + 127) / 128 * 128);
    const int i = threadIdx.x;
    const bool noisy = nz.amp != nullptr;
    int row = blockIdx.x;
    if (i == 0) {
        mbar_init(bar, 1);
        pdl_wait(); // the product spectra are the wire pass's
        mbar_arrive_expect_tx(bar, row_bytes);
        bulk_copy_g2s(stage, b.spec_inv + (size_t)row * b.spec_stride, row_bytes, bar);
    }
    pdl_wait();
    __syncthreads();
    uint32_t parity = 0;
    float2 tws[E];
    split_twiddles<E>(tws, load_tw(b.tw_real, i)); // the same for every row this thread works on
    for (; row < g.n_wires; row += gridDim.x) {
        mbar_wait(bar, parity);
        parity ^= 1u;
        if (noisy) {
            const int noise_plane = plane_of_row(b.planes, row);
            const uint32_t wire = (uint32_t)(row - b.planes.row0[noise_plane]); // the plane's own wire and seed (A26)
            const uint64_t noise_seed = nz.seed[noise_plane];
            // one Philox call gives the phases of four consecutive frequency bins (A17): a thread takes whole calls
            for (int q = i; q < N / 4; q += NT) {
                const uint4 words = noise_words(noise_seed, wire, (uint32_t)q);
                const float4 a = __ldg(reinterpret_cast<const float4 *>(nz.amp) + q);
                float4 *x = reinterpret_cast<float4 *>(stage + 4 * q);
                float4 lo = x[0], hi = x[1];
                float sn, cs;
                noise_sincos(noise_phase(words.x), &sn, &cs), lo.x = fmaf(a.x, cs, lo.x), lo.y = fmaf(a.x, sn, lo.y);
                noise_sincos(noise_phase(words.y), &sn, &cs), lo.z = fmaf(a.y, cs, lo.z), lo.w = fmaf(a.y, sn, lo.w);
                noise_sincos(noise_phase(words.z), &sn, &cs), hi.x = fmaf(a.z, cs, hi.x), hi.y = fmaf(a.z, sn, hi.y);
                noise_sincos(noise_phase(words.w), &sn, &cs), hi.z = fmaf(a.w, cs, hi.z), hi.w = fmaf(a.w, sn, hi.w);
                x[0] = lo, x[1] = hi;
            }
            if (i == 0) stage[N] = cadd(stage[N], noise_bin(nz, noise_seed, wire, (uint32_t)N));
            __syncthreads();
        }
        // Z_k = (X_k + conj X_{N-k}) + i exp(+2 pi i k / 2N) (X_k - conj X_{N-k});  inverse FFT of Z = even + i odd
        float2 v[E];
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const int k = i + e * NT;
            float2 xk = stage[k], xn = stage[N - k];
            if (k == 0) xk.y = 0.f, xn.y = 0.f; // imaginary parts of the DC and Nyquist bins do not reach a real output
            const float2 s = make_float2(xk.x + xn.x, xk.y - xn.y);
            const float2 d = make_float2(xk.x - xn.x, xk.y + xn.y);
            const float2 w = tws[e]; // (cos, -sin)
            const float2 t = make_float2(w.x * d.x + w.y * d.y, w.x * d.y - w.y * d.x);
            v[e] = make_float2(s.x - t.y, s.y + t.x);
        }
        __syncthreads(); // every thread is done with the staged row and with last row's exchange buffer
        const int next = row + gridDim.x;
        if (i == 0 && next < g.n_wires) {
            fence_proxy_async(); // the generic-proxy accesses to the stage above precede the async-proxy refill
            mbar_arrive_expect_tx(bar, row_bytes);
            bulk_copy_g2s(stage, b.spec_inv + (size_t)next * b.spec_stride, row_bytes, bar);
        }
        fft_block<N, 1, E, +1, 1, RowCfg<N, false>::r32>(v, smem, i, 0, b.tw_row, false);
        float2 *dst = reinterpret_cast<float2 *>(b.M + (size_t)row * g.n_ticks);
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const int pt = i + e * NT;
            if (2 * pt < g.n_ticks) dst[pt] = v[e];
        }
    }
}

template <typename K>
cudaError_t set_smem(K kernel, int bytes)
{
    if (bytes <= 48 * 1024) return cudaSuccess;
    return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
}

constexpr int kTmaSmemCap = 200 * 1024;
template <int NN>
cudaError_t configure_tma()
{
    if constexpr (RowTma<NN>::enabled) {
        return cudaFuncSetAttribute(rows_inverse_tma_kernel<NN>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                    kTmaSmemCap);
    }
    return cudaSuccess;
}

// the TMA-staged kernel wants 16-byte aligned rows (bulk copies) and float2 stores into M
template <int NN>
bool inverse_tma_ok(GridDims g, const ConvBuffers &b)
{
    if constexpr (!RowTma<NN>::enabled) return false;
    return g.n_ticks % 2 == 0 && reinterpret_cast<uintptr_t>(b.M) % 8 == 0 &&
           reinterpret_cast<uintptr_t>(b.spec_inv) % 16 == 0 && RowTma<NN>::smem_bytes(b.spec_stride * 8) <= kTmaSmemCap;
}
template <int NN>
void launch_inverse_tma(GridDims g, ConvBuffers b, NoiseArgs nz, cudaStream_t st)
{
    if constexpr (RowTma<NN>::enabled) {
        const int stage = b.spec_stride * 8;
        launch_pdl(rows_inverse_tma_kernel<NN>, RowTma<NN>::grid(g.n_wires, stage, b.sm_count), RowTma<NN>::threads,
                   RowTma<NN>::smem_bytes(stage), st, g, b, nz);
    }
}

#define WCSIM_ROW_SIZES(X) X(16) X(32) X(64) X(128) X(256) X(512) X(1024) X(2048) X(4096) X(8192) X(16384)
#define WCSIM_COL_SIZES(X) X(16) X(32) X(64) X(128) X(256) X(512) X(1024) X(2048) X(4096) X(8192)

} // namespace

bool conv_sizes_supported(int pad_w, int pad_t)
{
    const int n = pad_t / 2;
    bool row_ok = false, col_ok = false;
#define X(NN) row_ok = row_ok || (n == NN);
    WCSIM_ROW_SIZES(X)
#undef X
#define X(NN) col_ok = col_ok || (pad_w == NN);
    WCSIM_COL_SIZES(X)
#undef X
    return row_ok && col_ok && pad_t == 2 * n;
}

cudaError_t conv_configure(int pad_w, int pad_t)
{
    cudaError_t err = cudaSuccess;
    switch (pad_t / 2) {
#define X(NN)                                                                                                          \
    case NN:                                                                                                           \
        if (err == cudaSuccess) err = set_smem(rows_forward_kernel<NN, true>, RowCfg<NN>::smem_bytes);                 \
        if (err == cudaSuccess) err = set_smem(rows_forward_kernel<NN, false>, RowCfg<NN>::smem_bytes);                \
        if (err == cudaSuccess) err = set_smem(rows_inverse_kernel<NN, true>, RowCfg<NN, false>::smem_bytes);                 \
        if (err == cudaSuccess) err = set_smem(rows_inverse_kernel<NN, false>, RowCfg<NN, false>::smem_bytes);                \
        if (err == cudaSuccess) err = configure_tma<NN>();                                                             \
        break;
        WCSIM_ROW_SIZES(X)
#undef X
    default:
        return cudaErrorInvalidValue;
    }
    switch (pad_w) {
#define X(NN)                                                                                                          \
    case NN:                                                                                                           \
        if (err == cudaSuccess) err = set_smem(cols_kernel<NN>, ColCfg<NN>::smem_bytes);                               \
        break;
        WCSIM_COL_SIZES(X)
#undef X
    default:
        return cudaErrorInvalidValue;
    }
    return err;
}

static bool rows_vectorisable(GridDims g, const void *p)
{
    return (g.n_ticks % 2 == 0) && (reinterpret_cast<uintptr_t>(p) % 8 == 0);
}

cudaError_t launch_rows_forward(GridDims g, int pad_t, ConvBuffers b, cudaStream_t st)
{
    const bool vec = rows_vectorisable(g, b.S);
    int tail = 0; // first CTA of the last wave (pdl.cuh): from the resident CTAs per SM of this row length
    switch (pad_t / 2) {
#define X(NN)                                                                                                          \
    case NN:                                                                                                           \
        tail = pdl_tail_from(g.n_wires, (long long)b.sm_count * RowCfg<NN>::min_ctas);                                 \
        if (vec)                                                                                                       \
            launch_pdl(rows_forward_kernel<NN, true>, g.n_wires, RowCfg<NN>::threads, RowCfg<NN>::smem_bytes, st, g, b, tail); \
        else                                                                                                           \
            launch_pdl(rows_forward_kernel<NN, false>, g.n_wires, RowCfg<NN>::threads, RowCfg<NN>::smem_bytes, st, g, b, tail); \
        break;
        WCSIM_ROW_SIZES(X)
#undef X
    default:
        return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

cudaError_t launch_cols(GridDims g, int pad_w, int pad_t, ConvBuffers b, cudaStream_t st)
{
    (void)pad_t;
    switch (pad_w) {
#define X(NN)                                                                                                          \
    case NN:                                                                                                           \
        cols_kernel<NN><<<b.spec_stride / ColCfg<NN>::C, ColCfg<NN>::threads, ColCfg<NN>::smem_bytes, st>>>(g, b);     \
        break;
        WCSIM_COL_SIZES(X)
#undef X
    default:
        return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

int wires_chunk() { return kWiresD; }
int wires_rows_per_group() { return kWiresO * kWiresRG; }

// zero rows the direct wire kernel may read below wire 0 / above wire n_wires-1 of the row spectra
void wires_halo(int n_rw, int *below, int *above)
{
    const int c = (n_rw - 1) / 2;
    const int rt_rows = (n_rw + kWiresD - 1) / kWiresD * kWiresD;
    *below = rt_rows - 1 - c; // lowest row read: 0 + c - (rt_rows - D) - (D - 1)
    *above = kWiresO - 1 + c; // highest: (n_wires - 1) + (O - 1) + c, from the last, ragged row group
}

cudaError_t launch_wires(GridDims g, int pad_t, ConvBuffers b, cudaStream_t st)
{
    constexpr int O = kWiresO;
    const int nk = pad_t / 2 + 1;
    const dim3 block(32, kWiresRG), grid((nk + 31) / 32, b.planes.grp0[b.planes.n]); // row groups of all planes
    // BASELINE.json's paddings and response widths (21 wires -> 3 chunks of 7 offsets, 41 -> 6) get immediate-offset loads and an
    // unrolled chunk loop; anything else takes the generic instance
    const int key = b.impact_K == 1 ? b.rt_rows / kWiresD * 100000 + b.spec_stride : -1;
    const int tail = pdl_tail_from((long long)grid.x * grid.y, (long long)b.sm_count * kWiresCtas);
    cudaError_t err = cudaSuccess;
    switch (key) {
    case kWiresNch21 * 100000 + 1024 / 2 + 8: err = launch_pdl(wires_kernel<O, kWiresD, kWiresNch21, 1024 / 2 + 8>, grid, block, 0, st, g, b, nk, tail); break;
    case kWiresNch21 * 100000 + 8192 / 2 + 8: err = launch_pdl(wires_kernel<O, kWiresD, kWiresNch21, 8192 / 2 + 8>, grid, block, 0, st, g, b, nk, tail); break;
    case kWiresNch41 * 100000 + 16384 / 2 + 8: err = launch_pdl(wires_kernel<O, kWiresD, kWiresNch41, 16384 / 2 + 8>, grid, block, 0, st, g, b, nk, tail); break;
    default: err = launch_pdl(wires_kernel<O, kWiresD, 0, 0>, grid, block, 0, st, g, b, nk, tail); break;
    }
    return err != cudaSuccess ? err : cudaGetLastError();
}

cudaError_t launch_rows_inverse(GridDims g, int pad_t, ConvBuffers b, NoiseArgs noise, bool use_spec, bool accumulate,
                                cudaStream_t st)
{
    const bool vec = rows_vectorisable(g, b.M);
    switch (pad_t / 2) {
#define X(NN)                                                                                                          \
    case NN:                                                                                                           \
        if (use_spec && !accumulate && inverse_tma_ok<NN>(g, b))                                                       \
            launch_inverse_tma<NN>(g, b, noise, st);                                                                   \
        else if (vec)                                                                                                  \
            rows_inverse_kernel<NN, true><<<g.n_wires, RowCfg<NN, false>::threads, RowCfg<NN, false>::smem_bytes, st>>>(             \
                g, b, noise, use_spec, accumulate);                                                                    \
        else                                                                                                           \
            rows_inverse_kernel<NN, false><<<g.n_wires, RowCfg<NN, false>::threads, RowCfg<NN, false>::smem_bytes, st>>>(            \
                g, b, noise, use_spec, accumulate);                                                                    \
        break;
        WCSIM_ROW_SIZES(X)
#undef X
    default:
        return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

} // namespace wcsim

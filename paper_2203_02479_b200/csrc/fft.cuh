// fft.cuh -- shared-memory Stockham FFT engine used by the three convolution kernels (Eq. 2).
//
// One CTA transforms C independent length-N complex sequences ("columns", C fastest in memory).  Every thread owns
// E elements of one sequence in registers, at points  pt = i + e*(N/E), e = 0..E-1  (i = its butterfly lane).  A pass
// of radix R does E/R in-register butterflies per thread; between passes the data is exchanged through shared
// memory in Stockham (autosort) order, so the input of the first pass and the output of the last pass both sit at
// the same natural-order points pt = i + e*(N/E).  That is what lets the column kernel multiply by the response
// spectrum and start the inverse transform without leaving registers, and lets first loads / last stores go
// straight to global memory, coalesced.
//
// Everything here is __host__ __device__ so that tests/test_fft_engine_host.py can run the same index logic on the
// CPU (threads emulated by loops) against numpy.fft.
#pragma once
#include <cuda_runtime.h>
#include <math.h>

#ifndef WCSIM_HD
#define WCSIM_HD __host__ __device__ __forceinline__
#endif

namespace wcsim {

WCSIM_HD float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
WCSIM_HD float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
WCSIM_HD float2 cmul(float2 a, float2 b) { return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
WCSIM_HD float2 cconj(float2 a) { return make_float2(a.x, -a.y); }

// multiply by exp(DIR * i * pi/2): DIR = -1 (forward) gives -i*a, DIR = +1 (inverse) gives +i*a
template <int DIR>
WCSIM_HD float2 mul_qi(float2 a)
{
    return DIR < 0 ? make_float2(a.y, -a.x) : make_float2(-a.y, a.x);
}

// multiply by exp(DIR * 2 pi i * m / 16) for a compile-time m
template <int DIR, int M>
WCSIM_HD float2 mul_w16(float2 a)
{
    constexpr int m = ((M % 16) + 16) % 16;
    constexpr float C1 = 0.92387953251128673848f, S1 = 0.38268343236508978178f, H = 0.70710678118654752440f;
    if constexpr (m == 0) return a;
    else if constexpr (m == 4) return mul_qi<DIR>(a);
    else if constexpr (m == 8) return make_float2(-a.x, -a.y);
    else if constexpr (m == 12) return mul_qi<-DIR>(a);
    else if constexpr (m == 2) { // (1 + DIR i)/sqrt2
        return DIR < 0 ? make_float2((a.x + a.y) * H, (a.y - a.x) * H) : make_float2((a.x - a.y) * H, (a.y + a.x) * H);
    } else if constexpr (m == 6) { // (-1 + DIR i)/sqrt2
        return DIR < 0 ? make_float2((a.y - a.x) * H, -(a.x + a.y) * H) : make_float2(-(a.x + a.y) * H, (a.x - a.y) * H);
    } else {
        constexpr float c = (m == 1) ? C1 : (m == 3) ? S1 : (m == 5) ? -S1 : (m == 7) ? -C1 : (m == 9) ? -C1
                          : (m == 10) ? -H : (m == 11) ? -S1 : (m == 13) ? S1 : (m == 14) ? H : /*15*/ C1;
        constexpr float s = (m == 1) ? S1 : (m == 3) ? C1 : (m == 5) ? C1 : (m == 7) ? S1 : (m == 9) ? -S1
                          : (m == 10) ? -H : (m == 11) ? -C1 : (m == 13) ? -C1 : (m == 14) ? -H : /*15*/ -S1;
        // exp(DIR i theta) = c + DIR i s
        return DIR < 0 ? make_float2(a.x * c + a.y * s, a.y * c - a.x * s) : make_float2(a.x * c - a.y * s, a.y * c + a.x * s);
    }
}

template <int DIR>
WCSIM_HD void fft2(float2 &a0, float2 &a1)
{
    float2 t = a0;
    a0 = cadd(t, a1);
    a1 = csub(t, a1);
}

// X[q] = sum_m a_m exp(DIR 2 pi i m q / 4), in place
template <int DIR>
WCSIM_HD void fft4(float2 &a0, float2 &a1, float2 &a2, float2 &a3)
{
    float2 s02 = cadd(a0, a2), d02 = csub(a0, a2), s13 = cadd(a1, a3), d13 = mul_qi<DIR>(csub(a1, a3));
    a0 = cadd(s02, s13);
    a1 = cadd(d02, d13);
    a2 = csub(s02, s13);
    a3 = csub(d02, d13);
}

// in-register radix-R transforms, natural order in and out
template <int R, int DIR>
struct Butterfly;

template <int DIR>
struct Butterfly<2, DIR> {
    static WCSIM_HD void run(float2 (&x)[2]) { fft2<DIR>(x[0], x[1]); }
};
template <int DIR>
struct Butterfly<4, DIR> {
    static WCSIM_HD void run(float2 (&x)[4]) { fft4<DIR>(x[0], x[1], x[2], x[3]); }
};
template <int DIR>
struct Butterfly<8, DIR> {
    static WCSIM_HD void run(float2 (&x)[8])
    {
        fft4<DIR>(x[0], x[2], x[4], x[6]); // E_q at x[2q]
        fft4<DIR>(x[1], x[3], x[5], x[7]); // O_q at x[2q+1]
        float2 o0 = x[1], o1 = mul_w16<DIR, 2>(x[3]), o2 = mul_w16<DIR, 4>(x[5]), o3 = mul_w16<DIR, 6>(x[7]);
        float2 e0 = x[0], e1 = x[2], e2 = x[4], e3 = x[6];
        x[0] = cadd(e0, o0); x[4] = csub(e0, o0);
        x[1] = cadd(e1, o1); x[5] = csub(e1, o1);
        x[2] = cadd(e2, o2); x[6] = csub(e2, o2);
        x[3] = cadd(e3, o3); x[7] = csub(e3, o3);
    }
};
template <int DIR>
struct Butterfly<16, DIR> {
    static WCSIM_HD void run(float2 (&x)[16])
    {
        // b[r][q] = sum_m x[r+4m] W4^{mq}, left at x[r + 4q]
        fft4<DIR>(x[0], x[4], x[8], x[12]);
        fft4<DIR>(x[1], x[5], x[9], x[13]);
        fft4<DIR>(x[2], x[6], x[10], x[14]);
        fft4<DIR>(x[3], x[7], x[11], x[15]);
        // c[r][q] = W16^{rq} b[r][q]
        x[5] = mul_w16<DIR, 1>(x[5]);   x[6] = mul_w16<DIR, 2>(x[6]);   x[7] = mul_w16<DIR, 3>(x[7]);
        x[9] = mul_w16<DIR, 2>(x[9]);   x[10] = mul_w16<DIR, 4>(x[10]); x[11] = mul_w16<DIR, 6>(x[11]);
        x[13] = mul_w16<DIR, 3>(x[13]); x[14] = mul_w16<DIR, 6>(x[14]); x[15] = mul_w16<DIR, 9>(x[15]);
        // X[q + 4s] = sum_r W4^{rs} c[r][q], left at x[4q + s]
        fft4<DIR>(x[0], x[1], x[2], x[3]);
        fft4<DIR>(x[4], x[5], x[6], x[7]);
        fft4<DIR>(x[8], x[9], x[10], x[11]);
        fft4<DIR>(x[12], x[13], x[14], x[15]);
        // transpose 4x4 to natural order: X[q + 4s] <- x[4q + s]
        float2 t;
        t = x[1];  x[1] = x[4];   x[4] = t;
        t = x[2];  x[2] = x[8];   x[8] = t;
        t = x[3];  x[3] = x[12];  x[12] = t;
        t = x[6];  x[6] = x[9];   x[9] = t;
        t = x[7];  x[7] = x[13];  x[13] = t;
        t = x[11]; x[11] = x[14]; x[14] = t;
    }
};

// w * exp(-2 pi i e / 32) for a compile-time e in 0..15: the real-row split needs exp(-2 pi i (i + e N/16) / (2N)) =
// exp(-2 pi i i / (2N)) exp(-2 pi i e / 32) at a thread's 16 points, i.e. one table load and 15 constant rotations instead
// of 16 loads (the row kernels are bound by the load/store path)
template <int EIDX, int DIR = -1>
WCSIM_HD float2 rot32(float2 w)
{
    constexpr float C[16] = {1.0f, 0.98078528040323044913f, 0.92387953251128675613f, 0.83146961230254523708f,
                             0.70710678118654752440f, 0.55557023301960222474f, 0.38268343236508977173f, 0.19509032201612826785f,
                             0.0f, -0.19509032201612826785f, -0.38268343236508977173f, -0.55557023301960222474f,
                             -0.70710678118654752440f, -0.83146961230254523708f, -0.92387953251128675613f, -0.98078528040323044913f};
    constexpr float S[16] = {0.0f, 0.19509032201612826785f, 0.38268343236508977173f, 0.55557023301960222474f,
                             0.70710678118654752440f, 0.83146961230254523708f, 0.92387953251128675613f, 0.98078528040323044913f,
                             1.0f, 0.98078528040323044913f, 0.92387953251128675613f, 0.83146961230254523708f,
                             0.70710678118654752440f, 0.55557023301960222474f, 0.38268343236508977173f, 0.19509032201612826785f};
    if constexpr (EIDX == 0) return w;
    else if constexpr (DIR < 0) return make_float2(w.x * C[EIDX] + w.y * S[EIDX], w.y * C[EIDX] - w.x * S[EIDX]); // (a + ib)(c - is)
    else return make_float2(w.x * C[EIDX] - w.y * S[EIDX], w.y * C[EIDX] + w.x * S[EIDX]);                         // (a + ib)(c + is)
}
// w * exp(-2 pi i e / 64) for a compile-time e in 0..31 (the split twiddles of a thread that keeps 32 points)
template <int EIDX>
WCSIM_HD float2 rot64(float2 w)
{
    constexpr float C[32] = {1.0f, 0.99518472667219688624f, 0.98078528040323044913f, 0.95694033573220886494f,
                             0.92387953251128675613f, 0.88192126434835502971f, 0.83146961230254523708f, 0.77301045336273696081f,
                             0.70710678118654752440f, 0.63439328416364549822f, 0.55557023301960222474f, 0.47139673682599764856f,
                             0.38268343236508977173f, 0.29028467725446236764f, 0.19509032201612826785f, 0.09801714032956060199f,
                             0.0f, -0.09801714032956060199f, -0.19509032201612826785f, -0.29028467725446236764f,
                             -0.38268343236508977173f, -0.47139673682599764856f, -0.55557023301960222474f, -0.63439328416364549822f,
                             -0.70710678118654752440f, -0.77301045336273696081f, -0.83146961230254523708f, -0.88192126434835502971f,
                             -0.92387953251128675613f, -0.95694033573220886494f, -0.98078528040323044913f, -0.99518472667219688624f};
    constexpr float S[32] = {0.0f, 0.09801714032956060199f, 0.19509032201612826785f, 0.29028467725446236764f,
                             0.38268343236508977173f, 0.47139673682599764856f, 0.55557023301960222474f, 0.63439328416364549822f,
                             0.70710678118654752440f, 0.77301045336273696081f, 0.83146961230254523708f, 0.88192126434835502971f,
                             0.92387953251128675613f, 0.95694033573220886494f, 0.98078528040323044913f, 0.99518472667219688624f,
                             1.0f, 0.99518472667219688624f, 0.98078528040323044913f, 0.95694033573220886494f,
                             0.92387953251128675613f, 0.88192126434835502971f, 0.83146961230254523708f, 0.77301045336273696081f,
                             0.70710678118654752440f, 0.63439328416364549822f, 0.55557023301960222474f, 0.47139673682599764856f,
                             0.38268343236508977173f, 0.29028467725446236764f, 0.19509032201612826785f, 0.09801714032956060199f};
    if constexpr (EIDX == 0) return w;
    else return make_float2(w.x * C[EIDX] + w.y * S[EIDX], w.y * C[EIDX] - w.x * S[EIDX]);
}
// the E split twiddles of thread i (E = 16 or 32 points per thread): tw[e] = exp(-2 pi i (i + e N/E) / (2N))
template <int E, int I = 0>
WCSIM_HD void split_twiddles(float2 (&tw)[E], float2 w0)
{
    static_assert(E == 16 || E == 32, "the row kernels keep 16 or 32 points per thread");
    if constexpr (I < E) {
        if constexpr (E == 16) tw[I] = rot32<I>(w0);
        else tw[I] = rot64<I>(w0);
        split_twiddles<E, I + 1>(tw, w0);
    }
}

// radix 32 from two radix-16 transforms of the even and odd inputs: X[q] = E_q + W32^q O_q, X[q+16] = E_q - W32^q O_q
template <int DIR, int Q = 0>
WCSIM_HD void combine32(float2 (&x)[32], const float2 (&ev)[16], const float2 (&od)[16])
{
    if constexpr (Q < 16) {
        const float2 t = rot32<Q, DIR>(od[Q]);
        x[Q] = cadd(ev[Q], t);
        x[Q + 16] = csub(ev[Q], t);
        combine32<DIR, Q + 1>(x, ev, od);
    }
}
template <int DIR>
struct Butterfly<32, DIR> {
    static WCSIM_HD void run(float2 (&x)[32])
    {
        float2 ev[16], od[16];
#pragma unroll
        for (int q = 0; q < 16; ++q) ev[q] = x[2 * q], od[q] = x[2 * q + 1];
        Butterfly<16, DIR>::run(ev);
        Butterfly<16, DIR>::run(od);
        combine32<DIR>(x, ev, od);
    }
};

constexpr int ilog2(int n) { return n <= 1 ? 0 : 1 + ilog2(n >> 1); }

// radix of the pass that starts with P points already combined: the first pass takes the odd bits, the rest are 16.
// R32 (threads that keep 32 points): a single odd bit is not spent on a radix-2 pass with a shared-memory exchange of its
// own but folded into a radix-32 first pass (N = 2.16.16.16 becomes 32.16.16: one exchange fewer).
template <int N, int P, bool R32 = false>
struct PassRadix {
    static constexpr int rem = ilog2(N) % 4;
    static constexpr int value = (P == 1 && rem != 0) ? ((R32 && rem == 1) ? 32 : (1 << rem)) : 16;
};

// shared-memory index (in float2 units) of point pt of column c: one float2*C of padding after every 16 points,
// which spreads the radix-strided writes of the first passes over all banks
// (SH = 5: one float2 after every 32 points, for the exchange that follows a radix-32 pass)
template <int C, int SH = 4>
WCSIM_HD int smem_index(int pt, int c)
{
    return (pt + (pt >> SH)) * C + c;
}
template <int N, int C>
struct SmemSize {
    static constexpr int float2s = (N + (N >> 4) + 1) * C;
};

WCSIM_HD float2 load_tw(const float2 *__restrict__ tw, int idx)
{
#ifdef __CUDA_ARCH__
    return __ldg(tw + idx);
#else
    return tw[idx];
#endif
}

// Twiddle tables, one per pass, laid out so that a warp's loads coalesce: for the pass that starts with P points
// already combined (P > 1; its radix is 16) the factor of input r of the butterfly with k = b mod P sits at
//   tw[tw_offset(N, P) + (r-1) P + k] = exp(-2 pi i r k / (16 P)),   r = 1..15, k < P.
// Lanes of a warp hold consecutive k, so each of the 15 loads touches P-contiguous entries (a flat table indexed
// r*k*step would cost up to 16 L1 wavefronts per load instead of 1-2).
constexpr int first_radix(int n) { return (ilog2(n) % 4) ? (1 << (ilog2(n) % 4)) : 16; }
constexpr int tw_offset(int n, int P)
{
    int off = 0;
    for (int p = first_radix(n); p < P; p *= 16) off += 15 * p;
    return off;
}
constexpr int tw_size(int n) { return tw_offset(n, n) > 0 ? tw_offset(n, n) : 1; }

// host-side builder of the table above (fp64 angles, rounded once)
inline void build_pass_twiddles(int n, float2 *out)
{
    int off = 0;
    for (int p = first_radix(n); p < n; p *= 16) {
        for (int r = 1; r < 16; ++r)
            for (int k = 0; k < p; ++k) {
                const double a = -2.0 * 3.14159265358979323846 * (double)r * (double)k / (16.0 * (double)p);
                out[off + (r - 1) * p + k] = make_float2((float)cos(a), (float)sin(a));
            }
        off += 15 * p;
    }
}

// One pass: twiddle + butterflies on the registers.  TWP: form eleven of the fifteen twiddles of a butterfly as products of
// the other four instead of loading all fifteen.
template <int N, int E, int R, int P, int DIR, bool TWP = true>
WCSIM_HD void fft_pass(float2 (&v)[E], int i, const float2 *__restrict__ tw)
{
    constexpr int NB = E / R;
    static_assert(NB >= 1 && NB * R == E, "radix must divide the per-thread element count");
#pragma unroll
    for (int u = 0; u < NB; ++u) {
        float2 x[R];
#pragma unroll
        for (int r = 0; r < R; ++r) x[r] = v[u + r * NB];
        if constexpr (P > 1) {
            static_assert(R == 16, "passes after the first are radix 16");
            const int b = i + u * (N / E);
            const int k = b & (P - 1);
            constexpr int off = tw_offset(N, P);
            if constexpr (!TWP) {
#pragma unroll
                for (int r = 1; r < R; ++r) {
                    float2 w = load_tw(tw, off + (r - 1) * P + k);
                    if (DIR > 0) w.y = -w.y;
                    x[r] = cmul(x[r], w);
                }
            } else {
                // The row kernels are bound by the load/store path (L1/TEX 74 % busy in `ncu`), not by arithmetic: only
                // w^1, w^2, w^4, w^8 are loaded and the other eleven powers are products of them (at most three
                // multiplications deep: ~2e-7 relative, the size of the transform's own fp32 rounding).
                float2 w[R];
#pragma unroll
                for (int r = 1; r < R; r <<= 1) {
                    w[r] = load_tw(tw, off + (r - 1) * P + k);
                    if (DIR > 0) w[r].y = -w[r].y;
                }
                w[3] = cmul(w[1], w[2]);
                w[5] = cmul(w[1], w[4]);
                w[6] = cmul(w[2], w[4]);
                w[7] = cmul(w[3], w[4]);
#pragma unroll
                for (int r = 1; r < 8; ++r) w[8 + r] = cmul(w[r], w[8]);
#pragma unroll
                for (int r = 1; r < R; ++r) x[r] = cmul(x[r], w[r]);
            }
        }
        Butterfly<R, DIR>::run(x);
#pragma unroll
        for (int r = 0; r < R; ++r) v[u + r * NB] = x[r];
    }
}

// Stockham scatter of a finished pass into shared memory: butterfly b, output r goes to point (b-k)R + k + rP
template <int N, int C, int E, int R, int P, int SH = 4>
WCSIM_HD void fft_store(const float2 (&v)[E], float2 *smem, int i, int c)
{
    constexpr int NB = E / R;
#pragma unroll
    for (int u = 0; u < NB; ++u) {
        const int b = i + u * (N / E);
        const int k = b & (P - 1);
        const int j = (b - k) * R + k;
#pragma unroll
        for (int r = 0; r < R; ++r) smem[smem_index<C, SH>(j + r * P, c)] = v[u + r * NB];
    }
}

// gather of the next pass's inputs: points i + e*(N/E)
template <int N, int C, int E, int SH = 4>
WCSIM_HD void fft_load(float2 (&v)[E], const float2 *smem, int i, int c)
{
#pragma unroll
    for (int e = 0; e < E; ++e) v[e] = smem[smem_index<C, SH>(i + e * (N / E), c)];
}

#ifdef __CUDACC__
// Whole transform from registers to registers (device only: uses __syncthreads).  On entry v holds the input at
// points i + e*(N/E); on exit it holds the transform at the same points.  `smem` has SmemSize<N,C>::float2s
// entries.  SYNC_FIRST: set when other threads may still be reading `smem` from earlier work.
template <int N, int C, int E, int DIR, int P = 1, bool R32 = false>
__device__ __forceinline__ void fft_block(float2 (&v)[E], float2 *smem, int i, int c, const float2 *__restrict__ tw,
                                          bool sync_first)
{
    constexpr int R = PassRadix<N, P, R32>::value;
    constexpr int SH = R32 ? 5 : 4;
    // twiddles by products where loads are what binds: the row transforms (a warp's lanes are 32 different k) and the long
    // column transforms; the short column transforms (few distinct k per warp: cheap loads) keep their 15 loads
    // (measured: 512-point columns 13.5 us with loads, 17.4 us with products; 1024: 55.6 / 47.5 us; 4096: 598 / 528 us)
    fft_pass<N, E, R, P, DIR, (C == 1 || N >= 1024)>(v, i, tw);
    if constexpr (P * R < N) {
        if (P > 1 || sync_first) __syncthreads();
        fft_store<N, C, E, R, P, SH>(v, smem, i, c);
        __syncthreads();
        fft_load<N, C, E, SH>(v, smem, i, c);
        fft_block<N, C, E, DIR, P * R, R32>(v, smem, i, c, tw, true);
    }
}
#endif

} // namespace wcsim

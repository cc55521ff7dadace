// raster.cu -- steps a1-a3 of the hot path: Raster, charge fluctuation, Scatter-add
// (Section 2.2; Section 3.1 for the binomial fluctuation).
//
// One warp owns one depo at a time (the SoA layout of PAPER.md:72 makes the depo the unit of parallelism).  The
// lanes evaluate erf at consecutive bin edges of one axis, a shuffle turns neighbouring edges into bin weights
// ("erf bin edges once per axis"), and the patch p_ij = wt_i wx_j is formed in registers: lanes run along the tick
// axis (contiguous in S), the wire index is broadcast by shuffle.  Nothing of the patch is ever written to HBM
// except the final adds into S.
//
//   fluctuate = 0: fp32 weights (erff), value q * (wt * wx)
//   fluctuate = 1: fp64 weights (erf), p = wt * wx, integer draw B(N, p; Philox word of the absolute bin)
//
// Two scatter modes:
//   atomic: red.global.add.f32 straight into S
//   tiled : depos are grouped by the grid tiles their patch overlaps (count / scan / fill), one CTA per tile
//           accumulates its depos in shared memory in 2^-24 fixed point (integer adds: order independent, so the
//           result is bitwise reproducible) and adds the tile to S once.
#include "internal.h"
#include "rng.cuh"
#include <type_traits>

namespace wcsim {

namespace {

constexpr int kChunk = 31;             // bins per warp pass on one axis (32 edges)
constexpr int kTileW = 16, kTileT = 256;
constexpr double kFixScale = 16777216.0; // 2^24

struct Extent {
    int lo, hi; // clipped [lo, hi); empty if lo >= hi
};

// floor(c - n s) .. floor(c + n s) + 1 (A2), clipped to [clip_lo, clip_hi); every operation rounded separately
__device__ __forceinline__ Extent axis_extent(double centre, double sigma, double nsigma, int clip_lo, int clip_hi)
{
    const double h = __dmul_rn(nsigma, sigma);
    double lo = floor(__dsub_rn(centre, h));
    double hi = __dadd_rn(floor(__dadd_rn(centre, h)), 1.0);
    lo = fmax(lo, (double)clip_lo);
    hi = fmin(hi, (double)clip_hi);
    Extent e;
    if (lo < hi) {
        e.lo = (int)lo;
        e.hi = (int)hi;
    } else {
        e.lo = 0;
        e.hi = 0;
    }
    return e;
}

__device__ __forceinline__ bool depo_valid(float t0, float x0, float st, float sx, float q)
{
    return isfinite(t0) && isfinite(x0) && isfinite(st) && isfinite(sx) && isfinite(q) && st >= 0.0f && sx >= 0.0f;
}

// weights of bins base .. base+30 in lanes 0 .. 30:  1/2 [erf((i+1-c)/(sqrt2 s)) - erf((i-c)/(sqrt2 s))]   (A1, A4)
template <typename T>
__device__ __forceinline__ T axis_weights(int base, double centre, double sigma, int lane)
{
    T w;
    if (sigma < 1e-6) { // uniform over the warp
        w = (floor(centre) == (double)(base + lane)) ? T(1) : T(0);
    } else {
        T E;
        const double d = __dsub_rn((double)(base + lane), centre);
        if constexpr (sizeof(T) == 8) {
            const double s = __dmul_rn(1.4142135623730951, sigma);
            E = erf(__ddiv_rn(d, s));
        } else {
            const float inv = 1.0f / (1.41421356f * (float)sigma);
            E = erff((float)d * inv);
        }
        const T Eh = __shfl_down_sync(0xffffffffu, E, 1);
        w = T(0.5) * (Eh - E);
    }
    return w;
}

struct GlobalSink {
    float *S;
    int n_ticks;
    __device__ __forceinline__ void add(int wire, int tick, float v) const
    {
        atomicAdd(S + (size_t)wire * n_ticks + tick, v); // result unused -> RED.E.ADD.F32
    }
};

struct TileSink {
    unsigned long long *acc; // shared memory, [kTileW][kTileT]
    int w0, k0;
    __device__ __forceinline__ void add(int wire, int tick, float v) const
    {
        const long long q = __double2ll_rn((double)v * kFixScale);
        atomicAdd(acc + (wire - w0) * kTileT + (tick - k0), (unsigned long long)q);
    }
};

// Rasters depo (t0, x0, st, sx, q) into the clip window [w_lo, w_hi) x [k_lo, k_hi) (already inside the grid).
// Returns the number of bins this lane deposited; *lane_total accumulates the lane's signed draws.
template <bool FLUCT, typename Sink>
__device__ __forceinline__ unsigned int raster_depo(float t0f, float x0f, float stf, float sxf, float qf, uint64_t id,
                                                    uint64_t seed, double nsigma, int n_ticks, int w_lo, int w_hi,
                                                    int k_lo, int k_hi, const Sink &sink, int lane, int *lane_total)
{
    using T = typename std::conditional<FLUCT, double, float>::type;
    const double T0 = t0f, X0 = x0f, ST = stf, SX = sxf;
    const Extent et = axis_extent(T0, ST, nsigma, k_lo, k_hi);
    const Extent ex = axis_extent(X0, SX, nsigma, w_lo, w_hi);
    if (et.lo >= et.hi || ex.lo >= ex.hi) return 0;
    const double Ntr = floor(fabs((double)qf) + 0.5);
    const double sgn = (qf < 0.0f) ? -1.0 : 1.0;
    unsigned int drawn = 0;
    for (int xc = ex.lo; xc < ex.hi; xc += kChunk) {
        const T wx = axis_weights<T>(xc, X0, SX, lane);
        const int nj = min(kChunk, ex.hi - xc);
        for (int tc = et.lo; tc < et.hi; tc += kChunk) {
            const T wt = axis_weights<T>(tc, T0, ST, lane);
            const int tick = tc + lane;
            const bool act = lane < kChunk && tick < et.hi;
            for (int j = 0; j < nj; ++j) {
                const T wxj = __shfl_sync(0xffffffffu, wx, j);
                if (act) {
                    const int wire = xc + j;
                    ++drawn;
                    if constexpr (FLUCT) {
                        const double p = __dmul_rn(wt, wxj);
                        const uint64_t g = (uint64_t)wire * (uint64_t)n_ticks + (uint64_t)tick;
                        const uint4 words = fluct_words(seed, id, g >> 2);
                        const double k = binomial_draw(Ntr, p, pick_word(words, (uint32_t)g & 3u));
                        if (k != 0.0) {
                            const double v = sgn * k;
                            *lane_total += (int)v;
                            sink.add(wire, tick, (float)v);
                        }
                    } else {
                        sink.add(wire, tick, qf * (wt * wxj));
                    }
                }
            }
        }
    }
    return drawn;
}

__device__ __forceinline__ int warp_sum(int v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ unsigned long long warp_sum(unsigned long long v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// ------------------------------------------------------------------------------------------------------------------
// atomic mode: persistent grid, warp w takes depos w, w + n_warps, ...
// ------------------------------------------------------------------------------------------------------------------
template <bool FLUCT>
__global__ void __launch_bounds__(256) raster_atomic_kernel(GridDims g, DepoArrays d, long long n, uint64_t id_base,
                                                            uint64_t seed, double nsigma, float *__restrict__ S,
                                                            int *__restrict__ totals, Counters *counters)
{
    const int lane = threadIdx.x & 31;
    const long long warp = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const long long n_warps = ((long long)gridDim.x * blockDim.x) >> 5;
    const GlobalSink sink{S, g.n_ticks};
    unsigned long long drawn = 0, skipped = 0;
    for (long long i = warp; i < n; i += n_warps) {
        const float t0 = __ldg(d.t0 + i), x0 = __ldg(d.x0 + i), st = __ldg(d.sigma_t + i), sx = __ldg(d.sigma_x + i),
                    q = __ldg(d.q + i);
        int tot = 0;
        if (depo_valid(t0, x0, st, sx, q)) {
            drawn += raster_depo<FLUCT>(t0, x0, st, sx, q, id_base + (uint64_t)i, seed, nsigma, g.n_ticks, 0, g.n_wires,
                                        0, g.n_ticks, sink, lane, &tot);
        } else {
            skipped += (lane == 0);
        }
        if (totals != nullptr) {
            tot = warp_sum(tot);
            if (lane == 0) totals[i] = tot;
        }
    }
    drawn = warp_sum(drawn);
    skipped = warp_sum(skipped);
    if (lane == 0) {
        if (drawn) atomicAdd(&counters->bins_drawn, drawn);
        if (skipped) atomicAdd(&counters->depos_skipped, skipped);
    }
}

// ------------------------------------------------------------------------------------------------------------------
// tiled mode
// ------------------------------------------------------------------------------------------------------------------
struct TileRange {
    int w0, w1, t0, t1; // tile index ranges [w0, w1] x [t0, t1]; empty if w0 > w1
};

__device__ __forceinline__ TileRange depo_tiles(GridDims g, DepoArrays d, long long i, double nsigma)
{
    TileRange r{0, -1, 0, -1};
    const float t0 = __ldg(d.t0 + i), x0 = __ldg(d.x0 + i), st = __ldg(d.sigma_t + i), sx = __ldg(d.sigma_x + i),
                q = __ldg(d.q + i);
    if (!depo_valid(t0, x0, st, sx, q)) return r;
    const Extent et = axis_extent(t0, st, nsigma, 0, g.n_ticks);
    const Extent ex = axis_extent(x0, sx, nsigma, 0, g.n_wires);
    if (et.lo >= et.hi || ex.lo >= ex.hi) return r;
    r.w0 = ex.lo / kTileW;
    r.w1 = (ex.hi - 1) / kTileW;
    r.t0 = et.lo / kTileT;
    r.t1 = (et.hi - 1) / kTileT;
    return r;
}

__global__ void tile_count_kernel(GridDims g, DepoArrays d, long long n, double nsigma, TileScratch ts)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const TileRange r = depo_tiles(g, d, i, nsigma);
    for (int tw = r.w0; tw <= r.w1; ++tw)
        for (int tt = r.t0; tt <= r.t1; ++tt) atomicAdd(ts.tile_count + (size_t)tw * ts.tiles_t + tt, 1u);
}

// exclusive scan of tile_count[0..n_tiles) in place, tile_count[n_tiles] = total, cursors = offsets; one CTA
__global__ void __launch_bounds__(1024) tile_scan_kernel(TileScratch ts)
{
    __shared__ unsigned int warp_tot[32];
    __shared__ unsigned int carry;
    const int n_tiles = ts.tiles_w * ts.tiles_t;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (int base = 0; base < n_tiles; base += 1024) {
        const int i = base + threadIdx.x;
        const unsigned int v = (i < n_tiles) ? ts.tile_count[i] : 0u;
        unsigned int incl = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const unsigned int t = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += t;
        }
        if (lane == 31) warp_tot[wid] = incl;
        __syncthreads();
        if (wid == 0) {
            unsigned int w = warp_tot[lane];
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const unsigned int t = __shfl_up_sync(0xffffffffu, w, o);
                if (lane >= o) w += t;
            }
            warp_tot[lane] = w; // inclusive over warps
        }
        __syncthreads();
        const unsigned int before = carry + (wid ? warp_tot[wid - 1] : 0u) + incl - v;
        if (i < n_tiles) {
            ts.tile_count[i] = before;
            ts.tile_cursor[i] = before;
        }
        __syncthreads();
        if (threadIdx.x == 0) carry += warp_tot[31];
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        ts.tile_count[n_tiles] = carry;
        *ts.total = carry;
    }
}

__global__ void tile_fill_kernel(GridDims g, DepoArrays d, long long n, double nsigma, TileScratch ts)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const TileRange r = depo_tiles(g, d, i, nsigma);
    for (int tw = r.w0; tw <= r.w1; ++tw)
        for (int tt = r.t0; tt <= r.t1; ++tt) {
            const unsigned int pos = atomicAdd(ts.tile_cursor + (size_t)tw * ts.tiles_t + tt, 1u);
            if (pos < ts.capacity) ts.entries[pos] = (unsigned int)i;
        }
}

template <bool FLUCT>
__global__ void __launch_bounds__(256) tile_accumulate_kernel(GridDims g, DepoArrays d, uint64_t id_base, uint64_t seed,
                                                              double nsigma, TileScratch ts, float *__restrict__ S,
                                                              int *__restrict__ totals, Counters *counters)
{
    __shared__ unsigned long long acc[kTileW * kTileT];
    const int tile = blockIdx.x;
    const unsigned int beg = ts.tile_count[tile], end = ts.tile_count[tile + 1];
    if (beg == end) return; // uniform over the CTA
    const int tw = tile / ts.tiles_t, tt = tile % ts.tiles_t;
    const int w0 = tw * kTileW, k0 = tt * kTileT;
    const int w1 = min(w0 + kTileW, g.n_wires), k1 = min(k0 + kTileT, g.n_ticks);
    for (int i = threadIdx.x; i < kTileW * kTileT; i += blockDim.x) acc[i] = 0ull;
    __syncthreads();
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, n_warps = blockDim.x >> 5;
    const TileSink sink{acc, w0, k0};
    unsigned long long drawn = 0;
    for (unsigned int e = beg + wid; e < end; e += n_warps) {
        const unsigned int i = ts.entries[e];
        const float t0 = __ldg(d.t0 + i), x0 = __ldg(d.x0 + i), st = __ldg(d.sigma_t + i), sx = __ldg(d.sigma_x + i),
                    q = __ldg(d.q + i);
        int tot = 0;
        drawn += raster_depo<FLUCT>(t0, x0, st, sx, q, id_base + (uint64_t)i, seed, nsigma, g.n_ticks, w0, w1, k0, k1,
                                    sink, lane, &tot);
        if (totals != nullptr) {
            tot = warp_sum(tot);
            if (lane == 0 && tot != 0) atomicAdd(totals + i, tot);
        }
    }
    drawn = warp_sum(drawn);
    if (lane == 0 && drawn) atomicAdd(&counters->bins_drawn, drawn);
    __syncthreads();
    for (int i = threadIdx.x; i < kTileW * kTileT; i += blockDim.x) {
        const int w = w0 + i / kTileT, k = k0 + i % kTileT;
        const long long q = (long long)acc[i];
        if (q != 0 && w < w1 && k < k1) {
            float *p = S + (size_t)w * g.n_ticks + k;
            *p = *p + (float)((double)q * (1.0 / kFixScale));
        }
    }
}

// counts depos skipped as invalid (tiled mode; the atomic kernel counts them itself)
__global__ void count_invalid_kernel(DepoArrays d, long long n, Counters *counters)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const bool bad = (i < n) && !depo_valid(__ldg(d.t0 + i), __ldg(d.x0 + i), __ldg(d.sigma_t + i),
                                            __ldg(d.sigma_x + i), __ldg(d.q + i));
    const unsigned int m = __ballot_sync(0xffffffffu, bad);
    if ((threadIdx.x & 31) == 0 && m) atomicAdd(&counters->depos_skipped, (unsigned long long)__popc(m));
}

} // namespace

cudaError_t launch_raster_atomic(GridDims g, DepoArrays d, long long n, uint64_t id_base, uint64_t seed, int fluctuate,
                                 double nsigma, float *S, int *depo_totals, Counters *counters, int sm_count,
                                 cudaStream_t st)
{
    if (n <= 0) return cudaSuccess;
    const int threads = 256, warps_per_cta = threads / 32;
    long long ctas = (n + warps_per_cta - 1) / warps_per_cta;
    const long long max_ctas = (long long)sm_count * 8; // 2048 threads per SM resident
    if (ctas > max_ctas) ctas = max_ctas;
    if (fluctuate)
        raster_atomic_kernel<true><<<(unsigned)ctas, threads, 0, st>>>(g, d, n, id_base, seed, nsigma, S, depo_totals,
                                                                      counters);
    else
        raster_atomic_kernel<false><<<(unsigned)ctas, threads, 0, st>>>(g, d, n, id_base, seed, nsigma, S, depo_totals,
                                                                       counters);
    return cudaGetLastError();
}

cudaError_t launch_tile_count(GridDims g, DepoArrays d, long long n, double nsigma, TileScratch ts, cudaStream_t st)
{
    if (n <= 0) return cudaSuccess;
    tile_count_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(g, d, n, nsigma, ts);
    return cudaGetLastError();
}

cudaError_t launch_tile_scan(TileScratch ts, cudaStream_t st)
{
    tile_scan_kernel<<<1, 1024, 0, st>>>(ts);
    return cudaGetLastError();
}

cudaError_t launch_tile_fill(GridDims g, DepoArrays d, long long n, double nsigma, TileScratch ts, cudaStream_t st)
{
    if (n <= 0) return cudaSuccess;
    tile_fill_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(g, d, n, nsigma, ts);
    return cudaGetLastError();
}

cudaError_t launch_tile_accumulate(GridDims g, DepoArrays d, uint64_t id_base, uint64_t seed, int fluctuate,
                                   double nsigma, TileScratch ts, float *S, int *depo_totals, Counters *counters,
                                   cudaStream_t st)
{
    const int n_tiles = ts.tiles_w * ts.tiles_t;
    if (fluctuate)
        tile_accumulate_kernel<true><<<n_tiles, 256, 0, st>>>(g, d, id_base, seed, nsigma, ts, S, depo_totals, counters);
    else
        tile_accumulate_kernel<false><<<n_tiles, 256, 0, st>>>(g, d, id_base, seed, nsigma, ts, S, depo_totals, counters);
    return cudaGetLastError();
}

cudaError_t launch_count_invalid(DepoArrays d, long long n, Counters *counters, cudaStream_t st)
{
    if (n <= 0) return cudaSuccess;
    count_invalid_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(d, n, counters);
    return cudaGetLastError();
}

void tile_shape(int *tile_w, int *tile_t)
{
    *tile_w = kTileW;
    *tile_t = kTileT;
}

} // namespace wcsim

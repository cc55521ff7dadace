// raster.cu -- steps a1-a3 of the hot path: Raster, charge fluctuation, Scatter-add
// (Section 2.2; Section 3.1 for the binomial fluctuation).
//
// Every scatter mode runs the same batch bodies (raster_flat_body with fluctuation off, raster_quad_body with it on): a warp
// takes a batch of 16 depos, one per lane (the SoA layout of PAPER.md:72 makes the depo the unit of parallelism and the
// loads coalesce; lanes 16..31 own none).  Each owning lane works out its depo's patch extent, clipped to the batch's
// window (the plane, or a tile of it); a warp scan lays all bin EDGES of the batch's patches end to end and all 32 lanes
// evaluate erf over that flat list ("erf bin edges once per axis"; own table erf, erf_table.cuh), leaving the values in
// the warp's shared-memory scratch; then the lanes walk the flat list of the batch's BINS (fluctuation off) or QUADS
// (on: aligned groups of four absolute bins, one Philox call each), 32 at a time, forming p_ij = wt_i wx_j from four edge
// values.  All lanes are busy whatever the patch shapes are (patches are 1-5 wires x 1-16 ticks in BASELINE.json's
// configs).  With fluctuation on, bins are sorted by the routine that will draw them (rounded normal / inversion in three
// mu bands / exact) into five per-warp shared-memory queues and drawn 32 at a time from one queue by straight-line code:
// guarded fp32 estimates first (rng.cuh), the fp64 routines for the ~1 % of bins a guard does not accept.
// A patch with more edges than the scratch holds falls back to the one-warp-per-depo walk (raster_depo), which chunks
// it.  Nothing of a patch is ever written to HBM except the final adds into S.
//
// raster_depo (patches too big for the scratch): one warp owns one depo.  The lanes evaluate erf at consecutive bin
// edges of one axis, a shuffle turns neighbouring edges into bin weights, lanes run along the tick axis (contiguous in
// S), the wire index is broadcast by shuffle.
//
//   fluctuate = 0: fp32 weights (erff), value q * (wt * wx)
//   fluctuate = 1: fp64 weights (erf), p = wt * wx, integer draw B(N, p; Philox word of the absolute bin)
//   fluctuate = 2: the same with the normal-approximation draw of the paper's Kokkos port (reading A21)
//
// Scatter modes:
//   atomic: raster_batch_kernel, persistent warps: two batches by the warp's index in the grid, then batches of 4 depos
//           from a device counter (guided scheduling); fp32 reductions (REDG.E.ADD.F32) straight into S.
//           raster_planes_kernel: the same for the stacked planes of a multi-plane plan, one launch for all planes.
//   fixed : the atomic kernel adding in 2^-24 fixed point into a 64-bit grid (integer reductions: order independent, so the
//           result is bitwise reproducible), folded into S by tile_finalize_kernel.
//   tiled : depos are listed under the (at most 4) grid tiles their patch overlaps (count / scan / fill), up to 8 CTAs per
//           tile run the batch body over its depos, clipped to the tile, accumulating in shared memory in 2^-24 fixed point
//           and adding the tile into the fixed-point grid once; patches over more than 4 tiles go through the atomic kernel
//           into the same grid; everything stream-ordered.
#include "internal.h"
#include "erf_table.cuh"
#include "pdl.cuh"
#include "rng.cuh"
#include <type_traits>
#include <mutex>
#include <cstdio>
#include <cstdlib>

namespace wcsim {

namespace {

__device__ double g_erf_tab[(kErfDegree + 1) * kErfIntervals]; // erf_table.cuh; filled by raster_configure()

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

// sum of the axis weights over the whole extent floor(c - n s) .. floor(c + n s) + 1, from its two outer edges (A24)
__device__ __forceinline__ double axis_norm(double centre, double sigma, double nsigma)
{
    if (sigma < 1e-6) return 1.0;
    const double h = __dmul_rn(nsigma, sigma), s = 1.4142135623730951 * sigma;
    const double lo = floor(__dsub_rn(centre, h)), hi = __dadd_rn(floor(__dadd_rn(centre, h)), 1.0);
    return 0.5 * (erf_from_table(g_erf_tab, fast_div(hi - centre, s)) - erf_from_table(g_erf_tab, fast_div(lo - centre, s)));
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
            E = erf_from_table(g_erf_tab, __ddiv_rn(d, s));
        } else {
            const float inv = 1.0f / (1.41421356f * (float)sigma);
            E = erff((float)d * inv);
        }
        const T Eh = __shfl_down_sync(0xffffffffu, E, 1);
        w = T(0.5) * (Eh - E);
    }
    return w;
}

// Where a bin's value goes.  index() is the code of a bin kept in the draw queues (< 2^30), add_at() the accumulation.
struct GlobalSink {
    float *S;
    int n_ticks;
    __device__ __forceinline__ uint32_t index(int wire, int tick) const
    {
        return (uint32_t)wire * (uint32_t)n_ticks + (uint32_t)tick;
    }
    __device__ __forceinline__ void add_at(uint32_t idx, float v) const
    {
        atomicAdd(S + idx, v); // result unused -> RED.E.ADD.F32
    }
    __device__ __forceinline__ void add(int wire, int tick, float v) const { add_at(index(wire, tick), v); }
    __device__ __forceinline__ GlobalSink shifted(int rows) const { return GlobalSink{S + (size_t)rows * n_ticks, n_ticks}; }
};

// the same adds in 2^-24 fixed point into a 64-bit grid (RED.ADD.64: order independent); tile_finalize_kernel folds it into S
struct FixSink {
    unsigned long long *fix;
    int n_ticks;
    __device__ __forceinline__ uint32_t index(int wire, int tick) const
    {
        return (uint32_t)wire * (uint32_t)n_ticks + (uint32_t)tick;
    }
    __device__ __forceinline__ void add_at(uint32_t idx, float v) const
    {
        atomicAdd(fix + idx, (unsigned long long)__double2ll_rn((double)v * kFixScale));
    }
    __device__ __forceinline__ void add(int wire, int tick, float v) const { add_at(index(wire, tick), v); }
    __device__ __forceinline__ FixSink shifted(int rows) const { return FixSink{fix + (size_t)rows * n_ticks, n_ticks}; }
};

template <bool FIX>
__device__ __forceinline__ auto make_grid_sink(float *grid, int n_ticks)
{
    if constexpr (FIX) return FixSink{reinterpret_cast<unsigned long long *>(grid), n_ticks};
    else return GlobalSink{grid, n_ticks};
}

struct TileSink {
    unsigned long long *acc; // shared memory, [kTileW][kTileT]
    int w0, k0;
    __device__ __forceinline__ uint32_t index(int wire, int tick) const
    {
        return (uint32_t)((wire - w0) * kTileT + (tick - k0));
    }
    __device__ __forceinline__ void add_at(uint32_t idx, float v) const
    {
        // a 64-bit shared-memory atomic add is a compare-and-swap loop (ATOMS.CAST.SPIN.64); two native 32-bit adds with
        // the carry of the low word do the same sum modulo 2^64, in any order
        const unsigned long long q = (unsigned long long)__double2ll_rn((double)v * kFixScale);
        const unsigned int lo = (unsigned int)q, hi = (unsigned int)(q >> 32);
        unsigned int *a = reinterpret_cast<unsigned int *>(acc + idx); // little endian: a[0] low word
        const unsigned int old = atomicAdd(a, lo);
        const unsigned int h = hi + ((old + lo < old) ? 1u : 0u);
        if (h) atomicAdd(a + 1, h);
    }
    __device__ __forceinline__ void add(int wire, int tick, float v) const { add_at(index(wire, tick), v); }
    __device__ __forceinline__ TileSink shifted(int) const { return *this; } // tiles belong to one plane
};

// the clip window of a batch: the plane, or one tile of it.  row_off: the plane's first row in a stacked multi-plane grid
// (wire indices, Philox bins and the window are the plane's own; only the sink index carries the offset)
struct Clip {
    int w_lo, w_hi, k_lo, k_hi;
    int row_off = 0;
};

// Rasters depo (t0, x0, st, sx, q) into the clip window [w_lo, w_hi) x [k_lo, k_hi) (already inside the grid).
// Returns the number of bins this lane deposited; *lane_total accumulates the lane's signed draws.
template <bool FLUCT, typename Sink>
__device__ __noinline__ unsigned int raster_depo(float t0f, float x0f, float stf, float sxf, float qf, uint64_t id,
                                                    uint64_t seed, double nsigma, int n_ticks, int w_lo, int w_hi,
                                                    int k_lo, int k_hi, const Sink &sink, int lane, int *lane_total,
                                                    bool normal_only, double inv_norm)
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
                        const double p = __dmul_rn(wt, wxj) * inv_norm; // inv_norm = 1 unless patches are renormalised (A24)
                        const uint64_t g = (uint64_t)wire * (uint64_t)n_ticks + (uint64_t)tick;
                        const uint4 words = fluct_words(seed, id, g >> 2);
                        const double k = binomial_draw(Ntr, p, pick_word(words, (uint32_t)g & 3u), normal_only);
                        if (k != 0.0) {
                            const double v = sgn * k;
                            *lane_total += (int)v;
                            sink.add(wire, tick, (float)v);
                        }
                    } else {
                        sink.add(wire, tick, qf * (wt * wxj) * (float)inv_norm);
                    }
                }
            }
        }
    }
    return drawn;
}

// ---- tiles of the deterministic sort-by-tile mode (the kernels are further down) ----
constexpr int kSliceEntries = 256;  // listed depos per slice of a hot tile, at least
constexpr int kMaxListedTiles = 4; // a depo is listed in at most this many tiles; bigger patches go through the fixed-point grid
struct TileRange {
    int w0, w1, t0, t1; // tile index ranges [w0, w1] x [t0, t1]; empty if w0 > w1
    __device__ __forceinline__ int count() const { return w0 > w1 || t0 > t1 ? 0 : (w1 - w0 + 1) * (t1 - t0 + 1); }
};
__device__ __forceinline__ TileRange depo_tile_range(GridDims g, float t0, float x0, float st, float sx, float q, double nsigma)
{
    TileRange r{0, -1, 0, -1};
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
// the tiles a depo is LISTED in: none if it touches more than kMaxListedTiles
__device__ __forceinline__ TileRange depo_tiles(GridDims g, DepoArrays d, long long i, double nsigma)
{
    TileRange r = depo_tile_range(g, __ldg(d.t0 + i), __ldg(d.x0 + i), __ldg(d.sigma_t + i), __ldg(d.sigma_x + i),
                                  __ldg(d.q + i), nsigma);
    if (r.count() > kMaxListedTiles) r = TileRange{0, -1, 0, -1};
    return r;
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
// batches: a warp takes kBatchDepos depos at a time, one per lane
// ------------------------------------------------------------------------------------------------------------------
constexpr int kBatchWarps = 4;          // warps per CTA
#ifndef WCSIM_BATCH_SHIFT
#define WCSIM_BATCH_SHIFT 4
#endif
#ifndef WCSIM_FLUCT_CTAS
#define WCSIM_FLUCT_CTAS 5
#endif
constexpr int kBatchShift = WCSIM_BATCH_SHIFT;          // log2 of the depos a warp fetches at a time (lanes beyond that own no depo):
constexpr int kBatchDepos = 1 << kBatchShift; // small batches keep the per-warp serial path short and the load balanced
constexpr int kTailDepos = 4, kTailPerWarp = 2; // guided scheduling of the last batches (raster_batch_kernel)
constexpr uint32_t kBinMirror = 1u << 30, kBinNegative = 1u << 31, kBinMask = kBinMirror - 1u; // grid < 2^30 bins

// largest d in [0, kBatchDepos) with off[d] <= x (off is an exclusive prefix over the depos of a batch; entries from
// kBatchDepos on all hold the total, which is > x)
__device__ __forceinline__ int owner_of(const int *off, int x)
{
    int lo = 0;
#pragma unroll
    for (int step = kBatchDepos / 2; step > 0; step >>= 1)
        if (off[lo + step] <= x) lo += step;
    return lo;
}

__device__ __forceinline__ int warp_incl_scan(int v, int lane)
{
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, v, o);
        if (lane >= o) v += t;
    }
    return v;
}

// ---- fluctuation off: flat lists of edges and of bins -----------------------------------------------------------
constexpr int kEdgeCap = 128; // edge values per warp scratch (8 patches of 16 x 5 bins need 184: two sub-batches)
struct FlatScratch {
    float edge[kEdgeCap];
    int eoff[33], boff[33];
};

// One batch of up to kBatchDepos depos, one per lane (lane l < count owns a depo, the others own none), fluctuation off:
// extents clipped to `clip`, erf at the flat list of all bin edges, then q wt_i wx_j over the flat list of all bins.
// Shared by the atomic kernel (clip = the grid, sink = S) and the tiled kernel (clip = a tile, sink = the tile's
// fixed-point accumulators).
template <typename Sink>
__device__ __forceinline__ void raster_flat_body(GridDims g, Clip clip, const Sink &sink, float t0, float x0, float st,
                                                 float sx, float q, bool valid, double nsigma, bool normalize,
                                                 FlatScratch &sc, unsigned int &drawn, int lane)
{
    const double T0 = t0, X0 = x0, ST = st, SX = sx;
    Extent et{0, 0}, ex{0, 0};
    if (valid) {
        et = axis_extent(T0, ST, nsigma, clip.k_lo, clip.k_hi);
        ex = axis_extent(X0, SX, nsigma, clip.w_lo, clip.w_hi);
    }
    const bool live = et.lo < et.hi && ex.lo < ex.hi;
    // renormalised patches (reading A24): 1 / (W_t W_x), W = the axis weights summed over the whole, unclipped extent
    double inv_norm = 1.0;
    if (normalize && live) inv_norm = __ddiv_rn(1.0, axis_norm(T0, ST, nsigma) * axis_norm(X0, SX, nsigma));
    const int nt = live ? et.hi - et.lo : 0, nx = live ? ex.hi - ex.lo : 0;
    const bool big = nt + nx + 2 > kEdgeCap || (long long)nt * nx > (1 << 24);
    const int ne = (live && !big) ? nt + nx + 2 : 0, nb = (live && !big) ? nt * nx : 0;
    const int eincl = warp_incl_scan(ne, lane), bincl = warp_incl_scan(nb, lane);
    __syncwarp();
    sc.eoff[lane] = eincl - ne;
    sc.boff[lane] = bincl - nb;
    if (lane == 31) {
        sc.eoff[32] = eincl;
        sc.boff[32] = bincl;
    }
    __syncwarp();
    drawn += (unsigned int)nb;

    // patches too big for the scratch: the whole warp walks them one at a time
    unsigned int big_mask = __ballot_sync(0xffffffffu, live && big);
    while (big_mask) {
        const int src = __ffs(big_mask) - 1;
        big_mask &= big_mask - 1;
        int tot = 0;
        drawn += raster_depo<false>(__shfl_sync(0xffffffffu, t0, src), __shfl_sync(0xffffffffu, x0, src),
                                    __shfl_sync(0xffffffffu, st, src), __shfl_sync(0xffffffffu, sx, src),
                                    __shfl_sync(0xffffffffu, q, src), 0ull, 0ull, nsigma, g.n_ticks, clip.w_lo, clip.w_hi,
                                    clip.k_lo, clip.k_hi, sink, lane, &tot, false,
                                    normalize ? __shfl_sync(0xffffffffu, inv_norm, src) : 1.0);
    }

    // sub-batches of consecutive depos whose edges fit the scratch (normally all at once)
    int d0 = 0;
    while (d0 < 32) {
        const int ebase = sc.eoff[d0];
        const unsigned int fits = __ballot_sync(0xffffffffu, lane >= d0 && eincl - ebase <= kEdgeCap);
        const int d1 = d0 + __popc(fits); // eincl is monotone: the fitting lanes are d0 .. d1-1, at least one
        const int etot = sc.eoff[d1] - ebase, bbase = sc.boff[d0], btot = sc.boff[d1] - bbase;
        // ---- edges: erf((edge - centre) / (sqrt2 sigma)), flat over the sub-batch -------------------------------
        for (int e0 = 0; e0 < etot; e0 += 32) {
            const int e = e0 + lane;
            const bool act = e < etot;
            const int own = owner_of(sc.eoff, ebase + (act ? e : 0));
            const int le = ebase + e - sc.eoff[own];
            const int nto = __shfl_sync(0xffffffffu, nt, own);
            const bool on_t = le <= nto;
            const int lo_t = __shfl_sync(0xffffffffu, et.lo, own), lo_x = __shfl_sync(0xffffffffu, ex.lo, own);
            const float ct = __shfl_sync(0xffffffffu, t0, own), cx = __shfl_sync(0xffffffffu, x0, own);
            const float sgt = __shfl_sync(0xffffffffu, st, own), sgx = __shfl_sync(0xffffffffu, sx, own);
            const double centre = (double)(on_t ? ct : cx), sigma = (double)(on_t ? sgt : sgx);
            const int coord = on_t ? lo_t + le : lo_x + (le - nto - 1);
            float E;
            if (sigma < 1e-6) { // all weight in bin floor(centre) (A4): a step from -1 to +1 after that bin's low edge
                E = ((double)coord <= floor(centre)) ? -1.0f : 1.0f;
            } else {
                const double dd = __dsub_rn((double)coord, centre);
                const float inv = 1.0f / (1.41421356f * (float)sigma);
                E = erff((float)dd * inv);
            }
            if (act) sc.edge[e] = E;
        }
        __syncwarp();
        // ---- bins: q wt_i wx_j, flat over the sub-batch -----------------------------------------------------------
        for (int b0 = 0; b0 < btot; b0 += 32) {
            const int b = b0 + lane;
            const bool act = b < btot;
            const int own = owner_of(sc.boff, bbase + (act ? b : 0));
            const int l = bbase + b - sc.boff[own];
            const int nto = __shfl_sync(0xffffffffu, nt, own);
            const int lo_t = __shfl_sync(0xffffffffu, et.lo, own), lo_x = __shfl_sync(0xffffffffu, ex.lo, own);
            // wire index in the patch, l / nto: (l + 1/2) / nto is at least 1/(2 nto) away from an integer, far more
            // than the rounding of the product below for l < 2^22 (a flat-path patch has < 2^14 bins)
            const int j = act ? __float2int_rz(((float)l + 0.5f) * __frcp_rn((float)max(nto, 1))) : 0;
            const int ii = act ? l - j * nto : 0;                              // tick index in the patch
            const float *E = sc.edge + (sc.eoff[own] - ebase);
            const float wt = 0.5f * (E[ii + 1] - E[ii]);
            const float wx = 0.5f * (E[nto + 1 + j + 1] - E[nto + 1 + j]);
            const float qq = __shfl_sync(0xffffffffu, q, own);
            const float scale = normalize ? (float)__shfl_sync(0xffffffffu, inv_norm, own) : 1.0f;
            if (act) sink.add(lo_x + j, lo_t + ii, qq * (wt * wx) * scale);
        }
        __syncwarp();
        d0 = d1;
    }
}

// ---- fluctuation on: quads ------------------------------------------------------------------------------------------
// One Philox call gives the words of four consecutive absolute grid bins (reading A8), so the unit of work of the front
// end is a QUAD: (depo, wire row of its patch, aligned group of four bins g>>2 of that row).  A lane finds its depo once,
// calls Philox once, loads the wire weight once and then classifies its (up to) four bins:
//   * k known without a draw (p <= 0, p >= 1, N = 0, or u <= 1 - mu, which implies u <= (1-p)^N): added at once;
//   * everything else is pushed to one of five per-warp shared-memory queues and drawn from there 32 bins at a time by
//     straight-line code, all lanes busy:
//     NORMAL  (mu >= 16, or the normal-approximation sampler): the guarded fp32 estimate of rng.cuh;
//     INV_A/B/C (mu < 2 / < 6 / < 16): the guarded fp32 inversion of rng.cuh with 8 / 16 / 32 terms;
//     EXACT   whatever the fp32 guards do not accept (~1 %), and bins not eligible for them: the fp64 routines.
// The edges of a batch are laid out per depo as [3 pad][nt+1 tick edges][3 pad][nx+1 wire edges], so that the loads of a
// quad never need a bounds check (pad values only ever reach bins that are masked off).
#ifndef WCSIM_KUNROLL
#define WCSIM_KUNROLL 1
#endif
constexpr int kQuadUnroll = WCSIM_KUNROLL; // unroll factor of the loop over the four bins of a quad
#ifndef WCSIM_EDGE_CAP
#define WCSIM_EDGE_CAP 400
#endif
// Edge values a warp's scratch holds.  The atomic kernels take 400: a whole 16-depo batch of BASELINE.json's patches
// (<= 16 + 5 + 2 edges and 6 pad slots each) then fits at once -- with 192 every batch was cut into two or three
// sub-batches whose edge and quad passes ran with a quarter of their lanes empty (configs[1] 66.2 -> 64.6 us, configs[4]
// 6.48 -> 6.23 ms).  The tile kernel keeps 192: with 8 warps and the tile's accumulators two of its CTAs must fit an SM.
constexpr int kQuadEdgeCap = WCSIM_EDGE_CAP, kTileEdgeCap = 192, kEdgePad = 3;
constexpr int kQueueCap = 64; // entries per queue: at most 31 left over + 32 pushed
enum QuadQueue : int { kQNorm = 0, kQInvA = 1, kQInvB = 2, kQInvC = 3, kQExact = 4, kNumQuadQueues = 5 };
constexpr int kQTotal = kNumQuadQueues * kQueueCap;

struct alignas(16) DepoRec {
    int lo_t, lo_x;  // first tick / wire of the clipped patch
    uint32_t shape;  // nt | nx << 8 | nq << 16 | (q < 0) << 31
    int ebase;       // index of the patch's first pad slot in QuadScratch::edge
    float t0, x0, N; // centre; N = floor(|q| + 1/2) (a float q makes it a float)
    uint32_t idx;    // index of the depo in the call (relative to the batch's dbase)
    double inv_t, inv_x; // 1 / (sqrt2 sigma); 0: sigma < 1e-6 (A4)
};

template <int CAP>
struct QuadScratch {
    double edge[CAP + 8]; // + slack: a quad past the end of a row may read up to 3 slots beyond the last pad
    DepoRec rec[kBatchDepos];
    double inv_norm[kBatchDepos];
    int eoff[33], qoff[33];
};
// queue entry: 20 bytes (24 with per-depo totals); queue c holds entries c kQueueCap .. c kQueueCap + fill - 1
template <bool TOT>
struct QuadQueues {
    double p[kQTotal];     // after the mirror: 0 < p <= 1/2 (normal-approximation sampler: 0 < p < 1)
    float N[kQTotal];      // exact queue: -N marks a bin of the inversion class (mu < 16)
    uint32_t w[kQTotal];   // after the mirror
    uint32_t bin[kQTotal]; // sink index | kBinMirror | kBinNegative
    uint32_t depo[TOT ? kQTotal : 1];
    alignas(16) int fill[8]; // entries in each of the five queues (kQNorm .. kQExact); pushed to with shared-memory atomics
};
template <bool TOT, int CAP>
struct QuadWarp {
    QuadScratch<CAP> sc;
    QuadQueues<TOT> q;
};
// the fills while the queues are drained (registers, uniform over the warp): the four fp32 queues (kQNorm .. kQInvC) and
// the exact queue.  Between drains the fills live in QuadQueues::fill.
struct QuadCounts {
    int fast[4];
    int exact;
};
template <bool TOT, int CAP>
__device__ __forceinline__ void queues_init(QuadWarp<TOT, CAP> &ws, int lane)
{
    if (lane < 8) ws.q.fill[lane] = 0;
    __syncwarp();
}

template <bool TOT, typename Sink>
__device__ __forceinline__ void commit_draw(const Sink &sink, int *__restrict__ totals, uint32_t fb, float N, float k,
                                            uint32_t depo)
{
    if (fb & kBinMirror) k = N - k;
    if (k != 0.0f) {
        const float v = (fb & kBinNegative) ? -k : k;
        sink.add_at(fb & kBinMask, v);
        if constexpr (TOT) atomicAdd(totals + depo, (int)v);
    }
}

// the exact queue: the fp64 routines of rng.cuh, 32 bins at a time (out of line: it is rare).  Returns the new fill.
template <bool TOT, typename Sink>
__device__ __noinline__ int drain_exact(QuadQueues<TOT> *Qp, int count, bool everything, Sink sink, int *__restrict__ totals,
                                        int lane)
{
    QuadQueues<TOT> &Q = *Qp;
    while (count >= 32 || (everything && count > 0)) {
        const int take = min(32, count);
        count -= take;
        if (lane < take) {
            const int e = kQExact * kQueueCap + count + lane;
            const float Nq = Q.N[e];
            const double N = (double)fabsf(Nq), p = Q.p[e];
            const uint32_t w = Q.w[e];
            const double k = Nq < 0.0f               ? draw_inversion(N, p, w)
                             : word_is_central(w) ? draw_normal_central(N, p, w)
                                                  : draw_normal_tail(N, p, w);
            commit_draw<TOT>(sink, totals, Q.bin[e], fabsf(Nq), (float)k, TOT ? Q.depo[e] : 0u);
        }
        __syncwarp();
    }
    return count;
}

// one group of up to 32 bins from the top of fp32 queue QI; bins the guard does not accept move to the exact queue
template <int QI, bool TOT, typename Sink>
__device__ __forceinline__ void drain_fast_group(QuadQueues<TOT> &Q, QuadCounts &qc, const Sink &sink, int *__restrict__ totals,
                                                 int lane)
{
    const int fill = qc.fast[QI];
    const int take = min(32, fill);
    qc.fast[QI] = fill - take;
    const int e = QI * kQueueCap + fill - take + lane;
    bool rej = false;
    if (lane < take) {
        const double p = Q.p[e];
        const float N = Q.N[e];
        const uint32_t w = Q.w[e];
        float kv;
        bool ok;
        if constexpr (QI == kQNorm) ok = p <= 0.5 && fast_normal_draw(N, p, __dmul_rn((double)N, p), w, kv);
        else if constexpr (QI == kQInvA) ok = inv_fast_draw<8>(N, p, w, kv);
        else if constexpr (QI == kQInvB) ok = inv_fast_draw<16>(N, p, w, kv);
        else ok = inv_fast_draw<32>(N, p, w, kv);
        if (ok) commit_draw<TOT>(sink, totals, Q.bin[e], N, kv, TOT ? Q.depo[e] : 0u);
        rej = !ok;
    }
    const unsigned int mr = __ballot_sync(0xffffffffu, rej);
    if (mr) { // the exact queue holds < 32 entries here
        if (rej) {
            const int x = kQExact * kQueueCap + qc.exact + __popc(mr & ((1u << lane) - 1u));
            Q.p[x] = Q.p[e], Q.w[x] = Q.w[e], Q.bin[x] = Q.bin[e];
            Q.N[x] = QI == kQNorm ? Q.N[e] : -Q.N[e]; // -N: inversion class
            if constexpr (TOT) Q.depo[x] = Q.depo[e];
        }
        qc.exact += __popc(mr);
        __syncwarp();
        if (qc.exact >= 32) qc.exact = drain_exact<TOT>(&Q, qc.exact, false, sink, totals, lane);
    }
}

// The queues.  Called (from one place) when one of them holds a warp's worth of work: every queue with 32 or more entries
// is worked off in groups of 32; with `finish`, everything.
template <bool TOT, int CAP, typename Sink>
__device__ __forceinline__ void drain_queues(QuadWarp<TOT, CAP> &ws, int4 fills, int fill_exact, bool finish, const Sink &sink,
                                             int *__restrict__ totals, int lane)
{
    QuadQueues<TOT> &Q = ws.q;
    QuadCounts qc{{fills.x, fills.y, fills.z, fills.w}, fill_exact}; // what the caller has just read from Q.fill
    const int due = finish ? 1 : 32; // a queue is due when it holds a warp's worth (finish: anything)
    // the exact queue first if it is what is full: the groups below may each add up to 32 rejected bins to it
    if (qc.exact >= 32) qc.exact = drain_exact<TOT>(&Q, qc.exact, false, sink, totals, lane);
    while (qc.fast[kQNorm] >= due) drain_fast_group<kQNorm, TOT>(Q, qc, sink, totals, lane);
    while (qc.fast[kQInvA] >= due) drain_fast_group<kQInvA, TOT>(Q, qc, sink, totals, lane);
    while (qc.fast[kQInvB] >= due) drain_fast_group<kQInvB, TOT>(Q, qc, sink, totals, lane);
    while (qc.fast[kQInvC] >= due) drain_fast_group<kQInvC, TOT>(Q, qc, sink, totals, lane);
    if (qc.exact >= 32 || (finish && qc.exact > 0)) qc.exact = drain_exact<TOT>(&Q, qc.exact, finish, sink, totals, lane);
    __syncwarp(); // every lane has read its entries
    if (lane == 0) {
        *reinterpret_cast<int4 *>(Q.fill) = make_int4(qc.fast[0], qc.fast[1], qc.fast[2], qc.fast[3]);
        Q.fill[kQExact] = qc.exact;
    }
    __syncwarp();
}

// One batch of up to kBatchDepos depos, one per lane (lanes >= kBatchDepos own none), fluctuation on.  The call-wide index
// of the depo of lane l is dbase + l, or dbase + dl (of lane l) when the batch comes from an index list (INDIRECT).
// `flush`: the caller has no more batches (the lanes then carry no depo): every queue is emptied before the call returns.
// NORMAL_ONLY: the normal-approximation sampler of reading A21 (no inversion branch, no mirror).
template <bool NORMAL_ONLY, bool TOT, bool INDIRECT, int CAP, typename Sink>
__device__ __forceinline__ void raster_quad_body(GridDims g, Clip clip, const Sink &sink, float t0, float x0, float st,
                                                 float sx, float q, bool valid, long long dbase, uint32_t dl,
                                                 uint64_t id_base, uint64_t seed, double nsigma, bool normalize,
                                                 int *__restrict__ totals, QuadWarp<TOT, CAP> &ws, bool flush,
                                                 unsigned int &drawn, int lane)
{
    constexpr bool normal_only = NORMAL_ONLY;
    QuadScratch<CAP> &sc = ws.sc;
    QuadQueues<TOT> &Q = ws.q;
    const double T0 = t0, X0 = x0, ST = st, SX = sx;
    Extent et{0, 0}, ex{0, 0};
    if (valid) {
        et = axis_extent(T0, ST, nsigma, clip.k_lo, clip.k_hi);
        ex = axis_extent(X0, SX, nsigma, clip.w_lo, clip.w_hi);
    }
    const bool live = et.lo < et.hi && ex.lo < ex.hi;
    const int nt = live ? et.hi - et.lo : 0, nx = live ? ex.hi - ex.lo : 0;
    const bool big = nt + nx + 2 + 2 * kEdgePad > CAP || nt > 255 || nx > 255;
    const bool flat = live && !big;
    // quads per wire row: with n_ticks a multiple of 4 every row of a patch starts at the same offset in its quad
    const bool aligned = (g.n_ticks & 3) == 0;
    const int nq = aligned ? ((((et.lo & 3) + nt - 1) >> 2) + 1) : (((nt + 2) >> 2) + 1);
    const int ne = flat ? nt + nx + 2 : 0, nqs = flat ? nx * nq : 0;
    const int eincl = warp_incl_scan(ne, lane), qincl = warp_incl_scan(nqs, lane);
    const uint32_t didx = INDIRECT ? dl : (uint32_t)lane;
    __syncwarp();
    sc.eoff[lane] = eincl - ne;
    sc.qoff[lane] = qincl - nqs;
    if (lane == 31) {
        sc.eoff[32] = eincl;
        sc.qoff[32] = qincl;
    }
    if (lane < kBatchDepos) {
        DepoRec rc;
        rc.lo_t = et.lo, rc.lo_x = ex.lo;
        rc.shape = (uint32_t)nt | ((uint32_t)nx << 8) | ((uint32_t)nq << 16) | (q < 0.0f ? 0x80000000u : 0u);
        rc.ebase = 0;
        rc.t0 = t0, rc.x0 = x0, rc.N = (float)floor(fabs((double)q) + 0.5), rc.idx = didx;
        rc.inv_t = ST < 1e-6 ? 0.0 : fast_rcp(1.4142135623730951 * ST);
        rc.inv_x = SX < 1e-6 ? 0.0 : fast_rcp(1.4142135623730951 * SX);
        sc.rec[lane] = rc;
        // renormalised patches (reading A24): 1 / (W_t W_x), W = the axis weights summed over the whole, unclipped extent
        if (normalize)
            sc.inv_norm[lane] = flat ? __ddiv_rn(1.0, axis_norm(T0, ST, nsigma) * axis_norm(X0, SX, nsigma)) : 1.0;
    }
    __syncwarp();
    if (flat) drawn += (unsigned int)(nt * nx);

    // patches too big for the scratch: the whole warp walks them one at a time (fp64 sampler per bin)
    unsigned int big_mask = __ballot_sync(0xffffffffu, live && big);
    while (big_mask) {
        const int src = __ffs(big_mask) - 1;
        big_mask &= big_mask - 1;
        int tot = 0;
        const long long dio = dbase + (long long)__shfl_sync(0xffffffffu, didx, src);
        double inv_norm = 1.0;
        if (normalize) {
            if (lane == src) inv_norm = __ddiv_rn(1.0, axis_norm(T0, ST, nsigma) * axis_norm(X0, SX, nsigma));
            inv_norm = __shfl_sync(0xffffffffu, inv_norm, src);
        }
        drawn += raster_depo<true>(__shfl_sync(0xffffffffu, t0, src), __shfl_sync(0xffffffffu, x0, src),
                                   __shfl_sync(0xffffffffu, st, src), __shfl_sync(0xffffffffu, sx, src),
                                   __shfl_sync(0xffffffffu, q, src), id_base + (uint64_t)dio, seed, nsigma, g.n_ticks,
                                   clip.w_lo, clip.w_hi, clip.k_lo, clip.k_hi, sink.shifted(clip.row_off), lane, &tot,
                                   normal_only, inv_norm);
        if (totals != nullptr) {
            tot = warp_sum(tot);
            if (lane == 0 && tot != 0) atomicAdd(totals + dio, tot);
        }
    }

    // sub-batches of consecutive depos whose padded edge lists fit the scratch (normally the whole batch)
    int d0 = 0;
    while (d0 < 32) {
        const int ebase = sc.eoff[d0];
        const unsigned int fits = __ballot_sync(
            0xffffffffu, lane >= d0 && eincl - ebase + 2 * kEdgePad * (min(lane, kBatchDepos - 1) - d0 + 1) <= CAP);
        const int d1 = d0 + __popc(fits); // monotone: the fitting lanes are d0 .. d1-1, at least one
        const int etot = sc.eoff[d1] - ebase, qbase = sc.qoff[d0], qtot = sc.qoff[d1] - qbase;
        if (lane >= d0 && lane < d1 && lane < kBatchDepos) sc.rec[lane].ebase = eincl - ne - ebase + 2 * kEdgePad * (lane - d0);
        __syncwarp();
        // ---- edges: erf((edge - centre) / (sqrt2 sigma)) in fp64, flat over the sub-batch ---------------------------
        for (int e0 = 0; e0 < etot; e0 += 32) {
            const int e = e0 + lane;
            const bool act = e < etot;
            const int own = owner_of(sc.eoff, ebase + (act ? e : 0));
            const int le = ebase + e - sc.eoff[own];
            const DepoRec &rc = sc.rec[own];
            const int4 a = *reinterpret_cast<const int4 *>(&rc.lo_t);
            const float2 ctr = *reinterpret_cast<const float2 *>(&rc.t0);
            const double2 inv2 = *reinterpret_cast<const double2 *>(&rc.inv_t);
            const int nto = a.z & 255;
            const bool on_t = le <= nto;
            const int coord = on_t ? a.x + le : a.y + (le - nto - 1);
            const double centre = (double)(on_t ? ctr.x : ctr.y), inv = on_t ? inv2.x : inv2.y;
            double E;
            if (inv == 0.0) { // all weight in bin floor(centre) (A4): a step from -1 to +1 after that bin's low edge
                E = ((double)coord <= floor(centre)) ? -1.0 : 1.0;
            } else {
                E = erf_from_table(g_erf_tab, __dsub_rn((double)coord, centre) * inv);
            }
            if (act) sc.edge[a.w + kEdgePad + le + (on_t ? 0 : kEdgePad)] = E;
        }
        __syncwarp();
        // ---- quads (one more, empty pass when flushing, so that the queues are drained from this one place) -----------
        const bool flush_here = flush && d1 >= 32;
        for (int s0 = 0; s0 < qtot || (flush_here && s0 == 0); s0 += 32) {
            const int s = s0 + lane;
            const bool act = s < qtot;
            const int own = owner_of(sc.qoff, qbase + (act ? s : 0));
            const int l = act ? qbase + s - sc.qoff[own] : 0;
            const DepoRec &rc = sc.rec[own];
            const int4 a = *reinterpret_cast<const int4 *>(&rc.lo_t);
            const float4 bq = *reinterpret_cast<const float4 *>(&rc.t0);
            const float Nf = bq.z;
            const int nto = a.z & 255, nqo = (a.z >> 16) & 255;
            // wire row of the quad, l / nq: (l + 1/2) / nq is at least 1/(2 nq) away from an integer, far more than the
            // rounding of the product for l < 2^16
            const int j = __float2int_rz(((float)l + 0.5f) * __frcp_rn((float)max(nqo, 1)));
            const int qi = l - j * nqo;
            const int wire = a.y + j;
            const uint32_t g0 = (uint32_t)wire * (uint32_t)g.n_ticks + (uint32_t)a.x; // absolute bin of the row's first tick
            const uint32_t gq = (g0 >> 2) + (uint32_t)qi;
            const int ii0 = (int)(4u * gq - g0); // patch tick index of the quad's first bin: -3 .. nt-1
            const double *E = sc.edge + a.w + kEdgePad + ii0;
            const double *Ex = sc.edge + a.w + 2 * kEdgePad + nto + 1 + j;
            const double wxq = 0.25 * (Ex[1] - Ex[0]); // wx / 2: p = (wx / 2) (E_t[i+1] - E_t[i])
            const double inv_n = normalize ? sc.inv_norm[own] : 1.0;
            const uint32_t dio = (uint32_t)dbase + __float_as_uint(bq.w); // index of the depo in the call (< 2^32: totals)
            const uint4 words = fluct_words(seed, id_base + (uint64_t)(dbase + (long long)__float_as_uint(bq.w)), (uint64_t)gq);
            const uint32_t idx0 = sink.index(wire + clip.row_off, a.x) + (uint32_t)ii0; // sink index of the quad's first bin (mod 2^32)
            const uint32_t neg = a.z < 0 ? kBinNegative : 0u;
            const bool live_q = act && Nf > 0.0f; // N = 0 draws nothing
            uint32_t w0 = words.x, w1 = words.y, w2 = words.z, w3 = words.w;
#pragma unroll kQuadUnroll
            for (int k = 0; k < 4; ++k) {
                uint32_t w = w0; // the word of this bin; the others move up
                w0 = w1, w1 = w2, w2 = w3;
                const bool v = live_q && (unsigned)(ii0 + k) < (unsigned)nto;
                double p = __dmul_rn(__dsub_rn(E[k + 1], E[k]), wxq); // = wt wx: the two factors 1/2 are exact scalings
                p = __dmul_rn(p, inv_n); // inv_n = 1 unless patches are renormalised (A24): an exact no-op then
                const bool all = p >= 1.0; // every electron lands here
                const bool mirror = !normal_only && p > 0.5 && !all;
                if (mirror) {
                    p = __dsub_rn(1.0, p);
                    w = ~w;
                }
                const float muf = (float)__dmul_rn((double)Nf, p); // class boundaries below: see the note on `cls`
                const bool small = !normal_only && __dmul_rn((double)Nf, p) < 16.0;
                // u <= 1 - mu implies u <= (1-p)^N = F(0), i.e. k = 0 (Bernoulli); in fp32 with a margin that covers the
                // roundings of u, mu and their sum (3 x 2^-24)
                const bool quick = small && fmaf((float)w, 2.3283064365386963e-10f, 1.1641532182693481e-10f) + muf <= 0.9999996f;
                const bool draw = v && p > 0.0 && !all && !quick;
                // k = N without a draw: p >= 1, or k = 0 of the mirrored draw
                if (v && (all || (quick && mirror))) {
                    sink.add_at(idx0 + k, neg ? -Nf : Nf);
                    if constexpr (TOT) atomicAdd(totals + dio, (int)(neg ? -Nf : Nf));
                }
                // The queue.  mu < 16 against mu >= 16 is the sampler's own branch and is decided in fp64 (`small`); the
                // bands of the inversion only choose how many terms the fp32 routine sums, so fp32 mu is good enough
                // (a bin next to a band edge that needs more terms than its band has fails the guard and is redone).
                int cls = !small ? kQNorm : !inv_fast_eligible(Nf, p) ? kQExact : muf < 2.0f ? kQInvA : muf < 6.0f ? kQInvB : kQInvC;
                if (!draw) cls = -1;
                // push: a shared-memory atomic on the queue's fill hands every lane its slot (the order of the entries in a
                // queue does not matter: each carries all it needs, and the adds into S are order independent or exact)
                if (cls >= 0) {
                    const int pos = cls * kQueueCap + atomicAdd(&Q.fill[cls], 1);
                    Q.p[pos] = p;
                    Q.N[pos] = (cls == kQExact && small) ? -Nf : Nf;
                    Q.w[pos] = w;
                    Q.bin[pos] = (idx0 + k) | neg | (mirror ? kBinMirror : 0u);
                    if constexpr (TOT) Q.depo[pos] = dio;
                }
                __syncwarp();
                const int4 f = *reinterpret_cast<const int4 *>(Q.fill); // every fill is < 64: bit 5 says "a warp's worth"
                const int fx = Q.fill[kQExact];
                const bool last = flush_here && k == 3 && s0 + 32 >= qtot;
                if ((((f.x | f.y) | (f.z | f.w) | fx) & 32) | (int)last) drain_queues(ws, f, fx, last, sink, totals, lane);
            }
        }
        __syncwarp();
        d0 = d1;
    }
}

// shared memory of the batch kernels
template <bool FLUCT, bool TOT>
struct BatchSmem {
    FlatScratch scratch[kBatchWarps];
};
template <bool TOT>
struct BatchSmem<true, TOT> {
    QuadWarp<TOT, kQuadEdgeCap> warp[kBatchWarps];
};

// ------------------------------------------------------------------------------------------------------------------
// atomic mode: persistent warps; a warp's first batch is its own index in the grid, further ones come from a device
// counter (guided: kBatchDepos depos at a time, kTailDepos at a time near the end)
// ------------------------------------------------------------------------------------------------------------------
// FLUCT: 0 off, 1 binomial (reading A6), 2 normal approximation (reading A21)
template <int FLUCT, bool TOT, bool FIX>
__global__ void __launch_bounds__(kBatchWarps * 32, FLUCT ? WCSIM_FLUCT_CTAS : 8) raster_batch_kernel(GridDims g, DepoArrays d, long long n,
                                                                        uint64_t id_base, uint64_t seed, double nsigma,
                                                                        float *__restrict__ S, int *__restrict__ totals,
                                                                        Counters *counters, bool normalize, int4 sched)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    BatchSmem<FLUCT != 0, TOT> &sm = *reinterpret_cast<BatchSmem<FLUCT != 0, TOT> *>(smem_raw);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    // FIX: S points at the 64-bit fixed-point grid (deterministic mode without tiles)
    using Sink = typename std::conditional<FIX, FixSink, GlobalSink>::type;
    const Sink sink = make_grid_sink<FIX>(S, g.n_ticks);
    const Clip clip{0, g.n_wires, 0, g.n_ticks};
    // guided batches: kBatchDepos depos at a time, then kTailDepos at a time for the last kTailPerWarp depos per warp of the
    // grid, so that the warps run out of work within a short batch of one another (on configs[1] a warp gets only
    // 3-4 batches of 8)
    const long long n_warps_grid = (long long)gridDim.x * kBatchWarps;
    const int tail_size = sched.x, n_static = sched.z;
    const bool big_only = sched.w != 0; // the tiled mode's pass over the depos that are too big to be listed by tile
    const long long tail_depos = n_warps_grid * sched.y < n ? n_warps_grid * sched.y : n;
    const long long big_batches = (n - tail_depos) >> kBatchShift;
    const long long big_depos = big_batches << kBatchShift;
    const long long n_batches = big_batches + (n - big_depos + tail_size - 1) / tail_size;
    unsigned int drawn = 0, skipped = 0; // per lane
    if constexpr (FLUCT != 0) queues_init(sm.warp[wid], lane);
    // the grid is one wave, so the next kernel's CTAs may take the slots this one frees as it drains.  As a
    // programmatic dependent itself it only overlaps a preceding KERNEL's tail: copies and memsets ahead of it in the
    // stream are still fully ordered (checked with 300 host-buffer plane-events of changing depos, 0 mismatches)
    pdl_trigger();
    pdl_wait();

    // The first batch of a warp is its index in the grid: all warps start at once, and thousands of atomics on one
    // counter would queue up behind one another for microseconds (same-address atomics are served one every ~2 ns; with
    // every batch fetched from the counter the fetch was 42 % of the stall samples of the unfluctuated raster on
    // configs[1]).  Later batches come from the counter, which keeps the load balanced.
    // (Fetching the NEXT batch's index early to hide the round trip was tried: a warp then sits on a batch while it
    // works on another, and the load balance suffers more than the latency costs.)
    long long batch = (long long)blockIdx.x * kBatchWarps + wid;
    int round = 0;
    for (;;) {
        const bool more = batch < n_batches;
        const long long first = batch < big_batches ? batch << kBatchShift : big_depos + (batch - big_batches) * tail_size;
        const int count = batch < big_batches ? kBatchDepos : tail_size;
        const long long i = first + lane;
        float t0 = 0.f, x0 = 0.f, st = 0.f, sx = 0.f, q = 0.f;
        bool valid = false;
        if (more && lane < count && i < n) {
            t0 = d.t0[i], x0 = d.x0[i], st = d.sigma_t[i], sx = d.sigma_x[i], q = d.q[i]; // plain loads: pdl.cuh
            valid = depo_valid(t0, x0, st, sx, q);
            if (big_only) valid = valid && depo_tile_range(g, t0, x0, st, sx, q, nsigma).count() > kMaxListedTiles;
            else skipped += !valid; // (the tiled mode counts invalid depos in its own pass)
        }
        // fluctuated: one more call without depos after the last batch empties the warp's draw queues
        if constexpr (FLUCT)
            raster_quad_body<FLUCT == 2, TOT, false>(g, clip, sink, t0, x0, st, sx, q, valid, first, 0u, id_base, seed, nsigma,
                                                     normalize, totals, sm.warp[wid], !more, drawn, lane);
        else if (more)
            raster_flat_body(g, clip, sink, t0, x0, st, sx, q, valid, nsigma, normalize, sm.scratch[wid], drawn, lane);
        if (!more) break;
        if (++round < n_static) {
            batch += n_warps_grid;
        } else if (n_static * n_warps_grid >= n_batches) {
            batch = n_batches; // the static rounds cover every batch: no fetch (one more pass empties the draw queues)
        } else {
            if (lane == 0) batch = n_static * n_warps_grid + (long long)atomicAdd(&counters->next_batch, 1ull);
            batch = __shfl_sync(0xffffffffu, batch, 0);
        }
    }
    const unsigned long long drawn_w = warp_sum((unsigned long long)drawn), skipped_w = warp_sum((unsigned long long)skipped);
    if (lane == 0) {
        if (drawn_w) atomicAdd(&counters->bins_drawn, drawn_w);
        if (skipped_w) atomicAdd(&counters->depos_skipped, skipped_w);
        // the last warp to leave re-arms the batch counter for the next launch on this stream (every warp has made its
        // last fetch before it adds itself here)
        const unsigned long long n_warps = (unsigned long long)gridDim.x * kBatchWarps;
        if (atomicAdd(&counters->warps_done, 1ull) == n_warps - 1) {
            counters->next_batch = 0ull;
            counters->warps_done = 0ull;
        }
    }
}

// ------------------------------------------------------------------------------------------------------------------
// The planes of a multi-plane plan in ONE launch (one plane-event does not fill the
// device).  The batch list is the concatenation of the planes' batch lists; a warp looks its batch's plane up (uniform
// over the warp) and runs the same batch body with that plane's depo arrays, wire count and row offset in the stacked
// grid.  Depo ids and Philox bins are the plane's own, so the result equals the planes rastered one by one.
// ------------------------------------------------------------------------------------------------------------------
template <int FLUCT, bool FIX>
__global__ void __launch_bounds__(kBatchWarps * 32, FLUCT ? WCSIM_FLUCT_CTAS : 8)
    raster_planes_kernel(int n_ticks, const __grid_constant__ RasterPlanes P, double nsigma,
                         float *__restrict__ S, Counters *counters, bool normalize, int n_static)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    BatchSmem<FLUCT != 0, false> &sm = *reinterpret_cast<BatchSmem<FLUCT != 0, false> *>(smem_raw);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    using Sink = typename std::conditional<FIX, FixSink, GlobalSink>::type;
    const Sink sink = make_grid_sink<FIX>(S, n_ticks);
    const long long n_warps_grid = (long long)gridDim.x * kBatchWarps;
    const long long n_batches = P.batch0[P.n];
    unsigned int drawn = 0, skipped = 0; // per lane
    if constexpr (FLUCT != 0) queues_init(sm.warp[wid], lane);
    pdl_trigger();
    pdl_wait();
    long long batch = (long long)blockIdx.x * kBatchWarps + wid;
    int round = 0;
    for (;;) {
        const bool more = batch < n_batches;
        int pl = 0;
        if (more)
            while (pl + 1 < P.n && batch >= P.batch0[pl + 1]) ++pl;
        const long long first = more ? (batch - P.batch0[pl]) << kBatchShift : 0;
        const long long i = first + lane;
        float t0 = 0.f, x0 = 0.f, st = 0.f, sx = 0.f, q = 0.f;
        bool valid = false;
        if (more && lane < kBatchDepos && i < P.count[pl]) {
            const DepoArrays &d = P.d[pl];
            t0 = d.t0[i], x0 = d.x0[i], st = d.sigma_t[i], sx = d.sigma_x[i], q = d.q[i]; // plain loads: pdl.cuh
            valid = depo_valid(t0, x0, st, sx, q);
            skipped += !valid;
        }
        const GridDims g{P.n_wires[pl], n_ticks};
        const Clip clip{0, g.n_wires, 0, n_ticks, P.row0[pl]};
        if constexpr (FLUCT)
            raster_quad_body<FLUCT == 2, false, false>(g, clip, sink, t0, x0, st, sx, q, valid, first, 0u, 0ull, P.seed[pl], nsigma,
                                                       normalize, nullptr, sm.warp[wid], !more, drawn, lane);
        else if (more)
            raster_flat_body(g, clip, sink.shifted(clip.row_off), t0, x0, st, sx, q, valid, nsigma, normalize,
                             sm.scratch[wid], drawn, lane);
        if (!more) break;
        if (++round < n_static) {
            batch += n_warps_grid;
        } else if (n_static * n_warps_grid >= n_batches) {
            batch = n_batches; // every batch was assigned statically
        } else {
            if (lane == 0) batch = n_static * n_warps_grid + (long long)atomicAdd(&counters->next_batch, 1ull);
            batch = __shfl_sync(0xffffffffu, batch, 0);
        }
    }
    const unsigned long long drawn_w = warp_sum((unsigned long long)drawn), skipped_w = warp_sum((unsigned long long)skipped);
    if (lane == 0) {
        if (drawn_w) atomicAdd(&counters->bins_drawn, drawn_w);
        if (skipped_w) atomicAdd(&counters->depos_skipped, skipped_w);
        const unsigned long long n_warps = (unsigned long long)gridDim.x * kBatchWarps;
        if (atomicAdd(&counters->warps_done, 1ull) == n_warps - 1) { // the last warp re-arms the batch counter
            counters->next_batch = 0ull;
            counters->warps_done = 0ull;
        }
    }
}

// ------------------------------------------------------------------------------------------------------------------
// tiled mode
// ------------------------------------------------------------------------------------------------------------------
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
        // a tile is split over several CTAs only when it lists well over the average: twice the mean, at least kSliceEntries
        const unsigned int twice_mean = (unsigned int)(2ull * carry / (unsigned int)(n_tiles > 0 ? n_tiles : 1));
        *ts.slice_dev = twice_mean > (unsigned int)kSliceEntries ? twice_mean : (unsigned int)kSliceEntries;
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

// Up to kTileSlices CTAs per tile (one per kSliceEntries listed depos, so that the hot tiles along a track do not
// serialise on one CTA).  A CTA's warps take their slice of the tile's depos (the index list built by count / scan /
// fill) eight at a time and run the same flat-list batch body as the atomic kernel, clipped to the tile and
// accumulating into fixed-point shared-memory accumulators; at the end the CTA adds its non-zero accumulators into the
// global fixed-point grid `fix` (64-bit integer atomics: order independent), and tile_finalize_kernel folds `fix`
// into S with one float add per bin.
constexpr int kTileWarps = 8, kTileSlices = 8;
template <bool FLUCT, bool TOT>
struct TileSmem {
    unsigned long long acc[kTileW * kTileT];
    FlatScratch scratch[kTileWarps];
};
template <bool TOT>
struct TileSmem<true, TOT> {
    unsigned long long acc[kTileW * kTileT];
    QuadWarp<TOT, kTileEdgeCap> warp[kTileWarps];
};

template <int FLUCT, bool TOT>
__global__ void __launch_bounds__(kTileWarps * 32, 2) tile_accumulate_kernel(GridDims g, DepoArrays d, uint64_t id_base,
                                                                          uint64_t seed, double nsigma, TileScratch ts,
                                                                          float *__restrict__ S, int *__restrict__ totals,
                                                                          Counters *counters, bool normalize)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    TileSmem<FLUCT != 0, TOT> &sm = *reinterpret_cast<TileSmem<FLUCT != 0, TOT> *>(smem_raw);
    const int tile = blockIdx.x / kTileSlices, slice = blockIdx.x % kTileSlices;
    const unsigned int tile_beg = ts.tile_count[tile], tile_end = ts.tile_count[tile + 1];
    const unsigned int listed = tile_end - tile_beg;
    // a tile is split only when it lists well over the average (*ts.slice_dev = max(kSliceEntries, 2 x mean)): on an
    // evenly busy plane (configs[4]) slicing only adds clears, flushes and partial queue drains
    const unsigned int slice_entries = *ts.slice_dev;
    const unsigned int n_slices = min((unsigned int)kTileSlices, (listed + slice_entries - 1) / slice_entries);
    if ((unsigned int)slice >= n_slices) return; // uniform over the CTA (also: nothing listed)
    // equal slices in whole batches
    const unsigned int per = ((listed + n_slices - 1) / n_slices + kBatchDepos - 1) / kBatchDepos * kBatchDepos;
    const unsigned int beg = min(tile_beg + (unsigned int)slice * per, tile_end), end = min(beg + per, tile_end);
    if (beg == end) return;
    const int tw = tile / ts.tiles_t, tt = tile % ts.tiles_t;
    const int w0 = tw * kTileW, k0 = tt * kTileT;
    const int w1 = min(w0 + kTileW, g.n_wires), k1 = min(k0 + kTileT, g.n_ticks);
    for (int i = threadIdx.x; i < kTileW * kTileT; i += blockDim.x) sm.acc[i] = 0ull;
    __syncthreads();
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const TileSink sink{sm.acc, w0, k0};
    const Clip clip{w0, w1, k0, k1};
    unsigned int drawn = 0; // per lane
    if constexpr (FLUCT != 0) queues_init(sm.warp[wid], lane);
    for (unsigned int e0 = beg + (unsigned int)wid * kBatchDepos;; e0 += kTileWarps * kBatchDepos) {
        const bool more = e0 < end;
        float t0 = 0.f, x0 = 0.f, st = 0.f, sx = 0.f, q = 0.f;
        unsigned int i = 0;
        bool valid = false;
        if (more && lane < kBatchDepos && e0 + lane < end) {
            i = ts.entries[e0 + lane];
            t0 = __ldg(d.t0 + i), x0 = __ldg(d.x0 + i), st = __ldg(d.sigma_t + i), sx = __ldg(d.sigma_x + i), q = __ldg(d.q + i);
            valid = depo_valid(t0, x0, st, sx, q); // listed depos are valid; kept for symmetry with the atomic kernel
        }
        if constexpr (FLUCT)
            raster_quad_body<FLUCT == 2, TOT, true>(g, clip, sink, t0, x0, st, sx, q, valid, 0ll, i, id_base, seed, nsigma,
                                                    normalize, totals, sm.warp[wid], !more, drawn, lane);
        else if (more)
            raster_flat_body(g, clip, sink, t0, x0, st, sx, q, valid, nsigma, normalize, sm.scratch[wid], drawn, lane);
        if (!more) break;
    }
    const unsigned long long drawn_w = warp_sum((unsigned long long)drawn);
    if (lane == 0 && drawn_w) atomicAdd(&counters->bins_drawn, drawn_w);
    __syncthreads();
    for (int i = threadIdx.x; i < kTileW * kTileT; i += blockDim.x) {
        const int w = w0 + i / kTileT, k = k0 + i % kTileT;
        const unsigned long long q = sm.acc[i];
        if (q != 0ull && w < w1 && k < k1) atomicAdd(ts.fix + (size_t)w * g.n_ticks + k, q);
    }
}

__global__ void __launch_bounds__(256) tile_finalize_kernel(long long n_bins, unsigned long long *__restrict__ fix,
                                                            float *__restrict__ S)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_bins) return;
    const long long q = (long long)fix[i];
    if (q != 0) {
        S[i] = S[i] + (float)((double)q * (1.0 / kFixScale));
        fix[i] = 0ull;
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

static const double *erf_table_once()
{
    static double tab[(kErfDegree + 1) * kErfIntervals];
    static std::once_flag once;
    std::call_once(once, [] { build_erf_table(tab); });
    return tab;
}

void erf_table_host(const double *z, double *out, long long n)
{
    const double *tab = erf_table_once();
    for (long long i = 0; i < n; ++i) out[i] = erf_from_table(tab, z[i]);
}

// Once per device (under a mutex): later plans must not rewrite the table while other plans' kernels read it.
cudaError_t raster_configure(cudaStream_t st)
{
    static std::mutex mu;
    static bool done[64] = {};
    int dev = 0;
    cudaError_t err = cudaGetDevice(&dev);
    if (err != cudaSuccess) return err;
    std::lock_guard<std::mutex> lock(mu);
    if (dev >= 0 && dev < 64 && done[dev]) return cudaSuccess;
    err = cudaMemcpyToSymbolAsync(g_erf_tab, erf_table_once(), sizeof(double) * (kErfDegree + 1) * kErfIntervals, 0,
                                  cudaMemcpyHostToDevice, st);
    if (err != cudaSuccess) return err;
    err = cudaStreamSynchronize(st);
    if (err != cudaSuccess) return err;
#define WCSIM_RASTER_SMEM(F, T, X)                                                                                     \
    err = cudaFuncSetAttribute(raster_batch_kernel<F, T, X>, cudaFuncAttributeMaxDynamicSharedMemorySize,              \
                               (int)sizeof(BatchSmem<F != 0, T>));                                                     \
    if (err != cudaSuccess) return err;
    WCSIM_RASTER_SMEM(1, true, false)
    WCSIM_RASTER_SMEM(1, false, false)
    WCSIM_RASTER_SMEM(2, true, false)
    WCSIM_RASTER_SMEM(2, false, false)
    WCSIM_RASTER_SMEM(0, false, false)
    WCSIM_RASTER_SMEM(1, true, true)
    WCSIM_RASTER_SMEM(1, false, true)
    WCSIM_RASTER_SMEM(2, true, true)
    WCSIM_RASTER_SMEM(2, false, true)
    WCSIM_RASTER_SMEM(0, false, true)
#undef WCSIM_RASTER_SMEM
#define WCSIM_PLANES_SMEM(F, X)                                                                                        \
    err = cudaFuncSetAttribute(raster_planes_kernel<F, X>, cudaFuncAttributeMaxDynamicSharedMemorySize,                \
                               (int)sizeof(BatchSmem<F != 0, false>));                                                 \
    if (err != cudaSuccess) return err;
    WCSIM_PLANES_SMEM(0, false)
    WCSIM_PLANES_SMEM(1, false)
    WCSIM_PLANES_SMEM(2, false)
    WCSIM_PLANES_SMEM(0, true)
    WCSIM_PLANES_SMEM(1, true)
    WCSIM_PLANES_SMEM(2, true)
#undef WCSIM_PLANES_SMEM
#define WCSIM_TILE_SMEM(F, T)                                                                                          \
    err = cudaFuncSetAttribute(tile_accumulate_kernel<F, T>, cudaFuncAttributeMaxDynamicSharedMemorySize,              \
                               (int)sizeof(TileSmem<F != 0, T>));                                                      \
    if (err != cudaSuccess) return err;
    WCSIM_TILE_SMEM(1, true)
    WCSIM_TILE_SMEM(1, false)
    WCSIM_TILE_SMEM(2, true)
    WCSIM_TILE_SMEM(2, false)
    WCSIM_TILE_SMEM(0, false)
#undef WCSIM_TILE_SMEM
    if (dev >= 0 && dev < 64) done[dev] = true;
    return cudaSuccess;
}

template <int FLUCT, bool TOT, bool FIX>
static cudaError_t launch_raster_batch(GridDims g, DepoArrays d, long long n, uint64_t id_base, uint64_t seed, double nsigma,
                                       float *S, int *depo_totals, Counters *counters, int sm_count, cudaStream_t st,
                                       bool normalize, bool big_only)
{
    const size_t smem = sizeof(BatchSmem<FLUCT != 0, TOT>);
    const int fit = (int)((227u * 1024u) / (smem + 1024u)); // 227 KB per SM, 1 KB reserved per CTA
    const int cap = FLUCT ? WCSIM_FLUCT_CTAS : 8; // the kernel's __launch_bounds__
    const int ctas_per_sm = fit > cap ? cap : fit;
    const long long max_ctas = (long long)sm_count * (ctas_per_sm > 0 ? ctas_per_sm : 1);
    int4 sched = make_int4(kTailDepos, kTailPerWarp, 2, big_only ? 1 : 0);
    // A small call (fewer depos than kBatchDepos per resident warp) is latency bound: a warp works its batch off serially,
    // so the depos are spread over as many warps as there are, in batches of `per` < kBatchDepos depos each (the kernel's
    // "tail" batches, here for every depo).  configs[0]: 100 depos -> 100 one-depo batches instead of 7 batches of 16.
    long long n_batches = (n + kBatchDepos - 1) / kBatchDepos;
    const long long warp_slots = max_ctas * kBatchWarps;
    const long long per = (n + warp_slots - 1) / warp_slots;
    if (per < kBatchDepos) {
        sched = make_int4((int)(per > 0 ? per : 1), 1 << 24, 1, big_only ? 1 : 0); // every depo in a `per`-depo batch
        n_batches = (n + sched.x - 1) / sched.x;
    }
    long long ctas = (n_batches + kBatchWarps - 1) / kBatchWarps;
    if (ctas > max_ctas) ctas = max_ctas;
#ifdef WCSIM_SCHED_ENV // experiment knob, off in the shipped library: WCSIM_SCHED="tail depos,tail batches per warp,chunk,CTAs per SM"
    {
        int4 e4 = sched;
        int max_per_sm = 0;
        const char *e = getenv("WCSIM_SCHED");
        if (e && sscanf(e, "%d,%d,%d,%d", &e4.x, &e4.y, &e4.z, &max_per_sm) >= 3 && e4.x >= 1 && e4.x <= kBatchDepos &&
            e4.y >= 0 && e4.z >= 1) {
            sched = make_int4(e4.x, e4.y, e4.z, sched.w);
            if (max_per_sm > 0 && ctas > (long long)sm_count * max_per_sm) ctas = (long long)sm_count * max_per_sm;
        }
    }
#endif
    return launch_pdl(raster_batch_kernel<FLUCT, TOT, FIX>, (unsigned)ctas, kBatchWarps * 32, smem, st, g, d, n, id_base, seed,
                      nsigma, S, depo_totals, counters, normalize, sched);
}

template <bool FIX>
static cudaError_t launch_raster_grid(GridDims g, DepoArrays d, long long n, uint64_t id_base, uint64_t seed, int fluctuate,
                                      double nsigma, float *grid, int *depo_totals, Counters *counters, int sm_count,
                                      cudaStream_t st, bool big_only = false)
{
    if (n <= 0) return cudaSuccess;
    const bool normalize = (fluctuate & kRasterNormalize) != 0;
    fluctuate &= ~kRasterNormalize;
#define WCSIM_BATCH(F, T) launch_raster_batch<F, T, FIX>(g, d, n, id_base, seed, nsigma, grid, T ? depo_totals : nullptr, counters, sm_count, st, normalize, big_only)
    if (!fluctuate) return WCSIM_BATCH(0, false); // no draws, no per-depo integer totals
    if (fluctuate == 2) return depo_totals ? WCSIM_BATCH(2, true) : WCSIM_BATCH(2, false);
    return depo_totals ? WCSIM_BATCH(1, true) : WCSIM_BATCH(1, false);
#undef WCSIM_BATCH
}

cudaError_t launch_raster_atomic(GridDims g, DepoArrays d, long long n, uint64_t id_base, uint64_t seed, int fluctuate,
                                 double nsigma, float *S, int *depo_totals, Counters *counters, int sm_count,
                                 cudaStream_t st)
{
    return launch_raster_grid<false>(g, d, n, id_base, seed, fluctuate, nsigma, S, depo_totals, counters, sm_count, st);
}

cudaError_t launch_raster_fixed(GridDims g, DepoArrays d, long long n, uint64_t id_base, uint64_t seed, int fluctuate,
                                double nsigma, unsigned long long *fix, int *depo_totals, Counters *counters, int sm_count,
                                cudaStream_t st, bool big_only)
{
    return launch_raster_grid<true>(g, d, n, id_base, seed, fluctuate, nsigma, reinterpret_cast<float *>(fix), depo_totals,
                                    counters, sm_count, st, big_only);
}

int raster_batch_depos() { return kBatchDepos; }

template <int FLUCT, bool FIX>
static cudaError_t launch_raster_planes_t(int n_ticks, const RasterPlanes &planes, double nsigma, float *grid,
                                          Counters *counters, int sm_count, cudaStream_t st, bool normalize)
{
    const long long n_batches = planes.batch0[planes.n];
    if (n_batches <= 0) return cudaSuccess;
    const size_t smem = sizeof(BatchSmem<FLUCT != 0, false>);
    const int fit = (int)((227u * 1024u) / (smem + 1024u));
    const int cap = FLUCT ? WCSIM_FLUCT_CTAS : 8;
    const int ctas_per_sm = fit > cap ? cap : fit;
    long long ctas = (n_batches + kBatchWarps - 1) / kBatchWarps;
    const long long max_ctas = (long long)sm_count * (ctas_per_sm > 0 ? ctas_per_sm : 1);
    if (ctas > max_ctas) ctas = max_ctas;
    return launch_pdl(raster_planes_kernel<FLUCT, FIX>, (unsigned)ctas, kBatchWarps * 32, smem, st, n_ticks, planes, nsigma,
                      grid, counters, normalize, 2);
}

cudaError_t launch_raster_planes(int n_ticks, const RasterPlanes &planes, int fluctuate, double nsigma,
                                 void *grid, bool fixed, Counters *counters, int sm_count, cudaStream_t st)
{
    const bool normalize = (fluctuate & kRasterNormalize) != 0;
    fluctuate &= ~kRasterNormalize;
    float *gp = reinterpret_cast<float *>(grid);
#define WCSIM_PLANES(F) (fixed ? launch_raster_planes_t<F, true>(n_ticks, planes, nsigma, gp, counters, sm_count, st, normalize) \
                               : launch_raster_planes_t<F, false>(n_ticks, planes, nsigma, gp, counters, sm_count, st, normalize))
    if (!fluctuate) return WCSIM_PLANES(0);
    if (fluctuate == 2) return WCSIM_PLANES(2);
    return WCSIM_PLANES(1);
#undef WCSIM_PLANES
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

template <int FLUCT, bool TOT>
static cudaError_t launch_tile_accumulate_t(GridDims g, DepoArrays d, uint64_t id_base, uint64_t seed, double nsigma,
                                            TileScratch ts, float *S, int *depo_totals, Counters *counters, bool normalize,
                                            cudaStream_t st)
{
    const int n_tiles = ts.tiles_w * ts.tiles_t;
    tile_accumulate_kernel<FLUCT, TOT><<<n_tiles * kTileSlices, kTileWarps * 32, sizeof(TileSmem<FLUCT != 0, TOT>), st>>>(
        g, d, id_base, seed, nsigma, ts, S, depo_totals, counters, normalize);
    return cudaGetLastError();
}

cudaError_t launch_tile_accumulate(GridDims g, DepoArrays d, uint64_t id_base, uint64_t seed, int fluctuate,
                                   double nsigma, TileScratch ts, float *S, int *depo_totals, Counters *counters,
                                   cudaStream_t st)
{
    const bool normalize = (fluctuate & kRasterNormalize) != 0;
    fluctuate &= ~kRasterNormalize;
#define WCSIM_TILE(F, T) launch_tile_accumulate_t<F, T>(g, d, id_base, seed, nsigma, ts, S, T ? depo_totals : nullptr, counters, normalize, st)
    if (!fluctuate) return WCSIM_TILE(0, false);
    if (fluctuate == 2) return depo_totals ? WCSIM_TILE(2, true) : WCSIM_TILE(2, false);
    return depo_totals ? WCSIM_TILE(1, true) : WCSIM_TILE(1, false);
#undef WCSIM_TILE
}

cudaError_t launch_tile_finalize(GridDims g, TileScratch ts, float *S, cudaStream_t st)
{
    const long long n_bins = (long long)g.n_wires * g.n_ticks;
    tile_finalize_kernel<<<(unsigned)((n_bins + 255) / 256), 256, 0, st>>>(n_bins, ts.fix, S);
    return cudaGetLastError();
}

cudaError_t launch_count_invalid(DepoArrays d, long long n, Counters *counters, cudaStream_t st)
{
    if (n <= 0) return cudaSuccess;
    count_invalid_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(d, n, counters);
    return cudaGetLastError();
}

int tile_max_listed() { return kMaxListedTiles; }

void tile_shape(int *tile_w, int *tile_t)
{
    *tile_w = kTileW;
    *tile_t = kTileT;
}

} // namespace wcsim

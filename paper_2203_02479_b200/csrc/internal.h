// internal.h -- host-side declarations shared by the translation units of libwcsim (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace wcsim {

struct DepoArrays {
    const float *t0, *x0, *sigma_t, *sigma_x, *q;
};

struct GridDims {
    int n_wires, n_ticks;
};

// The planes of a plan, stacked along the wire axis (wcsim_plan_create_planes: the planes of one APA event go through one
// launch sequence; an ordinary plan has n = 1).  Plane p owns rows row0[p] .. row0[p+1]-1 of S, M and the
// product spectra; in the row-spectrum buffer its rows start at srow0[p], with the wire pass's zero halo rows in between.
constexpr int kMaxPlanes = 8;
struct PlaneTable {
    int n;
    int row0[kMaxPlanes + 1];
    int srow0[kMaxPlanes];
    int grp0[kMaxPlanes + 1]; // first row group (blockIdx.y of the direct wire pass) of plane p
};
__host__ __device__ inline int plane_of_row(const PlaneTable &t, int row)
{
    int p = 0;
    while (p + 1 < t.n && row >= t.row0[p + 1]) ++p;
    return p;
}

// device counters (wcsim_stats)
struct Counters {
    unsigned long long depos_skipped;
    unsigned long long bins_drawn;
    unsigned long long next_batch; // work counter of the atomic-mode raster kernel; the kernel leaves it at 0
    unsigned long long warps_done;
};

// ---- raster.cu ----
// `fluctuate` of the launchers below: 0 off, 1 binomial (A6), 2 normal approximation (A21), plus kRasterNormalize for
// renormalised patches (A24)
constexpr int kRasterNormalize = 4;
cudaError_t raster_configure(cudaStream_t st); // erf table and shared-memory attributes of the raster kernels (per plan)
void erf_table_host(const double *z, double *out, long long n); // the table erf of erf_table.cuh, evaluated on the host
// a1-a3, atomic mode: S[wire][tick] += patch of every depo (red.global.add.f32)
cudaError_t launch_raster_atomic(GridDims g, DepoArrays d, long long n, uint64_t id_base, uint64_t seed, int fluctuate,
                                 double nsigma, float *S, int *depo_totals, Counters *counters, int sm_count,
                                 cudaStream_t st);

// the same kernel adding in 2^-24 fixed point into a 64-bit grid (RED.ADD.64: order independent, so reproducible bit for
// bit whatever the order of the adds); launch_tile_finalize folds the grid into S afterwards
// big_only: raster only the depos whose patch touches more than tile_max_listed() tiles (the rest of the tiled mode's work)
cudaError_t launch_raster_fixed(GridDims g, DepoArrays d, long long n, uint64_t id_base, uint64_t seed, int fluctuate,
                                double nsigma, unsigned long long *fix, int *depo_totals, Counters *counters, int sm_count,
                                cudaStream_t st, bool big_only = false);

// a1-a3 for the planes of a multi-plane plan in ONE launch (atomic or fixed-point sink): plane p's depos are cut into
// batches batch0[p] .. batch0[p+1]-1, a warp's batch index says which plane (depo arrays, wire count, row offset in the
// stacked grid) it works on; depo ids and Philox bins are the plane's own, as if each plane were rastered by its own plan
struct RasterPlanes {
    int n;
    DepoArrays d[kMaxPlanes];
    long long count[kMaxPlanes];
    uint64_t seed[kMaxPlanes]; // Philox key of plane p's fluctuation draws (reading A26)
    long long batch0[kMaxPlanes + 1];
    int n_wires[kMaxPlanes];
    int row0[kMaxPlanes];
};
int raster_batch_depos(); // depos per batch (for batch0)
cudaError_t launch_raster_planes(int n_ticks, const RasterPlanes &planes, int fluctuate, double nsigma,
                                 void *grid, bool fixed, Counters *counters, int sm_count, cudaStream_t st);

// a1-a3, tiled mode (deterministic): scratch buffers are owned by the plan and grown by the caller
struct TileScratch {
    int tile_w, tile_t;           // tile shape in bins
    int tiles_w, tiles_t;         // tile counts
    unsigned int *tile_count;     // [n_tiles + 1] counts, then exclusive offsets
    unsigned int *tile_cursor;    // [n_tiles] fill cursors
    unsigned int *entries;        // [capacity] depo indices grouped by tile
    unsigned long long capacity;  // entries allocated: >= kMaxListedTiles * n of the call (a depo is listed in at most that
                                  // many tiles; one that touches more is rastered straight into `fix` by the atomic kernel)
    unsigned int *slice_dev;      // [1] DEVICE: listed depos per slice of a hot tile, set by tile_scan from the mean tile load
    unsigned long long *fix;      // [n_wires * n_ticks] 2^-24 fixed-point grid the tile CTAs add into; zero between calls
};
cudaError_t launch_tile_count(GridDims g, DepoArrays d, long long n, double nsigma, TileScratch ts, cudaStream_t st);
cudaError_t launch_tile_scan(TileScratch ts, cudaStream_t st);
cudaError_t launch_tile_fill(GridDims g, DepoArrays d, long long n, double nsigma, TileScratch ts, cudaStream_t st);
cudaError_t launch_count_invalid(DepoArrays d, long long n, Counters *counters, cudaStream_t st);
void tile_shape(int *tile_w, int *tile_t);
int tile_max_listed(); // kMaxListedTiles
cudaError_t launch_tile_accumulate(GridDims g, DepoArrays d, uint64_t id_base, uint64_t seed, int fluctuate,
                                   double nsigma, TileScratch ts, float *S, int *depo_totals, Counters *counters,
                                   cudaStream_t st);
// S += fix 2^-24, fix = 0 (after launch_tile_accumulate)
cudaError_t launch_tile_finalize(GridDims g, TileScratch ts, float *S, cudaStream_t st);

// ---- convolve.cu ----
struct ConvBuffers {
    const float *S;       // [n_wires][n_ticks]
    float *M;             // [n_wires][n_ticks]
    float2 *spec;         // [n_wires][spec_stride]  row spectra (FFT wire mode: then, in place, the product spectra);
                          // wires_halo() zero rows sit below row 0 and above row n_wires-1 of the allocation
    float2 *spec2;        // [n_wires][spec_stride]  product spectra of the direct wire mode
    const float2 *spec_inv; // what rows_inverse reads: spec (FFT wire mode) or spec2 (direct wire mode)
    const float2 *Rt;     // [rt_rows][spec_stride]  rfft_t(R[d]) / pad_t, rows d >= n_rw are zero (direct wire mode)
    int rt_rows, n_rw;    // rt_rows = n_rw rounded up to a multiple of wires_chunk()
    const float2 *Rhat;   // [pad_w][spec_stride]
    const float2 *tw_row; // per-pass twiddle tables of a pad_t/2-point FFT (fft.cuh)
    const float2 *tw_real;// [pad_t/2]  exp(-2 pi i j / pad_t)
    const float2 *tw_col; // per-pass twiddle tables of a pad_w-point FFT
    int spec_stride;      // pad_t/2 + 8
    int sm_count;         // SMs of the plan's device (grid size of the persistent row kernels)
    int impact_K;         // impact positions per wire (reading A25): the row spectra hold n_wires * impact_K fine rows, fine
                          // row x K + k = position k of wire x; Rt holds impact_K blocks of rt_rows rows.  1: whole wires
    PlaneTable planes;    // GridDims::n_wires of the convolution launchers is the stacked row count planes.row0[planes.n];
                          // Rt holds planes.n blocks of rt_rows rows, plane p's response at Rt + p rt_rows spec_stride
};
struct NoiseArgs {
    const float *amp; // DEVICE [pad_t/2 + 1], already scaled by pad_t^-1/2; NULL = no noise
    uint64_t seed[kMaxPlanes]; // Philox key of plane p's noise (reading A26); a single-seed call fills every entry alike
};
inline NoiseArgs noise_args(const float *amp, const uint64_t *seeds, int n_seeds)
{
    NoiseArgs nz{};
    nz.amp = amp;
    for (int p = 0; p < kMaxPlanes; ++p) nz.seed[p] = seeds[p < n_seeds ? p : n_seeds - 1];
    return nz;
}
bool conv_sizes_supported(int pad_w, int pad_t);
cudaError_t conv_configure(int pad_w, int pad_t); // sets the kernels' shared-memory attributes (once per plan)
cudaError_t launch_rows_forward(GridDims g, int pad_t, ConvBuffers b, cudaStream_t st);
cudaError_t launch_cols(GridDims g, int pad_w, int pad_t, ConvBuffers b, cudaStream_t st);
int wires_chunk(); // response offsets per register chunk of the direct wire-axis kernel
void wires_halo(int n_rw, int *below, int *above); // zero rows of `spec` that kernel reads outside [0, n_wires)
int wires_rows_per_group();                        // output wires per CTA of that kernel (PlaneTable::grp0)
cudaError_t launch_wires(GridDims g, int pad_t, ConvBuffers b, cudaStream_t st);
// M = (accumulate ? M : 0) + c2r(use_spec ? spec : 0  +  noise)
cudaError_t launch_rows_inverse(GridDims g, int pad_t, ConvBuffers b, NoiseArgs noise, bool use_spec, bool accumulate,
                                cudaStream_t st);

// ---- response.cu ---- (plan time)
// Rhat[kx][kt] = 1/(pad_w pad_t) sum_dx sum_dt R[dx+c][dt] exp(-2 pi i (kx dx / pad_w + kt dt / pad_t)), fp64 -> fp32
cudaError_t build_response_spectrum(const float *dev_R, int n_rw, int n_rt, int pad_w, int pad_t, int spec_stride,
                                    double2 *dev_tmp /* [n_rw][pad_t/2+1] */, float2 *dev_Rhat, cudaStream_t st);
// Rt[d][kt] = tmp[d][kt] / pad_t for d < n_rw, 0 for n_rw <= d < rt_rows (and in the padding columns); after the above
cudaError_t build_response_rows(const double2 *dev_tmp, int n_rw, int rt_rows, int pad_t, int spec_stride,
                                float2 *dev_Rt, cudaStream_t st);

// ---- drift.cu ---- (upstream of the raster: reading A22)
struct DriftInputs {
    const float *x, *y, *z, *t, *q;
};
struct DepoOutputs {
    float *t0, *x0, *sigma_t, *sigma_x, *q;
};
struct DriftParams {
    double v_drift, two_DL, two_DT, tick, t_origin, lifetime; // two_D* = 2 D 1e-6: cm^2/us
};
struct DriftPlane {
    double x_plane, cos_theta, sin_theta, pitch_origin, pitch;
    DepoOutputs out;
};
constexpr int kMaxDriftPlanes = 4;
struct DriftPlanes {
    int n;
    DriftPlane plane[kMaxDriftPlanes];
};
cudaError_t launch_drift(DriftInputs in, long long n, DriftParams prm, DriftPlanes planes, cudaStream_t st);
// p[0..n) = 0 by a kernel launched as a programmatic dependent (the raster after it overlaps its launch with the clear's tail)
cudaError_t launch_clear(float *p, long long n, int sm_count, cudaStream_t st);
// ideal ADC of reading A23: adc[i] = clamp(rint(M[i] gain + baseline), 0, 2^bits - 1); M 16-byte, adc 8-byte aligned
cudaError_t launch_digitize(const float *M, long long n, float gain, float baseline, int bits, short *adc, cudaStream_t st);

// ---- debug.cu ----
cudaError_t launch_debug_philox(const unsigned int *ctr, const unsigned int *key, unsigned int *out, long long n,
                                cudaStream_t st);
cudaError_t launch_debug_binomial(const double *N, const double *p, const unsigned int *w, double *k, long long n,
                                  bool normal_only, cudaStream_t st);

cudaError_t launch_debug_fast_normal(const double *N, const double *p, const unsigned int *w, double *k, int *ok,
                                     long long n, cudaStream_t st);
cudaError_t launch_debug_z32_scan(unsigned long long first, unsigned long long count, unsigned long long *out4,
                                  cudaStream_t st);

} // namespace wcsim

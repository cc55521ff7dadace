/*
 * wcsim.h -- C ABI of libwcsim: the data-parallel hot path of the Wire-Cell LArTPC signal
 * simulation on one wire plane, hand-written CUDA for sm_100a (NVIDIA B200).
 *
 *     M(t,x) = sum_{t',x'} R(t-t', x-x') S(t',x') + N(t,x)          PAPER.md:38-40, Section 2.1, Eq. (1)
 *
 * S is built from "ionization electron groups" (depos) by the Raster and Scatter-add tasks of
 * PAPER.md:54-58 (Section 2.2); the convolution follows the FFT route of PAPER.md:46-52 (Eq. 2);
 * N is the optional electronics-noise term of Eq. (1), model from BASELINE.json configs[3].
 * Where the paper is silent the readings A1..A26 of DESIGN.md apply; each call names the ones it uses.
 *
 * Conventions
 *   - Grids are wire-major, tick fastest: S[wire * n_ticks + tick], fp32.  Bin k covers [k, k+1) on both axes (A1).
 *   - Every pointer says HOST or DEVICE.  Device pointers must belong to the device that was current at
 *     wcsim_plan_create.  The library never takes ownership of a caller's buffer.
 *   - All work is enqueued on the plan's CUDA stream (the `cuda_stream` given at creation; 0/NULL = the legacy
 *     default stream) and returns without waiting, except wcsim_plan_create (synchronises once), wcsim_sync,
 *     wcsim_plan_destroy and the *_host convenience calls (they synchronise before returning).
 *   - Return value: WCSIM_OK (0) or a negative wcsim_status.  Nothing throws or aborts across this boundary.
 *     Asynchronous CUDA faults surface at the next synchronising call as WCSIM_ECUDA.
 *   - There is no CPU fallback: without a CUDA device every call that needs one returns WCSIM_ECUDA.
 */
#ifndef WCSIM_H
#define WCSIM_H

#ifdef __cplusplus
extern "C" {
#endif

typedef enum wcsim_status {
    WCSIM_OK = 0,
    WCSIM_EINVAL = -1, /* NULL pointer, non-positive size, even n_rwires, bad padding, nsigma <= 0, unknown mode,
                          n_wires * n_ticks >= 2^30 */
    WCSIM_ENOMEM = -2, /* host or device allocation failed */
    WCSIM_ECUDA = -3,  /* a CUDA runtime call or kernel failed; wcsim_last_cuda_error() gives the cudaError_t */
    WCSIM_ESTATE = -4, /* call not valid in the plan's current state */
    WCSIM_ETOOBIG = -5 /* wcsim_raster_scatter_noalloc only: n_wires * n_ticks exceeds WCSIM_NOALLOC_MAX_BINS */
} wcsim_status;

/* scatter_mode of wcsim_plan_create */
#define WCSIM_SCATTER_ATOMIC 0 /* fp32 red.global adds straight into S; order of equal-address adds is not fixed */
#define WCSIM_SCATTER_TILED 1  /* depos are binned by grid tile, each tile is accumulated in shared memory in
                                  integer / fixed-point arithmetic (order independent => bitwise reproducible)
                                  and stored once; "deterministic sort-by-tile mode" of BASELINE.json north_star.
                                  WCSIM_SCATTER_FIXED gives the same bits faster */
#define WCSIM_SCATTER_FIXED 2  /* the atomic mode's kernel adding in 2^-24 fixed point into a 64-bit grid (integer
                                  red.global adds: order independent => bitwise reproducible), folded into S by one
                                  pass; deterministic without sorting, 8 bytes per bin of extra device memory */

/* wire_mode of wcsim_set_wire_mode: how wcsim_convolve treats the wire axis of Eq. (2).  Both give the same M up to
 * fp32 rounding (the cropped result is the linear convolution either way). */
#define WCSIM_WIRES_AUTO 0   /* direct up to the measured crossover width (32 / 45 / 100 response wires for wire paddings
                                <= 512 / <= 2048 / larger), FFT beyond (default) */
#define WCSIM_WIRES_FFT 1    /* pad_w-point FFT, multiply by Rhat(w_t, w_x), inverse FFT: Eq. (2) literally */
#define WCSIM_WIRES_DIRECT 2 /* tick axis by FFT, wire axis by direct summation over the n_rwires response offsets:
                                Mhat(w_t, x) = sum_dx Rt(w_t, dx) Shat(w_t, x - dx) */

typedef struct wcsim_plan wcsim_plan; /* opaque; owns S, M, the spectra, the response spectrum, twiddles, tile lists */

/* FFT padding.  0 on an axis = automatic: the next power of two >= n_ticks + n_rticks - 1 (ticks) and
 * >= n_wires + (n_rwires-1)/2 (wires) (A13).  Explicit values must be powers of two that satisfy those bounds,
 * with ticks >= 32 and wires >= 16. */
typedef struct wcsim_pad {
    int wires;
    int ticks;
} wcsim_pad;

/* Depositions as a structure of arrays ("structures/objects of arrays").  DEVICE pointers,
 * n elements each, caller-owned, must stay valid until the enqueued work has run. */
typedef struct wcsim_depos {
    const float *t0;      /* centre on the drift-time axis, in ticks */
    const float *x0;      /* centre on the wire-pitch axis, in pitches */
    const float *sigma_t; /* Gaussian width in ticks, >= 0 */
    const float *sigma_x; /* Gaussian width in pitches, >= 0 */
    const float *q;       /* charge in electrons (sign is carried) */
} wcsim_depos;

/* Counters kept on the device, copied out by wcsim_get_stats (which synchronises). */
typedef struct wcsim_stats {
    unsigned long long depos_skipped; /* depos with a non-finite field or a negative sigma: skipped, not rastered */
    unsigned long long bins_drawn;    /* patch bins inside the grid that were deposited (or drawn) */
} wcsim_stats;

/*
 * p0 Plan ("the similarly transformed 2D detector response array R(omega_t, omega_x)").
 *   response : HOST, n_rwires x n_rticks floats, tick fastest.  Row (n_rwires-1)/2 is wire offset dx = 0 (A11),
 *              column dt = 0..n_rticks-1 is causal in time.  Copied; the caller may free it on return.
 *   n_rwires : odd.
 *   nsigma   : patch half-width in sigmas (A2), > 0; all BASELINE.json configs use 3.
 * Embeds R in the padded grid (wrap-around on the wire axis), transforms it in fp64 by the definition of the DFT,
 * folds the 1/(pad.wires*pad.ticks) of the inverse transform in (A14) and keeps it as fp32.  S and M start at zero.
 * On failure *out is NULL.
 */
int wcsim_plan_create(wcsim_plan **out, int n_wires, int n_ticks, const float *response, int n_rwires, int n_rticks,
                      wcsim_pad pad, float nsigma, int scatter_mode, void *cuda_stream);

/*
 * a1-a3 Raster + fluctuation + scatter-add (PAPER.md:82 for the binomial fluctuation).
 * For every depo d (id = depo_id_base + d): extent floor(c - nsigma s) .. floor(c + nsigma s) on each axis (A2),
 * per-axis bin weights 1/2 [erf((i+1-c)/(sqrt2 s)) - erf((i-c)/(sqrt2 s))] (sigma < 1e-6: all weight in bin
 * floor(c), A4), patch p_ij = wt_i wx_j with no renormalisation (A3).
 *   fluctuate = 0 : S[j][i] += q p_ij                         (weights in fp32)
 *   fluctuate = 1 : S[j][i] += sign(q) B(floor(|q|+1/2), p_ij; w)   (weights, p and the sampler in fp64; A6, A7)
 *                   with w the Philox4x32-10 word keyed (seed, id, absolute grid bin j*n_ticks+i) (A8).
 *   fluctuate = 2 : the same with the normal approximation the paper's Kokkos port uses (A21):
 *                   S[j][i] += sign(q) clamp(rint(N p + sqrt(N p (1-p)) Phi^-1(u)), 0, N), N = floor(|q|+1/2), for every mu.
 *                   Any other value: WCSIM_EINVAL.
 * Bins outside the grid are dropped and not drawn (A5).  S accumulates across calls; wcsim_clear zeroes it.
 *   depos           : struct of DEVICE pointers (the struct itself is read on the host during the call).
 *   dev_depo_totals : DEVICE, n int32, or NULL.  With fluctuate = 1 or 2 receives the signed sum of each depo's draws.
 * n = 0 is valid and does nothing.  Every mode only enqueues.  WCSIM_SCATTER_TILED lists a depo in the at most 4 tiles
 * its patch touches (so 4 n list entries always suffice and nothing is read back; the lists are grown, with one stream
 * synchronisation, when a call brings more depos than any before) and sends a patch that touches more tiles through the
 * fixed-point grid of WCSIM_SCATTER_FIXED instead; 4 n + 16 must be < 2^32.
 */
int wcsim_raster_scatter(wcsim_plan *plan, const wcsim_depos *depos, long long n, unsigned long long depo_id_base,
                         unsigned long long seed, int fluctuate, int *dev_depo_totals);

/* Renormalised patches (reading A24; PAPER.md:56 leaves the patch normalisation open): with `on` != 0
 * later wcsim_raster_scatter calls use p_ij = (wt_i wx_j) / (W_t W_x), W the sum of the axis weights over the whole
 * +-nsigma extent, so a patch that lies inside the grid carries exactly q (fluctuate = 0) or has sum p = 1.  Charge
 * falling outside the grid is still dropped (A5).  Default: off (reading A3). */
int wcsim_set_normalize(wcsim_plan *plan, int on);

/*
 * a4-a6 Convolution by Eq. (2): M = crop(irfft2(Rhat * rfft2(zero_pad(S)))).  S is preserved.
 * Equals the linear convolution of Eq. (1) on the n_wires x n_ticks window exactly, up to fp32 rounding (A10-A13).
 * If noise was armed with wcsim_arm_noise, it is added inside the last transform and the arm is cleared.
 */
int wcsim_convolve(wcsim_plan *plan);

/*
 * a7 Noise (Eq. (1)'s N(t,x); model of BASELINE.json configs[3]; A15-A17): per wire x, on the padded
 * tick length P, k = 0..P/2: Z_k = amp[k] exp(2 pi i u(seed, x, k)), u from Philox4x32-10;
 * N[x][t] = P^-1/2 [Re Z_0 + 2 sum_{0<k<P/2} Re(Z_k e^{2 pi i k t / P}) + Re Z_{P/2} (-1)^t];  M += N for t < n_ticks.
 *   amp : HOST, P/2+1 floats, or NULL for the built-in A(f) = 3 (f/f0) exp(-f/f0), f0 = 0.1 f_Nyquist.
 * wcsim_add_noise runs now, as its own pass over M.  wcsim_arm_noise defers it into the next wcsim_convolve,
 * where it costs no extra pass over M; both give the same M up to fp32 rounding.
 */
int wcsim_add_noise(wcsim_plan *plan, const float *amp, unsigned long long seed);
int wcsim_arm_noise(wcsim_plan *plan, const float *amp, unsigned long long seed);

/* Waits for the plan's stream, frees everything the plan owns.  NULL is accepted.  WCSIM_ESTATE (nothing freed) while a
 * wcsim_graph made from the plan has not been destroyed. */
int wcsim_plan_destroy(wcsim_plan *plan);

/* ---- accessories ---- */
int wcsim_clear(wcsim_plan *plan);       /* S = 0 (enqueued) */
int wcsim_clear_output(wcsim_plan *plan); /* M = 0 (enqueued) */
int wcsim_sync(wcsim_plan *plan);        /* waits for the plan's stream; returns the first deferred CUDA fault */
int wcsim_set_scatter_mode(wcsim_plan *plan, int scatter_mode);
int wcsim_set_wire_mode(wcsim_plan *plan, int wire_mode);
/* the route wcsim_convolve takes on this plan now: WCSIM_WIRES_DIRECT or WCSIM_WIRES_FFT (WCSIM_WIRES_AUTO resolved) */
int wcsim_get_wire_mode(const wcsim_plan *plan, int *resolved);
/* borrowed DEVICE pointers to n_wires*n_ticks floats, valid until wcsim_plan_destroy */
int wcsim_charge_ptr(wcsim_plan *plan, float **dev);
int wcsim_output_ptr(wcsim_plan *plan, float **dev);
int wcsim_get_dims(const wcsim_plan *plan, int *n_wires, int *n_ticks, int *pad_wires, int *pad_ticks);
int wcsim_get_stats(wcsim_plan *plan, wcsim_stats *out); /* synchronises */
int wcsim_reset_stats(wcsim_plan *plan);

/*
 * Stage timing (what bench.py's per-stage numbers and `roofline` come from).  While enabled, every call records a
 * CUDA event pair on the plan's stream around each stage it enqueues; wcsim_get_stage_times synchronises, adds the
 * finished spans up and returns, per stage, the total milliseconds and the number of spans (arrays of WCSIM_N_STAGES).
 */
#define WCSIM_STAGE_RASTER 0       /* a1-a3: the whole wcsim_raster_scatter call */
#define WCSIM_STAGE_ROWS_FORWARD 1 /* a4, tick axis */
#define WCSIM_STAGE_COLS 2         /* a4 wire axis + a5 multiply + a6 wire axis */
#define WCSIM_STAGE_ROWS_INVERSE 3 /* a6 tick axis (+ armed noise) */
#define WCSIM_STAGE_NOISE 4        /* a7 as its own pass (wcsim_add_noise) */
#define WCSIM_STAGE_CONVOLVE 5     /* the whole wcsim_convolve call as ONE span (level WCSIM_PROFILE_CALLS only) */
#define WCSIM_N_STAGES 6
/* level: 0 off; WCSIM_PROFILE_KERNELS: an event pair around every kernel of wcsim_convolve (the records sit between the
 * kernels, which are programmatic dependents of one another, and cost a few microseconds per plane-event);
 * WCSIM_PROFILE_CALLS: one pair around the whole wcsim_convolve call, nothing between its kernels (stage CONVOLVE).
 * wcsim_raster_scatter and wcsim_add_noise are one span each at either level. */
#define WCSIM_PROFILE_KERNELS 1
#define WCSIM_PROFILE_CALLS 2
int wcsim_set_profiling(wcsim_plan *plan, int level);
int wcsim_get_stage_times(wcsim_plan *plan, double *ms, unsigned long long *calls, int reset);
/* number of kernels of this library enqueued through `plan` so far (memsets and copies are not counted) */
int wcsim_get_launch_count(const wcsim_plan *plan, unsigned long long *out);

/*
 * End-to-end convenience with HOST buffers (what bench.py's `e2e` times): copies the five depo arrays
 * host->device, clears S, rasters+scatters, convolves (with noise if noise_seed_or_0 != 0 ... see `noise`),
 * copies M device->host, synchronises.
 *   host_* : HOST, n floats each (pinned memory makes the copies asynchronous)
 *   host_M : HOST, n_wires*n_ticks floats, written
 *   noise  : 0 = none, 1 = built-in amplitude spectrum with `noise_seed`
 */
int wcsim_simulate_host(wcsim_plan *plan, const float *host_t0, const float *host_x0, const float *host_sigma_t,
                        const float *host_sigma_x, const float *host_q, long long n, unsigned long long seed,
                        int fluctuate, int noise, unsigned long long noise_seed, float *host_M);
/*
 * The same, without the final synchronisation: everything (the host->device copies of the depos, the kernels and the
 * device->host copy of M) is enqueued on the plan's stream and the call returns.  host_M holds this plane-event's
 * M(t,x) (Eq. 1) once wcsim_sync(plan) has returned; the host depo arrays must stay valid and unchanged
 * until then, and must be pinned for the copies to be asynchronous.  Two or three plans on as many streams, used in turn,
 * overlap one event's device->host copy with the next event's copies and kernels (what bench.py's `e2e` does).
 * Errors: as wcsim_simulate_host; asynchronous CUDA errors surface at wcsim_sync.
 */
int wcsim_simulate_host_async(wcsim_plan *plan, const float *host_t0, const float *host_x0, const float *host_sigma_t,
                        const float *host_sigma_x, const float *host_q, long long n, unsigned long long seed,
                        int fluctuate, int noise, unsigned long long noise_seed, float *host_M);

/* The same round trip returning ADC codes instead of the fp32 M (wcsim_digitize below, reading A23): half the device->host
 * bytes.  host_adc: HOST, n_wires*n_ticks int16, written; valid after wcsim_sync(plan).  The codes are staged in a device
 * buffer the plan owns.  If the five host depo arrays follow one another in memory (one block of 5 n floats, as here), they
 * go over in one copy.  Errors: as wcsim_simulate_host_async; bits outside 1..15: WCSIM_EINVAL. */
int wcsim_simulate_host_adc_async(wcsim_plan *plan, const float *host_t0, const float *host_x0, const float *host_sigma_t,
                                  const float *host_sigma_x, const float *host_q, long long n, unsigned long long seed,
                                  int fluctuate, int noise, unsigned long long noise_seed, float gain, float baseline,
                                  int bits, short *host_adc);

/*
 * Several planes through ONE launch sequence (Section 3.3 and Fig. 4: "with one process
 * per GPU the GPU is under-utilized"; the planes of an anode are independent).  A multi-plane plan stacks
 * 1..8 planes of the same n_ticks, tick padding and response footprint (n_rwires x n_rticks) along the wire axis:
 * plane p owns rows first_row(p) .. first_row(p) + n_wires[p] - 1 of S and M (wcsim_get_plane_rows).  One raster launch
 * takes the depos of all planes, the row transforms run over all stacked rows, one direct wire pass applies every plane's
 * own response (planes never mix: each has its own zero halo rows), noise is keyed by the plane's own wire index.  Every
 * plane's S and M equal what a plan of that plane alone gives (same seeds; depo ids start at 0 in every plane).
 *   n_wires   : HOST, n_planes ints;  responses : HOST, n_planes pointers to n_rwires x n_rticks floats each.
 *   pad_ticks : 0 = automatic.  The wire axis is always done directly (WCSIM_WIRES_DIRECT), so there is no wire padding.
 *   scatter_mode : WCSIM_SCATTER_ATOMIC or WCSIM_SCATTER_FIXED (the tiled mode is per plane: WCSIM_EINVAL).
 * wcsim_clear, wcsim_convolve, wcsim_arm_noise / wcsim_add_noise (the same spectrum and seed for every plane; see the
 * *_planes variants below for a seed per plane),
 * wcsim_digitize, wcsim_charge_ptr / wcsim_output_ptr (the stacked grids) work on such a plan as on any other;
 * wcsim_raster_scatter and the *_host calls return WCSIM_ESTATE.
 */
int wcsim_plan_create_planes(wcsim_plan **out, int n_planes, const int *n_wires, int n_ticks,
                             const float *const *responses, int n_rwires, int n_rticks, int pad_ticks, float nsigma,
                             int scatter_mode, void *cuda_stream);
/* a1-a3 for all planes of the plan in one launch.  depos: HOST array of n_planes structs of DEVICE pointers; n: HOST,
 * n_planes counts (0 allowed).  Depo d of plane p has id d; the Philox bin is the plane's own wire * n_ticks + tick (A8).
 * Works on single-plane plans too (n_planes = 1).  No per-depo totals.  Errors: WCSIM_ESTATE in tiled scatter mode. */
int wcsim_raster_scatter_planes(wcsim_plan *plan, const wcsim_depos *depos, const long long *n, unsigned long long seed,
                                int fluctuate);
/* Independent planes (reading A26 of DESIGN.md; the simulation "treats each plane independently", PAPER.md:40
 * for N(t,x)): with ONE seed, equal (depo id, bin) pairs of different planes draw from the same Philox word and wire x of
 * every plane carries the same noise waveform -- fine for a test, wrong for physics.  These variants take one seed per
 * plane, seeds: HOST, n_planes values; plane p is then exactly what a single-plane plan gives with seeds[p] (Philox key =
 * seeds[p]; counters unchanged: depo id and the plane's own bin for the fluctuation, the plane's own wire for the noise).
 * Everything else as wcsim_raster_scatter_planes / wcsim_arm_noise / wcsim_add_noise.  NULL seeds: WCSIM_EINVAL. */
int wcsim_raster_scatter_planes_seeded(wcsim_plan *plan, const wcsim_depos *depos, const long long *n,
                                       const unsigned long long *seeds, int fluctuate);
int wcsim_arm_noise_planes(wcsim_plan *plan, const float *amp, const unsigned long long *seeds);
int wcsim_add_noise_planes(wcsim_plan *plan, const float *amp, const unsigned long long *seeds);
int wcsim_get_plane_rows(const wcsim_plan *plan, int plane, int *first_row, int *n_rows);

/*
 * Sub-wire "impact position" response binning (reading A25 of DESIGN.md; the patches are
 * "typically O(20x20) elements", which whole-wire bins do not give).  The charge grid is n_impact times finer along the
 * wire axis: fine row x * n_impact + k holds the charge arriving at impact position k of wire x, i.e. at pitch coordinate
 * [(x n_impact + k) / n_impact, +1/n_impact).  Depos given to such a plan carry x0 and sigma_x in units of
 * pitch / n_impact (wcsim_drift with pitch / n_impact as its pitch produces them); the raster, the fluctuation and the
 * Philox bin (fine row * n_ticks + tick) are those of a plane with n_wires * n_impact rows.  The response is given per
 * impact position and the measured waveform of a wire sums over its impact positions:
 *     M[x][t] = sum_k sum_dx sum_dt R_k[dx + c][dt] S[(x - dx) n_impact + k][t - dt]
 * (n_impact = 1: Eq. (1) as wcsim_plan_create computes it).  wcsim_convolve transforms the n_wires * n_impact fine rows
 * along ticks, applies the n_impact * n_rwires taps directly along wires, and inverts n_wires rows.
 *   responses : HOST, n_impact pointers to n_rwires x n_rticks floats (position k's response, layout as in wcsim_plan_create).
 * wcsim_charge_ptr gives the fine grid (wcsim_get_charge_dims: its rows), wcsim_output_ptr the n_wires x n_ticks M.
 * Errors: WCSIM_EINVAL (n_impact outside 1..64, n_wires * n_impact * n_ticks >= 2^30, ...).
 */
int wcsim_plan_create_impact(wcsim_plan **out, int n_wires, int n_ticks, int n_impact, const float *const *responses,
                             int n_rwires, int n_rticks, int pad_ticks, float nsigma, int scatter_mode, void *cuda_stream);
/* rows and ticks of the charge grid S (rows = n_wires * n_impact; the stacked rows of a multi-plane plan) */
int wcsim_get_charge_dims(const wcsim_plan *plan, int *rows, int *n_ticks, int *n_impact);

/*
 * Raster + fluctuation + scatter-add WITHOUT any device allocation, and without a plan (creating a plan allocates).
 *
 * For callers that cannot call cudaMalloc at the point where they need the charge grid: a plug-in of a host framework
 * that owns all device memory and forbids driver allocations while its event loop runs (an allocation takes a
 * device-wide lock and can synchronise every stream in the process, stalling the framework's other work), a
 * latency-bound acquisition thread that may not block in the driver, or a job so close to the memory limit that a late
 * allocation could fail.  Such a caller owns S (carved out of its own arena) and passes it in; the one thing the kernel
 * needs besides its inputs and outputs -- a 64-bit fixed-point accumulation grid of one word per bin plus a 256-byte
 * counter block -- is built into the library as a fixed device array instead of being allocated.
 *
 * The cost and the limit: that array is WCSIM_NOALLOC_MAX_BINS words (4 MiB) + 256 bytes, and every GPU on which the
 * process uses CUDA with libwcsim.so loaded holds it from then until the process exits, used or not.  A grid with
 * n_wires * n_ticks > WCSIM_NOALLOC_MAX_BINS is refused with WCSIM_ETOOBIG (nothing is enqueued, nothing is allocated to
 * make room); use a plan for larger grids.
 *
 * What it computes: exactly wcsim_raster_scatter on a plan in WCSIM_SCATTER_FIXED mode -- same kernel, same readings,
 * same Philox keys, bitwise reproducible -- on the device that is current on the calling thread:
 *     dev_S[wire * n_ticks + tick] += patch of every depo            (dev_S accumulates; the caller zeroes it when it wants)
 *   n_wires, n_ticks : the charge grid, n_wires * n_ticks <= WCSIM_NOALLOC_MAX_BINS.
 *   depos            : HOST struct of five DEVICE pointers, n floats each, caller-owned, read.
 *   depo_id_base, seed, fluctuate : as wcsim_raster_scatter (0 off, 1 binomial, 2 normal approximation).
 *   nsigma           : patch half-width in sigmas, > 0 (3 in all BASELINE.json configs).
 *   dev_S            : DEVICE, n_wires * n_ticks floats, caller-owned, read and written.
 *   cuda_stream      : the work is enqueued on it (memset of the scratch, raster kernel, fold into S) and the call returns.
 * Invalid depos (non-finite field, negative sigma) are skipped as everywhere else; their count is not available here
 * (there is no plan to ask), and there are no per-depo totals.
 *
 * First call on each device: it looks up the built-in array's device address, uploads the raster's erf table and sets
 * kernel attributes, and for that it synchronises cuda_stream once.  Make that first call (n = 1 on a scratch S will do)
 * during start-up, before the no-allocation phase and before any stream capture is begun on cuda_stream.  Later calls
 * only enqueue.
 *
 * Sharing: all calls on a device use the same built-in array, whatever their stream or thread.  Each call zeroes the
 * part it uses before its kernel runs, so stale contents of an earlier (even a failed) call never leak into S; but two
 * calls whose GPU work overlaps -- different streams, or different host threads on different streams -- write the same
 * words at once and corrupt each other's S.  Keep all calls on one stream, or order them with events.
 *
 * Errors: WCSIM_EINVAL (NULL dev_S or depo pointer with n > 0, non-positive dims, n < 0, fluctuate outside 0..2,
 * nsigma <= 0), WCSIM_ETOOBIG, WCSIM_ECUDA (wcsim_last_cuda_error is not updated by this call).  n = 0 returns WCSIM_OK
 * without touching the device.  Calls no cudaMalloc, cudaFree, or any library routine that allocates.
 */
#define WCSIM_NOALLOC_MAX_BINS 524288 /* e.g. 64 x 8192, 128 x 4096, 256 x 2048; configs[0] (64 x 512) is 1/16 of it */
int wcsim_raster_scatter_noalloc(int n_wires, int n_ticks, const wcsim_depos *depos, long long n,
                                 unsigned long long depo_id_base, unsigned long long seed, int fluctuate, float nsigma,
                                 float *dev_S, void *cuda_stream);

/*
 * CUDA graphs (a small plane-event is bound by launch latency).  Between wcsim_graph_begin and
 * wcsim_graph_end the plan's stream is in capture mode: wcsim_clear, wcsim_raster_scatter(_planes), wcsim_arm_noise
 * (built-in spectrum), wcsim_convolve, wcsim_add_noise (built-in), wcsim_digitize only RECORD their work (the kernels keep
 * their programmatic-dependent-launch edges); the graph replays that sequence on the plan's stream at every
 * wcsim_graph_launch, with the pointers and sizes recorded (the depo arrays must still be valid and may hold new values).
 * Not capturable (WCSIM_ESTATE while capturing): a first use of the fixed-point or tiled mode on the plan, or a tiled
 * call with more depos than any before (they allocate: run the call once outside the capture), custom noise spectra, anything that synchronises (wcsim_sync, wcsim_get_stats, the
 * *_host calls must not be called).  The plan's stream must not be the legacy default stream (WCSIM_ESTATE).
 * Stage timing is off inside a capture.  Destroy graphs before their plan: wcsim_plan_destroy returns WCSIM_ESTATE (and
 * frees nothing) while a graph made from the plan is alive.
 *
 * What a replay repeats.  Everything passed BY VALUE to the recorded calls is frozen in the graph: the fluctuation seed,
 * depo_id_base and the depo count n of wcsim_raster_scatter(_planes), the noise seed of wcsim_arm_noise / wcsim_add_noise,
 * gain / baseline / bits of wcsim_digitize.  Only the CONTENTS of the recorded device arrays are read afresh.  So plain
 * replays over new depos reuse the same Philox stream and the same noise realisation (Eq. (1)'s N(t,x),
 * PAPER.md:40): consecutive events would be statistically correlated.  For independent events give every event its own
 * seeds through wcsim_graph_update: wcsim_graph_begin, the same calls in the same order with the new seeds / counts /
 * pointers, then wcsim_graph_update(plan, graph) instead of wcsim_graph_end.  It ends the capture and rewrites the
 * parameters of the existing executable graph in place (no re-instantiation; launches of the old parameters that are
 * already enqueued are not affected).  If the recorded sequence is not the one the graph was made from (another call
 * order, another scatter mode, a tiled call, a different number of kernels) it returns WCSIM_ESTATE; the graph should then
 * be destroyed and made anew.  With NULL arguments (WCSIM_EINVAL), or a graph of another plan or no capture in progress
 * (WCSIM_ESTATE), the capture state is left as it was.
 */
typedef struct wcsim_graph wcsim_graph;
int wcsim_graph_begin(wcsim_plan *plan);
int wcsim_graph_end(wcsim_plan *plan, wcsim_graph **out); /* *out = NULL on failure */
int wcsim_graph_update(wcsim_plan *plan, wcsim_graph *graph);
int wcsim_graph_launch(wcsim_graph *graph);
int wcsim_graph_destroy(wcsim_graph *graph);

/*
 * Drift: the step upstream of the Raster ("After simulating the diffusion process along the drifting, each
 * ionization electron group is diffused into a 2D distribution along the drifting and wire pitch directions"; reading
 * A22).  One pass over n electron groups writes the depo arrays of n_planes planes (1..4):
 *   td = (x - x_plane)/v_drift;  t0 = (t + td - t_origin)/tick;  x0 = (y cos_theta + z sin_theta - pitch_origin)/pitch;
 *   sigma_t = sqrt(2 D_L td)/v_drift/tick;  sigma_x = sqrt(2 D_T td)/pitch;  q_out = q exp(-td/lifetime)
 * computed in fp64 and rounded once to fp32.  Units: cm and us, D_L and D_T in cm^2/s, q in electrons; lifetime <= 0
 * means no attenuation.  A group behind a plane (td < 0) gets NaN in that plane's five fields; wcsim_raster_scatter
 * skips and counts such depos.  No plan is involved.
 *   dev_x .. dev_q : DEVICE, n floats each, read.
 *   planes         : HOST array of n_planes geometry records (read during the call).
 *   out            : HOST array of n_planes wcsim_depos whose five DEVICE pointers (n floats each, caller-owned) are
 *                    written; the const in wcsim_depos is cast away for these.
 * Errors: WCSIM_EINVAL (NULL, n < 0, n_planes outside 1..4, non-positive v_drift / tick / pitch, negative D),
 * WCSIM_ECUDA.  Asynchronous on cuda_stream.
 */
typedef struct {
    double v_drift, D_L, D_T, tick, t_origin, lifetime;
} wcsim_drift_params;
typedef struct {
    double x_plane, cos_theta, sin_theta, pitch_origin, pitch;
} wcsim_plane_geom;
int wcsim_drift(const float *dev_x, const float *dev_y, const float *dev_z, const float *dev_t, const float *dev_q,
                long long n, const wcsim_drift_params *params, const wcsim_plane_geom *planes, int n_planes,
                const wcsim_depos *out, void *cuda_stream);

/*
 * Digitisation: the step downstream of M ("M(t,x) is the 'measured' value such as what is input to an
 * analog-to-digital converter (ADC) channel x at time t"; reading A23).  An ideal ADC of `bits` bits:
 *   dev_adc[x][t] = clamp(rint(M[x][t] * gain + baseline), 0, 2^bits - 1),  round half to even, fp32, NaN -> 0,
 * over the plan's output grid (after wcsim_convolve / wcsim_add_noise), enqueued on the plan's stream.
 *   dev_adc : DEVICE, n_wires*n_ticks int16, 8-byte aligned, caller-owned, written.
 * Errors: WCSIM_EINVAL (NULL, bits outside 1..15, misaligned dev_adc), WCSIM_ECUDA.
 */
int wcsim_digitize(wcsim_plan *plan, float gain, float baseline, int bits, short *dev_adc);

/* Test/diagnostic hooks: exact pieces of the path, exposed so that parity can be checked piecewise. */
/* out[4] (DEVICE, 4*n uint32) = Philox4x32-10(ctr = dev_ctr[4*i..], key = dev_key[2*i..]) for i < n */
int wcsim_debug_philox(const unsigned int *dev_ctr, const unsigned int *dev_key, unsigned int *dev_out, long long n,
                       void *cuda_stream);
/* The raster's own fp64 erf (a 48-interval degree-12 Taylor table, csrc/erf_table.cuh) evaluated on the HOST with the
 * same code the kernels run: out[i] = erf(z[i]).  HOST pointers, n elements each; no device is touched.  Used by the
 * CPU tests to pin the table against a library erf (bin weights of reading A2). */
int wcsim_debug_erf(const double *host_z, double *host_out, long long n);
/* dev_k[i] = B(dev_N[i], dev_p[i]; dev_w[i]) -- the device binomial sampler (fp64 in, fp64 integer-valued out) */
int wcsim_debug_binomial(const double *dev_N, const double *dev_p, const unsigned int *dev_w, double *dev_k,
                         long long n, void *cuda_stream);
/* dev_k[i] = G(dev_N[i], dev_p[i]; dev_w[i]) -- the normal-approximation draw of fluctuate = 2 (A21) */
int wcsim_debug_normal_draw(const double *dev_N, const double *dev_p, const unsigned int *dev_w, double *dev_k,
                         long long n, void *cuda_stream);
/* The guarded fp32 fast path of the rounded-normal draw (csrc/rng.cuh; the raster takes it for mu >= 16 and falls back
 * to the fp64 routine behind wcsim_debug_binomial when the guard rejects): dev_k[i] = its k, dev_ok[i] = 1 if the guard
 * accepted it (then k must equal the fp64 routine's), 0 if not.  dev_p in (0, 1/2]; DEVICE pointers, n elements. */
int wcsim_debug_fast_normal(const double *dev_N, const double *dev_p, const unsigned int *dev_w, double *dev_k,
                            int *dev_ok, long long n, void *cuda_stream);
/* Error of the fast path's fp32 normal quantile against the fp64 AS 241 routine over the 32-bit words
 * first_word .. first_word + n_words - 1 (first_word + n_words <= 2^32): dev_out4 (DEVICE, 4 doubles) receives
 * max |z32 - z64| and max |z64| over the words the fast path accepts, their number, and max |z32 - z64| / max(1, |z64|). */
int wcsim_debug_z32_scan(unsigned long long first_word, unsigned long long n_words, double *dev_out4, void *cuda_stream);
/* copy the response spectrum Rhat[kx][kt] (kx < pad_wires, kt <= pad_ticks/2) to HOST as interleaved re,im floats */
int wcsim_debug_response_spectrum(wcsim_plan *plan, float *host_out);

const char *wcsim_strerror(int status);
int wcsim_last_cuda_error(void); /* cudaError_t of the most recent WCSIM_ECUDA on this thread, else 0 */
const char *wcsim_version(void);

#ifdef __cplusplus
}
#endif
#endif /* WCSIM_H */
